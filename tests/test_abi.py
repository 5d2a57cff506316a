"""CPU (`-m "not gpu"`) checks of the boundary: libcheb_dm.so builds for sm_100a, loads without a GPU and
exports every symbol include/cheb_dm.h declares; the binding lists the same names; no compute calls."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "cheb_dm.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(cheb_dm_[a-z_A-Z0-9]+)\s*\(", src)))


def test_header_symbols_are_exported():
    from paper_2306_12616_b200 import binding
    names = _declared()
    assert "cheb_dm_plan" in names and "cheb_dm_coeffs" in names and "cheb_dm_compute" in names and "cheb_dm_trace" in names
    L = ctypes.CDLL(binding.lib_path()) if os.path.exists(binding.lib_path()) else binding.lib()
    L = binding.lib()
    for n in names:
        assert hasattr(L, n), n
    assert sorted(binding.EXPORTS) == names


def test_signatures_have_no_torch_types():
    src = open(os.path.join(ROOT, "include", "cheb_dm.h")).read()
    assert "torch" not in src.lower() and "at::" not in src
    assert 'extern "C"' in src


def test_strerror_and_no_device_behaviour():
    from paper_2306_12616_b200 import binding
    L = binding.lib()
    assert L.cheb_dm_strerror(0) == b"ok"
    assert b"bounds" in L.cheb_dm_strerror(5)
    import torch
    if not torch.cuda.is_available():
        h = ctypes.c_void_p()
        assert L.cheb_dm_plan(ctypes.byref(h), 16, 4, 0) == 3  # ECUDA: there is no CPU fallback
    # argument checks that precede any CUDA call
    h = ctypes.c_void_p()
    assert L.cheb_dm_plan(ctypes.byref(h), 0, 4, 0) == 1
    assert L.cheb_dm_plan(ctypes.byref(h), 4, 4, 3) == 6
    assert L.cheb_dm_destroy(None) == 1


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2306_12616_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "cheb_oracle" not in txt, f


def test_option_and_trace_structs_match_the_header():
    """The ctypes mirrors of cheb_dm_options_t / cheb_dm_trace_rec_t have the header's fields, in order, and its size."""
    from paper_2306_12616_b200 import binding
    src = open(os.path.join(ROOT, "include", "cheb_dm.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    body = re.search(r"typedef struct \{([^}]*)\} cheb_dm_options_t;", src).group(1)
    fields = re.findall(r"\bint\s+([a-z_]+)(\[\d+\])?\s*;", body)
    assert [f for f, _ in fields] == [n for n, _ in binding.Options._fields_]
    nints = sum(int(a.strip("[]")) if a else 1 for _, a in fields)
    assert ctypes.sizeof(binding.Options) == 4 * nints == 64
    body = re.search(r"typedef struct \{([^}]*)\} cheb_dm_trace_rec_t;", src).group(1)
    names = re.findall(r"\b([a-z_]+)\s*[,;]", body)
    assert names == [n for n, _ in binding.TraceRec._fields_]
    assert ctypes.sizeof(binding.TraceRec) == 4 * 4 + 5 * 8


def test_entry_points_reject_bad_arguments_before_any_cuda_work():
    from paper_2306_12616_b200 import binding
    L = binding.lib()
    for fn in (L.cheb_dm_check, L.cheb_dm_wait):
        assert fn(None, None) == 1                      # EINVAL: NULL plan
    assert L.cheb_dm_compute_host_async(None, None, None, None, None) == 1
    assert L.cheb_dm_get_options(None, None) == 1
    assert L.cheb_dm_set_trace(None, 1) == 1
    o = binding.Options(symmetric=3)
    h = ctypes.c_void_p()
    import torch
    if torch.cuda.is_available():
        assert L.cheb_dm_plan_ex(ctypes.byref(h), 8, 4, 0, ctypes.byref(o)) == 1   # bad option value
