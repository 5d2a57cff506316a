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
