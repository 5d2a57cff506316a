"""ctypes binding of include/cheb_dm.h (same names, marshalling only)."""
from __future__ import annotations

import ctypes as C
import os

from . import build as _build

OUTER_CHEBYSHEV, OUTER_POWER = 0, 1
SCHED_GROUPED, SCHED_SERIAL = 0, 1
PAIR_AUTO, PAIR_SERIAL, PAIR_BALANCED, PAIR_ALG1 = 0, 1, 2, 3
MAX_BATCH = 64
TILE_AUTO, TILE_128x128, TILE_128x64, TILE_64x64 = 0, 1, 2, 3
STATUS_NAMES = ["OK", "EINVAL", "EALLOC", "ECUDA", "ESTATE", "EBOUNDS", "EUNSUPPORTED", "ENOCONV", "ESIZE"]

EXPORTS = [
    "cheb_dm_plan", "cheb_dm_plan_ex", "cheb_dm_destroy", "cheb_dm_coeffs", "cheb_dm_compute",
    "cheb_dm_trace", "cheb_dm_get_bounds", "cheb_dm_get_coeffs", "cheb_dm_get_kp", "cheb_dm_get_T",
    "cheb_dm_moments", "cheb_dm_solve_mu", "cheb_dm_product", "cheb_dm_workspace_bytes",
    "cheb_dm_last_launch_count", "cheb_dm_flops_per_compute", "cheb_dm_strerror",
    "cheb_dm_compute_host", "cheb_dm_set_timing", "cheb_dm_product_ms", "cheb_dm_dmma_peak",
    "cheb_dm_set_trace", "cheb_dm_get_trace", "cheb_dm_get_options", "cheb_dm_check",
    "cheb_dm_compute_host_async", "cheb_dm_wait",
    "cheb_dm_compute_batch", "cheb_dm_compute_batch_host", "cheb_dm_compute_batch_host_async", "cheb_dm_trace_batch",
    "cheb_dm_get_scalars", "cheb_dm_solve", "cheb_dm_solve_batch", "cheb_dm_assemble", "cheb_dm_flops_per_solve",
    "cheb_dm_product_sliced", "cheb_dm_sliced_ops_per_compute", "cheb_dm_bounds_static",
]


class TraceRec(C.Structure):
    _fields_ = [("task", C.c_int), ("tm", C.c_int), ("tn", C.c_int), ("sm", C.c_int),
                ("t_claim", C.c_uint64), ("t_desc", C.c_uint64), ("t_first", C.c_uint64),
                ("t_kend", C.c_uint64), ("t_done", C.c_uint64)]


class Options(C.Structure):
    _fields_ = [("k", C.c_int), ("p", C.c_int), ("outer", C.c_int), ("sched", C.c_int),
                ("pairing", C.c_int), ("tile", C.c_int), ("fuse_sums", C.c_int),
                ("giant", C.c_int), ("symmetric", C.c_int), ("max_batch", C.c_int), ("ldh", C.c_int), ("ldd", C.c_int),
                ("moments", C.c_int), ("host_slots", C.c_int), ("sliced", C.c_int), ("sliced_solve", C.c_int)]


class ChebDMError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        name = STATUS_NAMES[status] if 0 <= status < len(STATUS_NAMES) else str(status)
        msg = lib().cheb_dm_strerror(status).decode() if _LIB is not None else ""
        super().__init__(f"{where}: CHEB_DM_{name} ({msg})")


_LIB = None


def lib_path() -> str:
    return _build.LIB_PATH


def lib():
    """Load libcheb_dm.so (building it in-tree with nvcc if it is missing or stale)."""
    global _LIB
    if _LIB is not None:
        return _LIB
    path = _build.LIB_PATH
    if _build.is_stale():
        try:
            _build.build()
        except Exception as e:  # no nvcc: use what is there, or fail loudly
            if not os.path.exists(path):
                raise RuntimeError(f"libcheb_dm.so is missing and could not be built: {e}") from e
    L = C.CDLL(path)
    vp, dp, ip = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int)
    L.cheb_dm_plan.argtypes = [C.POINTER(vp), C.c_int, C.c_int, C.c_int]
    L.cheb_dm_plan_ex.argtypes = [C.POINTER(vp), C.c_int, C.c_int, C.c_int, C.POINTER(Options)]
    L.cheb_dm_destroy.argtypes = [vp]
    L.cheb_dm_coeffs.argtypes = [vp, C.c_double, C.c_double, dp]
    L.cheb_dm_compute.argtypes = [vp, vp, vp, vp]
    L.cheb_dm_trace.argtypes = [vp, vp, vp, vp]
    L.cheb_dm_get_bounds.argtypes = [vp, dp, vp]
    L.cheb_dm_get_coeffs.argtypes = [vp, dp, dp, dp, vp]
    L.cheb_dm_get_kp.argtypes = [vp, ip, ip]
    L.cheb_dm_get_T.argtypes = [vp, C.c_int, vp, vp]
    L.cheb_dm_moments.argtypes = [vp, vp, dp, vp]
    L.cheb_dm_solve_mu.argtypes = [vp, C.c_double, C.c_double, C.c_int, dp, vp]
    L.cheb_dm_product.argtypes = [vp, C.c_double, vp, vp, C.c_double, vp, vp, vp]
    L.cheb_dm_workspace_bytes.argtypes = [vp, C.POINTER(C.c_size_t)]
    L.cheb_dm_last_launch_count.argtypes = [vp, ip]
    L.cheb_dm_flops_per_compute.argtypes = [vp, dp]
    L.cheb_dm_compute_host.argtypes = [vp, vp, vp, vp, vp]
    L.cheb_dm_set_timing.argtypes = [vp, C.c_int]
    L.cheb_dm_product_ms.argtypes = [vp, ip, dp]
    L.cheb_dm_dmma_peak.argtypes = [C.c_int, dp, vp]
    L.cheb_dm_get_options.argtypes = [vp, C.POINTER(Options)]
    L.cheb_dm_check.argtypes = [vp, vp]
    L.cheb_dm_compute_host_async.argtypes = [vp, vp, vp, vp, vp]
    L.cheb_dm_wait.argtypes = [vp, vp]
    L.cheb_dm_set_trace.argtypes = [vp, C.c_int]
    L.cheb_dm_get_trace.argtypes = [vp, C.POINTER(TraceRec), C.c_int, ip]
    pp = C.POINTER(vp)
    L.cheb_dm_compute_batch.argtypes = [vp, C.c_int, pp, pp, dp, vp]
    L.cheb_dm_compute_batch_host.argtypes = [vp, C.c_int, pp, pp, vp, dp, vp]
    L.cheb_dm_compute_batch_host_async.argtypes = [vp, C.c_int, pp, pp, vp, dp, vp]
    L.cheb_dm_trace_batch.argtypes = [vp, C.c_int, pp, vp, vp]
    L.cheb_dm_get_scalars.argtypes = [vp, C.c_int, dp, vp]
    L.cheb_dm_solve.argtypes = [vp, vp, C.c_double, C.c_int, vp, dp, vp]
    L.cheb_dm_solve_batch.argtypes = [vp, C.c_int, pp, dp, C.c_int, pp, dp, vp]
    L.cheb_dm_assemble.argtypes = [vp, C.c_int, dp, pp, vp]
    L.cheb_dm_flops_per_solve.argtypes = [vp, dp]
    L.cheb_dm_sliced_ops_per_compute.argtypes = [vp, dp]
    L.cheb_dm_product_sliced.argtypes = [vp, C.c_double, vp, vp, C.c_double, vp, vp, C.c_int, vp]
    L.cheb_dm_bounds_static.argtypes = [vp, C.c_int, C.c_longlong, vp, vp]
    for n in EXPORTS:
        getattr(L, n).restype = C.c_int
    L.cheb_dm_strerror.argtypes = [C.c_int]
    L.cheb_dm_strerror.restype = C.c_char_p
    _LIB = L
    return L


def _chk(status: int, where: str):
    if status != 0:
        raise ChebDMError(status, where)


def _darr(a):
    import numpy as np
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(C.POINTER(C.c_double))


def _parr(ptrs):
    """HOST array of raw addresses (ints) for the batched calls."""
    n = len(ptrs)
    return (C.c_void_p * n)(*[int(x) for x in ptrs])


def _dvec(vals):
    if vals is None:
        return None
    n = len(vals)
    return (C.c_double * n)(*[float(x) for x in vals])


def dmma_peak(iters: int = 20000, stream: int = 0) -> float:
    """FP64 tensor (DMMA.8x8x4) issue-rate peak of the current device in TFLOP/s (cheb_dm_dmma_peak)."""
    v = C.c_double()
    _chk(lib().cheb_dm_dmma_peak(iters, C.byref(v), stream), "cheb_dm_dmma_peak")
    return v.value


STATIC_MAX_N = 8192  # CHEB_DM_STATIC_MAX_N


def bounds_static(dH: int, N: int, ldh: int, d_bounds: int, stream: int = 0):
    """cheb_dm_bounds_static: Gershgorin bounds (a, b) of the device matrix dH into the 2 device doubles d_bounds; no
    plan, no allocation (scratch in a fixed device array: N <= STATIC_MAX_N, overlapping calls race)."""
    _chk(lib().cheb_dm_bounds_static(dH, N, ldh, d_bounds, stream), "cheb_dm_bounds_static")


class Plan:
    """cheb_dm_plan_t with the same calls as the C ABI.  Pointers are raw device addresses (int)."""

    def __init__(self, N: int, M: int, *, k: int = 0, p: int = 0, outer: int = OUTER_CHEBYSHEV,
                 sched: int = SCHED_GROUPED, pairing: int = PAIR_AUTO, tile: int = TILE_AUTO,
                 fuse_sums: int = 0, giant: int = 0, symmetric: int = 0, max_batch: int = 0, ldh: int = 0, ldd: int = 0,
                 moments: int = 0, host_slots: int = 0, sliced: int = 0, sliced_solve: int = 0, dtype: int = 0):
        self._h = C.c_void_p()
        self.N, self.M = N, M
        o = Options(k=k, p=p, outer=outer, sched=sched, pairing=pairing, tile=tile, fuse_sums=fuse_sums, giant=giant, symmetric=symmetric,
                    max_batch=max_batch, ldh=ldh, ldd=ldd, moments=moments, host_slots=host_slots, sliced=sliced, sliced_solve=sliced_solve)
        _chk(lib().cheb_dm_plan_ex(C.byref(self._h), N, M, dtype, C.byref(o)), "cheb_dm_plan_ex")
        kk, pp = C.c_int(), C.c_int()
        _chk(lib().cheb_dm_get_kp(self._h, C.byref(kk), C.byref(pp)), "cheb_dm_get_kp")
        self.k, self.p = kk.value, pp.value
        self.opts = Options()  # as resolved by the plan (tile, fuse_sums, giant, ...)
        _chk(lib().cheb_dm_get_options(self._h, C.byref(self.opts)), "cheb_dm_get_options")

    def destroy(self):
        if self._h:
            lib().cheb_dm_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def coeffs(self, beta: float, mu: float, bounds=None):
        if bounds is None:
            _chk(lib().cheb_dm_coeffs(self._h, beta, mu, None), "cheb_dm_coeffs")
        else:
            arr = (C.c_double * 2)(float(bounds[0]), float(bounds[1]))
            _chk(lib().cheb_dm_coeffs(self._h, beta, mu, arr), "cheb_dm_coeffs")

    def compute(self, dH: int, dD: int, stream: int = 0):
        _chk(lib().cheb_dm_compute(self._h, dH, dD, stream), "cheb_dm_compute")

    def compute_batch(self, dH, dD, mu=None, stream: int = 0):
        """dH, dD: sequences of device addresses; mu: sequence of floats or None (cheb_dm_compute_batch)."""
        n = len(dH)
        _chk(lib().cheb_dm_compute_batch(self._h, n, _parr(dH), _parr(dD), _dvec(mu), stream), "cheb_dm_compute_batch")

    def compute_batch_host(self, hH, hD, h_trace: int = 0, mu=None, stream: int = 0):
        n = len(hH)
        _chk(lib().cheb_dm_compute_batch_host(self._h, n, _parr(hH), _parr(hD), h_trace or None, _dvec(mu), stream),
             "cheb_dm_compute_batch_host")

    def compute_batch_host_async(self, hH, hD, h_trace: int = 0, mu=None, stream: int = 0):
        n = len(hH)
        _chk(lib().cheb_dm_compute_batch_host_async(self._h, n, _parr(hH), _parr(hD), h_trace or None, _dvec(mu), stream),
             "cheb_dm_compute_batch_host_async")

    def trace_batch(self, dD, d_out: int, stream: int = 0):
        _chk(lib().cheb_dm_trace_batch(self._h, len(dD), _parr(dD), d_out, stream), "cheb_dm_trace_batch")

    def solve(self, dH: int, n_occ: float, dD: int, iters: int = 100, want_mu: bool = True, stream: int = 0):
        """mu-inclusive solve (cheb_dm_solve); returns mu (synchronises) or None."""
        mu = C.c_double()
        _chk(lib().cheb_dm_solve(self._h, dH, float(n_occ), iters, dD, C.byref(mu) if want_mu else None, stream), "cheb_dm_solve")
        return mu.value if want_mu else None

    def solve_batch(self, dH, n_occ, dD, iters: int = 100, want_mu: bool = True, stream: int = 0):
        n = len(dH)
        mu = (C.c_double * n)()
        _chk(lib().cheb_dm_solve_batch(self._h, n, _parr(dH), _dvec(n_occ), iters, _parr(dD), mu if want_mu else None, stream),
             "cheb_dm_solve_batch")
        return [float(x) for x in mu] if want_mu else None

    def assemble(self, mu, dD, stream: int = 0):
        _chk(lib().cheb_dm_assemble(self._h, len(dD), _dvec(mu), _parr(dD), stream), "cheb_dm_assemble")

    def get_scalars(self, slot: int = 0, stream: int = 0):
        """(a, b, mu, N_e(mu)) of a slot after the last call."""
        out = (C.c_double * 4)()
        _chk(lib().cheb_dm_get_scalars(self._h, slot, out, stream), "cheb_dm_get_scalars")
        return tuple(float(x) for x in out)

    def flops_per_solve(self) -> float:
        v = C.c_double()
        _chk(lib().cheb_dm_flops_per_solve(self._h, C.byref(v)), "cheb_dm_flops_per_solve")
        return v.value

    def compute_host(self, hH: int, hD: int, h_trace: int = 0, stream: int = 0):
        """hH, hD, h_trace: HOST addresses (e.g. of pinned torch tensors / numpy arrays)."""
        _chk(lib().cheb_dm_compute_host(self._h, hH, hD, h_trace or None, stream), "cheb_dm_compute_host")

    def check(self, stream: int = 0):
        """Synchronise the stream and raise if the device flagged an error during the last compute."""
        _chk(lib().cheb_dm_check(self._h, stream), "cheb_dm_check")

    def set_trace(self, enable: bool):
        _chk(lib().cheb_dm_set_trace(self._h, int(bool(enable))), "cheb_dm_set_trace")

    def get_trace(self, max_records: int = 1 << 20):
        """Per-tile timeline of the last compute: list of dicts (times in ns of %globaltimer)."""
        buf = (TraceRec * max_records)()
        n = C.c_int()
        _chk(lib().cheb_dm_get_trace(self._h, buf, max_records, C.byref(n)), "cheb_dm_get_trace")
        return [{f: getattr(buf[i], f) for f, _ in TraceRec._fields_} for i in range(n.value)]

    def compute_host_async(self, hH: int, hD: int, h_trace: int = 0, stream: int = 0):
        """Pipelined compute_host: queue one solve (HOST addresses, pinned); results valid after wait()."""
        _chk(lib().cheb_dm_compute_host_async(self._h, hH, hD, h_trace or None, stream), "cheb_dm_compute_host_async")

    def wait(self, stream: int = 0):
        _chk(lib().cheb_dm_wait(self._h, stream), "cheb_dm_wait")

    def set_timing(self, enable: bool):
        _chk(lib().cheb_dm_set_timing(self._h, int(bool(enable))), "cheb_dm_set_timing")

    def product_ms(self):
        """(count, total_ms) of the product-kernel launches recorded since set_timing(True)."""
        n, v = C.c_int(), C.c_double()
        _chk(lib().cheb_dm_product_ms(self._h, C.byref(n), C.byref(v)), "cheb_dm_product_ms")
        return n.value, v.value

    def trace(self, dD: int, d_out: int, stream: int = 0):
        _chk(lib().cheb_dm_trace(self._h, dD, d_out, stream), "cheb_dm_trace")

    def get_bounds(self, stream: int = 0):
        out = (C.c_double * 2)()
        _chk(lib().cheb_dm_get_bounds(self._h, out, stream), "cheb_dm_get_bounds")
        return float(out[0]), float(out[1])

    def get_coeffs(self, stream: int = 0):
        import numpy as np
        n = self.k * self.p
        c, g, d = np.zeros(n), np.zeros(n), np.zeros(n)
        _chk(lib().cheb_dm_get_coeffs(self._h, c.ctypes.data_as(C.POINTER(C.c_double)),
                                      g.ctypes.data_as(C.POINTER(C.c_double)),
                                      d.ctypes.data_as(C.POINTER(C.c_double)), stream), "cheb_dm_get_coeffs")
        return c, g.reshape(self.k, self.p), d.reshape(self.k, self.p)

    def get_T(self, n: int, d_out: int, stream: int = 0):
        _chk(lib().cheb_dm_get_T(self._h, n, d_out, stream), "cheb_dm_get_T")

    def moments(self, dH: int, want_host: bool = True, stream: int = 0):
        import numpy as np
        if want_host:
            tau = np.zeros(self.k * self.p)
            _chk(lib().cheb_dm_moments(self._h, dH, tau.ctypes.data_as(C.POINTER(C.c_double)), stream),
                 "cheb_dm_moments")
            return tau
        _chk(lib().cheb_dm_moments(self._h, dH, None, stream), "cheb_dm_moments")
        return None

    def solve_mu(self, beta: float, n_occ: float, iters: int = 100, stream: int = 0) -> float:
        mu = C.c_double()
        _chk(lib().cheb_dm_solve_mu(self._h, beta, n_occ, iters, C.byref(mu), stream), "cheb_dm_solve_mu")
        return mu.value

    def product(self, alpha: float, dA: int, dB: int, beta: float, dC, d_out: int, stream: int = 0):
        _chk(lib().cheb_dm_product(self._h, alpha, dA, dB, beta, dC, d_out, stream), "cheb_dm_product")

    def product_sliced(self, alpha: float, dA: int, dB: int, beta: float, dC, d_out: int, symmetric: bool = False, stream: int = 0):
        _chk(lib().cheb_dm_product_sliced(self._h, alpha, dA, dB, beta, dC, d_out, 1 if symmetric else 0, stream), "cheb_dm_product_sliced")

    def sliced_ops_per_compute(self) -> float:
        v = C.c_double()
        _chk(lib().cheb_dm_sliced_ops_per_compute(self._h, C.byref(v)), "cheb_dm_sliced_ops_per_compute")
        return v.value

    def workspace_bytes(self) -> int:
        v = C.c_size_t()
        _chk(lib().cheb_dm_workspace_bytes(self._h, C.byref(v)), "cheb_dm_workspace_bytes")
        return v.value

    def last_launch_count(self) -> int:
        v = C.c_int()
        _chk(lib().cheb_dm_last_launch_count(self._h, C.byref(v)), "cheb_dm_last_launch_count")
        return v.value

    def flops_per_compute(self) -> float:
        v = C.c_double()
        _chk(lib().cheb_dm_flops_per_compute(self._h, C.byref(v)), "cheb_dm_flops_per_compute")
        return v.value
