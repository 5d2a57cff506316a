"""CPU oracle -- TEST INFRASTRUCTURE ONLY (see oracle/cheb_oracle.c header).

Thin ctypes/numpy wrapper around oracle/libcheb_oracle.so (plain C, built by oracle/build.py)
plus two pure-Python pieces that are small enough for loops:
  * algorithm1_schedule(k): the product list of Algorithm 1
  * nq_for(M): the quadrature size fixed by DESIGN.md reading A3

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It imports nothing from paper_2306_12616_b200.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from .build import build as _build, LIB_PATH as _LIB_PATH

_lib = None
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)


def _load():
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH) or os.path.getmtime(_LIB_PATH) < os.path.getmtime(
            os.path.join(os.path.dirname(__file__), "cheb_oracle.c")):
        _build()
    lib = C.CDLL(_LIB_PATH)
    lib.co_num_threads.restype = C.c_int
    lib.co_fermi.restype = C.c_double
    lib.co_fermi.argtypes = [C.c_double] * 3
    lib.co_matmul.argtypes = [C.c_int, _dp, _dp, _dp]
    lib.co_gershgorin.argtypes = [C.c_int, _dp, _dp, _dp]
    lib.co_scale.argtypes = [C.c_int, _dp, C.c_double, C.c_double, _dp]
    lib.co_jacobi_eig.restype = C.c_int
    lib.co_jacobi_eig.argtypes = [C.c_int, _dp, _dp, _dp, C.c_int, C.c_double]
    lib.co_dm_from_eig.argtypes = [C.c_int, _dp, _dp, C.c_double, C.c_double, _dp]
    lib.co_cheb_coeffs.argtypes = [C.c_double] * 4 + [C.c_int, C.c_int, _dp]
    lib.co_cheb_coeffs_of_samples.argtypes = [_dp, C.c_int, C.c_int, _dp]
    lib.co_dm_cheb.argtypes = [C.c_int, _dp, C.c_double, C.c_double, _dp, C.c_int, _dp, _dp]
    lib.co_dm_cheb_columns.argtypes = [C.c_int, _dp, C.c_double, C.c_double, _dp, C.c_int,
                                       C.c_int, _ip, _dp]
    lib.co_eval_cheb_sum.restype = C.c_double
    lib.co_dm_cheb_apply.argtypes = [C.c_int, _dp, C.c_double, C.c_double, _dp, C.c_int, C.c_int, _dp, _dp]
    lib.co_eval_cheb_sum.argtypes = [_dp, C.c_int, C.c_double]
    lib.co_a_matrix.argtypes = [C.c_int, _dp]
    lib.co_x_matrix.argtypes = [C.c_int, C.c_int, _dp, _dp]
    lib.co_back_substitute.restype = C.c_double
    lib.co_back_substitute.argtypes = [C.c_int, _dp, _dp, _dp]
    lib.co_d_from_c_via_X.argtypes = [C.c_int, C.c_int, _dp, _dp]
    lib.co_g_from_c.argtypes = [C.c_int, C.c_int, _dp, _dp]
    lib.co_d_from_g.argtypes = [C.c_int, C.c_int, _dp, _dp]
    lib.co_eval_eq4.restype = C.c_double
    lib.co_eval_eq4.argtypes = [C.c_int, C.c_int, _dp, C.c_double]
    lib.co_eval_eq6.restype = C.c_double
    lib.co_eval_eq6.argtypes = [C.c_int, C.c_int, _dp, C.c_double]
    lib.co_electron_count.restype = C.c_double
    lib.co_electron_count.argtypes = [_dp, C.c_double, C.c_double, C.c_double, C.c_double,
                                      C.c_int, C.c_int]
    lib.co_solve_mu.restype = C.c_double
    lib.co_solve_mu.argtypes = [_dp, C.c_double, C.c_double, C.c_double, C.c_int, C.c_int,
                                C.c_double, C.c_int]
    lib.co_solve_mu_exact.restype = C.c_double
    lib.co_solve_mu_exact.argtypes = [C.c_int, _dp, C.c_double, C.c_double, C.c_double,
                                      C.c_double, C.c_int]
    _lib = lib
    return lib


def _p(a):
    return a.ctypes.data_as(_dp)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads() -> int:
    return int(_load().co_num_threads())


def nq_for(M: int) -> int:
    """Quadrature size N_q = 2^ceil(log2(4M)) (reading A3)."""
    nq = 1
    while nq < 4 * M:
        nq *= 2
    return nq


def fermi(beta, mu, eps) -> float:
    return float(_load().co_fermi(beta, mu, eps))


def matmul(A, B):
    A, B = _f64(A), _f64(B)
    n = A.shape[0]
    Cm = np.empty((n, n))
    _load().co_matmul(n, _p(A), _p(B), _p(Cm))
    return Cm


def gershgorin(H):
    H = _f64(H)
    a, b = C.c_double(), C.c_double()
    _load().co_gershgorin(H.shape[0], _p(H), C.byref(a), C.byref(b))
    return a.value, b.value


def scale(H, a, b):
    H = _f64(H)
    X = np.empty_like(H)
    _load().co_scale(H.shape[0], _p(H), a, b, _p(X))
    return X


def jacobi_eig(H, max_sweeps=60, tol=1e-14):
    """Returns (E, V) with columns of V the eigenvectors (H V = V diag(E)); unsorted."""
    H = _f64(H)
    n = H.shape[0]
    E = np.empty(n)
    Vt = np.empty((n, n))
    sweeps = _load().co_jacobi_eig(n, _p(H), _p(E), _p(Vt), max_sweeps, tol)
    if sweeps < 0:
        raise RuntimeError("Jacobi did not converge")
    return E, Vt.T.copy()


def jacobi_sweeps(H, max_sweeps=60, tol=1e-14) -> int:
    """Runs co_jacobi_eig and returns its sweep count (-1: stopped at max_sweeps before off(H) <= tol |H|_F).
    For timing the eigensolver (bench.py's cpu_baseline): max_sweeps = 1 times one sweep."""
    H = _f64(H)
    n = H.shape[0]
    E = np.empty(n)
    Vt = np.empty((n, n))
    return int(_load().co_jacobi_eig(n, _p(H), _p(E), _p(Vt), max_sweeps, tol))


def dm_from_eig(E, V, beta, mu):
    E = _f64(E)
    Vt = _f64(np.asarray(V).T)
    n = E.shape[0]
    D = np.empty((n, n))
    _load().co_dm_from_eig(n, _p(E), _p(Vt), beta, mu, _p(D))
    return D


def dm_eig(H, beta, mu):
    """O-eig: D = V f(E) V^T via cyclic Jacobi (Eq. 1-2)."""
    E, V = jacobi_eig(H)
    return dm_from_eig(E, V, beta, mu)


def cheb_coeffs(beta, mu, a, b, M, Nq=None):
    Nq = nq_for(M) if Nq is None else Nq
    c = np.empty(M)
    _load().co_cheb_coeffs(beta, mu, a, b, M, Nq, _p(c))
    return c


def cheb_coeffs_of_samples(fvals, M):
    fvals = _f64(fvals)
    c = np.empty(M)
    _load().co_cheb_coeffs_of_samples(_p(fvals), M, fvals.shape[0], _p(c))
    return c


def dm_cheb(H, a, b, c, want_tau=False):
    """O-cheb: sum_{n<M} c_n T_n(X) by the naive three-term matrix recurrence."""
    H, c = _f64(H), _f64(c)
    n = H.shape[0]
    D = np.empty((n, n))
    tau = np.empty(c.shape[0]) if want_tau else None
    _load().co_dm_cheb(n, _p(H), a, b, _p(c), c.shape[0], _p(D), _p(tau) if want_tau else None)
    return (D, tau) if want_tau else D


def dm_cheb_columns(H, a, b, c, cols):
    H, c = _f64(H), _f64(c)
    n = H.shape[0]
    cols = np.ascontiguousarray(cols, dtype=np.int32)
    out = np.empty((cols.shape[0], n))
    _load().co_dm_cheb_columns(n, _p(H), a, b, _p(c), c.shape[0], cols.shape[0],
                               cols.ctypes.data_as(_ip), _p(out))
    return out


def dm_cheb_apply(H, a, b, c, V):
    """(sum_{n<M} c_n T_n(X)) applied to the rows of V (nvec x n) by the vector three-term recurrence."""
    H, c, V = _f64(H), _f64(c), _f64(V)
    n = H.shape[0]
    V = V.reshape(-1, n)
    out = np.empty_like(V)
    _load().co_dm_cheb_apply(n, _p(H), a, b, _p(c), c.shape[0], V.shape[0], _p(V), _p(out))
    return out


def eval_cheb_sum(c, x) -> float:
    c = _f64(c)
    return float(_load().co_eval_cheb_sum(_p(c), c.shape[0], x))


def a_matrix(p):
    A = np.empty((p, p))
    _load().co_a_matrix(p, _p(A))
    return A


def x_matrix(k, p):
    A = a_matrix(p)
    X = np.empty((k * p, k * p))
    _load().co_x_matrix(k, p, _p(A), _p(X))
    return X


def back_substitute(U, rhs):
    U, rhs = _f64(U), _f64(rhs)
    x = np.empty(rhs.shape[0])
    lower = _load().co_back_substitute(rhs.shape[0], _p(U), _p(rhs), _p(x))
    return x, float(lower)


def pad_coeffs(c, k, p):
    c = _f64(c)
    out = np.zeros(k * p)
    out[: c.shape[0]] = c
    return out


def d_from_c_via_X(k, p, c):
    c = pad_coeffs(c, k, p)
    d = np.empty((k, p))
    _load().co_d_from_c_via_X(k, p, _p(c), _p(d))
    return d


def g_from_c(k, p, c):
    c = pad_coeffs(c, k, p)
    g = np.empty((k, p))
    _load().co_g_from_c(k, p, _p(c), _p(g))
    return g


def d_from_g(k, p, g):
    g = _f64(g)
    d = np.empty((k, p))
    _load().co_d_from_g(k, p, _p(g), _p(d))
    return d


def eval_eq4(k, p, d, x) -> float:
    d = _f64(d)
    return float(_load().co_eval_eq4(k, p, _p(d), x))


def eval_eq6(k, p, d, x) -> float:
    d = _f64(d)
    return float(_load().co_eval_eq6(k, p, _p(d), x))


def electron_count(tau, beta, mu, a, b, Nq=None) -> float:
    tau = _f64(tau)
    M = tau.shape[0]
    Nq = nq_for(M) if Nq is None else Nq
    return float(_load().co_electron_count(_p(tau), beta, mu, a, b, M, Nq))


def solve_mu(tau, beta, a, b, n_occ, iters=100, Nq=None) -> float:
    tau = _f64(tau)
    M = tau.shape[0]
    Nq = nq_for(M) if Nq is None else Nq
    return float(_load().co_solve_mu(_p(tau), beta, a, b, M, Nq, float(n_occ), iters))


def solve_mu_exact(E, beta, lo, hi, n_occ, iters=100) -> float:
    E = _f64(E)
    return float(_load().co_solve_mu_exact(E.shape[0], _p(E), beta, lo, hi, float(n_occ), iters))


def choose_kp(M: int):
    """Block sizes per SURVEY 8(a): k = ceil(sqrt(M)), p = ceil(M/k) (minimum at
    k = m = sqrt(L+1); Eq. 4 holds for any k*p >= M with zero-padded c)."""
    k = 1
    while k * k < M:
        k += 1
    p = (M + k - 1) // k
    return k, p


def algorithm1_schedule(k: int):
    """Algorithm 1, followed line by line.  Returns a list of stages; each
    stage is a list of products (n, left, right, minus) meaning T_n = 2 T_left T_right - T_minus.
    Reading A7: for s = 1, u = 2^{s-2} is not an integer, so only T_2 = 2 T_1 T_1 - T_0 runs;
    the two loops apply for s >= 2."""
    stages = []
    if k < 2:
        return stages
    nstages = 0
    while (1 << nstages) < k:
        nstages += 1  # ceil(log2 k)
    for s in range(1, nstages + 1):
        prods = []
        if s == 1:
            prods.append((2, 1, 1, 0))
        else:
            u, v = 2 ** (s - 2), 2 ** (s - 1)
            for i in range(u + 1, v + 1):          # u < i <= v
                if i + u <= k:
                    prods.append((i + u, i, u, i - u))
            for i in range(u + 1, v + 1):
                if i + v <= k:
                    prods.append((i + v, v, i, v - i))
        stages.append(prods)
    return stages
