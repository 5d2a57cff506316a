"""Oracle-side construction of the parity cases (inputs and expected values come from oracle/ and
workloads/ only -- never from the CUDA path).

case(cfg, seed, n, M): H (seeded, workloads/), Gershgorin bounds, Jacobi spectrum, the chemical
potential that puts N_occ electrons into the M-term expansion (reading A9), the M
Chebyshev coefficients, D_cheb (naive recurrence), D_eig (Eq. 1-2) and the scalar
truncation error eps_trunc = max_i |f(eps_i) - p_M(x~_i)| (SURVEY 8(c) gates).
"""
import functools

import numpy as np

import oracle
import workloads


def moments_from_spectrum(E, a, b, M):
    """tau_n = tr T_n(X) = sum_i cos(n arccos x~_i) (definition of T_n; pin P8)."""
    xt = np.clip((2.0 * np.asarray(E, dtype=np.longdouble) - (a + b)) / (b - a), -1.0, 1.0)
    th = np.arccos(xt)
    n = np.arange(M, dtype=np.longdouble)[:, None]
    return np.asarray(np.cos(n * th[None, :]).sum(axis=1), dtype=np.float64)


@functools.lru_cache(maxsize=16)
def case(cfg, seed=0, n=None, M=None, full=True, bounds="gershgorin", mu_fixed=None):
    c = workloads.CONFIGS[cfg]
    H = workloads.hamiltonian(cfg, seed=seed, n=n)
    N = H.shape[0]
    M = c.M if M is None else M
    nocc = workloads.n_occ(cfg, N)
    if N <= 1200:
        E, V = oracle.jacobi_eig(H)
    else:  # library eigenvalues only (LAPACK as a primitive); no eigenvectors / D_eig at this size
        E, V = np.linalg.eigvalsh(H), None
    if bounds == "gershgorin":
        a, b = oracle.gershgorin(H)
    else:  # tight: spectrum widened by 1 %
        lo, hi = float(E.min()), float(E.max())
        w = 0.01 * (hi - lo)
        a, b = lo - w, hi + w
    tau = moments_from_spectrum(E, a, b, M)
    # mu_fixed: skip the bisection (100 x M x N_q long-double terms: minutes for M ~ 4600) and use the given value
    mu = oracle.solve_mu(tau, c.beta, a, b, nocc, iters=100) if mu_fixed is None else float(mu_fixed)
    coef = oracle.cheb_coeffs(c.beta, mu, a, b, M)
    out = dict(cfg=cfg, H=H, N=N, M=M, beta=c.beta, nocc=nocc, a=a, b=b, E=E, V=V, tau=tau, mu=mu, c=coef)
    xt = (2.0 * E - (a + b)) / (b - a)
    pM = np.array([oracle.eval_cheb_sum(coef, float(x)) for x in xt])
    fE = np.array([oracle.fermi(c.beta, mu, float(e)) for e in E])
    out["eps_trunc"] = float(np.max(np.abs(fE - pM)))
    out["trace_cheb_scalar"] = float(np.sum(pM))
    if full:
        out["D_cheb"] = oracle.dm_cheb(H, a, b, coef)
        if V is not None:
            out["D_eig"] = oracle.dm_from_eig(E, V, c.beta, mu)
    return out
