"""Seeded synthetic Hamiltonians for the BASELINE.json configs.

This module is the ONLY code shared by the CUDA path's tests/bench and the CPU oracle.
It holds input generation only -- none of the method's arithmetic (no Chebyshev, no
Fermi function, no bounds, no eigen-solves used for the method).  Inputs are data.

Recipe (SURVEY.md 8(c)-A12 reading of BASELINE.json `configs`):

  cfg0  N=128   open tight-binding chain, h[i,i+1] = h[i+1,i] = -1, plus a dense symmetric
                Gaussian coupling 0.01*N(0,1) (drawn for i<j, mirrored), diagonal U(-0.5,0.5).
                beta=20, M=64, N_occ=64, seed 0.
  cfg1  N=500   off-diagonals N(0,1/N) for i<j (mirrored), diagonal U(-1,1).
                beta=40, M=256, N_occ=250, seeds 0..3.
  cfg2  N=1000  H = Q^T diag(eps) Q, Q = orthogonal factor of a Gaussian matrix (QR, R's
                diagonal made positive), eps = N/2 levels U(-10,-0.25) and N/2 levels
                U(0.25,10) (gap 0.5 at 0).  beta=10, M=256, N_occ=500.
  cfg3  N=5000  off-diagonals N(0,1/N), diagonal U(-2,2).  beta=50, M=1024, N_occ=2500.
  cfg4  N=2000  H = Q^T diag(eps) Q, eps = floor(0.6N) levels N(0,0.01^2) and the rest
                U(-5,5) (high density of states at the Fermi level).
                beta=200, M=2048, N_occ=1000.

Every generator accepts `n` to produce the same *kind* of matrix at a reduced size (for
parity tests the oracle finishes in seconds); N_occ scales as n*N_occ/N.

Draw order with numpy.random.default_rng(seed) is fixed and documented per generator so
that the matrices are reproducible across machines.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class Config:
    name: str
    N: int
    beta: float
    M: int            # number of Chebyshev terms (BASELINE.json "m=... terms")
    N_occ: int
    seeds: tuple
    kind: str
    note: str


CONFIGS = {
    "cfg0": Config("cfg0", 128, 20.0, 64, 64, (0,), "chain",
                   "N=128 open chain -1 hopping + 0.01*N(0,1) dense, diag U(-0.5,0.5)"),
    "cfg1": Config("cfg1", 500, 40.0, 256, 250, (0, 1, 2, 3), "goe",
                   "N=500 GOE-like N(0,1/N) + diag U(-1,1)"),
    "cfg2": Config("cfg2", 1000, 10.0, 256, 500, (0,), "gapped",
                   "N=1000 Q^T diag(eps) Q, eps U[-10,10] with gap 0.5 at 0"),
    "cfg3": Config("cfg3", 5000, 50.0, 1024, 2500, (0,), "goe2",
                   "N=5000 N(0,1/N) + diag U(-2,2)"),
    "cfg4": Config("cfg4", 2000, 200.0, 2048, 1000, (0,), "highdos",
                   "N=2000 Q^T diag(eps) Q, 60% levels N(0,0.01^2), rest U(-5,5)"),
}


def _symmetrize_upper(G: np.ndarray) -> np.ndarray:
    """Keep the strict upper triangle of G and mirror it (diagonal zero)."""
    U = np.triu(G, 1)
    return U + U.T


def _random_orthogonal(rng: np.random.Generator, n: int) -> np.ndarray:
    """Q factor of an n x n Gaussian matrix with R's diagonal made positive."""
    G = rng.standard_normal((n, n))
    Q, R = np.linalg.qr(G)
    s = np.sign(np.diag(R))
    s[s == 0] = 1.0
    return Q * s[None, :]


def _gen_chain(rng, n):
    # draw order: dense Gaussian (n*n), then diagonal (n)
    G = rng.standard_normal((n, n))
    diag = rng.uniform(-0.5, 0.5, size=n)
    H = 0.01 * _symmetrize_upper(G)
    idx = np.arange(n - 1)
    H[idx, idx + 1] += -1.0
    H[idx + 1, idx] += -1.0
    H[np.arange(n), np.arange(n)] = diag
    return H


def _gen_goe(rng, n, diag_halfwidth):
    # draw order: dense Gaussian (n*n), then diagonal (n)
    G = rng.standard_normal((n, n)) / np.sqrt(n)
    diag = rng.uniform(-diag_halfwidth, diag_halfwidth, size=n)
    H = _symmetrize_upper(G)
    H[np.arange(n), np.arange(n)] = diag
    return H


def _from_spectrum(rng, eps):
    n = eps.shape[0]
    Q = _random_orthogonal(rng, n)
    H = (Q.T * eps[None, :]) @ Q
    return 0.5 * (H + H.T)


def _gen_gapped(rng, n):
    # draw order: lower levels (n//2), upper levels (n - n//2), Gaussian for Q (n*n)
    lo = rng.uniform(-10.0, -0.25, size=n // 2)
    hi = rng.uniform(0.25, 10.0, size=n - n // 2)
    eps = np.concatenate([lo, hi])
    return _from_spectrum(rng, eps)


def _gen_highdos(rng, n):
    # draw order: dense levels floor(0.6n) ~ N(0,0.01^2), rest U(-5,5), Gaussian for Q (n*n)
    nd = int(np.floor(0.6 * n))
    dense = 0.01 * rng.standard_normal(nd)
    rest = rng.uniform(-5.0, 5.0, size=n - nd)
    eps = np.concatenate([dense, rest])
    return _from_spectrum(rng, eps)


def hamiltonian(cfg: str, seed: int = 0, n: int | None = None) -> np.ndarray:
    """Return the dense symmetric float64 C-contiguous H for config `cfg` (optionally at size n)."""
    c = CONFIGS[cfg]
    n = c.N if n is None else int(n)
    rng = np.random.default_rng(seed)
    if c.kind == "chain":
        H = _gen_chain(rng, n)
    elif c.kind == "goe":
        H = _gen_goe(rng, n, 1.0)
    elif c.kind == "goe2":
        H = _gen_goe(rng, n, 2.0)
    elif c.kind == "gapped":
        H = _gen_gapped(rng, n)
    elif c.kind == "highdos":
        H = _gen_highdos(rng, n)
    else:  # pragma: no cover
        raise ValueError(c.kind)
    H = np.ascontiguousarray(H, dtype=np.float64)
    assert np.array_equal(H, H.T)
    return H


def n_occ(cfg: str, n: int | None = None) -> int:
    """Target electron count, scaled with the matrix size when n differs from the config's N."""
    c = CONFIGS[cfg]
    if n is None or n == c.N:
        return c.N_occ
    return max(1, int(round(n * c.N_occ / c.N)))


def random_symmetric(n: int, seed: int, scale: float = 1.0) -> np.ndarray:
    """Generic dense symmetric test matrix (uniform entries in [-scale, scale])."""
    rng = np.random.default_rng(seed)
    G = rng.uniform(-scale, scale, size=(n, n))
    return np.ascontiguousarray(0.5 * (G + G.T))
