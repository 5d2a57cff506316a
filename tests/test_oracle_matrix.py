"""Pins for the matrix-level oracle functions (oracle/cheb_oracle.c): O-eig (Jacobi + Eq. 1-2),
O-cheb (PAPER.md:91 with the three-term recurrence), Gershgorin, scaling, trace / mu.

Each test checks the oracle against something that is NOT the oracle: closed forms, a LAPACK
routine (numpy.linalg.eigh) as a textbook cross-check, brute force via Eq. 3 on 4x4 matrices
(series expm + Gauss-Jordan inverse written out here), invariants the mathematics fixes.
All CPU, `-m "not gpu"`.
"""
import math

import numpy as np
import pytest

import oracle
import workloads


# ------------------------------------------------------------------------------ O-eig pins (P4)
def test_jacobi_matches_lapack_and_is_orthogonal():
    H = workloads.hamiltonian("cfg1", seed=0, n=60)
    E, V = oracle.jacobi_eig(H)
    assert np.max(np.abs(H @ V - V * E[None, :])) < 1e-12
    assert np.max(np.abs(V.T @ V - np.eye(60))) < 1e-12
    assert np.max(np.abs(np.sort(E) - np.linalg.eigvalsh(H))) < 1e-12


def test_dm_eig_diagonal_H_is_fermi_of_diagonal():
    eps = np.array([-1.5, -0.2, 0.0, 0.3, 2.0])
    D = oracle.dm_eig(np.diag(eps), beta=7.0, mu=0.1)
    expect = 1.0 / (1.0 + np.exp(7.0 * (eps - 0.1)))
    assert np.max(np.abs(D - np.diag(expect))) < 1e-15


def test_dm_eig_2x2_closed_form():
    # H = [[h, t],[t, -h]] has eigenvalues +-r, r = sqrt(h^2+t^2); f(H) = f0 I + f1 H with
    # f0 = (f(r)+f(-r))/2 = 1/2 (mu=0), f1 = (f(r)-f(-r))/(2r).
    h, t, beta = 0.3, -0.8, 3.0
    r = math.hypot(h, t)
    f = lambda e: 1.0 / (1.0 + math.exp(beta * e))
    f1 = (f(r) - f(-r)) / (2 * r)
    H = np.array([[h, t], [t, -h]])
    D = oracle.dm_eig(H, beta=beta, mu=0.0)
    assert np.max(np.abs(D - (0.5 * np.eye(2) + f1 * H))) < 1e-15


def _expm_series(A):
    """exp(A) by scaling-and-squaring with a long Taylor series (independent of any eigensolver)."""
    s = max(0, int(math.ceil(math.log2(max(1.0, np.abs(A).sum(axis=1).max())))) + 4)
    B = A / 2.0 ** s
    term = np.eye(A.shape[0])
    out = np.eye(A.shape[0])
    for i in range(1, 40):
        term = term @ B / i
        out = out + term
    for _ in range(s):
        out = out @ out
    return out


def _gauss_jordan_inverse(A):
    n = A.shape[0]
    M = np.hstack([A.astype(float).copy(), np.eye(n)])
    for c in range(n):
        piv = c + int(np.argmax(np.abs(M[c:, c])))
        M[[c, piv]] = M[[piv, c]]
        M[c] /= M[c, c]
        for r in range(n):
            if r != c:
                M[r] -= M[r, c] * M[c]
    return M[:, n:]


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_dm_eig_4x4_bruteforce_eq3(seed):
    """Eq. 3: D = [I + exp(beta(H - mu I))]^{-1}, by a route with no eigenvectors."""
    H = workloads.random_symmetric(4, seed)
    beta, mu = 2.5, 0.15
    D_ref = _gauss_jordan_inverse(np.eye(4) + _expm_series(beta * (H - mu * np.eye(4))))
    D = oracle.dm_eig(H, beta=beta, mu=mu)
    assert np.max(np.abs(D - D_ref)) < 1e-12


def test_dm_eig_invariants_trace_commutator_idempotency():
    H = workloads.hamiltonian("cfg2", seed=0, n=40)    # gap of 0.5 at 0
    E, V = oracle.jacobi_eig(H)
    D = oracle.dm_from_eig(E, V, beta=10.0, mu=0.0)
    f = 1.0 / (1.0 + np.exp(10.0 * np.linalg.eigvalsh(H)))
    assert abs(np.trace(D) - f.sum()) < 1e-12                 # tr D = sum f(eps_i)
    assert np.max(np.abs(H @ D - D @ H)) < 1e-12              # [H, D] = 0
    assert np.max(np.abs(D - D.T)) < 1e-14
    # beta -> infinity with mu in the gap: projector onto the occupied levels
    Dinf = oracle.dm_from_eig(E, V, beta=1e6, mu=0.0)
    assert np.max(np.abs(Dinf @ Dinf - Dinf)) < 1e-12
    assert abs(np.trace(Dinf) - 20) < 1e-12


# ---------------------------------------------------------------------------- Gershgorin (P9)
def test_gershgorin_diagonal_and_chain_closed_forms():
    a, b = oracle.gershgorin(np.diag([3.0, -2.0, 0.5]))
    assert (a, b) == (-2.0, 3.0)
    n = 10
    H = np.zeros((n, n))
    idx = np.arange(n - 1)
    H[idx, idx + 1] = H[idx + 1, idx] = -1.0
    assert oracle.gershgorin(H) == (-2.0, 2.0)                # interior rows: 0 -+ (1+1)


@pytest.mark.parametrize("cfg", ["cfg0", "cfg1", "cfg2", "cfg3", "cfg4"])
def test_gershgorin_contains_spectrum(cfg):
    H = workloads.hamiltonian(cfg, seed=0, n=64)
    a, b = oracle.gershgorin(H)
    ev = np.linalg.eigvalsh(H)
    assert a <= ev[0] and ev[-1] <= b


def test_scale_maps_bounds_to_unit_interval():
    # X = (2H - (a+b)I)/(b-a): eigenvalue a -> -1, b -> +1 (reading A1 of PAPER.md:96)
    X = oracle.scale(np.diag([-3.0, 5.0, 1.0]), -3.0, 5.0)
    assert np.allclose(np.diag(X), [-1.0, 1.0, 0.0], atol=1e-16)
    H = workloads.random_symmetric(7, 3)
    X = oracle.scale(H, -4.0, 6.0)
    assert np.max(np.abs(X - (2 * H - 2.0 * np.eye(7)) / 10.0)) < 1e-16


# ------------------------------------------------------------------------------- O-cheb (P5)
def test_matmul_matches_blas():
    rng = np.random.default_rng(0)
    A, B = rng.standard_normal((37, 37)), rng.standard_normal((37, 37))
    assert np.max(np.abs(oracle.matmul(A, B) - A @ B)) < 1e-12
    # transposed-operand mistake would fail: A@B != B@A for generic matrices
    assert np.max(np.abs(oracle.matmul(A, B) - B @ A)) > 1e-3


def test_dm_cheb_diagonal_H_is_scalar_chebyshev_sum():
    eps = np.linspace(-1.8, 1.7, 9)
    a, b, beta, mu, M = -2.0, 2.0, 6.0, 0.2, 40
    c = oracle.cheb_coeffs(beta, mu, a, b, M)
    D = oracle.dm_cheb(np.diag(eps), a, b, c)
    xt = (2 * eps - (a + b)) / (b - a)
    expect = np.array([oracle.eval_cheb_sum(c, x) for x in xt])
    assert np.max(np.abs(D - np.diag(expect))) < 1e-14
    # N = 1
    D1 = oracle.dm_cheb(np.array([[0.4]]), a, b, c)
    assert abs(D1[0, 0] - oracle.eval_cheb_sum(c, 0.2)) < 1e-14


def test_dm_cheb_single_terms_are_chebyshev_polynomials_of_X():
    """c = e_n  =>  D = T_n(X) = V cos(n arccos x~) V^T (definition of T_n; LAPACK eigenvectors)."""
    H = workloads.random_symmetric(12, 5)
    a, b = oracle.gershgorin(H)
    w, V = np.linalg.eigh(H)
    xt = (2 * w - (a + b)) / (b - a)
    for n in (0, 1, 2, 3, 7):
        c = np.zeros(8)
        c[n] = 1.0
        D = oracle.dm_cheb(H, a, b, c)
        Tn = (V * np.cos(n * np.arccos(xt))[None, :]) @ V.T
        assert np.max(np.abs(D - Tn)) < 1e-13, n


@pytest.mark.parametrize("cfg", ["cfg0", "cfg1", "cfg4"])
def test_dm_cheb_equals_polynomial_of_eigenvalues(cfg):
    H = workloads.hamiltonian(cfg, seed=0, n=48)
    c0 = workloads.CONFIGS[cfg]
    a, b = oracle.gershgorin(H)
    M = 96
    c = oracle.cheb_coeffs(c0.beta, 0.05, a, b, M)
    D, tau = oracle.dm_cheb(H, a, b, c, want_tau=True)
    w, V = np.linalg.eigh(H)
    xt = (2 * w - (a + b)) / (b - a)
    pM = np.array([oracle.eval_cheb_sum(c, x) for x in xt])
    assert np.max(np.abs(D - (V * pM[None, :]) @ V.T)) < 1e-12
    assert np.max(np.abs(D - D.T)) < 1e-13
    assert np.max(np.abs(H @ D - D @ H)) < 1e-11
    # moments: tau_n = sum_i cos(n arccos x~_i), tau_0 = N  (P8)
    tau_ref = np.array([np.cos(n * np.arccos(xt)).sum() for n in range(M)])
    assert tau[0] == 48
    assert np.max(np.abs(tau - tau_ref)) < 1e-11
    assert abs(np.trace(D) - float(np.dot(c, tau))) < 1e-11   # tr D = sum c_n tau_n


def test_dm_cheb_columns_equal_full_matrix_columns():
    H = workloads.hamiltonian("cfg1", seed=1, n=33)
    a, b = oracle.gershgorin(H)
    c = oracle.cheb_coeffs(40.0, 0.0, a, b, 50)
    D = oracle.dm_cheb(H, a, b, c)
    cols = [0, 7, 32]
    out = oracle.dm_cheb_columns(H, a, b, c, cols)
    assert np.max(np.abs(out - D[:, cols].T)) < 1e-13


def test_dm_cheb_apply_equals_matrix_times_vectors_and_column_routine():
    """oracle.dm_cheb_apply (vector three-term recurrence) against the matrix route: D_cheb @ v for
    Gaussian and +-1 vectors, unit vectors = the column routine, M = 1 and M = 2 (no recurrence step), and a
    diagonal H where (D v)_i = p_M(x~_i) v_i with p_M by the definition T_n = cos(n arccos x)."""
    n = 33
    H = workloads.hamiltonian("cfg1", seed=1, n=n)
    a, b = oracle.gershgorin(H)
    c = oracle.cheb_coeffs(40.0, 0.02, a, b, 50)
    D = oracle.dm_cheb(H, a, b, c)
    rng = np.random.default_rng(5)
    V = np.vstack([rng.standard_normal((2, n)), rng.choice([-1.0, 1.0], size=(2, n))])
    out = oracle.dm_cheb_apply(H, a, b, c, V)
    assert np.max(np.abs(out - V @ D.T)) < 1e-13
    # a dropped term / wrong sign in the recurrence shows up at O(|c_n|) ~ 1e-2
    assert np.max(np.abs(out - V @ D.T)) < 1e-6 * np.max(np.abs(c[2:10]))
    E = np.eye(n)[[0, 7, 32]]
    assert np.max(np.abs(oracle.dm_cheb_apply(H, a, b, c, E) - oracle.dm_cheb_columns(H, a, b, c, [0, 7, 32]))) < 1e-14
    for M in (1, 2, 3):
        DM = oracle.dm_cheb(H, a, b, c[:M].copy())
        assert np.max(np.abs(oracle.dm_cheb_apply(H, a, b, c[:M].copy(), V) - V @ DM.T)) < 1e-14
    eps = np.linspace(-1.3, 0.9, 12)
    Hd = np.diag(eps)
    cd = oracle.cheb_coeffs(9.0, -0.1, -1.5, 1.0, 30)
    pm = np.array([oracle.eval_cheb_sum(cd, float((2 * e + 0.5) / 2.5)) for e in eps])
    v = rng.standard_normal((1, 12))
    assert np.max(np.abs(oracle.dm_cheb_apply(Hd, -1.5, 1.0, cd, v) - pm * v)) < 1e-13


# ---------------------------------------------------------------------------- truncation (P7)
def test_truncation_error_bounded_by_tail_and_decays_exponentially():
    """||D_cheb - D_eig||_max <= sum_{n>=M}|c_n|, decaying like exp(-pi M / beta~)
    (paper: 'exponential error decay').  Tight bounds, beta~ ~ 46."""
    H = workloads.hamiltonian("cfg1", seed=0, n=40)
    ev = np.linalg.eigvalsh(H)
    a, b = ev[0] - 0.05, ev[-1] + 0.05
    beta, mu = 20.0, 0.03
    D_eig = oracle.dm_eig(H, beta, mu)
    c_long = oracle.cheb_coeffs(beta, mu, a, b, 400)
    errs = []
    for M in (16, 32, 64, 128, 256):
        D = oracle.dm_cheb(H, a, b, c_long[:M].copy())
        # c_n from a larger Nq differ slightly from nq_for(M) ones; the tail bound uses c_long
        err = np.max(np.abs(D - D_eig))
        tail = np.sum(np.abs(c_long[M:])) + 1e-13
        assert err <= tail, (M, err, tail)
        errs.append(err)
    assert errs[0] > errs[1] > errs[2] > errs[3] > errs[4]
    beta_t = beta * (b - a) / 2
    rate = math.log(errs[1] / errs[2]) / 32.0            # per-term decay between M=32 and 64
    assert 0.5 * math.pi / beta_t < rate < 2.0 * math.pi / beta_t
    assert errs[4] < 1e-6


# ------------------------------------------------------------------------------ mu / trace (P8)
def test_solve_mu_hits_target_electron_count():
    H = workloads.hamiltonian("cfg0", seed=0, n=32)
    a, b = oracle.gershgorin(H)
    M, beta, nocc = 64, 20.0, 16
    c_any = oracle.cheb_coeffs(beta, 0.0, a, b, M)
    _, tau = oracle.dm_cheb(H, a, b, c_any, want_tau=True)
    mu = oracle.solve_mu(tau, beta, a, b, nocc)
    assert a < mu < b
    assert abs(oracle.electron_count(tau, beta, mu, a, b) - nocc) < 1e-9
    D = oracle.dm_cheb(H, a, b, oracle.cheb_coeffs(beta, mu, a, b, M))
    assert abs(np.trace(D) - nocc) < 1e-9
    # exact-spectrum counterpart agrees up to the truncation error of the expansion
    mu_ex = oracle.solve_mu_exact(np.linalg.eigvalsh(H), beta, a, b, nocc)
    f = 1.0 / (1.0 + np.exp(beta * (np.linalg.eigvalsh(H) - mu_ex)))
    assert abs(f.sum() - nocc) < 1e-9
    assert abs(mu - mu_ex) < 0.05
