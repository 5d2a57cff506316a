"""Pins for the oracle's scalar pipeline (a_{j,l}, X, g, d, c_n, Algorithm 1) -- CPU only.

Each test checks oracle/ against something the paper prints, a closed form, an independent
library routine or brute force -- never against the oracle's own formula retyped.
"""
import math

import numpy as np
import pytest
from numpy.polynomial import chebyshev as npcheb

import oracle


# ---------------------------------------------------------------- P1: a_{j,l} (Eq. 8-12)
def test_a_matrix_equals_eq12_printed(golden):
    A_paper = golden("eq12_A_matrix.txt")
    assert np.array_equal(oracle.a_matrix(5), A_paper)


def test_a_matrix_rows_equal_eq8_printed(golden):
    rows = golden("eq8_powers.txt")
    A = oracle.a_matrix(5)
    for r in rows:
        j = int(r[0])
        assert np.array_equal(A[j], r[1:])


def test_a_matrix_base_of_recurrence():
    # a_{0,0}=1, a_{1,0}=0, a_{1,1}=1
    A = oracle.a_matrix(3)
    assert A[0, 0] == 1.0 and A[1, 0] == 0.0 and A[1, 1] == 1.0


@pytest.mark.parametrize("p", [1, 2, 7, 16, 33])
def test_a_matrix_is_chebyshev_expansion_of_monomials(p):
    # closed form: T_k^j = y^j with y = T_k, and T_{lk} = T_l(y)  =>  row j = poly2cheb(y^j)
    A = oracle.a_matrix(p)
    for j in range(p):
        mono = np.zeros(j + 1)
        mono[j] = 1.0
        ref = np.zeros(p)
        ref[: j + 1] = npcheb.poly2cheb(mono)
        assert np.allclose(A[j], ref, rtol=1e-13, atol=1e-300)


def test_a_matrix_parity_zeros_and_lower_triangular():
    # a_{j,l} = 0 if j,l differ in parity; lower-triangular (Eq. 11)
    A = oracle.a_matrix(12)
    for j in range(12):
        for l in range(12):
            if l > j or (j - l) % 2 == 1:
                assert A[j, l] == 0.0
            else:
                assert A[j, l] > 0.0
    assert np.allclose(A.sum(axis=1), 1.0)  # T_k^j at y=1: all T_l(1)=1


# ---------------------------------------------------------------- P2: X, g, d (Eq. 4-6, 16-20)
def _cheb_mul(u, v):
    """Product of two Chebyshev series by Eq. (7): 2 T_n T_m = T_{n+m} + T_{|n-m|} -- brute force."""
    out = np.zeros(len(u) + len(v) - 1)
    for n, un in enumerate(u):
        for m, vm in enumerate(v):
            out[n + m] += 0.5 * un * vm
            out[abs(n - m)] += 0.5 * un * vm
    return out


def _expand_eq6_bruteforce(k, p, d):
    """Chebyshev coefficients of sum_j sum_i d_{i,j} T_k^j T_i (Eq. 6) by repeated Eq. (7)."""
    total = np.zeros(k * p)
    Tk = np.zeros(k + 1)
    Tk[k] = 1.0
    power = np.array([1.0])  # T_k^0
    for j in range(p):
        for i in range(k):
            Ti = np.zeros(i + 1)
            Ti[i] = 1.0
            term = d[i, j] * _cheb_mul(power, Ti)
            total[: len(term)] += term[: k * p]
            assert np.all(term[k * p:] == 0.0)
        power = _cheb_mul(power, Tk)
    return total


KP = [(1, 1), (2, 1), (1, 3), (2, 2), (3, 2), (2, 3), (5, 5), (4, 7), (7, 4), (8, 8)]


@pytest.mark.parametrize("k,p", KP)
def test_d_bruteforce_expansion_reproduces_c(k, p):
    rng = np.random.default_rng(100 * k + p)
    c = rng.standard_normal(k * p)
    d = oracle.d_from_c_via_X(k, p, c)
    c_back = _expand_eq6_bruteforce(k, p, d)
    assert np.allclose(c_back, c, rtol=0, atol=1e-12 * max(1.0, np.abs(d).max()))


@pytest.mark.parametrize("k,p", KP)
def test_two_solve_routes_agree(k, p):
    rng = np.random.default_rng(7 + 31 * k + p)
    c = rng.standard_normal(k * p)
    d1 = oracle.d_from_c_via_X(k, p, c)
    d2 = oracle.d_from_g(k, p, oracle.g_from_c(k, p, c))
    assert np.allclose(d1, d2, rtol=1e-12, atol=1e-13 * np.abs(d1).max())


@pytest.mark.parametrize("k,p", KP + [(16, 16), (6, 11)])
def test_eq4_equals_eq6_equals_direct_sum(k, p):
    rng = np.random.default_rng(k * 1000 + p)
    M = k * p
    c = rng.standard_normal(M) * np.exp(-0.15 * np.arange(M))  # decaying, like a real expansion
    d = oracle.d_from_c_via_X(k, p, c)
    scale = max(1.0, np.abs(d).max())
    for x in [-1.0, -0.83, -0.31, 0.0, 0.2, 0.5, 0.999, 1.0]:
        ref = sum(c[n] * math.cos(n * math.acos(x)) for n in range(M))  # definition of T_n
        assert abs(oracle.eval_cheb_sum(c, x) - ref) < 1e-13
        assert abs(oracle.eval_eq4(k, p, d, x) - ref) < 1e-12 * scale
        assert abs(oracle.eval_eq6(k, p, d, x) - ref) < 1e-12 * scale


def test_zero_padding_is_exact():
    # M not a multiple of k: pad c with zeros up to k*p; polynomial unchanged
    M = 23
    k, p = oracle.choose_kp(M)
    assert (k, p) == (5, 5)
    rng = np.random.default_rng(5)
    c = rng.standard_normal(M)
    d = oracle.d_from_c_via_X(k, p, c)
    for x in [-0.7, 0.05, 0.6]:
        assert abs(oracle.eval_eq4(k, p, d, x) - oracle.eval_cheb_sum(c, x)) < 1e-12


def test_x_matrix_structure():
    # PAPER.md:171-182 and Eq. 25: upper-triangular; the first block row carries
    # the I blocks without the 1/2; blocks are a_{j,l} / (w a_{j,l} I + 1/2 a_{j,l+1} J).
    k, p = 4, 5
    X = oracle.x_matrix(k, p)
    A = oracle.a_matrix(p)
    assert np.all(np.tril(X, -1) == 0.0)
    J = np.fliplr(np.eye(k - 1))
    for l in range(p):
        for j in range(p):
            blk = X[l * k:(l + 1) * k, j * k:(j + 1) * k]
            w = 1.0 if l == 0 else 0.5
            a1 = A[j, l + 1] if l + 1 < p else 0.0
            assert blk[0, 0] == A[j, l]
            assert np.all(blk[0, 1:] == 0) and np.all(blk[1:, 0] == 0)
            assert np.array_equal(blk[1:, 1:], w * A[j, l] * np.eye(k - 1) + 0.5 * a1 * J)
    # Appendix: last diagonal block = diag(a_{m-1,m-1}, 1/2 a_{m-1,m-1} I)
    last = X[(p - 1) * k:, (p - 1) * k:]
    assert np.array_equal(last, np.diag([A[p - 1, p - 1]] + [0.5 * A[p - 1, p - 1]] * (k - 1)))
    # Eq. 25: first block row, scalar row = a_{0,0} 0 a_{2,0} 0 a_{4,0}
    assert np.array_equal(X[0, ::k], A[:, 0])


def test_back_substitute_matches_numpy_solve():
    rng = np.random.default_rng(3)
    U = np.triu(rng.standard_normal((9, 9))) + 4 * np.eye(9)
    rhs = rng.standard_normal(9)
    x, lower = oracle.back_substitute(U, rhs)
    assert lower == 0.0
    assert np.allclose(x, np.linalg.solve(U, rhs), rtol=1e-12)


def test_choose_kp_matches_survey_table():
    assert oracle.choose_kp(64) == (8, 8)
    assert oracle.choose_kp(256) == (16, 16)
    assert oracle.choose_kp(1024) == (32, 32)
    assert oracle.choose_kp(2048) == (46, 45)
    assert oracle.choose_kp(1) == (1, 1)
    for M in range(1, 300):
        k, p = oracle.choose_kp(M)
        assert k * p >= M and k * (p - 1) < M


# ---------------------------------------------------------------- P3: c_n
def test_dct_closed_forms():
    Nq = 64
    x = np.cos(np.pi * (np.arange(Nq) + 0.5) / Nq)
    c = oracle.cheb_coeffs_of_samples(x * x, 6)               # x^2 = 1/2 T_0 + 1/2 T_2
    assert np.allclose(c, [0.5, 0, 0.5, 0, 0, 0], atol=1e-15)
    c = oracle.cheb_coeffs_of_samples(npcheb.chebval(x, [0, 0, 0, 0, 0, 1.0]), 8)  # T_5 -> e_5
    assert np.allclose(c, np.eye(8)[5], atol=1e-15)
    c = oracle.cheb_coeffs_of_samples(np.ones(Nq), 4)         # c_0 is NOT halved
    assert np.allclose(c, [1, 0, 0, 0], atol=1e-15)


def test_fermi_coeffs_match_numpy_chebinterpolate():
    # library cross-check: numpy interpolates at the same first-kind nodes
    beta, mu, a, b, M = 3.0, 0.2, -2.0, 2.5, 40
    Nq = oracle.nq_for(M)
    assert Nq == 256
    bt, mt = beta * (b - a) / 2, (2 * mu - (a + b)) / (b - a)
    ref = npcheb.chebinterpolate(lambda x: 1.0 / (1.0 + np.exp(bt * (x - mt))), Nq - 1)[:M]
    c = oracle.cheb_coeffs(beta, mu, a, b, M)
    assert np.allclose(c, ref, atol=2e-15)


def test_fermi_coeffs_limits_and_symmetry():
    c = oracle.cheb_coeffs(1e-9, 0.0, -1.0, 1.0, 16)     # beta~ -> 0: f -> 1/2
    assert abs(c[0] - 0.5) < 1e-9 and np.all(np.abs(c[1:]) < 1e-9)
    c = oracle.cheb_coeffs(25.0, 0.0, -1.0, 1.0, 64)     # mu~ = 0: f(x) - 1/2 odd
    assert abs(c[0] - 0.5) < 1e-15
    assert np.all(np.abs(c[2::2]) < 1e-15)
    assert np.all(c[1::4] < 0) and np.all(c[3::4][: 8] > 0)  # alternating odd coefficients
    # mu mapped correctly: mu at the centre of [a,b] gives mu~ = 0 as well
    c2 = oracle.cheb_coeffs(25.0 / 3.0, 4.0, 1.0, 7.0, 64)   # beta~ = 25, mu~ = 0
    assert np.allclose(c2, c, atol=1e-15)


def test_fermi_coeffs_decay_rate():
    # |c_n| ~ exp(-pi n / beta~); fit the slope over the odd coefficients
    bt = 30.0
    c = oracle.cheb_coeffs(bt, 0.0, -1.0, 1.0, 200)
    n = np.arange(41, 160, 2)
    slope = np.polyfit(n, np.log(np.abs(c[n])), 1)[0]
    assert abs(slope - (-math.pi / bt)) < 0.05 * math.pi / bt


def test_fermi_function():
    assert oracle.fermi(7.0, 0.3, 0.3) == 0.5
    assert oracle.fermi(1e4, 0.0, 1.0) == 0.0 and oracle.fermi(1e4, 0.0, -1.0) == 1.0
    for e in [-3.0, -0.2, 0.9]:
        assert abs(oracle.fermi(2.0, 0.1, e) + oracle.fermi(2.0, 0.1, 0.2 - e) - 1.0) < 1e-15
        assert abs(oracle.fermi(2.0, 0.1, e) - 1.0 / (1.0 + math.exp(2.0 * (e - 0.1)))) < 1e-15


# ---------------------------------------------------------------- Algorithm 1
def test_algorithm1_prints_eq22_23(golden):
    rows = golden("eq22_23_babysteps.txt").astype(int)
    st = oracle.algorithm1_schedule(4)
    flat = [p for s in st for p in s]
    assert [tuple(r) for r in rows] == flat


@pytest.mark.parametrize("k", [1, 2, 3, 4, 5, 8, 16, 31, 32, 45, 46, 64])
def test_algorithm1_schedule_properties(k):
    st = oracle.algorithm1_schedule(k)
    assert len(st) == (math.ceil(math.log2(k)) if k > 1 else 0)
    known = {0, 1}
    produced = []
    for s, prods in enumerate(st, start=1):
        assert len(prods) <= 2 ** (s - 1)
        new = set()
        for (n, l, r, m) in prods:
            assert l + r == n and abs(l - r) == m            # Eq. 7 with T_{a+b} = 2 T_a T_b - T_|a-b|
            assert {l, r, m} <= known                        # only data from earlier stages
            new.add(n)
            produced.append(n)
        known |= new
    assert sorted(produced) == list(range(2, k + 1))          # k-1 products, each once
