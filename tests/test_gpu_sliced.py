"""`-m gpu` parity of cheb_dm_product_sliced: Out = alpha A B + beta C with the FP64 operands sliced
into int8 digits and the digit products on tcgen05.mma kind::i8 (int32 accumulators in tensor memory).

Oracle: oracle.matmul (plain triple loop, FP64).  Tolerance: the rounding bound of an FP64 dot product of N terms
with |entries| <= 1, 4 N 2^-52 (the same gate as the DMMA product test), for S = 8 digits; fewer digits are checked
against the slicing bound K (S+1) 2^{-7S} of include/cheb_dm.h, which must also be REACHED within two orders (the
digits really are truncated: a kernel that silently used more precision, or a wrong bound, fails)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _imports():
    import oracle
    import paper_2306_12616_b200 as cd
    import workloads
    import gpu_util
    return oracle, cd, workloads, gpu_util


def _run(cd, gu, A, B, Cm, alpha, beta, S, same=False, symmetric=False):
    torch = gu.torch_cuda()
    N = A.shape[0]
    plan = cd.Plan(N, 4, sliced=S)
    dA = gu.to_dev(A)
    dB = dA if same else gu.to_dev(B)
    dC = gu.to_dev(Cm) if Cm is not None else None
    dO = torch.full((N, N), float("nan"), dtype=torch.float64, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    plan.product_sliced(alpha, dA.data_ptr(), dB.data_ptr(), beta, dC.data_ptr() if dC is not None else None, dO.data_ptr(), symmetric, st)
    torch.cuda.synchronize()
    plan.destroy()
    return dO.cpu().numpy()


@pytest.mark.parametrize("N", [1, 2, 7, 63, 64, 65, 128, 130, 200, 333, 500, 777])
def test_sliced_product_2AB_minus_C_eight_digits(N):
    oracle, cd, workloads, gu = _imports()
    A = workloads.random_symmetric(N, seed=10 + N)
    B = workloads.random_symmetric(N, seed=20 + N)
    Cm = workloads.random_symmetric(N, seed=30 + N)
    expect = 2.0 * oracle.matmul(A, B) - Cm
    got = _run(cd, gu, A, B, Cm, 2.0, -1.0, 8)
    err = float(np.max(np.abs(got - expect)))
    print(f"N={N}: max|err| = {err:.3e} (gate {4.0 * N * 2.0 ** -52 + 1e-15:.3e})")
    assert err <= 4.0 * N * 2.0 ** -52 + 1e-15


def test_sliced_square_without_C_and_graded_rows():
    """A = B (digits formed once), C = NULL, rows of very different magnitude (row-wise scales 2^{e_i})."""
    oracle, cd, workloads, gu = _imports()
    N = 300
    A = workloads.random_symmetric(N, seed=5)
    g = 2.0 ** np.linspace(-40, 3, N)
    A = (A * g[:, None]) * g[None, :]          # symmetric, |a_ij| <= g_i g_j
    expect = oracle.matmul(A, A)
    got = _run(cd, gu, A, None, None, 1.0, 0.0, 8, same=True)
    rowmax = np.max(np.abs(A), axis=1)
    bound = 4.0 * N * 2.0 ** -52 * rowmax[:, None] * rowmax[None, :]
    assert np.all(np.abs(got - expect) <= bound + 1e-300)


def test_sliced_zero_rows_zero_operand_and_extreme_exponents():
    """Degenerate scales: rows and columns that are entirely zero (scale of an empty row), an all-zero operand, and
    operands near both ends of the FP64 exponent range (2^-480 and 2^+480: the products stay representable)."""
    oracle, cd, workloads, gu = _imports()
    N = 150
    A = workloads.random_symmetric(N, seed=41)
    B = workloads.random_symmetric(N, seed=42)
    for i in (0, 17, 149):     # (both operands stay symmetric: the contract of cheb_dm_product_sliced)
        A[i, :] = 0.0
        A[:, i] = 0.0
        B[(i + 3) % N, :] = 0.0
        B[:, (i + 3) % N] = 0.0
    got = _run(cd, gu, A, B, None, 1.0, 0.0, 8)
    expect = oracle.matmul(A, B)
    assert np.max(np.abs(got - expect)) <= 4.0 * N * 2.0 ** -52
    assert np.all(got[[0, 17, 149], :] == 0.0) and np.all(got[:, [3, 20, 2]] == 0.0)
    Z = np.zeros((N, N))
    assert np.all(_run(cd, gu, Z, B, None, 2.0, 0.0, 8) == 0.0)
    Cm = workloads.random_symmetric(N, seed=43)
    assert np.array_equal(_run(cd, gu, A, Z, Cm, 2.0, -1.0, 8), -Cm)
    for e in (-480, 480):
        As, Bs = A * 2.0 ** e, B * 2.0 ** e
        got = _run(cd, gu, As, Bs, None, 1.0, 0.0, 8)
        assert np.all(np.isfinite(got))
        assert np.max(np.abs(got * 2.0 ** (-2 * e) - expect)) <= 4.0 * N * 2.0 ** -52


@pytest.mark.parametrize("S", [4, 5, 6, 7])
def test_sliced_fewer_digits_meet_and_reach_the_slicing_bound(S):
    oracle, cd, workloads, gu = _imports()
    N = 256
    A = workloads.random_symmetric(N, seed=77)
    B = workloads.random_symmetric(N, seed=78)
    expect = oracle.matmul(A, B)
    got = _run(cd, gu, A, B, None, 1.0, 0.0, S)
    ra, rb = np.max(np.abs(A), axis=1), np.max(np.abs(B), axis=1)
    sa, sb = 2.0 ** np.ceil(np.log2(ra)), 2.0 ** np.ceil(np.log2(rb))   # the power-of-two row scales
    bound = N * (S + 1) * 2.0 ** (-7 * S) * sa[:, None] * sb[None, :] * 4.0
    err = np.abs(got - expect)
    assert np.all(err <= bound)
    assert np.max(err / bound) >= 1e-3      # truncated digits leave an error of the predicted order, not FP64 rounding


@pytest.mark.parametrize("N", [64, 129, 200, 333, 700])
def test_sliced_symmetric_tiles_on_commuting_operands(N):
    """Operands that commute (polynomials of one X, like every product of the method: T_5(X) T_3(X), minus T_2(X)):
    lower-triangle tiles only, mirrored on store; every element is still written exactly once."""
    oracle, cd, workloads, gu = _imports()
    X = workloads.random_symmetric(N, seed=3 + N) / (0.6 * N ** 0.5 + 1.0)
    T = [np.eye(N), X]
    for n in range(2, 6):
        T.append(2.0 * oracle.matmul(X, T[-1]) - T[-2])
    expect = 2.0 * oracle.matmul(T[5], T[3]) - T[2]          # = T_8(X), symmetric
    got = _run(cd, gu, T[5], T[3], T[2], 2.0, -1.0, 8, symmetric=True)
    ra, rb = np.max(np.abs(T[5]), axis=1), np.max(np.abs(T[3]), axis=1)
    assert np.max(np.abs(got - expect)) <= 4.0 * N * 2.0 ** -52 * max(1.0, ra.max() * rb.max()) + 1e-15
    assert np.max(np.abs(got - got.T)) <= 8.0 * N * 2.0 ** -52 * max(1.0, ra.max() * rb.max())


def test_sliced_needs_the_plan_option():
    oracle, cd, workloads, gu = _imports()
    torch = gu.torch_cuda()
    plan = cd.Plan(64, 4)
    a = torch.zeros((64, 64), dtype=torch.float64, device="cuda")
    o = torch.zeros((64, 64), dtype=torch.float64, device="cuda")
    with pytest.raises(cd.ChebDMError) as ei:
        plan.product_sliced(1.0, a.data_ptr(), a.data_ptr(), 0.0, None, o.data_ptr(), False)
    assert ei.value.status == 6
    plan.destroy()
    with pytest.raises(cd.ChebDMError) as ei:
        cd.Plan(64, 4, sliced=9)
    assert ei.value.status == 1


# ----------------------------------------------------------------------------------------------
# the whole fixed-mu solve on the sliced path (plan option sliced_solve): same gates as the DMMA path
# ----------------------------------------------------------------------------------------------
SOLVE_CASES = [("cfg0", 0, 128, None, {}), ("cfg1", 0, 300, None, {}), ("cfg1", 1, 257, None, {}), ("cfg2", 0, 250, None, {}),
               ("cfg3", 0, 200, 1024, {}), ("cfg4", 0, 200, 2048, {}), ("cfg1", 2, 130, 60, dict(k=6, p=10)),
               ("cfg4", 0, 333, 2048, {}), ("cfg1", 3, 200, 64, dict(symmetric=1)), ("cfg0", 0, 128, None, dict(outer=1)),
               ("cfg1", 0, 150, 96, dict(pairing=1, k=24, p=4)), ("cfg1", 1, 150, 256, dict(pairing=3)), ("cfg3", 0, 150, 1024, dict(k=16, p=64))]


@pytest.mark.parametrize("cfg,seed,n,M,opts", SOLVE_CASES)
def test_sliced_solve_parity(cfg, seed, n, M, opts):
    """cheb_dm_compute with every product on tcgen05 kind::i8 (8 digits): max|D - D_cheb| <= 1e-10, |dtr| <= 1e-9."""
    import oracle_cases as oc
    oracle, cd, workloads, gu = _imports()
    case = oc.case(cfg, seed, n, M)
    r = gu.gpu_solve(case["H"], case["beta"], case["mu"], case["M"], sliced_solve=1, **opts)
    dD = float(np.max(np.abs(r["D"] - case["D_cheb"])))
    dtr = abs(r["trace"] - float(np.trace(case["D_cheb"])))
    print(f"{cfg} n={case['N']} M={case['M']}: sliced solve max|dD| = {dD:.3e}, |dtr| = {dtr:.3e}")
    assert dD <= 1e-10
    assert dtr <= 1e-9
    assert np.max(np.abs(r["D"] - r["D"].T)) <= 1e-11


@pytest.mark.parametrize("cfg", ["cfg2", "cfg4", "cfg3"])
def test_sliced_solve_full_size(cfg):
    """Full-size parity of the sliced solve: every element for cfg2; sampled columns + probe vectors that touch every
    element for cfg4 / cfg3 (as tests/test_gpu_fullsize.py does for the DMMA path)."""
    import oracle_cases as oc
    oracle, cd, workloads, gu = _imports()
    whole = cfg == "cfg2"
    case = oc.case(cfg, 0, None, None, whole)
    N = case["N"]
    r = gu.gpu_solve(case["H"], case["beta"], case["mu"], case["M"], sliced_solve=1)
    D = r["D"]
    if whole:
        dD = float(np.max(np.abs(D - case["D_cheb"])))
        print(f"{cfg}: sliced solve, full matrix max|dD| = {dD:.3e}")
        assert dD <= 1e-10
    else:
        cols = np.unique(np.concatenate([[0, N - 1], np.random.default_rng(7).integers(0, N, size=1)])).astype(np.int32)
        want = oracle.dm_cheb_columns(case["H"], case["a"], case["b"], case["c"], cols)
        dcol = float(np.max(np.abs(D[:, cols].T - want)))
        rng = np.random.default_rng(11)
        V = np.vstack([rng.standard_normal((2, N)), rng.choice([-1.0, 1.0], size=(2, N))])
        want = oracle.dm_cheb_apply(case["H"], case["a"], case["b"], case["c"], V)
        err = np.max(np.abs(V @ D.T - want), axis=1) / np.max(np.abs(V), axis=1)
        print(f"{cfg}: sliced solve, columns max|dD| = {dcol:.3e}, probes {err}")
        assert dcol <= 1e-10
        assert np.all(err <= 1e-10 * np.sqrt(N))
    dtr = abs(r["trace"] - case["trace_cheb_scalar"])
    print(f"{cfg}: sliced solve |tr D - sum_i p_M(x_i)| = {dtr:.3e}")
    assert dtr <= 1e-9
    assert np.max(np.abs(D - D.T)) <= 1e-11


@pytest.mark.parametrize("cfg,seed,n,M,opts", [("cfg1", 0, 300, None, {}), ("cfg2", 0, 250, None, {}), ("cfg3", 0, 200, 1024, {}),
                                                ("cfg4", 0, 200, 2048, {}), ("cfg1", 2, 130, 60, dict(k=6, p=10)), ("cfg1", 0, 64, 12, dict(k=6, p=2)),
                                                ("cfg1", 1, 70, 8, dict(k=8, p=1)), ("cfg1", 1, 70, 6, dict(k=1, p=6)), ("cfg0", 0, 33, 9, dict(k=3, p=3))])
def test_sliced_mu_inclusive_solve(cfg, seed, n, M, opts):
    """cheb_dm_solve / cheb_dm_moments / cheb_dm_assemble on a sliced_solve plan: baby block and giant block on the int8
    path, moments by the Gram kernel, bisection, nested giant steps; (tau, mu, D) against the oracle as in test_gpu_solve."""
    oracle, cd, workloads, gu = _imports()
    torch = gu.torch_cuda()
    c = workloads.CONFIGS[cfg]
    H = workloads.hamiltonian(cfg, seed=seed, n=n)
    N = H.shape[0]
    M = c.M if M is None else M
    nocc = workloads.n_occ(cfg, N)
    a, b = oracle.gershgorin(H)
    _, tau = oracle.dm_cheb(H, a, b, np.zeros(M), want_tau=True)
    mu_or = oracle.solve_mu(tau, c.beta, a, b, nocc, iters=100)
    D_or = oracle.dm_cheb(H, a, b, oracle.cheb_coeffs(c.beta, mu_or, a, b, M))
    plan = cd.Plan(N, M, sliced_solve=1, **opts)
    st = torch.cuda.current_stream().cuda_stream
    dH = gu.to_dev(H)
    dD = torch.full((N, N), float("nan"), dtype=torch.float64, device="cuda")
    plan.coeffs(c.beta, 123.0, None)
    mu = plan.solve(dH.data_ptr(), nocc, dD.data_ptr(), 100, True, st)
    plan.check(st)
    assert abs(mu - mu_or) <= 1e-10 * max(1.0, b - a)
    D = dD.cpu().numpy()
    err = float(np.max(np.abs(D - D_or)))
    print(f"{cfg} n={N} M={M}: sliced cheb_dm_solve mu={mu:.12f} (oracle {mu_or:.12f}) max|dD|={err:.3e}")
    assert err <= 1e-10
    assert abs(float(np.trace(D)) - nocc) <= 1e-7
    tau_gpu = plan.moments(dH.data_ptr(), True, st)[:M]
    assert np.max(np.abs(tau_gpu - tau)) <= 1e-10 * N
    mu2 = mu_or + 0.05
    plan.assemble([mu2], [dD.data_ptr()], st)
    torch.cuda.synchronize()
    D2 = oracle.dm_cheb(H, a, b, oracle.cheb_coeffs(c.beta, mu2, a, b, M))
    assert np.max(np.abs(dD.cpu().numpy() - D2)) <= 1e-10
    plan.destroy()


def test_sliced_mu_inclusive_solve_full_size_cfg2():
    """cheb_dm_solve on a sliced_solve plan at full size (cfg2, N=1000): (mu, D) against the oracle, every element."""
    import oracle_cases as oc
    oracle, cd, workloads, gu = _imports()
    torch = gu.torch_cuda()
    case = oc.case("cfg2", 0, None, None, True)
    N, M = case["N"], case["M"]
    plan = cd.Plan(N, M, sliced_solve=1)
    st = torch.cuda.current_stream().cuda_stream
    dH = gu.to_dev(case["H"])
    dD = torch.full((N, N), float("nan"), dtype=torch.float64, device="cuda")
    plan.coeffs(case["beta"], 0.0, None)
    mu = plan.solve(dH.data_ptr(), case["nocc"], dD.data_ptr(), 100, True, st)
    plan.check(st)
    assert abs(mu - case["mu"]) <= 1e-10 * (case["b"] - case["a"])
    D = dD.cpu().numpy()
    err = float(np.max(np.abs(D - case["D_cheb"])))
    print(f"cfg2: sliced cheb_dm_solve mu = {mu:.12f} (oracle {case['mu']:.12f}), max|dD| = {err:.3e}")
    assert err <= 1e-10
    assert abs(float(np.trace(D)) - case["nocc"]) <= 1e-6
    plan.destroy()


@pytest.mark.parametrize("n,M,k,p,ldh,ldd", [(130, 12, 12, 1, 130, 137), (65, 8, 1, 8, 66, 65), (200, 9, 3, 3, 208, 203), (129, 2, 2, 1, 129, 129)])
def test_sliced_solve_degenerate_shapes_and_pitches(n, M, k, p, ldh, ldd):
    """p = 1 (no product in the outer sum: D = G_0, written through the mirroring copy of the lower-triangle sums), k = 1 (no
    baby step: the multiplier is X itself), padded and odd pitches of H and D; the padding of D is never written."""
    oracle, cd, workloads, gu = _imports()
    torch = gu.torch_cuda()
    st = torch.cuda.current_stream().cuda_stream
    H = workloads.hamiltonian("cfg1", seed=5, n=n)
    a, b = oracle.gershgorin(H)
    beta, mu = 6.0, 0.05
    D_or = oracle.dm_cheb(H, a, b, oracle.cheb_coeffs(beta, mu, a, b, M))
    Hp = np.full((n, ldh), 4.25)
    Hp[:, :n] = H
    dH = gu.to_dev(Hp)
    dD = torch.full((n, ldd), -7.0, dtype=torch.float64, device="cuda")
    dtr = torch.zeros(1, dtype=torch.float64, device="cuda")
    plan = cd.Plan(n, M, k=k, p=p, ldh=ldh, ldd=ldd, sliced_solve=1)
    assert (plan.k, plan.p) == (k, p)
    plan.coeffs(beta, mu, None)
    plan.compute(dH.data_ptr(), dD.data_ptr(), st)
    plan.trace(dD.data_ptr(), dtr.data_ptr(), st)
    plan.check(st)
    got = dD.cpu().numpy()
    assert np.max(np.abs(got[:, :n] - D_or)) <= 1e-10
    assert np.all(got[:, n:] == -7.0)
    assert abs(float(dtr.item()) - float(np.trace(D_or))) <= 1e-9
    assert np.max(np.abs(got[:, :n] - got[:, :n].T)) <= 1e-11
    plan.destroy()


def test_sliced_product_beyond_the_register_resident_slicing_kernel():
    """N = 6200 > 6144 columns: the slicing pass falls back to the two-pass kernel (rows no longer fit the registers of a
    block).  Sampled elements against exact dot products (math.fsum), the whole matrix against the DMMA product."""
    import math
    oracle, cd, workloads, gu = _imports()
    torch = gu.torch_cuda()
    N = 6200
    st = torch.cuda.current_stream().cuda_stream
    rs = np.random.RandomState(6200)
    A = rs.standard_normal((N, N))
    A = (A + A.T) * 0.5
    A /= np.abs(A).max()
    B = rs.standard_normal((N, N))
    B = (B + B.T) * 0.5
    B /= np.abs(B).max()
    dA, dB = gu.to_dev(A), gu.to_dev(B)
    dO = torch.full((N, N), float("nan"), dtype=torch.float64, device="cuda")
    dR = torch.full((N, N), float("nan"), dtype=torch.float64, device="cuda")
    plan = cd.Plan(N, 4, sliced=8)
    plan.product_sliced(1.0, dA.data_ptr(), dB.data_ptr(), 0.0, None, dO.data_ptr(), False, st)
    plan.product(1.0, dA.data_ptr(), dB.data_ptr(), 0.0, None, dR.data_ptr(), st)
    torch.cuda.synchronize()
    got, ref = dO.cpu().numpy(), dR.cpu().numpy()
    tol = 4.0 * N * 2.0 ** -52
    for i, j in zip(rs.randint(0, N, 300), rs.randint(0, N, 300)):
        exact = math.fsum(A[i, :] * B[:, j])
        assert abs(got[i, j] - exact) <= tol and abs(ref[i, j] - exact) <= tol, (i, j)
    for i in (0, N - 1):       # first and last row and column entirely
        exact = np.array([math.fsum(A[i, :] * B[:, j]) for j in range(0, N, 7)])
        assert np.max(np.abs(got[i, ::7] - exact)) <= tol and np.max(np.abs(got[::7, i] - np.array([math.fsum(A[r, :] * B[:, i]) for r in range(0, N, 7)]))) <= tol
    assert np.max(np.abs(got - ref)) <= 2.0 * tol
    plan.destroy()
