"""`-m gpu` parity tests: the CUDA path, called through the C ABI (include/cheb_dm.h via the ctypes
binding), against the CPU oracle on the same seeded inputs.

Gates (BASELINE.json north_star):
    max|D_gpu - D_cheb| <= 1e-10,  |tr D_gpu - tr D_cheb| <= 1e-9,
    max|D_gpu - D_eig|  <= eps_trunc(config) + 1e-9  (eps_trunc from oracle scalars).
Every expected value comes from oracle/ (tests/oracle_cases.py); nothing flows from the GPU into it.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL_D = 1e-10
TOL_TR = 1e-9


def _imports():
    import oracle
    import paper_2306_12616_b200 as cd
    import workloads
    import gpu_util
    import oracle_cases
    return oracle, cd, workloads, gpu_util, oracle_cases


# ----------------------------------------------------------------------------------------------
# a-4/a-6 kernel: one product with the fused 2AB - C epilogue (Eq. 7), all tile shapes, ragged sizes
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("tile", [1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11, 12])
@pytest.mark.parametrize("N", [1, 2, 7, 64, 65, 130, 200, 333])
def test_product_2AB_minus_C(N, tile):
    oracle, cd, workloads, gu, _ = _imports()
    torch = gu.torch_cuda()
    A = workloads.random_symmetric(N, seed=10 + N)
    B = workloads.random_symmetric(N, seed=20 + N)
    Cm = workloads.random_symmetric(N, seed=30 + N)
    expect = 2.0 * oracle.matmul(A, B) - Cm
    plan = cd.Plan(N, 4, tile=tile)
    dA, dB, dC = gu.to_dev(A), gu.to_dev(B), gu.to_dev(Cm)
    dO = torch.full((N, N), float("nan"), dtype=torch.float64, device="cuda")
    plan.product(2.0, dA.data_ptr(), dB.data_ptr(), -1.0, dC.data_ptr(), dO.data_ptr(),
                 torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    got = dO.cpu().numpy()
    # |entries| <= 1, N-term dot products: rounding <= ~N * 2^-52 each side
    assert np.max(np.abs(got - expect)) <= 4.0 * N * 2.0 ** -52 + 1e-15
    plan.destroy()


# ----------------------------------------------------------------------------------------------
# a-1: Gershgorin bounds + rescale
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,n", [("cfg0", 128), ("cfg1", 301), ("cfg2", 200), ("cfg3", 500), ("cfg4", 130)])
def test_gershgorin_bounds_and_rescale(cfg, n):
    oracle, cd, workloads, gu, _ = _imports()
    torch = gu.torch_cuda()
    H = workloads.hamiltonian(cfg, seed=0, n=n)
    a, b = oracle.gershgorin(H)
    r = gu.gpu_solve(H, 5.0, 0.0, 8, keep_plan=True)
    ga, gb = r["bounds"]
    scale = max(abs(a), abs(b))
    assert abs(ga - a) <= n * 2.0 ** -52 * scale and abs(gb - b) <= n * 2.0 ** -52 * scale
    # T_1 = X = (2H - (a+b)I)/(b-a)  (reading A1), with the GPU's own bounds
    dX = torch.empty((n, n), dtype=torch.float64, device="cuda")
    r["plan"].get_T(1, dX.data_ptr(), torch.cuda.current_stream().cuda_stream)
    X = oracle.scale(H, a, b)
    assert np.max(np.abs(dX.cpu().numpy() - X)) <= 1e-14
    r["plan"].destroy()


@pytest.mark.parametrize("n,ldh", [(4999, 4999), (4999, 5000), (4802, 4802)])
def test_gershgorin_bounds_and_rescale_rows_shared_by_warps(n, ldh):
    """a-1 at N ~ 5000, where 16 warps of a block share a row of H in the bounds and rescale passes: odd N (the last
    column apart), odd pitch (scalar loads) and even pitch (16-byte loads).  M = 4: the products are not the point."""
    oracle, cd, workloads, gu, _ = _imports()
    torch = gu.torch_cuda()
    st = torch.cuda.current_stream().cuda_stream
    H = workloads.hamiltonian("cfg3", seed=1, n=n)
    a, b = oracle.gershgorin(H)
    Hp = np.full((n, ldh), 3.25)
    Hp[:, :n] = H
    dH = gu.to_dev(Hp)
    dD = torch.empty((n, n), dtype=torch.float64, device="cuda")
    plan = cd.Plan(n, 4, ldh=ldh)
    plan.coeffs(5.0, 0.0, None)
    plan.compute(dH.data_ptr(), dD.data_ptr(), st)
    plan.check(st)
    ga, gb = plan.get_bounds(st)
    scale = max(abs(a), abs(b))
    assert abs(ga - a) <= n * 2.0 ** -52 * scale and abs(gb - b) <= n * 2.0 ** -52 * scale
    dX = torch.empty((n, n), dtype=torch.float64, device="cuda")
    plan.get_T(1, dX.data_ptr(), st)
    torch.cuda.synchronize()
    assert np.max(np.abs(dX.cpu().numpy() - oracle.scale(H, a, b))) <= 1e-14
    plan.destroy()


def test_gershgorin_degenerate_identity_widens():
    _, cd, _, gu, _ = _imports()
    H = 3.0 * np.eye(40)
    r = gu.gpu_solve(H, 2.0, 3.0, 6)
    assert r["bounds"] == (2.0, 4.0)
    # X = 0 => D = p_M(0) I ~ f(mu) I = 0.5 I up to truncation
    assert np.max(np.abs(r["D"] - np.diag(np.diag(r["D"])))) == 0.0


# ----------------------------------------------------------------------------------------------
# a-2 / a-3: coefficient tables computed on the device
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("M,k,p", [(64, 0, 0), (256, 0, 0), (2048, 0, 0), (1024, 0, 0), (30, 5, 7), (7, 7, 1), (5, 1, 5)])
def test_coefficient_tables(M, k, p):
    oracle, cd, workloads, gu, _ = _imports()
    H = workloads.hamiltonian("cfg1", seed=1, n=48)
    beta, mu, bounds = 40.0, 0.07, (-20.0, 21.0)
    outer = cd.OUTER_POWER if M <= 64 else cd.OUTER_CHEBYSHEV
    r = gu.gpu_solve(H, beta, mu, M, bounds=bounds, keep_plan=True, k=k, p=p, outer=outer)
    plan = r["plan"]
    c, g, d = plan.get_coeffs()
    kk, pp = plan.k, plan.p
    c_or = oracle.pad_coeffs(oracle.cheb_coeffs(beta, mu, bounds[0], bounds[1], M), kk, pp)
    assert np.max(np.abs(c - c_or)) <= 2e-15
    g_or = oracle.g_from_c(kk, pp, c_or)
    assert np.max(np.abs(g - g_or)) <= 1e-14
    if outer == cd.OUTER_POWER:
        d_or = oracle.d_from_g(kk, pp, g_or)
        assert np.max(np.abs(d - d_or)) <= 1e-13 * max(1.0, np.max(np.abs(d_or)))
    plan.destroy()


# ----------------------------------------------------------------------------------------------
# a-4: baby steps T_2..T_k (Eq. 7, 22-23, Algorithm 1) vs the three-term recurrence of the oracle
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("pairing", [0, 1, 2, 3])
@pytest.mark.parametrize("k", [2, 3, 5, 8, 11])
def test_baby_steps_match_three_term_recurrence(k, pairing):
    oracle, cd, workloads, gu, _ = _imports()
    torch = gu.torch_cuda()
    n = 150
    H = workloads.hamiltonian("cfg1", seed=2, n=n)
    a, b = oracle.gershgorin(H)
    r = gu.gpu_solve(H, 10.0, 0.0, k * 3, bounds=(a, b), keep_plan=True, k=k, p=3, pairing=pairing)
    X = oracle.scale(H, a, b)
    Tm, Tc = np.eye(n), X
    dT = torch.empty((n, n), dtype=torch.float64, device="cuda")
    for j in range(2, k + 1):
        Tn = 2.0 * oracle.matmul(X, Tc) - Tm
        Tm, Tc = Tc, Tn
        r["plan"].get_T(j, dT.data_ptr(), torch.cuda.current_stream().cuda_stream)
        assert np.max(np.abs(dT.cpu().numpy() - Tc)) <= 1e-13, j
    r["plan"].destroy()


# ----------------------------------------------------------------------------------------------
# whole path at reduced sizes (several tiles + ragged tail), every config kind
# ----------------------------------------------------------------------------------------------
SMALL = [("cfg0", 0, 128, None), ("cfg1", 0, 300, None), ("cfg1", 3, 257, None), ("cfg2", 0, 250, None),
         ("cfg3", 0, 200, 1024), ("cfg4", 0, 200, 2048)]


def _check(case, r):
    dD = np.max(np.abs(r["D"] - case["D_cheb"]))
    dtr = abs(r["trace"] - float(np.trace(case["D_cheb"])))
    assert dD <= TOL_D, dD
    assert dtr <= TOL_TR, dtr
    assert abs(float(np.trace(case["D_cheb"])) - case["nocc"]) <= 1e-7  # mu solved on the trace
    if "D_eig" in case:
        assert np.max(np.abs(r["D"] - case["D_eig"])) <= case["eps_trunc"] + 1e-9
    assert np.max(np.abs(r["D"] - r["D"].T)) <= 1e-11
    return dD, dtr


@pytest.mark.parametrize("cfg,seed,n,M", SMALL)
def test_parity_reduced_size_device_gershgorin(cfg, seed, n, M):
    """The hot path as bench.py runs it: bounds=None (Gershgorin on the device)."""
    oracle, cd, workloads, gu, oc = _imports()
    case = oc.case(cfg, seed, n, M)
    r = gu.gpu_solve(case["H"], case["beta"], case["mu"], case["M"])
    assert abs(r["bounds"][0] - case["a"]) <= n * 2.0 ** -52 * abs(case["a"])
    assert abs(r["bounds"][1] - case["b"]) <= n * 2.0 ** -52 * abs(case["b"])
    _check(case, r)


@pytest.mark.parametrize("tile", [1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11, 12])
@pytest.mark.parametrize("sched", [0, 1])
def test_parity_tiles_and_schedulers(tile, sched):
    oracle, cd, workloads, gu, oc = _imports()
    case = oc.case("cfg1", 0, 300, None)
    r = gu.gpu_solve(case["H"], case["beta"], case["mu"], case["M"], bounds=(case["a"], case["b"]), tile=tile, sched=sched)
    _check(case, r)


@pytest.mark.parametrize("giant", [1, 2])
@pytest.mark.parametrize("fuse", [1, 2])
@pytest.mark.parametrize("symmetric", [1, 2])
@pytest.mark.parametrize("cfg,n,outer", [("cfg1", 300, 0), ("cfg1", 257, 0), ("cfg2", 95, 0), ("cfg0", 128, 1), ("cfg1", 33, 0)])
def test_parity_giant_generic_and_resident(giant, fuse, cfg, n, outer, symmetric):
    """a-6: the giant steps in the generic grouped kernel and in the resident-multiplier kernel (N <= 512: T_k rows
    kept in shared memory, two column panels per CTA as independent chains), odd / ragged sizes, odd panel counts."""
    oracle, cd, workloads, gu, oc = _imports()
    case = oc.case(cfg, 0, n, None)
    r = gu.gpu_solve(case["H"], case["beta"], case["mu"], case["M"], giant=giant, fuse_sums=fuse, outer=outer, symmetric=symmetric,
                     keep_plan=True)
    assert r["plan"].opts.giant == giant and r["plan"].opts.symmetric == symmetric
    r["plan"].destroy()
    _check(case, r)


@pytest.mark.parametrize("fuse", [1, 2])
@pytest.mark.parametrize("outer", [0, 1])
def test_parity_fused_and_preformed_sums(fuse, outer):
    """a-5: epilogue-fused vs batched pre-formed low-order sums (Eq. 21) give the same D."""
    oracle, cd, workloads, gu, oc = _imports()
    case = oc.case("cfg0", 0, 128, None) if outer == 1 else oc.case("cfg2", 0, 250, None)
    r = gu.gpu_solve(case["H"], case["beta"], case["mu"], case["M"], bounds=(case["a"], case["b"]), fuse_sums=fuse, outer=outer)
    _check(case, r)
    r = gu.gpu_solve(case["H"], case["beta"], case["mu"], case["M"], fuse_sums=fuse, outer=outer, k=5, p=(case["M"] + 4) // 5, tile=2)
    _check(case, r)


@pytest.mark.parametrize("tile,n", [(4, 700), (5, 700), (6, 1500), (7, 700), (3, 700), (1, 1500), (8, 1500), (11, 700), (12, 700), (11, 257), (12, 129)])
def test_grouped_equals_serial_bitwise_many_tiles_per_task(tile, n):
    """a-8: with more tiles per product than resident CTAs every CTA streams several tiles back to back and the
    producer runs ahead of the consumers; the grouped schedule must reproduce the serial one bit for bit (fixed
    summation order).  Regression test for a shared-memory stage handed back while loads were still in flight."""
    oracle, cd, workloads, gu, oc = _imports()
    H = workloads.hamiltonian("cfg4", seed=0, n=n)
    ref = gu.gpu_solve(H, 200.0, 0.0, 64, tile=tile, sched=1)
    for _ in range(3):
        r = gu.gpu_solve(H, 200.0, 0.0, 64, tile=tile, sched=0, giant=1)
        assert np.array_equal(r["D"], ref["D"])


def test_parity_power_outer_recursion_eq4():
    """Eq. 4 literally (S_j + T_k acc), stable when the expansion is short (reading A6)."""
    oracle, cd, workloads, gu, oc = _imports()
    case = oc.case("cfg0", 0, 128, None)
    r = gu.gpu_solve(case["H"], case["beta"], case["mu"], case["M"], bounds=(case["a"], case["b"]), outer=cd.OUTER_POWER)
    _check(case, r)


def test_parity_serial_pairing_and_nonsquare_kp():
    oracle, cd, workloads, gu, oc = _imports()
    case = oc.case("cfg2", 0, 250, None)
    for kw in (dict(pairing=1), dict(pairing=3), dict(k=32, p=8), dict(k=8, p=32), dict(k=20, p=13), dict(k=256, p=1), dict(k=1, p=256)):
        r = gu.gpu_solve(case["H"], case["beta"], case["mu"], case["M"], bounds=(case["a"], case["b"]), **kw)
        _check(case, r)


# (config, reduced n, M): tight bounds (spectrum widened by 1 %) and M ~ 4.4 beta~ rounded up
# cfg4 (beta~ ~ 1010 even with tight bounds): mu fixed at the centre of its dense level cluster instead of the bisection
CONVERGED = [("cfg0", 128, 208, None), ("cfg1", 300, 512, None), ("cfg2", 250, 480, None), ("cfg3", 200, 720, None),
             ("cfg4", 200, 4608, 0.0)]


@pytest.mark.parametrize("cfg,n,M,mu_fixed", CONVERGED)
def test_converged_variant_meets_1e6_vs_diagonalisation(cfg, n, M, mu_fixed):
    """North-star's "<= 1e-6 vs the diagonalisation DM", one demonstration per config kind: holds with tight bounds
    and enough terms; with Gershgorin bounds the configs' own M are far from converged."""
    oracle, cd, workloads, gu, oc = _imports()
    case = oc.case(cfg, 0, n, M, True, "tight", mu_fixed)
    assert case["eps_trunc"] <= 1e-6, case["eps_trunc"]
    r = gu.gpu_solve(case["H"], case["beta"], case["mu"], case["M"], bounds=(case["a"], case["b"]))
    assert np.max(np.abs(r["D"] - case["D_cheb"])) <= TOL_D
    assert abs(r["trace"] - float(np.trace(case["D_cheb"]))) <= TOL_TR
    if mu_fixed is None:
        assert abs(float(np.trace(case["D_cheb"])) - case["nocc"]) <= 1e-7  # mu solved on the trace
    assert np.max(np.abs(r["D"] - case["D_eig"])) <= 1e-6


# ----------------------------------------------------------------------------------------------
# edge cases
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N,M", [(1, 1), (1, 9), (2, 2), (3, 1), (5, 3), (17, 2), (63, 10), (129, 25)])
def test_edge_sizes(N, M):
    oracle, cd, workloads, gu, _ = _imports()
    H = workloads.random_symmetric(N, seed=N * 100 + M, scale=2.0)
    a, b = oracle.gershgorin(H)
    if a == b:
        a, b = a - 1.0, b + 1.0
    beta, mu = 3.0, 0.1
    c = oracle.cheb_coeffs(beta, mu, a, b, M)
    D = oracle.dm_cheb(H, a, b, c)
    r = gu.gpu_solve(H, beta, mu, M)
    assert np.max(np.abs(r["D"] - D)) <= TOL_D
    assert abs(r["trace"] - np.trace(D)) <= TOL_TR


def test_diagonal_H_gives_scalar_polynomial_on_diagonal():
    oracle, cd, workloads, gu, _ = _imports()
    eps = np.linspace(-1.7, 2.3, 70)
    H = np.diag(eps)
    beta, mu, M = 6.0, 0.2, 48
    r = gu.gpu_solve(H, beta, mu, M)
    a, b = r["bounds"]
    assert (a, b) == (eps[0], eps[-1])  # Gershgorin is exact for diagonal H (pin P9)
    c = oracle.cheb_coeffs(beta, mu, a, b, M)
    want = np.array([oracle.eval_cheb_sum(c, float((2 * e - (a + b)) / (b - a))) for e in eps])
    assert np.max(np.abs(np.diag(r["D"]) - want)) <= 1e-13
    assert np.max(np.abs(r["D"] - np.diag(np.diag(r["D"])))) <= 1e-15


def test_bitwise_reproducible():
    oracle, cd, workloads, gu, oc = _imports()
    H = workloads.hamiltonian("cfg1", seed=1, n=300)
    r1 = gu.gpu_solve(H, 40.0, 0.01, 256)
    r2 = gu.gpu_solve(H, 40.0, 0.01, 256)
    assert np.array_equal(r1["D"], r2["D"]) and r1["trace"] == r2["trace"]


def test_plan_reuse_with_new_mu_and_new_H():
    oracle, cd, workloads, gu, oc = _imports()
    torch = gu.torch_cuda()
    n, M = 180, 100
    plan = cd.Plan(n, M)
    st = torch.cuda.current_stream().cuda_stream
    dD = torch.empty((n, n), dtype=torch.float64, device="cuda")
    for seed, mu in ((0, -0.2), (1, 0.3), (0, 0.05)):
        H = workloads.hamiltonian("cfg1", seed=seed, n=n)
        a, b = oracle.gershgorin(H)
        dH = gu.to_dev(H)
        plan.coeffs(25.0, mu, (a, b))
        plan.compute(dH.data_ptr(), dD.data_ptr(), st)
        torch.cuda.synchronize()
        D = oracle.dm_cheb(H, a, b, oracle.cheb_coeffs(25.0, mu, a, b, M))
        assert np.max(np.abs(dD.cpu().numpy() - D)) <= TOL_D
    plan.destroy()


def test_status_codes():
    oracle, cd, workloads, gu, _ = _imports()
    torch = gu.torch_cuda()
    import ctypes as C
    L = cd.lib()
    h = C.c_void_p()
    assert L.cheb_dm_plan(C.byref(h), 0, 4, 0) == 1          # EINVAL
    assert L.cheb_dm_plan(C.byref(h), 8, 0, 0) == 1
    assert L.cheb_dm_plan(C.byref(h), 8, 4, 7) == 6          # EUNSUPPORTED
    o = cd.Options(k=2, p=1)
    assert L.cheb_dm_plan_ex(C.byref(h), 8, 4, 0, C.byref(o)) == 1  # k*p < M
    assert L.cheb_dm_plan(C.byref(h), 8, 4, 0) == 0
    d = torch.zeros((8, 8), dtype=torch.float64, device="cuda")
    e = torch.zeros((8, 8), dtype=torch.float64, device="cuda")
    assert L.cheb_dm_compute(h, d.data_ptr(), e.data_ptr(), None) == 4   # ESTATE: no coeffs yet
    bad = (C.c_double * 2)(1.0, 1.0)
    assert L.cheb_dm_coeffs(h, 1.0, 0.0, bad) == 5           # EBOUNDS
    assert L.cheb_dm_coeffs(h, -1.0, 0.0, None) == 1
    assert L.cheb_dm_coeffs(h, float("nan"), 0.0, None) == 1
    assert L.cheb_dm_coeffs(h, 1.0, 0.0, None) == 0
    assert L.cheb_dm_compute(h, d.data_ptr(), d.data_ptr(), None) == 1   # aliasing
    assert L.cheb_dm_compute(h, None, e.data_ptr(), None) == 1
    mu = C.c_double()
    assert L.cheb_dm_solve_mu(h, 1.0, 4.0, 50, C.byref(mu), None) == 4   # ESTATE: no moments
    assert L.cheb_dm_destroy(h) == 0
    # non-finite H under Gershgorin -> EBOUNDS on read-back
    plan = cd.Plan(8, 4)
    Hn = np.eye(8)
    Hn[2, 3] = Hn[3, 2] = np.inf
    dH = gu.to_dev(Hn)
    plan.coeffs(1.0, 0.0, None)
    plan.compute(dH.data_ptr(), e.data_ptr(), torch.cuda.current_stream().cuda_stream)
    with pytest.raises(cd.ChebDMError) as ei:
        plan.get_bounds()
    assert ei.value.status == 5
    plan.destroy()


def test_sticky_device_flags_survive_later_computes():
    """a device-side error of ANY solve of a pipeline is reported by the one check at its end (the flags are
    sticky and cleared by the check), not erased by the next compute's front end."""
    oracle, cd, workloads, gu, _ = _imports()
    torch = gu.torch_cuda()
    st = torch.cuda.current_stream().cuda_stream
    n = 40
    good = gu.to_dev(workloads.hamiltonian("cfg1", seed=0, n=n))
    Hb = workloads.hamiltonian("cfg1", seed=1, n=n)
    Hb[3, 4] = Hb[4, 3] = np.inf
    bad = gu.to_dev(Hb)
    dD = torch.empty((n, n), dtype=torch.float64, device="cuda")
    plan = cd.Plan(n, 16)
    plan.coeffs(5.0, 0.0, None)
    plan.compute(bad.data_ptr(), dD.data_ptr(), st)
    plan.compute(good.data_ptr(), dD.data_ptr(), st)
    plan.compute(good.data_ptr(), dD.data_ptr(), st)
    with pytest.raises(cd.ChebDMError) as ei:
        plan.check(st)
    assert ei.value.status == 5       # EBOUNDS from the first of the three computes
    plan.check(st)                    # reported once, then cleared
    plan.compute(good.data_ptr(), dD.data_ptr(), st)
    plan.check(st)
    plan.destroy()


def test_enoconv_guard_of_the_power_basis_recursion():
    """Eq. 4 literally (OUTER_POWER): d_{i,p-1} = 2^p c (Eq. 12, a_{j,j} = 2^{1-j}).  Reading A6: when
    max|d| 2^-52 p > 1e-12 the device sets a flag and cheb_dm_check returns ENOCONV (cfg4 kind, M = 2048: max|d| ~ 1e13
    and the result is wrong at the 1e-4 level); short expansions (cfg0) pass."""
    oracle, cd, workloads, gu, oc = _imports()
    torch = gu.torch_cuda()
    st = torch.cuda.current_stream().cuda_stream
    H = workloads.hamiltonian("cfg4", seed=0, n=200)
    dH = gu.to_dev(H)
    dD = torch.empty((200, 200), dtype=torch.float64, device="cuda")
    plan = cd.Plan(200, 2048, outer=cd.OUTER_POWER)
    plan.coeffs(200.0, 0.0, None)
    plan.compute(dH.data_ptr(), dD.data_ptr(), st)
    with pytest.raises(cd.ChebDMError) as ei:
        plan.check(st)
    assert ei.value.status == 7
    _, _, d = plan.get_coeffs(st)
    a, b = oracle.gershgorin(H)
    d_or = oracle.d_from_g(plan.k, plan.p, oracle.g_from_c(plan.k, plan.p, oracle.pad_coeffs(oracle.cheb_coeffs(200.0, 0.0, a, b, 2048), plan.k, plan.p)))
    assert np.max(np.abs(d_or)) * 2.0 ** -52 * plan.p > 1e-12          # the oracle's table trips the same rule
    plan.destroy()
    case = oc.case("cfg0", 0, 128, None)
    r = gu.gpu_solve(case["H"], case["beta"], case["mu"], case["M"], outer=cd.OUTER_POWER)   # gpu_solve calls check
    _check(case, r)
    # the Chebyshev-basis recursion (default) never computes d and never trips
    r = gu.gpu_solve(H, 200.0, 0.0, 2048)
    assert np.all(np.isfinite(r["D"]))


@pytest.mark.parametrize("n,ldh,ldd", [(130, 136, 133), (257, 258, 300), (64, 64, 70), (33, 40, 33)])
def test_leading_dimension_options(n, ldh, ldd):
    """Options ldh / ldd: H and D inside larger device arrays, even and odd pitches."""
    oracle, cd, workloads, gu, oc = _imports()
    torch = gu.torch_cuda()
    st = torch.cuda.current_stream().cuda_stream
    H = workloads.hamiltonian("cfg1", seed=4, n=n)
    a, b = oracle.gershgorin(H)
    M, beta, mu = 48, 30.0, 0.04
    D_or = oracle.dm_cheb(H, a, b, oracle.cheb_coeffs(beta, mu, a, b, M))
    Hp = np.full((n, ldh), 7.77)          # the padding must never be read as data
    Hp[:, :n] = H
    dH = gu.to_dev(Hp)
    dD = torch.full((n, ldd), -5.0, dtype=torch.float64, device="cuda")
    dtr = torch.zeros(1, dtype=torch.float64, device="cuda")
    for giant in (1, 2):
        plan = cd.Plan(n, M, ldh=ldh, ldd=ldd, giant=giant)
        plan.coeffs(beta, mu, None)
        plan.compute(dH.data_ptr(), dD.data_ptr(), st)
        plan.trace(dD.data_ptr(), dtr.data_ptr(), st)
        plan.check(st)
        got = dD.cpu().numpy()
        assert np.max(np.abs(got[:, :n] - D_or)) <= TOL_D
        assert np.all(got[:, n:] == -5.0)                      # the padding of D is never written
        assert abs(float(dtr.item()) - float(np.trace(D_or))) <= TOL_TR
        assert plan.get_bounds(st) == pytest.approx((a, b), rel=1e-14)
        plan.destroy()
    with pytest.raises(cd.ChebDMError):
        cd.Plan(n, M, ldh=n - 1)


def test_cuda_graph_capture_and_replay():
    """cheb_dm_compute + cheb_dm_trace allocate nothing, read no environment and never
    synchronise, so the whole solve (cooperative launches included) is capturable; replays on new H contents are
    bit-identical to eager calls.  Both the resident-kernel path and the generic one, and a batch."""
    oracle, cd, workloads, gu, oc = _imports()
    torch = gu.torch_cuda()
    n, M, beta = 300, 100, 40.0
    Hs = [workloads.hamiltonian("cfg1", seed=s, n=n) for s in range(3)]
    for opts in (dict(), dict(giant=1), dict(max_batch=2)):
        nb = opts.get("max_batch", 1)
        plan = cd.Plan(n, M, **opts)
        plan.coeffs(beta, 0.03, None)
        dH = [torch.empty((n, n), dtype=torch.float64, device="cuda") for _ in range(nb)]
        dD = [torch.empty((n, n), dtype=torch.float64, device="cuda") for _ in range(nb)]
        dtr = torch.zeros(nb, dtype=torch.float64, device="cuda")
        eager = []
        st = torch.cuda.current_stream().cuda_stream
        for H in Hs:
            for x in dH:
                x.copy_(torch.from_numpy(H))
            plan.compute_batch([x.data_ptr() for x in dH], [x.data_ptr() for x in dD], None, st)
            plan.trace_batch([x.data_ptr() for x in dD], dtr.data_ptr(), st)
            torch.cuda.synchronize()
            eager.append((dD[0].cpu().numpy().copy(), float(dtr[0].item())))
        side = torch.cuda.Stream()
        g = torch.cuda.CUDAGraph()
        torch.cuda.synchronize()
        with torch.cuda.graph(g, stream=side):
            cs = torch.cuda.current_stream().cuda_stream
            plan.compute_batch([x.data_ptr() for x in dH], [x.data_ptr() for x in dD], None, cs)
            plan.trace_batch([x.data_ptr() for x in dD], dtr.data_ptr(), cs)
        for rep in range(2):
            for H, (D_e, tr_e) in zip(Hs, eager):
                for x in dH:
                    x.copy_(torch.from_numpy(H))
                for x in dD:
                    x.fill_(float("nan"))
                g.replay()
                torch.cuda.synchronize()
                for x in dD:
                    assert np.array_equal(x.cpu().numpy(), D_e)
                assert float(dtr[nb - 1].item()) == tr_e
        plan.check(st)
        del g
        plan.destroy()


def test_resident_kernel_guard_on_large_k():
    """the resident giant-step kernel stages k * 16 coefficients inside its idle TMA rings (80 KB): plans with
    k > 640 must fall back to the generic kernel instead of overrunning into the mbarriers."""
    oracle, cd, workloads, gu, oc = _imports()
    n, M = 64, 1400
    H = workloads.hamiltonian("cfg1", seed=0, n=n)
    a, b = oracle.gershgorin(H)
    D_or = oracle.dm_cheb(H, a, b, oracle.cheb_coeffs(15.0, 0.02, a, b, M))
    for k, want in ((700, 1), (640, 2)):
        r = gu.gpu_solve(H, 15.0, 0.02, M, k=k, p=(M + k - 1) // k, keep_plan=True)
        assert r["plan"].opts.giant == want
        r["plan"].destroy()
        assert np.max(np.abs(r["D"] - D_or)) <= TOL_D


# ----------------------------------------------------------------------------------------------
# a-7: trace, moments, mu
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,n,M,kp,tile", [("cfg0", 128, 64, (0, 0), 0), ("cfg1", 200, 256, (0, 0), 0), ("cfg2", 150, 60, (6, 10), 0),
                                              ("cfg4", 130, 90, (9, 10), 0), ("cfg1", 64, 12, (12, 1), 0), ("cfg1", 64, 12, (3, 4), 0),
                                              ("cfg1", 700, 64, (0, 0), 1), ("cfg1", 500, 256, (0, 0), 0), ("cfg2", 1000, 256, (0, 0), 0)])
def test_moments_and_mu(cfg, n, M, kp, tile):
    oracle, cd, workloads, gu, oc = _imports()
    torch = gu.torch_cuda()
    H = workloads.hamiltonian(cfg, seed=0, n=n)
    beta = workloads.CONFIGS[cfg].beta
    nocc = workloads.n_occ(cfg, n)
    a, b = oracle.gershgorin(H)
    _, tau_or = oracle.dm_cheb(H, a, b, np.zeros(M), want_tau=True)
    plan = cd.Plan(n, M, k=kp[0], p=kp[1], tile=tile)
    dH = gu.to_dev(H)
    st = torch.cuda.current_stream().cuda_stream
    plan.coeffs(beta, 0.0, (a, b))
    tau = plan.moments(dH.data_ptr(), True, st)[:M]
    assert np.max(np.abs(tau - tau_or)) <= 1e-10 * n
    mu_gpu = plan.solve_mu(beta, nocc, 100, st)
    mu_or = oracle.solve_mu(tau_or, beta, a, b, nocc, iters=100)
    # the electron count at the GPU's mu must hit the target as well as the oracle's own root does
    ne_gpu = oracle.electron_count(tau_or, beta, mu_gpu, a, b)
    ne_or = oracle.electron_count(tau_or, beta, mu_or, a, b)
    assert abs(ne_gpu - nocc) <= max(1e-8, 10 * abs(ne_or - nocc))
    plan.destroy()


def test_trace_kernel():
    oracle, cd, workloads, gu, _ = _imports()
    torch = gu.torch_cuda()
    for n in (1, 33, 500, 1025):
        A = workloads.random_symmetric(n, seed=n)
        plan = cd.Plan(n, 4)
        dA = gu.to_dev(A)
        out = torch.zeros(1, dtype=torch.float64, device="cuda")
        plan.trace(dA.data_ptr(), out.data_ptr(), torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        assert abs(out.item() - float(np.sum(np.diag(A).astype(np.longdouble)))) <= 1e-13 * n
        plan.destroy()


def test_trace_records_and_resolved_options():
    """Tracing aid (cheb_dm_set_trace / cheb_dm_get_trace) and cheb_dm_get_options: one record per work item with
    ordered timestamps; tracing does not change the result."""
    oracle, cd, workloads, gu, oc = _imports()
    torch = gu.torch_cuda()
    case = oc.case("cfg1", 0, 300, None)
    for giant in (1, 2):
        r = gu.gpu_solve(case["H"], case["beta"], case["mu"], case["M"], giant=giant, keep_plan=True)
        plan, dH = r["plan"], r["dH"]
        assert plan.opts.giant == giant and plan.opts.k == plan.k and plan.opts.tile == 4 and plan.opts.fuse_sums in (1, 2)
        st = torch.cuda.current_stream().cuda_stream
        dD = torch.empty_like(dH)
        plan.set_trace(True)
        plan.compute(dH.data_ptr(), dD.data_ptr(), st)
        torch.cuda.synchronize()
        recs = plan.get_trace()
        assert np.array_equal(dD.cpu().numpy(), r["D"])
        # 64x32 tiles of a 300x300 product: 5 x 10, of which 30 touch the lower triangle (symmetric-tile skipping);
        # the resident giant-step kernel works on the 55 lower-triangle tiles of the 10 x 10 tiles of 32x32
        nbaby_items = (plan.k - 1) * 30
        ngiant_items = plan.p * (55 if giant == 2 else 30)
        assert len(recs) == nbaby_items + ngiant_items
        for rec in recs:
            assert 0 < rec["t_desc"] <= rec["t_kend"] <= rec["t_done"]
            assert 0 <= rec["sm"] < 200
        plan.set_trace(False)
        plan.destroy()


@pytest.mark.parametrize("tile,n", [(0, 300), (0, 257), (1, 700), (6, 333), (8, 500), (9, 641), (3, 200), (7, 129), (11, 300), (11, 257), (12, 641), (12, 129)])
def test_symmetric_tile_skipping(tile, n):
    """Section 8(f)-3: only the tiles touching the lower triangle are computed, the rest is mirrored.  Same D as the full
    computation up to rounding, symmetric, parity with the oracle unchanged."""
    oracle, cd, workloads, gu, oc = _imports()
    H = workloads.hamiltonian("cfg1", seed=1, n=n)
    a, b = oracle.gershgorin(H)
    M = 40
    c = oracle.cheb_coeffs(40.0, 0.05, a, b, M)
    D_or = oracle.dm_cheb(H, a, b, c)
    on = gu.gpu_solve(H, 40.0, 0.05, M, tile=tile, symmetric=2, giant=1)
    off = gu.gpu_solve(H, 40.0, 0.05, M, tile=tile, symmetric=1, giant=1)
    assert np.max(np.abs(on["D"] - D_or)) <= TOL_D
    assert np.max(np.abs(off["D"] - D_or)) <= TOL_D
    assert np.max(np.abs(on["D"] - off["D"])) <= 1e-13
    assert np.max(np.abs(on["D"] - on["D"].T)) <= 1e-14   # mirrored blocks exactly, diagonal tiles to rounding
    for sym in (2, 1):                                              # default giant kernel for this size (resident if N <= 512)
        res = gu.gpu_solve(H, 40.0, 0.05, M, tile=tile, symmetric=sym)
        assert np.max(np.abs(res["D"] - D_or)) <= TOL_D
        assert np.max(np.abs(res["D"] - res["D"].T)) <= 1e-14


def test_host_entry_points_sync_and_pipelined():
    """cheb_dm_compute_host and the pipelined cheb_dm_compute_host_async / cheb_dm_wait (batch of 5 solves with
    different H and mu through two staging slots) give the same D and tr D as the device-resident call."""
    oracle, cd, workloads, gu, oc = _imports()
    torch = gu.torch_cuda()
    n, M = 300, 64
    Hs = [workloads.hamiltonian("cfg1", seed=s, n=n) for s in range(5)]
    mus = [0.01 * s for s in range(5)]
    st = torch.cuda.current_stream().cuda_stream
    plan = cd.Plan(n, M)
    ref = []
    for H, mu in zip(Hs, mus):
        dH = gu.to_dev(H)
        dD = torch.empty_like(dH)
        plan.coeffs(40.0, mu, None)
        plan.compute(dH.data_ptr(), dD.data_ptr(), st)
        torch.cuda.synchronize()
        ref.append(dD.cpu().numpy())
    hH = [torch.from_numpy(H).pin_memory() for H in Hs]
    hD = [torch.empty((n, n), dtype=torch.float64).pin_memory() for _ in Hs]
    htr = torch.zeros(5, dtype=torch.float64).pin_memory()
    for i in range(5):
        plan.coeffs(40.0, mus[i], None)
        plan.compute_host_async(hH[i].data_ptr(), hD[i].data_ptr(), htr[i:].data_ptr(), st)
    plan.wait(st)
    for i in range(5):
        assert np.array_equal(hD[i].numpy(), ref[i])
        assert abs(float(htr[i]) - float(np.trace(ref[i]))) <= 1e-10
    out = torch.empty((n, n), dtype=torch.float64).pin_memory()
    tr1 = torch.zeros(1, dtype=torch.float64).pin_memory()
    plan.coeffs(40.0, mus[2], None)
    plan.compute_host(hH[2].data_ptr(), out.data_ptr(), tr1.data_ptr(), st)
    assert np.array_equal(out.numpy(), ref[2])
    plan.destroy()


def test_several_plans_alive_at_once_and_launched_on_separate_streams():
    """A later plan must not change what an earlier one needs (kernel attributes are per kernel, not per plan: a plan for a
    smaller N once lowered the resident kernel's shared-memory opt-in), and plans launched on separate streams run
    concurrently without sharing anything but the GPU."""
    oracle, cd, workloads, gu, _ = _imports()
    torch = gu.torch_cuda()
    specs = [(500, 8, {}), (200, 12, {}), (129, 10, dict(max_batch=2)), (300, 9, dict(sliced_solve=1))]
    plans, data = [], []
    for n, M, opts in specs:                      # the N = 500 plan first, smaller ones after it
        plan = cd.Plan(n, M, **opts)
        plan.coeffs(7.0, 0.03, None)
        nb = opts.get("max_batch", 1)
        Hs = [workloads.hamiltonian("cfg1", seed=40 + n + q, n=n) for q in range(nb)]
        plans.append(plan)
        data.append((Hs, [gu.to_dev(h) for h in Hs], [torch.full((n, n), float("nan"), dtype=torch.float64, device="cuda") for _ in Hs]))
    streams = [torch.cuda.Stream() for _ in specs]
    torch.cuda.synchronize()
    for rep in range(2):
        for (n, M, opts), plan, (Hs, dH, dD), s in zip(specs, plans, data, streams):
            if len(Hs) == 1:
                plan.compute(dH[0].data_ptr(), dD[0].data_ptr(), s.cuda_stream)
            else:
                plan.compute_batch([x.data_ptr() for x in dH], [x.data_ptr() for x in dD], [0.03] * len(Hs), s.cuda_stream)
    torch.cuda.synchronize()
    for (n, M, opts), plan, (Hs, dH, dD), s in zip(specs, plans, data, streams):
        plan.check(s.cuda_stream)
        for H, d in zip(Hs, dD):
            a, b = oracle.gershgorin(H)
            assert np.max(np.abs(d.cpu().numpy() - oracle.dm_cheb(H, a, b, oracle.cheb_coeffs(7.0, 0.03, a, b, M)))) <= TOL_D
        plan.destroy()
