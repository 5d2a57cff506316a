"""`-m gpu` parity of the mu-inclusive path: cheb_dm_solve = bounds, baby block and giant block once,
moments by the Gram kernel, bisection on the device, D = G_0 + sum_l G_l U_l as one long-K product; cheb_dm_assemble
re-assembles D for new chemical potentials from the resident blocks.

Oracle side (no value flows from the GPU into it): tau_n = tr T_n(X) from the naive matrix recurrence
(oracle.dm_cheb(..., want_tau=True)), mu by oracle.solve_mu (the 100-halving bisection of reading A9), D by
oracle.dm_cheb with that mu."""
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
    return oracle, cd, workloads, gpu_util


def _oracle_solution(oracle, workloads, cfg, seed, n, M):
    H = workloads.hamiltonian(cfg, seed=seed, n=n)
    N = H.shape[0]
    c = workloads.CONFIGS[cfg]
    M = c.M if M is None else M
    nocc = workloads.n_occ(cfg, N)
    a, b = oracle.gershgorin(H)
    _, tau = oracle.dm_cheb(H, a, b, np.zeros(M), want_tau=True)
    mu = oracle.solve_mu(tau, c.beta, a, b, nocc, iters=100)
    D = oracle.dm_cheb(H, a, b, oracle.cheb_coeffs(c.beta, mu, a, b, M))
    return dict(H=H, N=N, M=M, beta=c.beta, nocc=nocc, a=a, b=b, tau=tau, mu=mu, D=D)


CASES = [("cfg0", 0, 128, None, {}), ("cfg1", 0, 300, None, {}), ("cfg1", 1, 257, None, {}), ("cfg2", 0, 250, None, {}),
         ("cfg3", 0, 200, 1024, {}), ("cfg4", 0, 200, 2048, {}), ("cfg1", 2, 130, 60, dict(k=6, p=10)),
         ("cfg1", 0, 64, 12, dict(k=12, p=1)), ("cfg1", 0, 64, 12, dict(k=1, p=12)), ("cfg1", 0, 64, 12, dict(k=6, p=2)),
         ("cfg2", 0, 150, 70, dict(k=2, p=35, tile=3)), ("cfg1", 3, 700, 64, dict(tile=1)), ("cfg1", 3, 333, 64, dict(symmetric=1)),
         # power-basis outer recursion (Eq. 4): the long-K assembly still runs on the Chebyshev table g (its operands are U_l = T_l(T_k))
         ("cfg1", 2, 127, 10, dict(k=3, p=4, outer=1)), ("cfg0", 0, 128, None, dict(outer=1))]


@pytest.mark.parametrize("cfg,seed,n,M,opts", CASES)
def test_solve_mu_inclusive_parity(cfg, seed, n, M, opts):
    oracle, cd, workloads, gu = _imports()
    torch = gu.torch_cuda()
    o = _oracle_solution(oracle, workloads, cfg, seed, n, M)
    N = o["N"]
    plan = cd.Plan(N, o["M"], **opts)
    st = torch.cuda.current_stream().cuda_stream
    dH = gu.to_dev(o["H"])
    dD = torch.full((N, N), float("nan"), dtype=torch.float64, device="cuda")
    dtr = torch.zeros(1, dtype=torch.float64, device="cuda")
    plan.coeffs(o["beta"], 123.0, None)  # the mu given here is ignored by cheb_dm_solve
    mu = plan.solve(dH.data_ptr(), o["nocc"], dD.data_ptr(), 100, True, st)
    plan.trace(dD.data_ptr(), dtr.data_ptr(), st)
    plan.check(st)
    a, b, mu_dev, ne = plan.get_scalars(0, st)
    assert mu == mu_dev
    # the electron count at the GPU's mu hits the target as well as the oracle's own root does (oracle-side evaluation)
    ne_gpu = oracle.electron_count(o["tau"], o["beta"], mu, o["a"], o["b"])
    ne_or = oracle.electron_count(o["tau"], o["beta"], o["mu"], o["a"], o["b"])
    assert abs(ne_gpu - o["nocc"]) <= max(1e-8, 10 * abs(ne_or - o["nocc"]))
    assert abs(mu - o["mu"]) <= 1e-10 * max(1.0, abs(o["b"] - o["a"]))
    D = dD.cpu().numpy()
    assert np.max(np.abs(D - o["D"])) <= TOL_D
    assert abs(float(dtr.item()) - float(np.trace(o["D"]))) <= TOL_TR
    assert abs(float(dtr.item()) - o["nocc"]) <= 1e-7
    assert np.max(np.abs(D - D.T)) <= 1e-11
    # moments left on the device by the same call chain (cheb_dm_moments shares the code): compare tau too
    tau = plan.moments(dH.data_ptr(), True, st)[: o["M"]]
    assert np.max(np.abs(tau - o["tau"])) <= 1e-10 * N
    # new chemical potentials from the resident blocks
    for mu2 in (o["mu"] + 0.05, o["a"] + 0.3 * (o["b"] - o["a"])):
        plan.assemble([mu2], [dD.data_ptr()], st)
        torch.cuda.synchronize()
        D2 = oracle.dm_cheb(o["H"], o["a"], o["b"], oracle.cheb_coeffs(o["beta"], mu2, o["a"], o["b"], o["M"]))
        assert np.max(np.abs(dD.cpu().numpy() - D2)) <= TOL_D
    plan.destroy()


def test_solve_batch_parity_and_equals_single():
    """cheb_dm_solve_batch: three matrices with different targets in one set of launches; same mu and D (bitwise) as
    the single-matrix call on a batch plan, parity with the oracle for each."""
    oracle, cd, workloads, gu = _imports()
    torch = gu.torch_cuda()
    sols = [_oracle_solution(oracle, workloads, "cfg1", s, 200, 100) for s in range(3)]
    noccs = [100.0, 90.0, 111.0]
    for o, no in zip(sols, noccs):
        o["mu"] = oracle.solve_mu(o["tau"], o["beta"], o["a"], o["b"], no, iters=100)
        o["D"] = oracle.dm_cheb(o["H"], o["a"], o["b"], oracle.cheb_coeffs(o["beta"], o["mu"], o["a"], o["b"], o["M"]))
    plan = cd.Plan(200, 100, max_batch=4)
    st = torch.cuda.current_stream().cuda_stream
    dH = [gu.to_dev(o["H"]) for o in sols]
    dD = [torch.empty((200, 200), dtype=torch.float64, device="cuda") for _ in sols]
    plan.coeffs(sols[0]["beta"], 0.0, None)
    mus = plan.solve_batch([x.data_ptr() for x in dH], noccs, [x.data_ptr() for x in dD], 100, True, st)
    plan.check(st)
    Ds = [d.cpu().numpy() for d in dD]
    for o, mu, D in zip(sols, mus, Ds):
        assert abs(mu - o["mu"]) <= 1e-10 * (o["b"] - o["a"])
        assert np.max(np.abs(D - o["D"])) <= TOL_D
    one = torch.empty((200, 200), dtype=torch.float64, device="cuda")
    mu1 = plan.solve(dH[1].data_ptr(), noccs[1], one.data_ptr(), 100, True, st)
    assert mu1 == mus[1] and np.array_equal(one.cpu().numpy(), Ds[1])
    plan.destroy()


def test_solve_needs_the_moments_option_and_call_order():
    oracle, cd, workloads, gu = _imports()
    torch = gu.torch_cuda()
    H = workloads.hamiltonian("cfg1", seed=0, n=64)
    dH, dD = gu.to_dev(H), torch.empty((64, 64), dtype=torch.float64, device="cuda")
    plan = cd.Plan(64, 16, moments=1)
    plan.coeffs(10.0, 0.0, None)
    for call in (lambda: plan.solve(dH.data_ptr(), 32, dD.data_ptr()), lambda: plan.moments(dH.data_ptr()),
                 lambda: plan.assemble([0.0], [dD.data_ptr()])):
        with pytest.raises(cd.ChebDMError) as ei:
            call()
        assert ei.value.status == 6  # EUNSUPPORTED
    plan.destroy()
    plan = cd.Plan(64, 16)
    plan.coeffs(10.0, 0.0, None)
    with pytest.raises(cd.ChebDMError) as ei:
        plan.assemble([0.0], [dD.data_ptr()])      # no blocks in the workspace yet
    assert ei.value.status == 4
    plan.solve(dH.data_ptr(), 32, dD.data_ptr())
    plan.assemble([0.1], [dD.data_ptr()])
    plan.compute(dH.data_ptr(), dD.data_ptr())      # a fixed-mu compute overwrites the blocks' bookkeeping
    with pytest.raises(cd.ChebDMError) as ei:
        plan.assemble([0.0], [dD.data_ptr()])
    assert ei.value.status == 4
    plan.destroy()


def test_assemble_after_new_coeffs_beta_keeps_the_blocks_new_bounds_do_not():
    """The blocks a solve leaves behind are polynomials of X(a, b): cheb_dm_coeffs with a new beta keeps them (assemble gives
    the D of the new beta), with new bounds or a new bounds mode it invalidates them (ESTATE) -- never a D for the old
    scaling."""
    oracle, cd, workloads, gu = _imports()
    torch = gu.torch_cuda()
    st = torch.cuda.current_stream().cuda_stream
    n, M = 129, 14
    H = workloads.hamiltonian("cfg1", seed=6, n=n)
    a, b = oracle.gershgorin(H)
    dH, dD = gu.to_dev(H), torch.empty((n, n), dtype=torch.float64, device="cuda")
    plan = cd.Plan(n, M)
    plan.coeffs(5.0, 0.0, None)
    plan.solve(dH.data_ptr(), 0.4 * n, dD.data_ptr(), 100, True, st)
    plan.coeffs(12.0, 0.0, None)                     # beta only
    plan.assemble([0.2], [dD.data_ptr()], st)
    plan.check(st)
    D_or = oracle.dm_cheb(H, a, b, oracle.cheb_coeffs(12.0, 0.2, a, b, M))
    assert np.max(np.abs(dD.cpu().numpy() - D_or)) <= 1e-10
    plan.coeffs(12.0, 0.0, (a - 1.0, b + 1.0))       # explicit bounds: another X
    for call in (lambda: plan.assemble([0.2], [dD.data_ptr()], st), lambda: plan.solve_mu(12.0, 0.4 * n, 100, st)):
        with pytest.raises(cd.ChebDMError) as ei:
            call()
        assert ei.value.status == 4
    plan.solve(dH.data_ptr(), 0.4 * n, dD.data_ptr(), 100, True, st)    # blocks for the explicit bounds
    plan.assemble([0.2], [dD.data_ptr()], st)
    plan.check(st)
    D_or = oracle.dm_cheb(H, a - 1.0, b + 1.0, oracle.cheb_coeffs(12.0, 0.2, a - 1.0, b + 1.0, M))
    assert np.max(np.abs(dD.cpu().numpy() - D_or)) <= 1e-10
    plan.coeffs(12.0, 0.0, None)                     # back to Gershgorin bounds: stale again
    with pytest.raises(cd.ChebDMError) as ei:
        plan.assemble([0.2], [dD.data_ptr()], st)
    assert ei.value.status == 4
    plan.destroy()


def test_cuda_graph_capture_of_the_mu_inclusive_sliced_and_static_entry_points():
    """cheb_dm_solve[_batch] with mu_out = NULL (mu never leaves the device), cheb_dm_assemble, the sliced solve and
    cheb_dm_bounds_static allocate nothing and never synchronise: each is captured into a CUDA graph and its replays on new
    H contents are bit-identical to the eager calls."""
    oracle, cd, workloads, gu = _imports()
    torch = gu.torch_cuda()
    n, M, beta = 200, 30, 12.0
    Hs = [workloads.hamiltonian("cfg1", seed=s, n=n) for s in range(3)]

    def blocks_plan():
        p = cd.Plan(n, M)
        p.coeffs(beta, 0.02, None)
        d, o = gu.to_dev(Hs[0]), torch.empty((n, n), dtype=torch.float64, device="cuda")
        p.solve(d.data_ptr(), 80.0, o.data_ptr(), 100, True, 0)
        return p

    cases = [
        ("solve", lambda: cd.Plan(n, M), 1, lambda p, dH, dD, st: p.solve(dH[0].data_ptr(), 80.0, dD[0].data_ptr(), 100, False, st)),
        ("solve_batch", lambda: cd.Plan(n, M, max_batch=2), 2,
         lambda p, dH, dD, st: p.solve_batch([x.data_ptr() for x in dH], [80.0, 80.0], [x.data_ptr() for x in dD], 100, False, st)),
        ("sliced compute", lambda: cd.Plan(n, M, sliced_solve=1), 1, lambda p, dH, dD, st: p.compute(dH[0].data_ptr(), dD[0].data_ptr(), st)),
        ("sliced solve", lambda: cd.Plan(n, M, sliced_solve=1), 1,
         lambda p, dH, dD, st: p.solve(dH[0].data_ptr(), 80.0, dD[0].data_ptr(), 100, False, st)),
        ("assemble", blocks_plan, 1, lambda p, dH, dD, st: p.assemble([0.07], [dD[0].data_ptr()], st)),
    ]
    for name, make_plan, nb, call in cases:
        plan = make_plan()
        plan.coeffs(beta, 0.02, None)
        dH = [torch.empty((n, n), dtype=torch.float64, device="cuda") for _ in range(nb)]
        dD = [torch.empty((n, n), dtype=torch.float64, device="cuda") for _ in range(nb)]
        st = torch.cuda.current_stream().cuda_stream
        eager = []
        for H in Hs:
            for x in dH:
                x.copy_(torch.from_numpy(H))
            call(plan, dH, dD, st)
            torch.cuda.synchronize()
            eager.append([d.cpu().numpy().copy() for d in dD])
        side, g = torch.cuda.Stream(), torch.cuda.CUDAGraph()
        torch.cuda.synchronize()
        with torch.cuda.graph(g, stream=side):
            call(plan, dH, dD, torch.cuda.current_stream().cuda_stream)
        for H, De in zip(Hs, eager):
            for x in dH:
                x.copy_(torch.from_numpy(H))
            for x in dD:
                x.fill_(float("nan"))
            g.replay()
            torch.cuda.synchronize()
            for d, e in zip(dD, De):
                assert np.array_equal(d.cpu().numpy(), e), name
        plan.check(st)
        del g
        plan.destroy()
    # the no-allocation bounds entry point (its reason to exist: callers under capture)
    d, out = gu.to_dev(Hs[1]), torch.zeros(2, dtype=torch.float64, device="cuda")
    cd.bounds_static(d.data_ptr(), n, n, out.data_ptr(), 0)
    torch.cuda.synchronize()
    e = out.cpu().numpy().copy()
    side, g = torch.cuda.Stream(), torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        cd.bounds_static(d.data_ptr(), n, n, out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    out.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), e) and tuple(e) == pytest.approx(oracle.gershgorin(Hs[1]), rel=1e-13)
