"""`-m gpu` parity of the batched path (many independent small Hamiltonians):
cheb_dm_compute_batch runs nbatch solves in one set of grouped launches.  Every matrix of a batch is compared
element by element with the oracle's naive M-term sum (oracle.dm_cheb) on the same seeded input, with its own
Gershgorin bounds and its own chemical potential.  Expected values come from oracle/ only."""
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


def _run_batch(cd, gu, Hs, beta, mus, M, nb_plan=None, **opts):
    torch = gu.torch_cuda()
    n = Hs[0].shape[0]
    plan = cd.Plan(n, M, max_batch=nb_plan or len(Hs), **opts)
    st = torch.cuda.current_stream().cuda_stream
    dH = [gu.to_dev(H) for H in Hs]
    dD = [torch.full((n, n), float("nan"), dtype=torch.float64, device="cuda") for _ in Hs]
    dtr = torch.zeros(len(Hs), dtype=torch.float64, device="cuda")
    plan.coeffs(beta, 0.0, None)
    plan.compute_batch([x.data_ptr() for x in dH], [x.data_ptr() for x in dD], mus, st)
    plan.trace_batch([x.data_ptr() for x in dD], dtr.data_ptr(), st)
    plan.check(st)
    torch.cuda.synchronize()
    scal = [plan.get_scalars(s, st) for s in range(len(Hs))]
    return plan, [d.cpu().numpy() for d in dD], dtr.cpu().numpy(), scal


def _compare(case, D, tr, scal):
    n = case["N"]
    assert abs(scal[0] - case["a"]) <= n * 2.0 ** -52 * abs(case["a"]) and abs(scal[1] - case["b"]) <= n * 2.0 ** -52 * abs(case["b"])
    assert scal[2] == case["mu"]
    dD = float(np.max(np.abs(D - case["D_cheb"])))
    dtr = abs(float(tr) - float(np.trace(case["D_cheb"])))
    assert dD <= TOL_D, dD
    assert dtr <= TOL_TR, dtr
    assert np.max(np.abs(D - D.T)) <= 1e-11
    return dD, dtr


def test_batch_cfg1_four_seeds_full_size_full_matrix():
    """The headline workload of bench.py: the four seeds of cfg1 (N=500, M=256) as ONE batch, every element of every D."""
    oracle, cd, workloads, gu, oc = _imports()
    cases = [oc.case("cfg1", s, None, None, True) for s in range(4)]
    plan, Ds, trs, scal = _run_batch(cd, gu, [c["H"] for c in cases], cases[0]["beta"], [c["mu"] for c in cases], cases[0]["M"])
    assert plan.opts.max_batch == 4
    worst = max(_compare(c, D, tr, sc)[0] for c, D, tr, sc in zip(cases, Ds, trs, scal))
    print("cfg1 x4 batch: max|dD| =", worst, "tile", plan.opts.tile)
    plan.destroy()


@pytest.mark.parametrize("tile", [0, 3, 4, 5, 7, 9, 10, 11, 12])
def test_batch_ragged_n257_three_of_four_slots(tile):
    """nbatch < max_batch, odd N (ragged tiles, padded leading dimension), a different mu per matrix."""
    oracle, cd, workloads, gu, oc = _imports()
    cases = [oc.case("cfg1", s, 257, None, True) for s in (3, 1, 2)]
    plan, Ds, trs, scal = _run_batch(cd, gu, [c["H"] for c in cases], cases[0]["beta"], [c["mu"] for c in cases], cases[0]["M"],
                                     nb_plan=4, tile=tile)
    for c, D, tr, sc in zip(cases, Ds, trs, scal):
        _compare(c, D, tr, sc)
    plan.destroy()


def test_batch_front_end_rows_shared_by_warps():
    """Eight matrices of N = 801: the cooperative front end has 37 blocks per matrix, so two warps share a row (odd N:
    the last column apart).  Bounds, D and trace of every matrix against the oracle."""
    oracle, cd, workloads, gu, oc = _imports()
    cases = [oc.case("cfg2", s % 2, 801, 32, True) for s in range(8)]
    plan, Ds, trs, scal = _run_batch(cd, gu, [c["H"] for c in cases], cases[0]["beta"], [c["mu"] for c in cases], cases[0]["M"])
    for c, D, tr, sc in zip(cases, Ds, trs, scal):
        _compare(c, D, tr, sc)
    plan.destroy()


@pytest.mark.parametrize("fuse,symmetric,outer,sched", [(1, 2, 0, 0), (2, 2, 0, 0), (1, 1, 0, 0), (2, 1, 0, 0), (0, 0, 1, 0), (0, 0, 0, 1)])
def test_batch_cfg0_x8_variants(fuse, symmetric, outer, sched):
    """cfg0 (N=128: one or two tiles per product) x 8, sums fused / pre-formed, with and without symmetric tiles,
    the power-basis outer recursion of Eq. 4 and the serial (one launch per product level) ablation scheduler."""
    oracle, cd, workloads, gu, oc = _imports()
    base = oc.case("cfg0", 0, 128, None, True)
    cases = [base] + [oc.case("cfg0", s, 128, None, True) for s in range(1, 8)]
    plan, Ds, trs, scal = _run_batch(cd, gu, [c["H"] for c in cases], base["beta"], [c["mu"] for c in cases], base["M"],
                                     fuse_sums=fuse, symmetric=symmetric, outer=outer, sched=sched)
    for c, D, tr, sc in zip(cases, Ds, trs, scal):
        _compare(c, D, tr, sc)
    plan.destroy()


def test_batch_equals_single_solves_bitwise_and_is_reproducible():
    """A matrix gets the same D (bit for bit) whether it is solved alone in the generic kernel or inside a batch, in
    any slot, and repeated batches are bitwise reproducible: the summation order of a tile does not depend on the
    schedule.  Many back-to-back epilogue-only tiles (giant level l = p-1 of every slot) and K loops that fit the
    free ring (N <= 256: ktiles <= STAGES) exercise the per-slot "stored" barriers of the persistent kernel."""
    oracle, cd, workloads, gu, oc = _imports()
    torch = gu.torch_cuda()
    n, M, beta = 256, 100, 30.0
    Hs = [workloads.hamiltonian("cfg1", seed=s, n=n) for s in range(6)]
    mus = [0.02 * s - 0.05 for s in range(6)]
    singles = [gu.gpu_solve(H, beta, mu, M, giant=1, tile=4)["D"] for H, mu in zip(Hs, mus)]
    for rep in range(4):
        plan, Ds, trs, scal = _run_batch(cd, gu, Hs[::-1] if rep % 2 else Hs, beta, mus[::-1] if rep % 2 else mus, M, nb_plan=6, tile=4)
        got = Ds[::-1] if rep % 2 else Ds
        for a, b in zip(singles, got):
            assert np.array_equal(a, b)
        plan.destroy()


def test_batch_host_entry_points():
    """cheb_dm_compute_batch_host (synchronous) and the pipelined _async form + cheb_dm_wait against the device call."""
    oracle, cd, workloads, gu, oc = _imports()
    torch = gu.torch_cuda()
    n, M, beta = 200, 64, 40.0
    Hs = [workloads.hamiltonian("cfg1", seed=s, n=n) for s in range(3)]
    mus = [0.01, -0.02, 0.03]
    plan, ref, trs, _ = _run_batch(cd, gu, Hs, beta, mus, M, nb_plan=3, host_slots=2)
    st = torch.cuda.current_stream().cuda_stream
    hH = [torch.from_numpy(H).pin_memory() for H in Hs]
    for rounds in range(3):  # three queued batches through the two staging sets
        hD = [[torch.empty((n, n), dtype=torch.float64).pin_memory() for _ in Hs] for _ in range(3)]
        htr = [torch.zeros(3, dtype=torch.float64).pin_memory() for _ in range(3)]
        for q in range(3):
            plan.compute_batch_host_async([x.data_ptr() for x in hH], [x.data_ptr() for x in hD[q]], htr[q].data_ptr(), mus, st)
        plan.wait(st)
        for q in range(3):
            for i in range(3):
                assert np.array_equal(hD[q][i].numpy(), ref[i])
                assert abs(float(htr[q][i]) - float(trs[i])) <= 1e-12
    out = [torch.empty((n, n), dtype=torch.float64).pin_memory() for _ in Hs]
    tr1 = torch.zeros(3, dtype=torch.float64).pin_memory()
    plan.compute_batch_host([x.data_ptr() for x in hH], [x.data_ptr() for x in out], tr1.data_ptr(), mus, st)
    for i in range(3):
        assert np.array_equal(out[i].numpy(), ref[i])
    plan.destroy()


def test_batch_argument_checks():
    oracle, cd, workloads, gu, oc = _imports()
    torch = gu.torch_cuda()
    plan = cd.Plan(16, 4, max_batch=2)
    plan.coeffs(1.0, 0.0, None)
    a = torch.zeros((16, 16), dtype=torch.float64, device="cuda")
    b = torch.zeros((16, 16), dtype=torch.float64, device="cuda")
    c = torch.zeros((16, 16), dtype=torch.float64, device="cuda")
    for args in (([a.data_ptr()] * 3, [b.data_ptr(), c.data_ptr(), a.data_ptr()], None),   # nbatch > max_batch
                 ([a.data_ptr(), a.data_ptr()], [b.data_ptr(), b.data_ptr()], None),       # two outputs alias
                 ([a.data_ptr()], [a.data_ptr()], None),                                    # D aliases H
                 ([a.data_ptr()], [b.data_ptr()], [float("nan")])):
        with pytest.raises(cd.ChebDMError) as ei:
            plan.compute_batch(*args)
        assert ei.value.status == 1
    with pytest.raises(cd.ChebDMError) as ei:
        cd.Plan(16, 4, max_batch=65)
    assert ei.value.status == 1
    plan.destroy()


@pytest.mark.parametrize("n,tile", [(200, 0), (129, 4), (64, 7), (300, 0)])
def test_single_solves_on_a_batch_plan(n, tile):
    """cheb_dm_compute, cheb_dm_compute_batch with nbatch = 1 and cheb_dm_compute_host on a plan made with max_batch = 3 at
    N < 450, where the batch's giant-step tasks gather the sums in their epilogues: the resident-multiplier kernel (which
    reads pre-formed sums) must not take such a solve."""
    oracle, cd, workloads, gu, oc = _imports()
    torch = gu.torch_cuda()
    st = torch.cuda.current_stream().cuda_stream
    M, beta, mu = 24, 9.0, 0.04
    H = workloads.hamiltonian("cfg1", seed=2, n=n)
    a, b = oracle.gershgorin(H)
    D_or = oracle.dm_cheb(H, a, b, oracle.cheb_coeffs(beta, mu, a, b, M))
    plan = cd.Plan(n, M, max_batch=3, tile=tile)
    plan.coeffs(beta, mu, None)
    dH = gu.to_dev(H)
    dD = torch.full((n, n), float("nan"), dtype=torch.float64, device="cuda")
    plan.compute(dH.data_ptr(), dD.data_ptr(), st)
    plan.check(st)
    assert np.max(np.abs(dD.cpu().numpy() - D_or)) <= TOL_D
    dD.fill_(float("nan"))
    plan.compute_batch([dH.data_ptr()], [dD.data_ptr()], [mu], st)
    plan.check(st)
    assert np.max(np.abs(dD.cpu().numpy() - D_or)) <= TOL_D
    hH = torch.from_numpy(H.copy()).pin_memory()
    hD = torch.empty((n, n), dtype=torch.float64).pin_memory()
    plan.compute_host(hH.data_ptr(), hD.data_ptr(), 0, st)
    assert np.max(np.abs(hD.numpy() - D_or)) <= TOL_D
    plan.destroy()
