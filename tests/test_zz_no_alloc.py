"""`-m gpu` test of cheb_dm_bounds_static (include/cheb_dm.h): the Gershgorin bounds entry point that allocates nothing
(scratch in a file-scope static device array).  Its output is compared with the existing path -- the bounds the fused
front end of cheb_dm_compute leaves in the plan (cheb_dm_get_bounds) -- and with the oracle, within the tolerance of
tests/test_gpu_parity.py::test_gershgorin_bounds_and_rescale (N 2^-52 max(|a|, |b|)), on two calls in a row: the second
on a SMALLER matrix, so that the rows the first call left in the shared scratch would show if they were read.

Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _existing_path_bounds(cd, gu, H):
    torch = gu.torch_cuda()
    n = H.shape[0]
    st = torch.cuda.current_stream().cuda_stream
    plan = cd.Plan(n, 4)
    plan.coeffs(5.0, 0.0, None)
    dH = gu.to_dev(H)
    dD = torch.empty((n, n), dtype=torch.float64, device="cuda")
    plan.compute(dH.data_ptr(), dD.data_ptr(), st)
    plan.check(st)
    ab = plan.get_bounds(st)
    plan.destroy()
    return ab


def test_bounds_static_matches_the_plan_path_two_calls_in_a_row():
    import oracle
    import paper_2306_12616_b200 as cd
    import workloads
    import gpu_util as gu
    torch = gu.torch_cuda()
    st = torch.cuda.current_stream().cuda_stream
    # second call smaller than the first (stale rows in the scratch), odd N with an odd pitch, then the degenerate H = cI
    cases = [(workloads.hamiltonian("cfg2", seed=3, n=1000), 1000), (workloads.hamiltonian("cfg1", seed=1, n=301), 301),
             (workloads.hamiltonian("cfg3", seed=0, n=257), 260), (3.0 * np.eye(40), 40)]
    expect = [(_existing_path_bounds(cd, gu, H), oracle.gershgorin(H)) for H, _ in cases[:3]]
    outs, keep = [], []
    for H, ld in cases:                      # the calls follow one another on one stream, nothing in between
        n = H.shape[0]
        Hp = np.full((n, ld), 9.5)           # the padding must never be read as data
        Hp[:, :n] = H
        dH = gu.to_dev(Hp)
        out = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
        cd.bounds_static(dH.data_ptr(), n, ld, out.data_ptr(), st)
        keep.append(dH)
        outs.append(out)
    torch.cuda.synchronize()
    for (H, _), out, (plan_ab, or_ab) in zip(cases[:3], outs[:3], expect):
        n = H.shape[0]
        a, b = (float(x) for x in out.cpu().numpy())
        tol = n * 2.0 ** -52 * max(abs(or_ab[0]), abs(or_ab[1]))
        assert abs(a - plan_ab[0]) <= tol and abs(b - plan_ab[1]) <= tol, (n, a, b, plan_ab)
        assert abs(a - or_ab[0]) <= tol and abs(b - or_ab[1]) <= tol, (n, a, b, or_ab)
    assert tuple(outs[3].cpu().numpy()) == (2.0, 4.0)   # widened like the solve (reading A2-iv)


def test_bounds_static_rejects_sizes_beyond_the_scratch():
    import paper_2306_12616_b200 as cd
    import gpu_util as gu
    torch = gu.torch_cuda()
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    buf = torch.zeros(16, dtype=torch.float64, device="cuda")   # never read: the size check comes first
    with pytest.raises(cd.ChebDMError) as ei:
        cd.bounds_static(buf.data_ptr(), cd.STATIC_MAX_N + 1, cd.STATIC_MAX_N + 1, out.data_ptr(), 0)
    assert ei.value.status == 8 and "8192" in str(ei.value)
    with pytest.raises(cd.ChebDMError) as ei:
        cd.bounds_static(buf.data_ptr(), 4, 3, out.data_ptr(), 0)
    assert ei.value.status == 1
    # the largest size runs: H = 0 except a unit diagonal -> a == b == 1, widened to (0, 2)
    n = cd.STATIC_MAX_N
    dH = torch.eye(n, dtype=torch.float64, device="cuda")
    cd.bounds_static(dH.data_ptr(), n, n, out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert tuple(out.cpu().numpy()) == (0.0, 2.0)
