"""`-m gpu` parity at BASELINE.json's full sizes, in the launch configuration bench.py times (default
plan options, Gershgorin bounds on the device): sampled columns of D against the oracle's column
recurrence (oracle.dm_cheb_columns: the same M-term sum applied to unit vectors), plus properties that
hold at any size (symmetry, tr D = N_occ because mu was solved on the trace, [H, D] = 0).

mu is an oracle-side input: tau_n from library eigenvalues (definition of T_n), oracle.solve_mu.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

FULL = [("cfg1", 0), ("cfg1", 1), ("cfg1", 2), ("cfg1", 3), ("cfg2", 0), ("cfg4", 0), ("cfg3", 0)]


@pytest.mark.parametrize("cfg,seed", FULL)
def test_full_size_sampled_columns(cfg, seed):
    import oracle
    import gpu_util as gu
    import oracle_cases as oc
    case = oc.case(cfg, seed, None, None, False)
    N, M = case["N"], case["M"]
    r = gu.gpu_solve(case["H"], case["beta"], case["mu"], M)
    assert abs(r["bounds"][0] - case["a"]) <= N * 2.0 ** -52 * abs(case["a"])
    assert abs(r["bounds"][1] - case["b"]) <= N * 2.0 ** -52 * abs(case["b"])
    D = r["D"]
    # columns spread over first / interior / last tiles (ragged tail included)
    ncols = 3 if N >= 2000 else 8
    cols = np.unique(np.concatenate([[0, N - 1], np.random.default_rng(7).integers(0, N, size=ncols - 2)])).astype(np.int32)
    want = oracle.dm_cheb_columns(case["H"], case["a"], case["b"], case["c"], cols)
    got = D[:, cols].T
    assert np.max(np.abs(got - want)) <= 1e-10
    # properties at any size
    assert np.max(np.abs(D - D.T)) <= 1e-11
    assert abs(r["trace"] - case["trace_cheb_scalar"]) <= 1e-9      # tr p_M(X) = sum_i p_M(x~_i)
    assert abs(r["trace"] - case["nocc"]) <= 1e-6                   # mu was solved on the trace
    assert abs(r["trace"] - float(np.trace(D))) <= 1e-9
    rows = cols[:2]
    comm = case["H"][rows, :] @ D - (D[rows, :] @ case["H"])
    assert np.max(np.abs(comm)) <= 1e-9 * max(1.0, np.max(np.abs(case["H"])) * N ** 0.5)


def test_cfg4_balanced_pairing_tightens_the_trace():
    """Reading A7b: with the balanced pairing of the baby steps (same stages and cost as Algorithm 1) the rounding left
    by Algorithm 1's squaring chains on cfg4 (|dtr| = 7.7e-10 of the 1e-9 gate) drops by two orders of magnitude."""
    import oracle
    import gpu_util as gu
    import oracle_cases as oc
    case = oc.case("cfg4", 0, None, None, False)
    r = gu.gpu_solve(case["H"], case["beta"], case["mu"], case["M"], pairing=2)
    assert abs(r["trace"] - case["trace_cheb_scalar"]) <= 5e-11
    cols = np.array([0, 777, case["N"] - 1], dtype=np.int32)
    want = oracle.dm_cheb_columns(case["H"], case["a"], case["b"], case["c"], cols)
    assert np.max(np.abs(r["D"][:, cols].T - want)) <= 1e-10
