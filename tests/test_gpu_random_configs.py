"""`-m gpu`: seeded random plan configurations (N, M, (k, p), tile, pairing, outer form, scheduling, batch, sliced, the
mu-inclusive calls) through the C ABI against the oracle's naive M-term sum, max|D - D_cheb| <= 1e-10 each.  The hand-picked
cases of the other files cover the shapes that matter; this one covers the combinations nobody picked (it found two: the
long-K assembly with the power-basis outer option, and sliced plans with p = 1).  Small N and M: the whole file runs in
seconds.  Expected values come from oracle/ only."""
import random

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _one_case(rng, it, big):
    import oracle
    import paper_2306_12616_b200 as cd
    import workloads
    import gpu_util as gu
    torch = gu.torch_cuda()
    st = torch.cuda.current_stream().cuda_stream
    n = rng.choice([300, 449, 450, 451, 500, 512, 513, 577, 640]) if big else \
        rng.choice([1, 2, 3, 7, 16, 31, 32, 33, 63, 64, 65, 96, 100, 127, 128, 129, 160, 200, 257])
    k = rng.choice([0, 1, 2, 3, 4, 5, 7, 8, 12])
    p = rng.choice([0, 1, 2, 3, 4, 5, 9])
    M = rng.randint(1, 40) if (k == 0 or p == 0) else rng.randint(max(1, k * (p - 1) + 1), k * p)
    if big and (k == 0 or p == 0):
        M = rng.randint(1, 14)
    if big and k * p > 16:
        k, p, M = 4, 4, rng.randint(13, 16)
    opts = {}
    mode = rng.choice(["plain", "plain", "batch", "sliced", "solve", "solve_batch", "sliced_solve_mu"])
    if rng.random() < 0.3:
        opts["tile"] = rng.choice([1, 2, 3, 4, 5, 6, 7, 9, 10, 11, 12])
    if rng.random() < 0.2:
        opts["symmetric"] = 1
    if rng.random() < 0.15 and mode not in ("sliced", "sliced_solve_mu") and (p == 0 or p <= 5) and M <= 25:
        opts["outer"] = 1          # power basis: small p only (the guard ENOCONV covers the rest, tests/test_gpu_parity.py)
    if rng.random() < 0.2:
        opts["fuse_sums"] = rng.choice([1, 2])
    if rng.random() < 0.2:
        opts["giant"] = rng.choice([1, 2])
    if rng.random() < 0.2:
        opts["pairing"] = rng.choice([1, 2, 3])
    if rng.random() < 0.15:
        opts["sched"] = 1
    nb = rng.choice([2, 3, 5]) if "batch" in mode else 1
    if nb > 1:
        opts["max_batch"] = nb + rng.choice([0, 1])
    if mode in ("sliced", "sliced_solve_mu"):
        opts["sliced_solve"] = 1
    desc = f"case {it}: n={n} M={M} k={k} p={p} mode={mode} opts={opts}"
    Hs = [workloads.hamiltonian("cfg1", seed=it * 7 + s, n=n) for s in range(nb)]
    beta = rng.choice([2.0, 8.0, 20.0])
    plan = cd.Plan(n, M, k=k, p=p, **opts)
    plan.coeffs(beta, 0.1, None)
    dH = [gu.to_dev(h) for h in Hs]
    dD = [torch.full((n, n), float("nan"), dtype=torch.float64, device="cuda") for _ in Hs]
    mus = [0.1 + 0.05 * s for s in range(nb)]
    nocc = max(0.3, 0.4 * n)
    if mode in ("plain", "sliced"):
        plan.compute(dH[0].data_ptr(), dD[0].data_ptr(), st)
        mus = [0.1]
    elif mode == "batch":
        plan.compute_batch([x.data_ptr() for x in dH], [x.data_ptr() for x in dD], mus, st)
    elif mode in ("solve", "sliced_solve_mu"):
        mus = [plan.solve(dH[0].data_ptr(), nocc, dD[0].data_ptr(), 100, True, st)]
    else:
        mus = list(plan.solve_batch([x.data_ptr() for x in dH], [nocc] * nb, [x.data_ptr() for x in dD], 100, True, st))
    plan.check(st)
    torch.cuda.synchronize()
    worst = 0.0
    for s in range(nb):
        a, b = oracle.gershgorin(Hs[s])
        if a == b:
            a, b = a - 1.0, b + 1.0
        D_or = oracle.dm_cheb(Hs[s], a, b, oracle.cheb_coeffs(beta, mus[s], a, b, M))
        worst = max(worst, float(np.max(np.abs(dD[s].cpu().numpy() - D_or))))
    plan.destroy()
    return desc, worst


@pytest.mark.parametrize("seed,count,big", [(1, 60, False), (2, 60, False), (3, 60, False), (11, 30, True)])
def test_random_configurations_against_the_oracle(seed, count, big):
    rng = random.Random(seed)
    failures = []
    for it in range(count):
        desc, worst = _one_case(rng, it, big)
        if not worst <= 1e-10:
            failures.append(f"{desc} -> max|dD| = {worst:.3e}")
    assert not failures, "\n".join(failures)
