"""`-m gpu`: seeded random CALL SEQUENCES on one plan (cheb_dm_coeffs with new beta / mu / bounds, fixed-mu solves alone, in
batches and from host buffers, the mu-inclusive calls, assemble, moments + solve_mu, a NaN input, tracing / timing toggles):
every D, tau and mu against the oracle, ESTATE / EBOUNDS exactly where include/cheb_dm.h says.  The single-call tests cover
the arithmetic; this covers what one call leaves behind for the next (it found two bugs: single solves on a batch plan, and
assemble after new bounds)."""
import random

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

OPS = ["coeffs", "compute", "batch", "solve", "solve_batch", "assemble", "moments", "host", "async", "nan", "toggle"]


def _sequence(rng, sq):
    import oracle
    import paper_2306_12616_b200 as cd
    import workloads
    import gpu_util as gu
    torch = gu.torch_cuda()
    st = torch.cuda.current_stream().cuda_stream

    def dm(H, ab_, beta, mu, M):
        return oracle.dm_cheb(H, ab_[0], ab_[1], oracle.cheb_coeffs(beta, mu, ab_[0], ab_[1], M))

    n = rng.choice([33, 64, 100, 129, 200, 450])
    M = rng.randint(3, 20) if n < 300 else rng.randint(3, 8)
    maxb = rng.choice([1, 3])
    opts = {}
    if rng.random() < 0.3:
        opts["sliced_solve"] = 1
        maxb = 1
    if rng.random() < 0.3:
        opts["tile"] = rng.choice([3, 4, 7, 9, 11, 12])
    if rng.random() < 0.2:
        opts["host_slots"] = 2
    plan = cd.Plan(n, M, max_batch=maxb, **opts)
    beta, mu, bounds = 5.0, 0.05, None
    plan.coeffs(beta, mu, bounds)
    Hs = [workloads.hamiltonian("cfg1", seed=sq * 11 + s, n=n) for s in range(3)]
    dHs = [gu.to_dev(h) for h in Hs]
    dDs = [torch.empty((n, n), dtype=torch.float64, device="cuda") for _ in range(3)]
    blocks_nb, blocks_H, log = 0, None, []

    def ab(H):
        return bounds if bounds is not None else oracle.gershgorin(H)

    for step in range(12):
        op = rng.choice(OPS)
        log.append(op)
        worst = 0.0
        if op == "coeffs":
            old = bounds
            beta, mu = rng.choice([3.0, 5.0, 12.0]), rng.uniform(-0.3, 0.3)
            bounds = None if rng.random() < 0.7 else (-8.0 - rng.random(), 8.0 + rng.random())
            if bounds != old:
                blocks_nb = 0          # new bounds make the blocks stale (include/cheb_dm.h, cheb_dm_assemble)
            plan.coeffs(beta, mu, bounds)
        elif op == "compute":
            i = rng.randrange(3)
            plan.compute(dHs[i].data_ptr(), dDs[0].data_ptr(), st)
            plan.check(st)
            worst = float(np.abs(dDs[0].cpu().numpy() - dm(Hs[i], ab(Hs[i]), beta, mu, M)).max())
            blocks_nb = 0
        elif op == "batch" and maxb > 1:
            nb = rng.choice([1, 2, 3])
            mus = [mu + 0.02 * s for s in range(nb)]
            plan.compute_batch([dHs[s].data_ptr() for s in range(nb)], [dDs[s].data_ptr() for s in range(nb)], mus, st)
            plan.check(st)
            for s in range(nb):
                worst = max(worst, float(np.abs(dDs[s].cpu().numpy() - dm(Hs[s], ab(Hs[s]), beta, mus[s], M)).max()))
            blocks_nb = 0
        elif op == "solve":
            i = rng.randrange(3)
            m = plan.solve(dHs[i].data_ptr(), 0.4 * n, dDs[0].data_ptr(), 100, True, st)
            plan.check(st)
            worst = float(np.abs(dDs[0].cpu().numpy() - dm(Hs[i], ab(Hs[i]), beta, m, M)).max())
            blocks_nb, blocks_H = 1, [Hs[i]]
        elif op == "solve_batch" and maxb > 1:
            nb = rng.choice([2, 3])
            ms = plan.solve_batch([dHs[s].data_ptr() for s in range(nb)], [0.4 * n] * nb, [dDs[s].data_ptr() for s in range(nb)], 100, True, st)
            plan.check(st)
            for s in range(nb):
                worst = max(worst, float(np.abs(dDs[s].cpu().numpy() - dm(Hs[s], ab(Hs[s]), beta, ms[s], M)).max()))
            blocks_nb, blocks_H = nb, Hs[:nb]
        elif op == "assemble":
            nb = blocks_nb if blocks_nb and rng.random() < 0.8 else (rng.choice([1, 2]) if maxb > 1 else 1)
            mus = [rng.uniform(-0.2, 0.2) for _ in range(nb)]
            if nb == blocks_nb:
                plan.assemble(mus, [dDs[s].data_ptr() for s in range(nb)], st)
                plan.check(st)
                for s in range(nb):
                    worst = max(worst, float(np.abs(dDs[s].cpu().numpy() - dm(blocks_H[s], ab(blocks_H[s]), beta, mus[s], M)).max()))
            else:
                with pytest.raises(cd.ChebDMError) as ei:
                    plan.assemble(mus, [dDs[s].data_ptr() for s in range(nb)], st)
                assert ei.value.status == 4, (log, nb, blocks_nb)
        elif op == "moments":
            i = rng.randrange(3)
            tau = plan.moments(dHs[i].data_ptr(), True, st)[:M]
            a, b = ab(Hs[i])
            _, tau_or = oracle.dm_cheb(Hs[i], a, b, np.zeros(M), want_tau=True)
            worst = float(np.abs(tau - tau_or).max()) / n
            blocks_nb, blocks_H = 1, [Hs[i]]
            m = plan.solve_mu(beta, 0.4 * n, 100, st)
            worst = max(worst, abs(m - oracle.solve_mu(tau_or, beta, a, b, 0.4 * n, iters=100)) / max(1.0, b - a))
        elif op in ("host", "async"):
            i = rng.randrange(3)
            hH = torch.from_numpy(Hs[i].copy()).pin_memory()
            hD = torch.empty((n, n), dtype=torch.float64).pin_memory()
            if op == "host":
                plan.compute_host(hH.data_ptr(), hD.data_ptr(), 0, st)
            else:
                plan.compute_host_async(hH.data_ptr(), hD.data_ptr(), 0, st)
                plan.compute_host_async(hH.data_ptr(), hD.data_ptr(), 0, st)
                plan.wait(st)
            worst = float(np.abs(hD.numpy() - dm(Hs[i], ab(Hs[i]), beta, mu, M)).max())
            blocks_nb = 0
        elif op == "nan" and bounds is None:
            Hn = Hs[0].copy()
            Hn[n // 2, n // 3] = Hn[n // 3, n // 2] = float("nan")
            dHn = gu.to_dev(Hn)
            plan.compute(dHn.data_ptr(), dDs[0].data_ptr(), st)
            with pytest.raises(cd.ChebDMError) as ei:
                plan.check(st)
            assert ei.value.status == 5, log     # EBOUNDS, reported once, then cleared
            blocks_nb = 0
        elif op == "toggle":
            plan.set_trace(rng.random() < 0.5)
            plan.set_timing(rng.random() < 0.5)
        assert worst <= 1e-10, f"seq {sq} n={n} M={M} max_batch={maxb} opts={opts}: step {step} ({op}) err {worst:.3e}; calls so far {log}"
    plan.destroy()


@pytest.mark.parametrize("seed,count", [(1, 25), (2, 25), (23, 25)])
def test_random_call_sequences_on_one_plan(seed, count):
    rng = random.Random(seed)
    for sq in range(count):
        _sequence(rng, sq)
