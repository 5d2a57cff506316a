#!/usr/bin/env python
"""bench.py -- density-matrix solves/sec of the dense Chebyshev Fermi-operator path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg1] [--impl ours|reference]

One "step" = one pass of the whole hot path (Gershgorin bounds + rescale, coefficient
tables, baby steps, giant steps with fused low-order sums, trace) over one batch of synthetic input
= one solve per seed of the workload (cfg1: seeds 0-3 -> a batch of 4 solves per step, ONE set of grouped
launches through cheb_dm_compute_batch), with mu fixed beforehand by the device's own mu-inclusive path.
That path (cheb_dm_solve_batch: baby block once, giant block, Gram-kernel moments, bisection on the device,
long-K assembly) is timed too and reported beside it (`mu_inclusive`).  Everything runs through the C ABI
(include/cheb_dm.h via the ctypes binding); torch supplies device memory, streams and events only.

Prints ONE JSON line (rank 0).  `value` = solves/s with inputs resident in HBM; `e2e` = the same through
cheb_dm_compute_batch_host_async with pinned HOST buffers (H2D + D2H inside the timed region); `roofline` = the
product kernels against the FP64 tensor (DMMA) peak; `cpu_baseline` = the oracle on the host cores.
Multi-GPU: replicas only -- every rank runs the same workload on its own GPU, no data-path
collective; value = all ranks' solves / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "dm_solves_per_sec"
UNIT = "solves/s"
FLUSH_BYTES = 512 << 20  # > 126 MB L2
# dram__bytes_read.sum + dram__bytes_write.sum of the product launches of one step, from the `ncu --set full` captures
# summarised under profiles/: read from the data file the capture step writes (never typed here).
TRAFFIC_FILE = os.path.join(ROOT, "profiles", "r02_traffic.json")


def ncu_traffic(name):
    try:
        with open(TRAFFIC_FILE) as f:
            ent = json.load(f).get(name)
        return (float(ent["dram_bytes_per_step"]), ent.get("source")) if ent else (None, None)
    except Exception:
        return None, None


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="cfg1", help="workload of the headline line (BASELINE.json configs[1] = cfg1)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--others", default="cfg0,cfg2,cfg4,cfg3", help="comma list of extra workloads reported under other_workloads ('' = none)")
    ap.add_argument("--batch", type=int, default=0, help="matrices per step (0 = the workload's seeds; cfg0: 16 seeds)")
    ap.add_argument("--no-batch", action="store_true", help="ablation: the step's solves as serial cheb_dm_compute calls")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sched", type=int, default=0)
    ap.add_argument("--tile", type=int, default=0)
    ap.add_argument("--fuse", type=int, default=0, help="fuse_sums option of the plan (0 auto, 1 epilogue-fused, 2 pre-formed)")
    ap.add_argument("--giant", type=int, default=0, help="giant option of the plan (0 auto, 1 generic, 2 resident-multiplier kernel)")
    ap.add_argument("--symmetric", type=int, default=0, help="symmetric-tile skipping (0 auto = on, 1 off, 2 on)")
    ap.add_argument("--sliced", type=int, default=0, help="S > 0: every product of cheb_dm_compute on the sliced int8 tensor path (tcgen05 kind::i8, S digits)")
    ap.add_argument("--k", type=int, default=0)
    ap.add_argument("--p", type=int, default=0)
    return ap.parse_args()


# ---------------------------------------------------------------------------------------------------
# clocks sampler (NVML in a thread; the recipe's nvidia-smi fields)
# ---------------------------------------------------------------------------------------------------
class ClockSampler:
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x10: "sync_boost"}

    def __init__(self, torch, device_index):
        self.samples = []  # (t, sm_mhz, reasons_mask, power_w)
        self.regions = []
        self.ok = False
        self._stop = threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            h = None
            try:
                uuid = str(torch.cuda.get_device_properties(device_index).uuid)
                h = pynvml.nvmlDeviceGetHandleByUUID(("GPU-" + uuid) if not uuid.startswith("GPU-") else uuid)
            except Exception:
                vis = os.environ.get("CUDA_VISIBLE_DEVICES")
                idx = int(vis.split(",")[device_index]) if vis and vis.split(",")[device_index].isdigit() else device_index
                h = pynvml.nvmlDeviceGetHandleByIndex(idx)
            self.h = h
            self.sm_max = int(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception as e:  # pragma: no cover
            self.err = repr(e)
        if self.ok:
            self.th = threading.Thread(target=self._run, daemon=True)
            self.th.start()

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                sm = int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    mask = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                pw = nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0
                self.samples.append((time.perf_counter(), sm, mask, pw))
            except Exception:
                pass
            time.sleep(0.01)

    def begin(self):
        self._t0 = time.perf_counter()

    def end(self):
        self.regions.append((self._t0, time.perf_counter()))

    def window(self, t0, t1):
        """Clocks inside one wall-clock window (the timed region of one arm)."""
        if not self.ok:
            return None
        inside = [x for x in self.samples if t0 <= x[0] <= t1]
        if not inside:
            return None
        sm = sorted(x[1] for x in inside)
        mask = 0
        for x in inside:
            mask |= x[2]
        return {"sm_mhz": sm[len(sm) // 2], "sm_min_mhz": sm[0], "power_w_max": max(x[3] for x in inside), "samples": len(inside),
                "reasons": [n for bit, n in self.REASONS.items() if mask & bit]}

    def summary(self):
        if not self.ok:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "note": "NVML unavailable"}
        self._stop.set()
        self.th.join(timeout=1.0)
        inside = [s for s in self.samples if any(a <= s[0] <= b for a, b in self.regions)]
        note = "sampled inside the timed regions (NVML, 10 ms period)"
        if len(inside) < 3:
            inside = self.samples
            note = "timed regions shorter than the sampling period: all samples of the run"
        sm = sorted(s[1] for s in inside)
        mask = 0
        for s in inside:
            mask |= s[2]
        reasons = [n for bit, n in self.REASONS.items() if mask & bit]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": self.sm_max, "reasons": reasons,
                "power_w_max": max((s[3] for s in inside), default=None), "samples": len(inside), "note": note}


# ---------------------------------------------------------------------------------------------------
# GPU arm
# ---------------------------------------------------------------------------------------------------
def workload_seeds(cfg, name, args):
    """cfg1: the four seeds of BASELINE.json; cfg0 (one tile per product): 16 seeded matrices of the same recipe
    form the batch; the others: their one seed."""
    n = args.batch if args.batch > 0 else (16 if name == "cfg0" else len(cfg.seeds))
    return tuple(cfg.seeds) if n == len(cfg.seeds) else tuple(range(n))


class Workload:
    """Device-resident inputs + a plan for one BASELINE.json config; mu per seed from the device's mu-inclusive path."""

    def __init__(self, torch, cd, workloads, name, args):
        self.torch, self.cd, self.name = torch, cd, name
        self.cfg = cfg = workloads.CONFIGS[name]
        self.N, self.M = cfg.N, cfg.M
        self.seeds = workload_seeds(cfg, name, args)
        self.units = len(self.seeds)
        self.batched = not args.no_batch
        self.st = torch.cuda.current_stream().cuda_stream
        self.plan = cd.Plan(cfg.N, cfg.M, sched=args.sched, tile=args.tile, k=args.k, p=args.p, fuse_sums=args.fuse, giant=args.giant,
                            symmetric=args.symmetric, max_batch=self.units if self.batched else 1, host_slots=2,
                            sliced=args.sliced, sliced_solve=1 if args.sliced else 0)
        self.hH, self.dH, self.dD, self.hD = [], [], [], []
        for seed in self.seeds:
            H = torch.from_numpy(workloads.hamiltonian(name, seed=seed))
            self.hH.append(H.pin_memory())
            self.dH.append(H.cuda())
            self.dD.append(torch.empty((cfg.N, cfg.N), dtype=torch.float64, device="cuda"))
            self.hD.append(torch.empty((cfg.N, cfg.N), dtype=torch.float64).pin_memory())
        self.pH, self.pD = [x.data_ptr() for x in self.dH], [x.data_ptr() for x in self.dD]
        self.phH, self.phD = [x.data_ptr() for x in self.hH], [x.data_ptr() for x in self.hD]
        self.dtr = torch.zeros(self.units, dtype=torch.float64, device="cuda")
        self.htr = torch.zeros(self.units, dtype=torch.float64).pin_memory()
        self.nocc = [float(cfg.N_occ)] * self.units
        # mu per seed: Gershgorin bounds -> blocks -> moments -> bisection, all on the device (cheb_dm_solve_batch)
        self.plan.coeffs(cfg.beta, 0.0, None)
        if self.batched:
            self.mu = self.plan.solve_batch(self.pH, self.nocc, self.pD, 100, True, self.st)
        else:
            self.mu = [self.plan.solve(self.pH[i], self.nocc[i], self.pD[i], 100, True, self.st) for i in range(self.units)]
        self.plan.check(self.st)
        self.launches_per_step = 0

    def step(self):
        if self.batched:
            self.plan.compute_batch(self.pH, self.pD, self.mu, self.st)
            self.plan.trace_batch(self.pD, self.dtr.data_ptr(), self.st)
            self.launches_per_step = self.plan.last_launch_count() + 1
            return
        n = 0
        for i in range(self.units):
            self.plan.coeffs(self.cfg.beta, self.mu[i], None)
            self.plan.compute(self.pH[i], self.pD[i], self.st)
            self.plan.trace(self.pD[i], self.dtr[i:].data_ptr(), self.st)
            n += self.plan.last_launch_count() + 1
        self.launches_per_step = n

    def step_mu_inclusive(self):
        # the whole "mu solved on the trace" path: nothing is known beforehand but beta and N_occ
        if self.batched:
            self.plan.solve_batch(self.pH, self.nocc, self.pD, 100, False, self.st)
            self.plan.trace_batch(self.pD, self.dtr.data_ptr(), self.st)
        else:
            for i in range(self.units):
                self.plan.solve(self.pH[i], self.nocc[i], self.pD[i], 100, False, self.st)
                self.plan.trace(self.pD[i], self.dtr[i:].data_ptr(), self.st)

    def step_host(self):
        # the batch of the step through the pipelined host entry point; every H2D / D2H of the step completes inside the
        # step (cheb_dm_wait)
        if self.batched:
            self.plan.compute_batch_host_async(self.phH, self.phD, self.htr.data_ptr(), self.mu, self.st)
        else:
            for i in range(self.units):
                self.plan.coeffs(self.cfg.beta, self.mu[i], None)
                self.plan.compute_host_async(self.phH[i], self.phD[i], self.htr[i:].data_ptr(), self.st)
        self.plan.wait(self.st)

    def step_host_queue(self):
        # the same call without the wait: consecutive steps pipeline through the plan's two staging sets (H2D of step
        # n+1 and D2H of step n-1 overlap the kernels of step n); the caller closes the timed region with plan.wait
        if self.batched:
            self.plan.compute_batch_host_async(self.phH, self.phD, self.htr.data_ptr(), self.mu, self.st)
        else:
            for i in range(self.units):
                self.plan.coeffs(self.cfg.beta, self.mu[i], None)
                self.plan.compute_host_async(self.phH[i], self.phD[i], self.htr[i:].data_ptr(), self.st)

    def h2d_bytes(self):
        return self.units * 8 * self.N * self.N

    def d2h_bytes(self):
        return self.units * (8 * self.N * self.N + 8)


def timed_steps(torch, step_fn, steps, warmup, flush, sampler=None, dist=None):
    """W untimed steps, then K steps each bracketed by CUDA events on the launching stream with an L2 flush
    (512 MiB memset) between them; returns total event milliseconds of the K steps."""
    for _ in range(warmup):
        flush.zero_()
        step_fn()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    if sampler:
        sampler.begin()
    evs = []
    for _ in range(steps):
        flush.zero_()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        step_fn()
        e1.record()
        evs.append((e0, e1))
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    if sampler:
        sampler.end()
    return sum(a.elapsed_time(b) for a, b in evs)


def timed_host_stream(torch, w, steps, warmup, dist=None):
    """End-to-end arm: `steps` consecutive steps through the pipelined host entry point inside ONE timed region (CUDA events
    on the launching stream; the closing event is recorded after cheb_dm_wait has seen every copy finish), so every step's
    H2D of its inputs from pinned host memory and D2H of its results lie inside the region.  No L2 flush: each step's inputs
    arrive from host memory.  Returns the total milliseconds."""
    for _ in range(warmup):
        w.step_host()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        w.step_host_queue()
    w.plan.wait(w.st)
    e1.record()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    return e0.elapsed_time(e1)


def max_over_ranks(torch, dist, ms):
    """Replicas only: the job's time is the slowest rank's; no data-path collective."""
    if dist is None:
        return ms
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([ms], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(world, units_per_step, steps, max_ms):
    """Whole-job solves/s: every rank processed units_per_step * steps solves in max_ms (weak scaling)."""
    return world * units_per_step * steps / (max_ms * 1e-3)


def measure_sliced(torch, cd, workloads, name, args, steps, warmup, flush, dist, world, int8_peak, sampler=None):
    """The same fixed-mu step with every product on the sliced int8 tensor path (tcgen05 kind::i8, plan option
    sliced_solve): solves/s, and the digit GEMMs' executed int8 operations against the int8 tensor peak."""
    import copy
    a2 = copy.copy(args)
    a2.sliced = 8
    w = Workload(torch, cd, workloads, name, a2)
    plan = w.plan
    plan.set_timing(True)
    for _ in range(warmup):
        w.step()
    torch.cuda.synchronize()
    plan.set_timing(True)
    t_w0 = time.perf_counter()
    total_ms = timed_steps(torch, w.step, steps, 0, flush, None, dist)
    t_w1 = time.perf_counter()
    n_rec, prod_ms = plan.product_ms()
    plan.set_timing(False)
    plan.check(w.st)
    total_ms = max_over_ranks(torch, dist, total_ms)
    ops = plan.sliced_ops_per_compute()
    kernel_ms = prod_ms / max(n_rec, 1)
    achieved = ops / (kernel_ms * 1e-3) * 1e-12
    mi_steps = max(2, min(steps, 5))
    mi_ms = max_over_ranks(torch, dist, timed_steps(torch, w.step_mu_inclusive, mi_steps, 1, flush, None, dist)) / mi_steps
    plan.check(w.st)
    tr_mi = [float(x) for x in w.dtr.cpu().tolist()]
    e2e_steps = max(3, min(steps, 10))
    e2e_ms = max_over_ranks(torch, dist, timed_host_stream(torch, w, e2e_steps, 1, dist))
    res = {"call": "cheb_dm_compute on a plan with sliced_solve = 1, sliced = 8 digits", "value": job_value(world, w.units, steps, total_ms), "unit": UNIT,
           "ms_per_solve": total_ms / steps / w.units, "tr_D": [float(x) for x in w.dtr.cpu().tolist()],
           "e2e": {"value": world * w.units * e2e_steps / (e2e_ms * 1e-3), "unit": UNIT},
           "mu_inclusive": {"call": "cheb_dm_solve on the same plan (baby block and giant block sliced, nested giant steps)", "ms_per_solve": mi_ms / w.units,
                            "value": world * w.units / (mi_ms * 1e-3), "unit": UNIT, "tr_D": tr_mi},
           "full_product_equivalent_tflops": (plan.k + plan.p - 2) * 2.0 * w.N ** 3 / (kernel_ms * 1e-3) * 1e-12,
           "roofline": {"bound": "tensor", "kernel": "oz_gemm_kernel<8> (tcgen05.mma kind::i8, 8 int32 accumulators in tensor memory) + oz_split_reg_kernel + form_sums",
                        "achieved": achieved, "peak": int8_peak, "unit": "TOP/s", "frac": achieved / int8_peak if int8_peak else None,
                        "peak_source": "MEASURED_PEAKS.json bf16_tflops (burst) x 2 (nominal int8 : bf16 ratio of the profiling guide)",
                        "kernel_ms": kernel_ms, "ops_per_launch": ops, "note": "kernel_ms spans all product launches of a solve, slicing passes and the sums pass included"},
           "gpu_launches_per_step": w.launches_per_step, "workspace_bytes": plan.workspace_bytes(),
           "clocks": sampler.window(t_w0, t_w1) if sampler else None}
    plan.destroy()
    del w
    torch.cuda.empty_cache()
    return res


def measure_graph_replay(torch, w, steps, flush, dist, world):
    """Extra arm (reported beside `value`, never instead of it): the same step -- cheb_dm_compute_batch + cheb_dm_trace_batch --
    captured ONCE into a CUDA graph (the calls allocate nothing and never synchronise) and replayed: what is left of a step
    when the host's launch gaps are gone.  None for the serial ablation (its per-solve cheb_dm_coeffs are host calls)."""
    if not w.batched:
        return None
    try:
        side, g = torch.cuda.Stream(), torch.cuda.CUDAGraph()
        torch.cuda.synchronize()
        with torch.cuda.graph(g, stream=side):
            cs = torch.cuda.current_stream().cuda_stream
            w.plan.compute_batch(w.pH, w.pD, w.mu, cs)
            w.plan.trace_batch(w.pD, w.dtr.data_ptr(), cs)
        n = max(3, min(steps, 10))
        ms = max_over_ranks(torch, dist, timed_steps(torch, g.replay, n, 2, flush, None, dist))
        w.plan.check(w.st)
        tr = [float(x) for x in w.dtr.cpu().tolist()]
        del g
        return {"value": world * w.units * n / (ms * 1e-3), "unit": UNIT, "ms_per_step": ms / n, "steps": n, "tr_D": tr,
                "how": "one step captured into a CUDA graph, replayed; CUDA events around each replay, L2 flush between replays"}
    except Exception as e:  # never let the extra arm take the bench line down
        torch.cuda.synchronize()
        return {"error": repr(e)[:200]}


def measure_workload(torch, cd, workloads, name, args, steps, warmup, flush, sampler, dist, peak_tf, world):
    w = Workload(torch, cd, workloads, name, args)
    plan = w.plan
    # device-resident arm (timing ring on: two event records per compute call, no host sync)
    plan.set_timing(True)
    for _ in range(warmup):
        w.step()
    torch.cuda.synchronize()
    plan.set_timing(True)  # resets the ring after warm-up
    t_w0 = time.perf_counter()
    total_ms = timed_steps(torch, w.step, steps, 0, flush, sampler, dist)
    t_w1 = time.perf_counter()
    n_rec, prod_ms = plan.product_ms()  # the timed compute calls only (at most the last 256 of them)
    plan.set_timing(False)
    plan.check(w.st)                     # sticky device flags of the whole timed region
    total_ms = max_over_ranks(torch, dist, total_ms)
    flops = plan.flops_per_compute()     # per matrix
    per_call = w.units if w.batched else 1
    ms_per_step = total_ms / steps
    value = job_value(world, w.units, steps, total_ms)
    kernel_ms = prod_ms / max(n_rec, 1)  # product launches of one compute call (a whole batch when batched)
    achieved = per_call * flops / (kernel_ms * 1e-3) * 1e-12 if kernel_ms > 0 else 0.0
    tr_D = [float(x) for x in w.dtr.cpu().tolist()]
    # mu-inclusive arm: cheb_dm_solve[_batch] (bounds, blocks, moments, bisection, assembly) + trace
    mi_steps = max(3, min(steps, 10))
    mi_ms = timed_steps(torch, w.step_mu_inclusive, mi_steps, max(1, min(warmup, 3)), flush, None, dist)
    mi_ms = max_over_ranks(torch, dist, mi_ms) / mi_steps
    plan.check(w.st)
    tr_D_mi = [float(x) for x in w.dtr.cpu().tolist()]
    # end-to-end arm: host buffers through the pipelined host entry point
    e2e_steps = max(3, min(steps, 10))
    e2e_ms = timed_host_stream(torch, w, e2e_steps, max(1, min(warmup, 3)), dist)
    e2e_ms = max_over_ranks(torch, dist, e2e_ms)
    # the same with a wait after every step (latency of ONE step from host buffers to host buffers, nothing overlapped)
    e2e_sync_ms = max_over_ranks(torch, dist, timed_steps(torch, w.step_host, e2e_steps, 1, flush, None, dist))
    graph_arm = measure_graph_replay(torch, w, steps, flush, dist, world)
    traffic, traffic_src = ncu_traffic(name)
    res = {
        "workload": name, "N": w.N, "M_terms": w.M, "k": plan.k, "p": plan.p, "solves_per_step": w.units,
        "batched": bool(w.batched and w.units > 1), "tile": plan.opts.tile, "giant_kernel": "resident" if (plan.opts.giant == 2 and per_call == 1) else "generic",
        "value": value, "ms_per_step": ms_per_step, "ms_per_solve": ms_per_step / w.units,
        "tflops_step": world * w.units * steps * flops / (total_ms * 1e-3) * 1e-12,
        "flops_per_solve": flops, "gpu_launches_per_step": w.launches_per_step,
        "roofline": {"bound": "tensor",
                     "kernel": ("gemm_dmma_kernel (persistent grouped FP64 DMMA GEMM: baby steps) + giant_resident_kernel (giant steps, "
                                "multiplier resident in shared memory)") if (plan.opts.giant == 2 and per_call == 1) else
                               "gemm_dmma_kernel (persistent grouped FP64 DMMA GEMM: baby-step launch + giant-step launch over the whole batch)",
                     "achieved": achieved, "peak": peak_tf, "unit": "TFLOP/s", "frac": achieved / peak_tf if peak_tf else None,
                     "traffic": traffic, "traffic_source": traffic_src, "kernel_ms": kernel_ms, "launches_timed": n_rec,
                     "kernel_share_of_step": (kernel_ms * (w.units / per_call)) / ms_per_step if ms_per_step > 0 else None,
                     "flops_per_launch": per_call * flops,
                     # context: what the same time would mean if every product were charged its full 2 N^3 flops
                     # (symmetric-tile skipping executes about half of them); not the roofline figure
                     "full_product_equivalent_tflops": (per_call * (plan.k + plan.p - 2) * 2.0 * w.N ** 3) / (kernel_ms * 1e-3) * 1e-12 if kernel_ms > 0 else None},
        "e2e": {"value": world * w.units * e2e_steps / (e2e_ms * 1e-3), "unit": UNIT,
                "h2d_bytes_per_step": w.h2d_bytes(), "d2h_bytes_per_step": w.d2h_bytes(), "steps": e2e_steps,
                "ms_per_step": e2e_ms / e2e_steps,
                "how": "consecutive steps through cheb_dm_compute[_batch]_host_async inside one timed region closed by cheb_dm_wait (two staging sets: copies of neighbouring steps overlap the kernels)",
                "one_step_latency_ms": e2e_sync_ms / e2e_steps,
                "one_step_value": world * w.units * e2e_steps / (e2e_sync_ms * 1e-3)},
        "mu_inclusive": {"call": "cheb_dm_solve_batch" if w.batched else "cheb_dm_solve", "ms_per_step": mi_ms, "ms_per_solve": mi_ms / w.units,
                         "value": world * w.units / (mi_ms * 1e-3), "unit": UNIT, "vs_fixed_mu": mi_ms / ms_per_step if ms_per_step > 0 else None,
                         "flops_per_solve": plan.flops_per_solve(), "tflops": w.units * plan.flops_per_solve() / (mi_ms * 1e-3) * 1e-12,
                         "products": plan.k + 2 * plan.p - 4, "tr_D": tr_D_mi},
        "graph_replay": graph_arm,
        "mu": w.mu, "tr_D": tr_D, "N_occ": w.cfg.N_occ, "seeds": list(w.seeds),
        "workspace_bytes": plan.workspace_bytes(),
        "clocks": sampler.window(t_w0, t_w1) if sampler else None,
    }
    plan.destroy()
    del w
    torch.cuda.empty_cache()
    return res


# ---------------------------------------------------------------------------------------------------
# CPU oracle arm (cpu_baseline leg and --impl reference)
# ---------------------------------------------------------------------------------------------------
def oracle_sample_setup(name):
    import numpy as np
    import oracle
    import workloads
    cfg = workloads.CONFIGS[name]
    H = workloads.hamiltonian(name, seed=cfg.seeds[0])
    a, b = oracle.gershgorin(H)
    return oracle, np, cfg, H, a, b


def oracle_time_terms(oracle, np, cfg, H, a, b, terms):
    """Seconds for the first `terms` terms of the oracle's naive recurrence (terms-2 plain products)."""
    c = np.zeros(terms)
    c[: min(terms, cfg.M)] = oracle.cheb_coeffs(cfg.beta, 0.0, a, b, cfg.M)[:terms]
    t0 = time.perf_counter()
    oracle.dm_cheb(H, a, b, c)
    return time.perf_counter() - t0


def oracle_rate(name, budget_s):
    """solves/s of O-cheb on this host, from a bounded sample extrapolated linearly in the product count."""
    oracle, np, cfg, H, a, b = oracle_sample_setup(name)
    t_probe = oracle_time_terms(oracle, np, cfg, H, a, b, 4)  # 2 products
    per_prod = max(t_probe / 2.0, 1e-6)
    terms = int(max(4, min(cfg.M, 2 + budget_s / per_prod)))
    t = oracle_time_terms(oracle, np, cfg, H, a, b, terms)
    per_prod = t / (terms - 2)
    t_solve = per_prod * (cfg.M - 2)
    full = terms >= cfg.M
    sample = (f"{name} seed {cfg.seeds[0]} (N={cfg.N}, M={cfg.M}): oracle.dm_cheb, first {terms} of {cfg.M} terms "
              f"({terms - 2} of {cfg.M - 2} naive products, {t:.2f} s)" + ("" if full else ", extrapolated linearly in the number of products"))
    return 1.0 / t_solve, sample, oracle.num_threads(), terms


def oracle_eig_rate(name, ref_sweep=None):
    """solves/s of O-eig (cyclic Jacobi + Eq. 1-2) on this host.  N <= 1000: ONE sweep is timed and multiplied by the
    sweeps a full run needs (counted on a 200 x 200 sample of the same kind); larger N: extrapolated from the
    N = 1000 sweep by (N/1000)^3.  Labelled accordingly."""
    import numpy as np
    import oracle
    import workloads
    cfg = workloads.CONFIGS[name]
    Hs = workloads.hamiltonian(name, seed=cfg.seeds[0], n=min(200, cfg.N))
    sweeps = max(1, oracle.jacobi_sweeps(Hs, 60, 1e-14))  # sweeps to off(H) <= 1e-14 |H|_F on the sample
    if cfg.N <= 1000:
        H = workloads.hamiltonian(name, seed=cfg.seeds[0])
        t0 = time.perf_counter()
        oracle.jacobi_sweeps(H, 1, 1e-14)
        t_sweep = time.perf_counter() - t0
        how = f"one Jacobi sweep at N={cfg.N} timed ({t_sweep:.2f} s) x {sweeps} sweeps (count from a 200x200 sample of the same kind)"
    else:
        t_sweep = (ref_sweep or 0.0) * (cfg.N / 1000.0) ** 3
        how = f"EXTRAPOLATED: one sweep at N=1000 ({ref_sweep:.2f} s) x (N/1000)^3 x {sweeps} sweeps"
    t = t_sweep * sweeps
    return (1.0 / t if t > 0 else None), how, t_sweep


def cpu_baselines(names, budget_s):
    """O-cheb (bounded sample, linear in the product count) and O-eig per workload, as SURVEY 8(d) specifies."""
    out, ref_sweep = {}, None
    for name in names:
        try:
            v, sample, cores, _ = oracle_rate(name, budget_s)
            ent = {"o_cheb": {"value": v, "unit": UNIT, "cores": cores, "sample": sample}}
            import workloads
            if workloads.CONFIGS[name].N == 1000 or ref_sweep is None:
                pass
            ve, how, t_sweep = oracle_eig_rate(name, ref_sweep)
            if workloads.CONFIGS[name].N == 1000:
                ref_sweep = t_sweep
            ent["o_eig"] = {"value": ve, "unit": UNIT, "cores": cores, "sample": how}
            out[name] = ent
        except Exception as e:  # pragma: no cover
            out[name] = {"error": repr(e)}
    return out


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import workloads
    name = args.config
    cfg = workloads.CONFIGS[name]
    oracle, np, cfg, H, a, b = oracle_sample_setup(name)
    t_probe = oracle_time_terms(oracle, np, cfg, H, a, b, 4)
    per_prod = max(t_probe / 2.0, 1e-6)
    budget_step = min(2.0, 150.0 / max(1, args.steps + args.warmup))
    terms = int(max(3, min(cfg.M, 2 + budget_step / per_prod)))
    for _ in range(args.warmup):
        oracle_time_terms(oracle, np, cfg, H, a, b, terms)
    ts = [oracle_time_terms(oracle, np, cfg, H, a, b, terms) for _ in range(args.steps)]
    per_prod = sum(ts) / len(ts) / (terms - 2)
    t_solve = per_prod * (cfg.M - 2)
    value = 1.0 / t_solve
    sample = (f"{name} seed {cfg.seeds[0]} (N={cfg.N}, M={cfg.M}): each step = oracle.dm_cheb over the first {terms} of {cfg.M} terms "
              f"({terms - 2} of {cfg.M - 2} naive products), solves/s extrapolated linearly in the number of products")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * sum(ts) / len(ts), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{name}: {cfg.note}; beta={cfg.beta}, M={cfg.M} terms, N_occ={cfg.N_occ}", "N": cfg.N, "M_terms": cfg.M},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ---------------------------------------------------------------------------------------------------
def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import paper_2306_12616_b200 as cd
    import workloads

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; --impl reference times the CPU oracle)")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        dist_mod.init_process_group(backend="nccl", device_id=torch.device("cuda", local))
        dist = dist_mod
    cd.lib()

    sampler = ClockSampler(torch, local) if rank == 0 else None
    flush = torch.empty(FLUSH_BYTES, dtype=torch.uint8, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    peak_tf = max(cd.dmma_peak(40000, st) for _ in range(3))

    try:
        int8_peak = 2.0 * float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))).get("bf16_tflops"))
    except Exception:
        int8_peak = 2.0 * 1590.0  # the profiling guide's fallback bf16 figure x 2
    main_res = measure_workload(torch, cd, workloads, args.config, args, args.steps, args.warmup, flush, sampler, dist, peak_tf, world)
    others = []
    for name in [s for s in args.others.split(",") if s and s != args.config]:
        big = workloads.CONFIGS[name].N >= 2000
        k_steps = max(2, min(args.steps, 5 if big else 10))
        others.append(measure_workload(torch, cd, workloads, name, args, k_steps, 3, flush, sampler, dist, peak_tf, world))
        if big and not args.sliced:
            # N >= 2000: the same step with the products on the sliced int8 tensor path, reported beside it
            others[-1]["sliced_int8"] = measure_sliced(torch, cd, workloads, name, args, k_steps, 3, flush, dist, world, int8_peak, sampler)
    peak_after = cd.dmma_peak(40000, st)
    # sustained DMMA peak: the same microbenchmark back to back for ~2 s (clocks settle under the power cap)
    t_end = time.perf_counter() + 2.0
    peak_sustained = peak_after
    while time.perf_counter() < t_end:
        peak_sustained = cd.dmma_peak(400000, st)

    if rank == 0:
        clocks = sampler.summary() if sampler else None
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except Exception:
            peaks = {}
        cfg = workloads.CONFIGS[args.config]
        line = {
            "metric": METRIC, "value": main_res["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": main_res["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{args.config}: {cfg.note}; beta={cfg.beta}, M={cfg.M} terms, N_occ={cfg.N_occ}, seeds {list(cfg.seeds)}; "
                                   "mu solved on the trace beforehand by cheb_dm_solve_batch (device moments + bisection); the step's solves run as one batch (cheb_dm_compute_batch)",
                       "N": cfg.N, "M_terms": cfg.M, "k": main_res["k"], "p": main_res["p"], "solves_per_step": main_res["solves_per_step"],
                       "batched": main_res["batched"], "tile": main_res["tile"], "giant_kernel": main_res["giant_kernel"],
                       "parallelism": "replicas only (one plan per GPU, no collective)" if world > 1 else "1 GPU",
                       "l2": "flushed between timed steps (512 MiB device memset outside the event brackets)",
                       "bounds": "Gershgorin on the device", "symmetric_tiles": bool(args.symmetric != 1),
                       "flops": "executed tensor flops only (lower-triangle tiles when symmetric_tiles)", "sched": "grouped persistent kernel" if args.sched == 0 else "serial launches"},
            "ms_per_solve": main_res["ms_per_solve"], "tflops": main_res["tflops_step"],
            "e2e": {k: main_res["e2e"][k] for k in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step", "how", "one_step_value", "one_step_latency_ms")},
            "gpu_launches": main_res["gpu_launches_per_step"] * args.steps,
            "roofline": dict(main_res["roofline"],
                             peak_source="cheb_dm_dmma_peak: live register-resident DMMA.8x8x4 microbenchmark on this GPU (MEASURED_PEAKS.json has no FP64 entry)",
                             peak_after_run=peak_after, peak_sustained=peak_sustained,
                             frac_of_sustained=(main_res["roofline"]["achieved"] / peak_sustained) if peak_sustained else None,
                             peak_alt_bf16_ratio=(peaks.get("bf16_tflops") or 0) * 40.0 / 2250.0 or None),
            "clocks": clocks,
            "mu": main_res["mu"], "tr_D": main_res["tr_D"], "mu_inclusive": main_res["mu_inclusive"],
            "graph_replay": main_res.get("graph_replay"),
            "other_workloads": others,
        }
        if not args.no_cpu_baseline and world == 1:
            v, sample, cores, _ = oracle_rate(args.config, 12.0)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}
            # per workload: O-cheb and O-eig; N = 1000 first so that the larger sizes can extrapolate its sweep
            names = [args.config] + [o["workload"] for o in others]
            order = sorted(names, key=lambda n: (workloads.CONFIGS[n].N != 1000, workloads.CONFIGS[n].N))
            per = cpu_baselines(order, 4.0)
            line["cpu_baseline"]["per_workload"] = {n: per[n] for n in names}
        print(json.dumps(line))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
