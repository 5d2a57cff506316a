"""Helpers for the `-m gpu` parity tests: device buffers (torch is plumbing only) and one solve
through the C ABI (paper_2306_12616_b200.Plan -> include/cheb_dm.h)."""
import numpy as np


def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


def to_dev(a):
    torch = torch_cuda()
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()


def gpu_solve(H, beta, mu, M, bounds=None, keep_plan=False, **opts):
    """cheb_dm_plan_ex -> cheb_dm_coeffs -> cheb_dm_compute -> cheb_dm_trace on the current stream.
    Returns dict(D, trace, bounds, plan?)."""
    import paper_2306_12616_b200 as cd
    torch = torch_cuda()
    N = H.shape[0]
    plan = cd.Plan(N, M, **opts)
    dH = to_dev(H)
    dD = torch.full((N, N), float("nan"), dtype=torch.float64, device="cuda")
    dtr = torch.zeros(1, dtype=torch.float64, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    plan.coeffs(beta, mu, bounds)
    plan.compute(dH.data_ptr(), dD.data_ptr(), st)
    plan.trace(dD.data_ptr(), dtr.data_ptr(), st)
    plan.check(st)   # no watchdog / bounds flag from the device
    torch.cuda.synchronize()
    out = {"D": dD.cpu().numpy(), "trace": float(dtr.item()), "bounds": plan.get_bounds(st),
           "k": plan.k, "p": plan.p, "launches": plan.last_launch_count()}
    if keep_plan:
        out["plan"] = plan
        out["dH"] = dH
    else:
        plan.destroy()
    return out
