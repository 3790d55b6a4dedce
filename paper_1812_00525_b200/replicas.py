"""Multi-GPU plumbing for bench.py: "replicas only".

north_star runs the path on one GPU with no domain decomposition and no halo exchange, so N ranks are N independent
replicas and there is no data-path collective.  The only cross-rank operations are the barrier around the timed region
and the reduction of the timing: whole-job throughput = (sum over ranks of the units processed) / (max over ranks of
the elapsed time).  Works with any torch.distributed backend (nccl on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def world():
    if dist.is_available() and dist.is_initialized():
        return dist.get_rank(), dist.get_world_size()
    return 0, 1


def barrier(device=None):
    if device is not None and torch.device(device).type == "cuda":
        torch.cuda.synchronize(device)
    if dist.is_available() and dist.is_initialized():
        dist.barrier()
        if device is not None and torch.device(device).type == "cuda":
            torch.cuda.synchronize(device)


def aggregate(units_local: float, seconds_local: float, device="cpu"):
    """Returns (total units over all ranks, max seconds over ranks, units/s of the whole job)."""
    rank, n = world()
    if n == 1:
        return float(units_local), float(seconds_local), float(units_local) / float(seconds_local)
    u = torch.tensor([float(units_local)], dtype=torch.float64, device=device)
    t = torch.tensor([float(seconds_local)], dtype=torch.float64, device=device)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(u.item()), float(t.item()), float(u.item()) / float(t.item())
