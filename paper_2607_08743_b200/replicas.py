"""Multi-GPU plumbing of the benchmark: "replicas only".

The path has no exchange step between patches, so N ranks advance N independent patches and nothing crosses the
data path. What does cross ranks is the timing: the step time is the MAX over ranks, the value the SUM of the
points all ranks advanced divided by that time. Works on any torch.distributed backend (nccl on GPUs, gloo in the
CPU tests)."""
from __future__ import annotations


def max_over_ranks(x: float, device=None) -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x: float, device=None) -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def whole_job_throughput(points_this_rank: int, steps: int, elapsed_ms_this_rank: float, device=None):
    """-> (Mpoint-updates/s of the whole job, max-over-ranks elapsed ms). Every rank gets the same answer."""
    ms = max_over_ranks(elapsed_ms_this_rank, device)
    pts = sum_over_ranks(float(points_this_rank), device)
    return pts * steps / (ms * 1e-3) / 1e6, ms
