"""Multi-GPU plumbing of the "replicas only" mode: N independent replicas of the
same problem, one process per GPU, NO data-path collective.  The only exchange is the timing reduction:
the step time of the job is the MAX over ranks, the throughput is the units all ranks processed divided
by that time.  Works on any torch.distributed backend (nccl on the GPU box, gloo in the CPU tests)."""
from __future__ import annotations


def max_over_ranks(seconds_or_ms: float, dist=None, device=None) -> float:
    """All-reduce(MAX) of one scalar; identity without a process group."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(seconds_or_ms)
    import torch
    t = torch.tensor([seconds_or_ms], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(units_per_rank: float, elapsed_s: float, world: int) -> float:
    """Whole-job throughput of `world` replicas that each processed `units_per_rank` units in (max) `elapsed_s`."""
    if elapsed_s <= 0:
        raise ValueError("elapsed time must be positive")
    return units_per_rank * world / elapsed_s
