"""Multi-GPU plumbing: events are independent, so ranks shard by event with no data-path
collective.  The only exchange is the timing reduction of bench.py: units summed over ranks,
elapsed time taken as the MAX over ranks."""
from __future__ import annotations


def aggregate_throughput(units_done: float, elapsed_ms: float, steps: int, world: int):
    """Returns (whole-job units per second, ms per step) with time = max over ranks, units = sum over ranks."""
    if world > 1:
        import torch
        import torch.distributed as dist
        dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
        t = torch.tensor([float(elapsed_ms)], dtype=torch.float64, device=dev)
        u = torch.tensor([float(units_done)], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(u, op=dist.ReduceOp.SUM)
        elapsed_ms, units_done = float(t.item()), float(u.item())
    return units_done / (elapsed_ms * 1e-3), elapsed_ms / max(1, steps)


def shard_events(n_events: int, rank: int, world: int):
    """Contiguous event ranges per rank (events never interact)."""
    lo = n_events * rank // world
    hi = n_events * (rank + 1) // world
    return range(lo, hi)
