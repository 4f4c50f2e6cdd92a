"""Rank sharding of the query axis: queries are independent, so a job over
n queries is cut in contiguous ranges, one per rank; the grid is replicated; no collective is on
the data path.  Only the timing is reduced (max over ranks)."""
from __future__ import annotations


def shard_range(n: int, rank: int, world: int) -> tuple[int, int]:
    """[lo, hi) of rank's contiguous share of n queries; shares differ by at most one query."""
    if world < 1 or not (0 <= rank < world) or n < 0:
        raise ValueError("bad shard arguments")
    base, rem = divmod(n, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def max_over_ranks(dist, seconds: float, device="cpu") -> float:
    """job time = the slowest rank's time (all_reduce MAX over the default process group)"""
    import torch
    t = torch.tensor([seconds], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
