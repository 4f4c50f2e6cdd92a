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


def vegas_allreduce(dist, sums, hist=None):
    """The one exchange step of the widened path: every rank samples its own share of an
    iteration's points, so the sums of eq. 1.74-1.75 and the refinement histograms (L913) are
    added over the ranks -- one all-reduce of 2 + ndim * nbins doubles per iteration (NCCL on GPUs, gloo in the CPU
    tests); every rank then refines the same grid from the same histogram."""
    dist.all_reduce(sums, op=dist.ReduceOp.SUM)
    if hist is not None:
        dist.all_reduce(hist, op=dist.ReduceOp.SUM)
    return sums, hist
