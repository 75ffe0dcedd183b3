"""Multi-GPU plumbing of the hot path.

Forest pairs are independent units and every output is an additive accumulator, so the path
shards with no exchange step.  bench.py gives every rank an independent catalogue of the same
shape (weak scaling); the only collectives are the reductions of (time, work) that the timing
contract needs.  Nothing here touches the method's arithmetic.
"""
from __future__ import annotations


def rank_seed(base_seed: int, rank: int) -> int | None:
    """Catalogue seed of a rank: rank 0 uses the config's own seed (None), others base + 1000 * rank."""
    return None if rank == 0 else int(base_seed) + 1000 * int(rank)


def aggregate(ms: float, units: float, device=None):
    """(max over ranks of ms, sum over ranks of units).  Works on any initialised process group
    (nccl on GPUs, gloo on CPU); without one it returns its arguments."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms), float(units)
    t = torch.tensor([float(ms), float(units)], dtype=torch.float64, device=device)
    tmax = t.clone()
    dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
    tsum = t.clone()
    dist.all_reduce(tsum, op=dist.ReduceOp.SUM)
    return float(tmax[0]), float(tsum[1])


def throughput(ms: float, units: float, device=None) -> float:
    """Whole-job units per second: all ranks' units over the slowest rank's time."""
    m, u = aggregate(ms, units, device)
    return u / (m * 1e-3)
