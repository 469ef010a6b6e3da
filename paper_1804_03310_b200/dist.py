"""Multi-GPU plumbing for bench.py: the walker step has no exchange step ("subsets which are
independently propagated"), so N GPUs run N independent replicas of the batch; the only cross-rank traffic is
the max-over-ranks of the measured time.  Works on any torch.distributed backend (nccl on GPUs, gloo in tests)."""
from __future__ import annotations


def rank_seed(base: int, rank: int) -> int:
    """Distinct, reproducible field seed per replica."""
    return int(base) + 7919 * int(rank)


def max_over_ranks(value: float, device=None) -> float:
    """MAX all-reduce of a scalar (identity when torch.distributed is not initialised)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank: int, world: int, seconds_max: float) -> float:
    """Aggregate throughput of `world` replicas that each processed `units_per_rank` units."""
    return world * units_per_rank / seconds_max
