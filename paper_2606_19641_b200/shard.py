"""World sharding and cross-rank timing reduction for multi-GPU runs (host logic only).

The render path has no exchange step ("rendering is local to each rank and requires no inter-rank
communication"): ranks own disjoint world ranges and never communicate on the data
path.  torch.distributed is used only for the timing barrier and the max-over-ranks reduction, so
these helpers work on any backend (NCCL on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations


def weak_world_range(rank: int, worlds_per_rank: int):
    """Weak scaling: every rank renders `worlds_per_rank` worlds with rank-disjoint global world ids."""
    if rank < 0 or worlds_per_rank < 1:
        raise ValueError("bad rank / worlds_per_rank")
    return rank * worlds_per_rank, worlds_per_rank


def strong_world_range(rank: int, world_size: int, n_worlds: int):
    """Strong scaling: contiguous, balanced partition of [0, n_worlds) (first ranks take the remainder)."""
    if not (0 <= rank < world_size) or n_worlds < 0:
        raise ValueError("bad rank / world_size / n_worlds")
    base, rem = divmod(n_worlds, world_size)
    begin = rank * base + min(rank, rem)
    return begin, base + (1 if rank < rem else 0)


def max_over_ranks(value: float, device=None) -> float:
    """Max of a per-rank scalar (device time of the timed region); identity without a process group."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(units_per_rank: int, steps: int, ms_per_rank: float, device=None) -> float:
    """Whole-job units/s: all ranks' units divided by the slowest rank's time."""
    import torch.distributed as dist
    n = dist.get_world_size() if (dist.is_available() and dist.is_initialized()) else 1
    ms = max_over_ranks(ms_per_rank, device)
    return n * units_per_rank * steps / (ms * 1e-3)
