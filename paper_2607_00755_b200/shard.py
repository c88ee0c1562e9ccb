"""Host-side sharding of a batch of distributions over ranks (one process per GPU).

The path partitions over B: every member f[b, :] is an independent problem (SURVEY.md section 8(e)
"parametric scans feasible on a single GPU").  Rank r of W therefore evaluates its own members with its own handle
and no data-path collective; the only exchange is the timing reduction (max over ranks) of bench.py.  Nothing here
touches the arithmetic of the method.
"""
from __future__ import annotations

import numpy as np


def member_range(n_members: int, rank: int, world: int) -> range:
    """Contiguous, balanced slice of `n_members` global members owned by `rank` (strong split of a fixed batch)."""
    if not (0 <= rank < world) or n_members < 0:
        raise ValueError("need 0 <= rank < world and n_members >= 0")
    base, rem = divmod(n_members, world)
    lo = rank * base + min(rank, rem)
    return range(lo, lo + base + (1 if rank < rem else 0))


def weak_member_ids(batch_per_rank: int, rank: int, world: int) -> np.ndarray:
    """Global member ids of rank `rank` when every rank evaluates `batch_per_rank` members (weak scaling):
    rank r owns r*B .. r*B+B-1, so the union over ranks is 0 .. W*B-1 without overlap."""
    if not (0 <= rank < world):
        raise ValueError("need 0 <= rank < world")
    return rank * batch_per_rank + np.arange(batch_per_rank, dtype=np.int64)


def max_over_ranks(values, dist=None, device=None):
    """Element-wise maximum of a list of floats over all ranks (`dist` = torch.distributed or None for one process).
    The tensor lives on `device` (a CUDA device for NCCL, None/CPU for gloo)."""
    import torch
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.cpu()]


def aggregate_rate(units_per_rank_per_step: int, world: int, steps: int, seconds_max_over_ranks: float) -> float:
    """Whole-job throughput: the units all ranks processed divided by the slowest rank's time."""
    return world * units_per_rank_per_step * steps / seconds_max_over_ranks
