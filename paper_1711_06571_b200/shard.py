"""Host-side sharding of the KF path across ranks.

Tracks (fit) and events (build) are independent -- "no correlation between particles", several events
in flight -- so the path shards with NO data-path collective: a rank owns a contiguous track range or a
set of whole events, bins its own events and keeps its results.  The only cross-rank traffic is the timing reduction.
Holds no KF arithmetic.
"""
from __future__ import annotations

import numpy as np


def track_range(n: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous, even split of n tracks: the first n % world ranks get one more.  -> [begin, end)"""
    assert 0 <= rank < world and n >= 0
    base, rem = divmod(n, world)
    begin = rank * base + min(rank, rem)
    return begin, begin + base + (1 if rank < rem else 0)


def assign_events(seed_counts, world: int) -> list[list[int]]:
    """Whole events to ranks, balanced by seed count: events in order of decreasing seed count (ties by index),
    each to the currently lightest rank (ties by rank).  Deterministic, so every rank computes the same table."""
    counts = np.asarray(seed_counts, dtype=np.int64)
    order = sorted(range(len(counts)), key=lambda e: (-int(counts[e]), e))
    load = [0] * world
    out: list[list[int]] = [[] for _ in range(world)]
    for e in order:
        r = min(range(world), key=lambda k: (load[k], k))
        out[r].append(e)
        load[r] += int(counts[e])
    return [sorted(v) for v in out]


def max_over_ranks(value: float, device="cpu") -> float:
    """MAX all-reduce of a scalar over the default process group (identity when torch.distributed is not initialised)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device="cpu") -> float:
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())
