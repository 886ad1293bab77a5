"""Event sharding for N > 1 GPUs.

(event, sector) tasks are independent through the whole path (sectors are
processed individually; L127: several events concurrently on one GPU), so the path shards
BY EVENT with no data-path collective: every rank tracks its own events, and the only
exchange is a gather of four counters for reporting.
"""
from __future__ import annotations

from typing import List, Sequence


def shard_events(n_events: int, world_size: int, rank: int) -> List[int]:
    """Contiguous block of events for ``rank``; sizes differ by at most one."""
    if world_size < 1 or not (0 <= rank < world_size):
        raise ValueError("need 0 <= rank < world_size")
    base, extra = divmod(n_events, world_size)
    start = rank * base + min(rank, extra)
    return list(range(start, start + base + (1 if rank < extra else 0)))


def merge_counts(per_rank: Sequence[Sequence[int]]) -> List[int]:
    """Element-wise sum of the per-rank (clusters, events, tracks, hits) tuples."""
    return [sum(col) for col in zip(*per_rank)]
