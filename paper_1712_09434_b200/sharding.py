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


def gather_counts(mine: Sequence[int]) -> List[int]:
    """Sum of the per-rank counters over the default process group (the ONLY exchange on the N > 1
    path; reporting, not data).  Works on gloo (CPU tensors) and nccl (tensors on the current device)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [int(v) for v in mine]
    dev = torch.device("cuda", torch.cuda.current_device()) if dist.get_backend() == "nccl" else torch.device("cpu")
    mine_t = torch.tensor([int(v) for v in mine], dtype=torch.int64, device=dev)
    parts = [torch.zeros_like(mine_t) for _ in range(dist.get_world_size())]
    dist.all_gather(parts, mine_t)
    return merge_counts([p.cpu().tolist() for p in parts])
