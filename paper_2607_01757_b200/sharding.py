"""Multi-GPU: batch sharding only.

Every image is independent through all five steps (the stereo pair is a batch of
identically shaped, independent images), so N GPUs = N contiguous slices of the batch dimension,
one process per GPU, and NO data-path collective.  The only exchange is optional: gathering the
fixed-shape padded outputs onto every rank for one consumer.
"""
from __future__ import annotations

from typing import Callable, Optional, Tuple

import torch


def shard_range(B: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous slice [lo, hi) of the batch owned by `rank` (sizes differ by at most one)."""
    if world < 1 or not (0 <= rank < world) or B < 0:
        raise ValueError("bad shard arguments")
    q, rem = divmod(B, world)
    lo = rank * q + min(rank, rem)
    return lo, lo + q + (1 if rank < rem else 0)


def sharded_extract(extract_fn: Callable, score: torch.Tensor, desc: Optional[torch.Tensor],
                    rank: int, world: int, gather: bool = False, group=None, **kw):
    """Runs `extract_fn(score[lo:hi], desc[lo:hi], **kw)` on this rank's slice.  With gather=True the
    per-rank outputs (dict of tensors with a leading batch dimension) are all-gathered and
    concatenated in rank order — the one optional collective."""
    lo, hi = shard_range(score.shape[0], rank, world)
    local = extract_fn(score[lo:hi], None if desc is None else desc[lo:hi], **kw) if hi > lo else None
    if not gather:
        return local
    import torch.distributed as dist
    parts = [None] * world
    dist.all_gather_object(parts, local, group=group)
    parts = [p for p in parts if p is not None]
    return {k: torch.cat([p[k] for p in parts], 0) for k in parts[0]}
