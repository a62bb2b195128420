"""Multi-GPU: batch sharding only.

Every image is independent through all five steps (the stereo pair is a batch of
identically shaped, independent images), so N GPUs = N contiguous slices of the batch dimension,
one process per GPU, and NO data-path collective.  The only exchange is optional: gathering the
fixed-shape padded outputs onto every rank for one consumer.
"""
from __future__ import annotations

import dataclasses
from typing import Callable, Dict, Optional, Tuple

import torch


def shard_range(B: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous slice [lo, hi) of the batch owned by `rank` (sizes differ by at most one)."""
    if world < 1 or not (0 <= rank < world) or B < 0:
        raise ValueError("bad shard arguments")
    q, rem = divmod(B, world)
    lo = rank * q + min(rank, rem)
    return lo, lo + q + (1 if rank < rem else 0)


def _as_dict(res) -> Dict[str, torch.Tensor]:
    """Per-rank result -> {field: tensor with a leading batch dimension}; None fields are dropped.
    Accepts the binding's DKDResult (a dataclass) or a plain dict."""
    if res is None:
        return {}
    if dataclasses.is_dataclass(res):
        d = {f.name: getattr(res, f.name) for f in dataclasses.fields(res)}
    elif isinstance(res, dict):
        d = dict(res)
    else:
        raise TypeError(f"sharded_extract: unsupported result type {type(res).__name__}")
    return {k: v for k, v in d.items() if isinstance(v, torch.Tensor)}


def sharded_extract(extract_fn: Callable, score: torch.Tensor, desc: Optional[torch.Tensor],
                    rank: int, world: int, gather: bool = False, group=None, **kw):
    """Runs `extract_fn(score[lo:hi], desc[lo:hi], **kw)` on this rank's slice and returns its result.

    With gather=True the per-rank outputs are all-gathered and concatenated in rank order into a dict of tensors
    covering the whole batch — the one optional collective.  The outputs are fixed-shape padded tensors
    (PAPER.md:139), so the exchange is a plain tensor all-gather: every rank pads its slice to the largest
    slice (sizes differ by at most one image), gathers in the tensors' own device / dtype (NCCL for CUDA
    tensors, gloo for CPU tensors), and trims.  An empty batch returns an empty dict."""
    B = score.shape[0]
    lo, hi = shard_range(B, rank, world)
    local = extract_fn(score[lo:hi], None if desc is None else desc[lo:hi], **kw) if hi > lo else None
    if not gather:
        return local
    import torch.distributed as dist
    sizes = [shard_range(B, r, world)[1] - shard_range(B, r, world)[0] for r in range(world)]
    if max(sizes) == 0:
        return {}
    mine = _as_dict(local)
    # ranks with an empty slice do not know the output fields: learn names / shapes / dtypes from the first
    # non-empty rank (rank 0 always owns images when the batch is not empty)
    meta = [None]
    if rank == 0:
        meta[0] = [(k, tuple(v.shape[1:]), str(v.dtype).replace("torch.", "")) for k, v in mine.items()]
    dist.broadcast_object_list(meta, src=0, group=group)
    ref_dev = next(iter(mine.values())).device if mine else None
    if ref_dev is None:
        ref_dev = score.device if score.is_cuda else torch.device("cpu")
    out = {}
    nmax = max(sizes)
    for name, tail, dt in meta[0]:
        dtype = getattr(torch, dt)
        buf = torch.zeros((nmax,) + tail, dtype=dtype, device=ref_dev)
        if name in mine:
            buf[: hi - lo] = mine[name]
        parts = [torch.empty_like(buf) for _ in range(world)]
        dist.all_gather(parts, buf, group=group)
        out[name] = torch.cat([p[:n] for p, n in zip(parts, sizes)], 0)
    return out
