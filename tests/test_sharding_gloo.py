"""N>1 path on CPU: world_size-2 gloo.  The batch shards across ranks with NO data-path collective
(DESIGN.md "Multi-GPU"); the optional output all-gather reassembles the unsharded result.  The
per-rank extractor here is the oracle (test infrastructure) standing in for the CUDA call."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2607_01757_b200.sharding import shard_range, sharded_extract


def test_shard_range_partitions_the_batch():
    for B in (0, 1, 2, 5, 64):
        for world in (1, 2, 3, 8):
            spans = [shard_range(B, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == B
            assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
            sizes = [hi - lo for lo, hi in spans]
            assert max(sizes) - min(sizes) <= 1


def _oracle_fn(score, desc, **kw):
    import oracle
    R = oracle.extract(score.numpy(), None if desc is None else desc.numpy(), **kw)
    return {"kpts": torch.from_numpy(R.kpts), "scores": torch.from_numpy(R.scores),
            "count": torch.from_numpy(R.count), "index": torch.from_numpy(R.index),
            "desc": torch.from_numpy(R.desc)}


def _dataclass_fn(score, desc, **kw):
    """Returns the binding's own result type (DKDResult), as DKD.extract does; `desc`/`offsets` may be None."""
    from paper_2607_01757_b200.binding import DKDResult
    d = _oracle_fn(score, desc, **kw)
    return DKDResult(kpts=d["kpts"].float(), scores=d["scores"], desc=None, count=d["count"], index=d["index"],
                     offsets=None)


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import synth
    score = synth.score_maps(5, 48, 64, 3, 0.1, 40)
    desc = synth.desc_maps(5, 48, 64, 16, 3, torch.float16)
    kw = dict(stride=1, r=2, thresh=0.2, top_k=32, T=0.1)
    got = sharded_extract(_oracle_fn, score, desc, rank, world, gather=True, **kw)
    # timing reduction used by bench.py: max over ranks
    t = torch.tensor([1.0 + rank], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    # the real return type (a dataclass with None fields), a batch smaller than the world, an empty batch
    got_dc = sharded_extract(_dataclass_fn, score, desc, rank, world, gather=True, **kw)
    got_one = sharded_extract(_dataclass_fn, score[:1], desc[:1], rank, world, gather=True, **kw)
    got_none = sharded_extract(_dataclass_fn, score[:0], desc[:0], rank, world, gather=True, **kw)
    local = sharded_extract(_dataclass_fn, score, desc, rank, world, gather=False, **kw)
    if rank == 0:
        want = _oracle_fn(score, desc, **kw)
        ok = all(torch.equal(got[k], want[k]) for k in want) and float(t) == float(world)
        ok = ok and sorted(got_dc) == ["count", "index", "kpts", "scores"]
        ok = ok and torch.equal(got_dc["index"], want["index"]) and torch.equal(got_dc["kpts"], want["kpts"].float())
        ok = ok and got_one["index"].shape[0] == 1 and torch.equal(got_one["index"][0], want["index"][0])
        ok = ok and got_none == {} and local.index.shape[0] == 3   # rank 0 owns 3 of the 5 images
        q.put(bool(ok))
    dist.barrier()
    dist.destroy_process_group()


def test_world_size_2_sharded_equals_unsharded():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    ok = q.get(timeout=180)
    for p in procs:
        p.join(60)
    assert ok and all(p.exitcode == 0 for p in procs)
