"""Host logic of the multi-GPU path: the (batch, kv head) partition, checked on one
process and on a world_size-2 `gloo` group on CPU.  The per-shard computation is stood in for by the CPU
oracle (this is a test: the product path has no CPU fallback): every rank computes only its own units, no
collective moves attention data, and the union of the shards equals the unsharded result."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
from paper_2606_06521_b200 import sharding as S
from paper_2606_06521_b200 import workloads as W


@pytest.mark.parametrize("B,Hq,Hkv,world", [(4, 32, 32, 8), (2, 64, 8, 8), (64, 32, 8, 8), (1, 4, 2, 3), (3, 6, 3, 2),
                                            (1, 2, 1, 4)])
def test_partition_covers_every_unit_once(B, Hq, Hkv, world):
    g = Hq // Hkv
    seen = np.zeros((B, Hkv), dtype=np.int32)
    sizes = []
    for r in range(world):
        sh = S.shard(r, world, B, Hq, Hkv)
        sizes.append(sh.hi - sh.lo)
        assert sum(p.kvh_hi - p.kvh_lo for p in sh.pieces) == sh.hi - sh.lo
        for p in sh.pieces:
            assert 0 <= p.kvh_lo < p.kvh_hi <= Hkv and (p.hq_lo, p.hq_hi) == (p.kvh_lo * g, p.kvh_hi * g)
            seen[p.b, p.kvh_lo:p.kvh_hi] += 1
    assert np.all(seen == 1)
    assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)


def test_unit_range_rejects_bad_ranks():
    with pytest.raises(ValueError):
        S.unit_range(2, 2, 10)
    with pytest.raises(ValueError):
        S.shard(0, 1, 1, 3, 2)


def _oracle_fwd(q, k, v, out, **kw):
    r = oracle.attention_fwd(np.ascontiguousarray(q), np.ascontiguousarray(k), np.ascontiguousarray(v), causal=True,
                             S=256.0, kv_order=1, mode=1, block_n=64, **kw)
    out[...] = r.out.reshape(out.shape)
    return r.uf_sink_block + r.uf_other_blocks


def _worker(rank, world, port, q, k, v, ret):
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        o = np.zeros(q.shape, dtype=np.float64)
        S.run_sharded(_oracle_fwd, q, k, v, o, rank, world)
        sh = S.shard(rank, world, q.shape[0], q.shape[1], k.shape[1])
        # the only communication of the path: barrier + max over ranks of the timing (bench.py)
        dist.barrier()
        t = torch.tensor([float(rank + 1)], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        assert t.item() == float(world)
        # test-only gather, to compare with the unsharded result on rank 0
        pieces = [None] * world
        dist.all_gather_object(pieces, (sh.lo, sh.hi, o))
        if rank == 0:
            ret.put(pieces)
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_union_equals_unsharded():
    B, Hq, Hkv, L, d = 3, 4, 2, 96, 64
    q, k, v = W.sink_qkv(B, Hq, Hkv, L, L, d, 6.0, seed=11)
    full = np.zeros(q.shape, dtype=np.float64)
    _oracle_fwd(q, k, v, full)
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    ret = ctx.SimpleQueue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q, k, v, ret)) for r in range(2)]
    for p in procs:
        p.start()
    pieces = ret.get()
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    g = Hq // Hkv
    merged = np.zeros_like(full).reshape(B * Hkv, g, L, d)
    covered = np.zeros(B * Hkv, dtype=np.int32)
    for lo, hi, o in pieces:
        o = o.reshape(B * Hkv, g, L, d)
        merged[lo:hi] = o[lo:hi]
        covered[lo:hi] += 1
        outside = np.ones(B * Hkv, dtype=bool)
        outside[lo:hi] = False
        assert np.all(o[outside] == 0)               # a rank never wrote another rank's rows
    assert np.all(covered == 1)
    assert np.array_equal(merged.reshape(full.shape), full)
