"""GPU parity of variable-length and paged KV-cache attention (the shape of the kernel the
paper simulates, attention_with_kvcache_prefill_fp8) against the oracle.  Interface work, no new
numerics: the oracle is run per batch element on that element's own rows and keys, gathered from the pages on the
host; memory past the end of a sequence holds large finite values to show it is masked."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_06521_b200 import workloads as W
import parity as P

pytestmark = pytest.mark.gpu


def build(kind, B, Hq, Hkv, Lq, lens_q, lens_k, page_size, seed, delta=9.0, paged=True):
    """Returns (device q, k, v, scales, block_table, per-batch oracle inputs)."""
    d = 128
    Lk = max(lens_k)
    max_pages = (Lk + page_size - 1) // page_size
    n_pages = B * max_pages + 3
    rng = np.random.default_rng(seed)
    perm = rng.permutation(n_pages)[:B * max_pages].reshape(B, max_pages).astype(np.int32)
    q, k, v = W.sink_qkv(B, Hq, Hkv, Lq, max_pages * page_size, d, delta, seed=seed)
    per_batch, sc = [], {}
    e4 = kind in ("e4m3", "decode")
    np_kv = np.uint8 if e4 else np.uint16
    fill = 0x7E if e4 else 0x7F00            # E4M3 448 / BF16 ~1.7e38: finite, and fatal if it were not masked
    pool_k = np.full((n_pages, Hkv, page_size, d), fill, dtype=np_kv)
    pool_v = np.full_like(pool_k, fill)
    dense_k = np.full((B, Hkv, max_pages * page_size, d), fill, dtype=np_kv)
    dense_v = np.full_like(dense_k, fill)
    qs_all, ks_all, vs_all = [], [], []
    q_dev = np.zeros((B, Hq, Lq, d), dtype=np.uint8 if kind == "e4m3" else np.uint16)
    for b in range(B):
        lq, lk = lens_q[b], lens_k[b]
        qb, kb, vb = q[b:b + 1, :, :lq], k[b:b + 1, :, :lk], v[b:b + 1, :, :lk]
        kw = {}
        if e4:
            kc, ks = oracle.quantize_e4m3(kb)
            vc, vs = oracle.quantize_e4m3(vb)
            kw.update(k_scale=ks, v_scale=vs)
            ks_all.append(ks[0]); vs_all.append(vs[0])
            if kind == "e4m3":
                qc, qs = oracle.quantize_e4m3(qb)
                kw.update(q_scale=qs)
                qs_all.append(qs[0])
                dt = oracle.DT_E4M3
            else:
                qc, dt = W.to_bf16_bits(qb), oracle.DT_BF16Q_E4M3KV
        else:
            qc, kc, vc, dt = W.to_bf16_bits(qb), W.to_bf16_bits(kb), W.to_bf16_bits(vb), oracle.DT_BF16
        q_dev[b, :, :lq] = qc[0]
        dense_k[b, :, :lk], dense_v[b, :, :lk] = kc[0], vc[0]
        for pg in range((lk + page_size - 1) // page_size):
            n = min(page_size, lk - pg * page_size)
            pool_k[perm[b, pg], :, :n] = kc[0, :, pg * page_size:pg * page_size + n]
            pool_v[perm[b, pg], :, :n] = vc[0, :, pg * page_size:pg * page_size + n]
        per_batch.append((qc, kc, vc, dt, kw))
    if e4:
        sc["k_scale"], sc["v_scale"] = np.stack(ks_all), np.stack(vs_all)
        if kind == "e4m3":
            sc["q_scale"] = np.stack(qs_all)
    bf = lambda a: P.to_dev(a, bf16=(a.dtype == np.uint16))
    tk, tv = (bf(pool_k), bf(pool_v)) if paged else (bf(dense_k), bf(dense_v))
    return bf(q_dev), tk, tv, {n: torch.from_numpy(a).to(P.dev()) for n, a in sc.items()}, \
        torch.from_numpy(perm).to(P.dev()), per_batch


def check_batches(r, per_batch, lens_q, Hq, Lq, causal, S, order, mode, bounds_of=None, **okw):
    d = 128
    o = r.o.float().cpu().numpy().astype(np.float64)
    rm, rs = r.row_max.cpu().numpy(), r.row_sum.cpu().numpy().astype(np.float64)
    tot_s = tot_o = 0
    for b, (qc, kc, vc, dt, kw) in enumerate(per_batch):
        lq = lens_q[b]
        nb = (kc.shape[2] + r.block_n - 1) // r.block_n
        sb = bounds_of(nb) if bounds_of else None
        ref = oracle.attention_fwd(qc, kc, vc, causal=causal, S=S, kv_order=order, mode=mode, in_dtype=dt,
                                   block_n=r.block_n, split_bounds=sb, **kw, **okw)
        got = o[b, :, :lq].reshape(-1, d)
        assert P.rel_l2(got, ref.out) <= P.REL_L2[mode], (b, P.rel_l2(got, ref.out))
        fin = np.isfinite(ref.row_max)
        tol = 1e-5 if mode != 2 else 1e-4
        assert np.allclose(rm[b, :, :lq].reshape(-1)[fin], ref.row_max[fin], rtol=tol, atol=tol)
        assert np.allclose(rs[b, :, :lq].reshape(-1), ref.row_sum, rtol=1e-5 if mode != 2 else 1e-3, atol=0)
        # rows past the end of the sequence: 0, -inf, 0
        assert np.all(o[b, :, lq:] == 0) and np.all(np.isneginf(rm[b, :, lq:])) and np.all(rs[b, :, lq:] == 0)
        tot_s, tot_o = tot_s + ref.uf_sink_block, tot_o + ref.uf_other_blocks
    assert np.all(np.isfinite(o))
    return tot_s, tot_o


@pytest.mark.parametrize("kind,mode", [("e4m3", 2), ("bf16", 1)])
@pytest.mark.parametrize("kernel,bn", [(1, 128), (2, 128), (2, 64)])
@pytest.mark.parametrize("paged", [False, True])
@pytest.mark.parametrize("order", [0, 1])
def test_varlen_paged_prefill(kind, mode, kernel, bn, paged, order):
    B, Hq, Hkv, Lq = 3, 4, 2, 300
    lens_q, lens_k = [300, 77, 130], [1000, 517, 130]
    tq, tk, tv, sc, table, per_batch = build(kind, B, Hq, Hkv, Lq, lens_q, lens_k, 256, seed=31, paged=paged)
    f = P.fa()
    kw = dict(seqlens_q=torch.tensor(lens_q, dtype=torch.int32, device=P.dev()),
              seqlens_k=torch.tensor(lens_k, dtype=torch.int32, device=P.dev()))
    if paged:
        kw.update(block_table=table, Lk=max(lens_k))
    r = f.fwd(tq, tk, tv, causal=True, S=256.0, kv_order=order, mode=mode, kernel=kernel, block_n=bn, want_stats=True,
              **sc, **kw)
    torch.cuda.synchronize()
    assert r.kernel_id == kernel and r.block_n == bn
    us, uo = check_batches(r, per_batch, lens_q, Hq, Lq, True, 256.0, order, mode)
    uf = r.underflow.cpu().numpy()
    slack = max(4, int(2e-3 * sum(lq * lk for lq, lk in zip(lens_q, lens_k)) * Hq))
    assert abs(int(uf[0]) - us) <= slack and abs(int(uf[1]) - uo) <= slack, (uf, us, uo)
    if order == 1:
        assert int(uf[1]) == 0 == uo


@pytest.mark.parametrize("ns", [0, 1, 4])
@pytest.mark.parametrize("page_size", [128, 512])
def test_paged_decode(ns, page_size):
    """Decode against a paged E4M3 KV cache with one new token per sequence and a different length per sequence; the
    block ranges of the splits follow each sequence's own block count (s * nb_b / ns)."""
    B, Hq, Hkv = 4, 8, 2
    lens_q, lens_k = [1, 1, 1, 1], [4096, 1000, 129, 2048]
    tq, tk, tv, sc, table, per_batch = build("decode", B, Hq, Hkv, 1, lens_q, lens_k, page_size, seed=33, delta=10.0)
    f = P.fa()
    r = f.fwd(tq, tk, tv, causal=False, S=256.0, kv_order=1, mode=2, num_splits=ns, want_stats=True, block_table=table,
              Lk=max(lens_k), seqlens_k=torch.tensor(lens_k, dtype=torch.int32, device=P.dev()), **sc)
    torch.cuda.synchronize()
    assert r.kernel_id == 3
    n = r.num_splits
    bounds = (lambda nb: [(s * nb) // n for s in range(n + 1)]) if n > 1 else None
    us, uo = check_batches(r, per_batch, lens_q, Hq, 1, False, 256.0, 1, 2, bounds_of=bounds)
    uf = r.underflow.cpu().numpy()
    assert abs(int(uf[0]) - us) <= 16 and int(uf[1]) == 0 == uo


def test_varlen_arguments():
    f = P.fa()
    tq, tk, tv, sc, table, _ = build("e4m3", 2, 2, 2, 128, [128, 64], [256, 256], 128, seed=35)
    with pytest.raises(f.Fp8AttnError) as e:      # a page smaller than the KV block
        f.fwd(tq, tk[:, :, :64].contiguous(), tv[:, :, :64].contiguous(), causal=True, S=256.0, kv_order=1, mode=2,
              block_table=table.repeat(1, 2).contiguous(), Lk=256, **sc)
    assert e.value.code == -5
    with pytest.raises(f.Fp8AttnError) as e:      # the table does not reach Lk
        f.fwd(tq, tk, tv, causal=True, S=256.0, kv_order=1, mode=2, block_table=table, Lk=1000, **sc)
    assert e.value.code == -2


@pytest.mark.parametrize("kernel", [1, 2])
def test_varlen_degenerate_lengths(kernel):
    """Empty sequences, a sequence with more query rows than keys (rows that see nothing), and full-length ones in
    the same call: the degenerate cases of the per-sequence geometry."""
    B, Hq, Hkv, Lq = 4, 2, 1, 260
    lens_q, lens_k = [0, 260, 200, 1], [300, 0, 120, 257]
    lens_k_build = [max(1, x) for x in lens_k]          # the builder needs one key; seqlens_k still says 0
    tq, tk, tv, sc, table, per_batch = build("e4m3", B, Hq, Hkv, Lq, [max(1, x) for x in lens_q], lens_k_build, 128,
                                             seed=41, paged=False)
    f = P.fa()
    r = f.fwd(tq, tk, tv, causal=True, S=256.0, kv_order=1, mode=2, kernel=kernel, want_stats=True,
              seqlens_q=torch.tensor(lens_q, dtype=torch.int32, device=P.dev()),
              seqlens_k=torch.tensor(lens_k, dtype=torch.int32, device=P.dev()), **sc)
    torch.cuda.synchronize()
    assert r.kernel_id == kernel
    o, rm, rs = r.o.cpu().numpy(), r.row_max.cpu().numpy(), r.row_sum.cpu().numpy()
    assert np.all(np.isfinite(o))
    for b in (0, 1):                                    # no query rows / no keys: nothing is computed
        assert np.all(o[b] == 0) and np.all(np.isneginf(rm[b])) and np.all(rs[b] == 0)
    # b = 2: 200 rows against 120 keys, bottom-right aligned: the first 80 rows see nothing
    assert np.all(o[2, :, :80] == 0) and np.all(np.isneginf(rm[2, :, :80]))
    for b in (2, 3):
        qc, kc, vc, dt, kw = per_batch[b]
        lq, lk = lens_q[b], lens_k[b]
        ref = oracle.attention_fwd(qc[:, :, :lq], kc[:, :, :lk], vc[:, :, :lk], causal=True, S=256.0, kv_order=1, mode=2,
                                   in_dtype=dt, block_n=r.block_n, **kw)
        got = o[b, :, :lq].reshape(-1, 128).astype(np.float64)
        assert P.rel_l2(got, ref.out) <= P.REL_L2[2]
        assert np.all(o[b, :, lq:] == 0)
