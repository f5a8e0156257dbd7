"""GPU parity of the split-KV decode kernel (kernel family 3, csrc/attn_decode.cuh) against the CPU
oracle run with the same split boundaries (reading R14): outputs, row statistics, and --
through the statistics instance of the kernel (same schedule) -- the E4M3 code of every P element by
element and both underflow counters; and against the general kernel."""
import numpy as np
import pytest
import torch

from paper_2606_06521_b200 import workloads as W
import parity as P

pytestmark = pytest.mark.gpu

SHAPES = [
    # B, Hq, Hkv, Lq, Lk, causal      (d = 128; (Hq/Hkv) * Lq <= 16 query rows per kv head)
    (2, 4, 2, 3, 1000, False),        # 6 rows -> 8-row instance, ragged tail block
    (1, 8, 2, 1, 517, False),         # GQA group of 4, one token
    (1, 16, 1, 1, 2048, False),       # 16 rows: the full N of the MMAs
    (2, 4, 2, 2, 700, True),          # two new tokens, causal: the last key is hidden from the first
    (1, 2, 2, 1, 128, False),         # exactly one block
    (3, 6, 3, 5, 1300, True),         # 10 rows -> 16-row instance
]


@pytest.mark.parametrize("shape", SHAPES)
@pytest.mark.parametrize("kind", ["e4m3", "decode"])
@pytest.mark.parametrize("ns", [0, 1, 3])
@pytest.mark.parametrize("order,S", [(1, 256.0), (0, 448.0)])
def test_decode_kernel_matches_oracle(shape, kind, ns, order, S):
    B, Hq, Hkv, Lq, Lk, causal = shape
    q, k, v = W.sink_qkv(B, Hq, Hkv, Lq, Lk, 128, 10.0, seed=7)
    case = P.make_case(q, k, v, kind)
    r = P.run_gpu(case, causal=causal, S=S, order=order, mode=2, num_splits=ns, kernel=3, underflow=False)
    nb = (Lk + 127) // 128
    assert r.kernel_id == 3 and r.block_n == 128
    assert 1 <= r.num_splits <= nb and r.split_bounds[0] == 0 and r.split_bounds[-1] == nb
    if ns:
        assert r.num_splits == min(ns, nb)
    ref = P.run_oracle(case, r, causal=causal, S=S, order=order, mode=2)
    P.check(case, r, ref, mode=2, label=f"decode {shape} {kind} ns={ns} S={S} order={order}", check_mse=False)
    # the statistics instance of the same kernel: every P code of one head against the oracle's (north_star:
    # >= 99.9 % identical in FP8 mode, never more than one code step apart; Alg. 1 line 9)
    # and both underflow counters over the whole call (Prop. 1)
    b, h = B - 1, Hq - 1
    ra = P.run_gpu(case, causal=causal, S=S, order=order, mode=2, num_splits=r.num_splits, kernel=3, underflow=True,
                   dump_head=(b, h))
    assert ra.kernel_id == 3 and ra.split_bounds == r.split_bounds
    assert torch.equal(ra.o, r.o) and torch.equal(ra.row_max, r.row_max) and torch.equal(ra.row_sum, r.row_sum)
    rows = (b * Hq + h) * Lq + np.arange(Lq)
    refc = P.run_oracle(case, ra, causal=causal, S=S, order=order, mode=2, rows=rows, want_codes=True)
    g = ra.p_codes.cpu().numpy()
    vis = refc.p_codes != 0xFF
    assert np.array_equal(g == 0xFF, ~vis), "mask pattern of the P dump differs"
    n_flip = int(np.sum(g[vis] != refc.p_codes[vis]))
    assert 1.0 - n_flip / max(1, int(vis.sum())) >= P.CODE_MATCH[2]
    assert np.abs(g[vis].astype(np.int32) - refc.p_codes[vis].astype(np.int32)).max(initial=0) <= 1
    uf = ra.underflow.cpu().numpy()
    slack = max(4, int(2e-3 * ref.n_nonsink_visible))
    assert abs(int(uf[0]) - ref.uf_sink_block) <= slack, (uf, ref.uf_sink_block)
    assert abs(int(uf[1]) - ref.uf_other_blocks) <= slack, (uf, ref.uf_other_blocks)
    if order == 1 and S == 256.0 and r.num_splits == 1:
        assert int(uf[1]) == 0 == ref.uf_other_blocks          # Thm 4
    # the general kernel with the same split layout
    g = P.run_gpu(case, causal=causal, S=S, order=order, mode=2, num_splits=r.num_splits, kernel=1)
    assert g.kernel_id == 1 and g.split_bounds == r.split_bounds
    og, od = g.o.cpu().numpy().astype(np.float64), r.o.cpu().numpy().astype(np.float64)
    assert P.rel_l2(od, og) <= 1e-3
    assert torch.allclose(g.row_max, r.row_max, rtol=1e-6, atol=1e-6)
    assert torch.allclose(g.row_sum, r.row_sum, rtol=1e-5, atol=0)


def test_decode_is_the_default_for_decode_shapes():
    q, k, v = W.sink_qkv(2, 8, 2, 1, 4096, 128, 10.0, seed=1)
    case = P.make_case(q, k, v, "decode")
    r = P.run_gpu(case, causal=False, S=256.0, order=1, mode=2, stats=False)
    assert r.kernel_id == 3
    assert r.n_launches == 1 + 1 + (1 if r.num_splits > 1 else 0)     # q quantiser (one fused launch), decode, combine
    r1 = P.run_gpu(case, causal=False, S=256.0, order=1, mode=2, stats=True)         # underflow counters wanted:
    assert r1.kernel_id == 3 and r1.num_splits == r.num_splits                        # the statistics instance
    g = P.run_gpu(case, causal=False, S=256.0, order=1, mode=2, stats=True, kernel=1, num_splits=r.num_splits)
    assert g.kernel_id == 1 and torch.equal(g.underflow, r1.underflow)
    f = P.fa()
    q2, k2, v2 = W.sink_qkv(1, 32, 1, 1, 256, 128, 10.0, seed=1)                     # 32 rows per kv head
    with pytest.raises(f.Fp8AttnError) as e:
        P.run_gpu(P.make_case(q2, k2, v2, "e4m3"), causal=False, S=256.0, order=1, mode=2, kernel=3, stats=False)
    assert e.value.code == -5


def test_decode_split_invariants():
    """row_max and row_sum do not depend on the split layout or the order (pins of the unpinned split path)."""
    q, k, v = W.sink_qkv(1, 8, 2, 1, 4096, 128, 10.0, seed=4)
    case = P.make_case(q, k, v, "decode")
    base = P.run_gpu(case, causal=False, S=256.0, order=1, mode=2, num_splits=1, kernel=3, underflow=False)
    for ns in (2, 5, 16):
        for order in (0, 1):
            r = P.run_gpu(case, causal=False, S=256.0, order=order, mode=2, num_splits=ns, kernel=3, underflow=False)
            assert torch.allclose(r.row_max, base.row_max, rtol=0, atol=1e-6)
            assert torch.allclose(r.row_sum, base.row_sum, rtol=1e-5, atol=0)
