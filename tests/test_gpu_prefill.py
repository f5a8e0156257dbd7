"""GPU parity of the warp-specialised prefill kernel (kernel family 2, csrc/attn_prefill.cuh)
against the CPU oracle on the same seeded inputs, and against the general kernel (family 1), which
carries the P-code dump: the two CUDA kernels implement the same Alg. 1 with the
same block size, so their outputs differ only through last-ulp effects."""
import numpy as np
import pytest
import torch

from paper_2606_06521_b200 import workloads as W
import parity as P

pytestmark = pytest.mark.gpu

SHAPES = [
    # B, Hq, Hkv, Lq, Lk, causal        (d = 128: the only head size of this kernel)
    (2, 4, 2, 130, 130, True),          # two tiles in one pair, the second nearly empty
    (1, 2, 2, 77, 300, True),           # Lq < Lk, bottom-right aligned, diagonal not block aligned
    (1, 1, 1, 300, 100, True),          # Lq > Lk: the first 200 rows see no key; second pair ragged
    (1, 2, 1, 600, 1000, False),        # three pairs, tail block of 104 keys
    (1, 2, 2, 512, 512, True),          # aligned causal
    (1, 3, 1, 1, 517, False),           # one query row (forced onto this kernel)
    (1, 2, 1, 257, 700, True),          # second pair has one row
    (1, 1, 1, 1280, 1280, True),        # ring wrap-around: 10 blocks > NS
    (1, 2, 1, 384, 1700, True),         # Lk - Lq not a multiple of the block: two partly masked blocks per tile
]


@pytest.mark.parametrize("shape", SHAPES)
@pytest.mark.parametrize("kind,mode", [("bf16", 1), ("e4m3", 2)])
@pytest.mark.parametrize("order,S", [(0, 16.0), (1, 256.0), (1, 448.0), (0, 1.0)])
@pytest.mark.parametrize("bn", [128, 64])
def test_prefill_kernel_matches_oracle(shape, kind, mode, order, S, bn):
    B, Hq, Hkv, Lq, Lk, causal = shape
    q, k, v = W.sink_qkv(B, Hq, Hkv, Lq, Lk, 128, 6.0, seed=5)
    case = P.make_case(q, k, v, kind)
    r = P.run_gpu(case, causal=causal, S=S, order=order, mode=mode, block_n=bn, num_splits=1, kernel=2,
                  underflow=False)
    assert r.kernel_id == 2 and r.block_n == bn and r.num_splits == 1
    ref = P.run_oracle(case, r, causal=causal, S=S, order=order, mode=mode)
    P.check(case, r, ref, mode=mode, label=f"prefill {shape} {kind} S={S} order={order}",
            check_mse=(Lq * Lk > 20000))
    if causal and Lq > Lk:
        o = r.o.cpu().numpy()
        assert np.all(o[:, :, :Lq - Lk] == 0)
        assert np.all(np.isneginf(r.row_max.cpu().numpy()[:, :, :Lq - Lk]))
        assert np.all(r.row_sum.cpu().numpy()[:, :, :Lq - Lk] == 0)
    # the general kernel on the same call: same semantics, same Bn
    g = P.run_gpu(case, causal=causal, S=S, order=order, mode=mode, block_n=bn, num_splits=1, kernel=1)
    assert g.kernel_id == 1
    og, op = g.o.cpu().numpy().astype(np.float64), r.o.cpu().numpy().astype(np.float64)
    assert P.rel_l2(op, og) <= (2e-4 if mode == 1 else 1e-3)
    assert torch.equal(torch.isfinite(g.row_max), torch.isfinite(r.row_max))
    fin = torch.isfinite(g.row_max)
    assert torch.allclose(g.row_max[fin], r.row_max[fin], rtol=1e-6, atol=1e-6)
    assert torch.allclose(g.row_sum, r.row_sum, rtol=2e-6, atol=0)


@pytest.mark.parametrize("shape", [(1, 2, 1, 600, 1000, False), (2, 4, 2, 130, 130, True), (1, 2, 1, 384, 1700, True),
                                   (1, 1, 1, 1280, 1280, True)])
@pytest.mark.parametrize("kind,mode", [("bf16", 1), ("e4m3", 2)])
@pytest.mark.parametrize("order,S", [(1, 256.0), (0, 1.0), (0, 448.0)])
@pytest.mark.parametrize("bn", [128, 64])
def test_prefill_kernel_p_codes_match_oracle(shape, kind, mode, order, S, bn):
    """The E4M3 code of every visible P of one head and the underflow counters, written by the throughput kernel
    itself (its statistics instance: same schedule, FMA-pipe exp2 share included; Bn = 128 and Bn = 64 kernels), against
    the oracle's:
    identical for >= 99.99 % (isolation) / 99.9 % (FP8 mode) of the visible elements and never more than one
    code step apart (north_star)."""
    B, Hq, Hkv, Lq, Lk, causal = shape
    q, k, v = W.sink_qkv(B, Hq, Hkv, Lq, Lk, 128, 7.0, seed=9)
    case = P.make_case(q, k, v, kind)
    b, h = B - 1, Hq - 1
    r = P.run_gpu(case, causal=causal, S=S, order=order, mode=mode, block_n=bn, num_splits=1, kernel=2,
                  underflow=True, dump_head=(b, h))
    assert r.kernel_id == 2 and r.p_codes is not None and r.underflow is not None
    # output, row statistics and the two underflow counters (Prop. 1) of the whole call
    P.check(case, r, P.run_oracle(case, r, causal=causal, S=S, order=order, mode=mode), mode=mode,
            label=f"prefill statistics instance {shape} {kind} S={S} order={order}", check_mse=False)
    rows = (b * Hq + h) * Lq + np.arange(Lq)
    ref = P.run_oracle(case, r, causal=causal, S=S, order=order, mode=mode, rows=rows, want_codes=True)
    g = r.p_codes.cpu().numpy()
    vis = ref.p_codes != 0xFF
    assert np.array_equal(g == 0xFF, ~vis), "mask pattern of the P dump differs"
    match = float(np.mean(g[vis] == ref.p_codes[vis]))
    assert match >= P.CODE_MATCH[mode], match
    step = np.abs(g[vis].astype(np.int32) - ref.p_codes[vis].astype(np.int32))
    assert step.max(initial=0) <= 1
    # the dump instance and the plain instance compute the same output
    r0 = P.run_gpu(case, causal=causal, S=S, order=order, mode=mode, block_n=bn, num_splits=1, kernel=2,
                   underflow=False)
    assert torch.equal(r0.o, r.o)


def test_prefill_is_the_default_for_prefill_shapes():
    q, k, v = W.sink_qkv(1, 2, 2, 256, 256, 128, 7.0, seed=1)
    case = P.make_case(q, k, v, "e4m3")
    r = P.run_gpu(case, causal=True, S=256.0, order=1, mode=2, stats=False)
    assert r.kernel_id == 2 and r.n_launches == 1
    r = P.run_gpu(case, causal=True, S=256.0, order=1, mode=2, stats=True)      # underflow counters wanted
    assert r.kernel_id == 1                                                      # automatic: general kernel
    r2 = P.run_gpu(case, causal=True, S=256.0, order=1, mode=2, stats=True, kernel=2)   # on request: this kernel
    assert r2.kernel_id == 2 and torch.equal(r2.underflow, r.underflow)
    f = P.fa()
    with pytest.raises(f.Fp8AttnError) as e:                                     # FP32 inputs: not this kernel
        P.run_gpu(P.make_case(q, k, v, "f32"), causal=True, S=256.0, order=1, mode=1, kernel=2, stats=False)
    assert e.value.code == -5


@pytest.mark.parametrize("kind,mode", [("bf16", 1), ("e4m3", 2)])
def test_prefill_subnormal_codes_and_saturation(kind, mode):
    """S = 1 forward puts most non-sink P values in the E4M3 subnormal range or at zero, S = 512 saturates
    the row maximum at 448 (reading R22): both ends of the code table go through P.V."""
    q, k, v = W.sink_qkv(1, 2, 2, 384, 384, 128, 5.0, seed=3)
    case = P.make_case(q, k, v, kind)
    for S in (1.0, 512.0):
        r = P.run_gpu(case, causal=False, S=S, order=0, mode=mode, block_n=128, num_splits=1, kernel=2,
                  underflow=False)
        ref = P.run_oracle(case, r, causal=False, S=S, order=0, mode=mode)
        P.check(case, r, ref, mode=mode, label=f"prefill S={S}")
