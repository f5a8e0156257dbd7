"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on
the same seeded inputs.  Small and medium shapes that span several tiles and ragged tails;
the full BASELINE sizes are in test_gpu_fullsize.py."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_06521_b200 import workloads as W
import parity as P

pytestmark = pytest.mark.gpu


# ------------------------------------------------------------------ primitives
@pytest.mark.parametrize("eb", [2, 1])
@pytest.mark.parametrize("a_in_tmem", [False, True])
@pytest.mark.parametrize("b_mn_major", [False, True])
@pytest.mark.parametrize("N", [64, 128])
def test_tcgen05_tile_gemm_matches_fp64(eb, a_in_tmem, b_mn_major, N):
    """The TMA / smem-descriptor / TMEM-operand helpers the attention kernels use give the exact
    product (inputs chosen so that FP32 accumulation is exact)."""
    f = P.fa()
    rng = np.random.default_rng(3)
    K = 256
    if b_mn_major and N < 128 // eb:
        pytest.skip("an MN-major B tile is at least one 128-byte run wide")
    if eb == 2:
        A = rng.integers(-8, 9, size=(128, K)).astype(np.float32)
        Bm = rng.integers(-8, 9, size=(N, K)).astype(np.float32)
        tA = torch.from_numpy(A).to(P.dev()).to(torch.bfloat16)
        tB = torch.from_numpy(Bm.T.copy() if b_mn_major else Bm).to(P.dev()).to(torch.bfloat16).contiguous()
    else:
        tab = np.concatenate([[0.0], oracle.e4m3_table()])
        ca = rng.integers(0, 0x40, size=(128, K)).astype(np.uint8) | (rng.integers(0, 2, size=(128, K)) << 7).astype(np.uint8)
        cb = rng.integers(0, 0x40, size=(N, K)).astype(np.uint8) | (rng.integers(0, 2, size=(N, K)) << 7).astype(np.uint8)
        A = np.where(ca & 0x80, -1.0, 1.0) * tab[ca & 0x7F]
        Bm = np.where(cb & 0x80, -1.0, 1.0) * tab[cb & 0x7F]
        tA = torch.from_numpy(ca).to(P.dev())
        tB = torch.from_numpy(cb.T.copy() if b_mn_major else cb).to(P.dev()).contiguous()
    D = f.debug_gemm(tA, tB, a_in_tmem, b_mn_major)
    torch.cuda.synchronize()
    ref = A.astype(np.float64) @ Bm.astype(np.float64).T
    got = D.cpu().numpy().astype(np.float64)
    assert np.allclose(got, ref, rtol=1e-5, atol=1e-5 * np.abs(ref).max())


def test_quantize_e4m3_bit_exact():
    """fp8attn_quantize_e4m3 == the oracle's per-(b,h) absmax/448 helper, code for code."""
    f = P.fa()
    rng = np.random.default_rng(11)
    x = rng.standard_normal((2, 3, 77, 128), dtype=np.float32) * 3.0
    x[0, 1] = 0.0                      # an all-zero slab: scale 1, codes 0
    x[1, 2, 5, 7] = -123.456           # absmax element is negative
    codes, scale = f.quantize_e4m3(torch.from_numpy(x).to(P.dev()))
    torch.cuda.synchronize()
    rc, rs = oracle.quantize_e4m3(x)
    assert np.array_equal(scale.cpu().numpy(), rs)
    assert np.array_equal(codes.cpu().numpy(), rc)
    assert codes.cpu().numpy()[1, 2, 5, 7] == 0xFE      # -448


# ------------------------------------------------------------------ BASELINE config 1
@pytest.mark.parametrize("S", [1.0, 256.0])
@pytest.mark.parametrize("order", [0, 1])
def test_cfg1_isolation(S, order):
    cfg = W.CONFIGS["cfg1"]
    q, k, v = W.config_qkv(cfg, seed=0)
    case = P.make_case(q, k, v, "f32")
    r = P.run_gpu(case, causal=False, S=S, order=order, mode=1, block_n=64, dump_head=(0, 0))
    assert r.block_n == 64 and r.num_splits == 1
    ref = P.run_oracle(case, r, causal=False, S=S, order=order, mode=1, want_codes=True)
    res = P.check(case, r, ref, mode=1, label=f"cfg1 S={S} order={order}")
    if order == 1 and S == 256.0:
        # Thm 4: reverse + S=256 -> no underflow outside the sink block
        assert res["underflow"][1] == 0 == ref.uf_other_blocks


@pytest.mark.parametrize("order", [0, 1])
def test_cfg1_nocast_is_softmax_attention(order):
    cfg = W.CONFIGS["cfg1"]
    q, k, v = W.config_qkv(cfg, seed=0)
    case = P.make_case(q, k, v, "f32")
    r = P.run_gpu(case, causal=False, S=256.0, order=order, mode=0, block_n=64)
    ref = P.run_oracle(case, r, causal=False, S=256.0, order=order, mode=0)
    P.check(case, r, ref, mode=0, label="cfg1 nocast")
    o = r.o.cpu().numpy().reshape(-1, cfg.d).astype(np.float64)
    assert P.rel_l2(o, ref.ref) <= 1e-5       # the plain definition


# ------------------------------------------------------------------ ragged shapes, masks, GQA
SHAPES = [
    # B, Hq, Hkv, Lq, Lk, d, causal
    (1, 2, 1, 200, 333, 64, False),
    (2, 4, 2, 130, 130, 128, True),
    (1, 2, 2, 77, 300, 128, True),      # Lq < Lk, bottom-right aligned
    (1, 1, 1, 300, 100, 64, True),      # Lq > Lk: the first 200 rows see no key
    (1, 3, 1, 1, 517, 128, False),      # one query row
    (1, 1, 1, 128, 64, 64, False),      # exactly one tile, one block
]


@pytest.mark.parametrize("shape", SHAPES)
@pytest.mark.parametrize("kind,mode", [("f32", 1), ("bf16", 1), ("f32", 0), ("bf16", 0), ("e4m3", 2)])
@pytest.mark.parametrize("order", [0, 1])
def test_ragged_shapes(shape, kind, mode, order):
    B, Hq, Hkv, Lq, Lk, d, causal = shape
    if kind == "e4m3" and d != 128:
        pytest.skip("E4M3 inputs are built for d=128")
    q, k, v = W.sink_qkv(B, Hq, Hkv, Lq, Lk, d, 6.0, seed=5)
    case = P.make_case(q, k, v, kind)
    bn = 64 if kind == "f32" else (64 if order == 0 else 128)
    S = 256.0 if order else 16.0
    r = P.run_gpu(case, causal=causal, S=S, order=order, mode=mode, block_n=bn, dump_head=(B - 1, Hq - 1))
    ref = P.run_oracle(case, r, causal=causal, S=S, order=order, mode=mode)
    P.check(case, r, ref, mode=mode, label=f"{shape} {kind} mode{mode}", check_mse=(Lq * Lk > 20000))
    if mode != 0:
        rows = ((B - 1) * Hq + Hq - 1) * Lq + np.arange(Lq)
        refh = P.run_oracle(case, r, causal=causal, S=S, order=order, mode=mode, rows=rows, want_codes=True)
        g = r.p_codes.cpu().numpy()
        vis = refh.p_codes != 0xFF
        assert np.array_equal(g == 0xFF, ~vis)
        match = float(np.mean(g[vis] == refh.p_codes[vis])) if vis.any() else 1.0
        assert match >= P.CODE_MATCH[mode], match
    # rows that see no key: zeros, row_max -inf, row_sum 0
    if causal and Lq > Lk:
        o = r.o.cpu().numpy()
        assert np.all(o[:, :, :Lq - Lk] == 0)
        assert np.all(np.isneginf(r.row_max.cpu().numpy()[:, :, :Lq - Lk]))
        assert np.all(r.row_sum.cpu().numpy()[:, :, :Lq - Lk] == 0)


# ------------------------------------------------------------------ S values incl. saturation
@pytest.mark.parametrize("S", [1.0, 16.0, 448.0, 512.0, 3.0])
def test_scale_values(S):
    """448 (not a power of two: double rounding of fl32(p*S)) and 512 (satfinite at 448, reading R22)."""
    q, k, v = W.sink_qkv(1, 2, 2, 256, 256, 128, 9.0, seed=2)
    case = P.make_case(q, k, v, "f32")
    r = P.run_gpu(case, causal=False, S=S, order=0, mode=1, block_n=64, dump_head=(0, 1))
    ref = P.run_oracle(case, r, causal=False, S=S, order=0, mode=1)
    P.check(case, r, ref, mode=1, label=f"S={S}")
    rows = 256 + np.arange(256)
    refh = P.run_oracle(case, r, causal=False, S=S, order=0, mode=1, rows=rows, want_codes=True)
    g = r.p_codes.cpu().numpy()
    assert float(np.mean(g == refh.p_codes)) >= 0.9999
    if S == 512.0:
        assert g.max() == 0x7E           # the row maximum p=1 saturates at 448


# ------------------------------------------------------------------ split-KV + combine
@pytest.mark.parametrize("kind,mode", [("f32", 1), ("e4m3", 2), ("decode", 2), ("bf16", 1)])
@pytest.mark.parametrize("ns", [1, 2, 3, 8])
@pytest.mark.parametrize("order", [0, 1])
def test_split_kv_matches_oracle(kind, mode, ns, order):
    B, Hq, Hkv, Lq, Lk, d = 2, 4, 2, 3, 1000, 128
    q, k, v = W.sink_qkv(B, Hq, Hkv, Lq, Lk, d, 10.0, seed=9)
    case = P.make_case(q, k, v, kind)
    bn = 64 if kind == "f32" else 128
    r = P.run_gpu(case, causal=False, S=256.0, order=order, mode=mode, block_n=bn, num_splits=ns)
    nb = (Lk + bn - 1) // bn
    assert r.num_splits == min(ns, nb) and r.split_bounds[0] == 0 and r.split_bounds[-1] == nb
    ref = P.run_oracle(case, r, causal=False, S=256.0, order=order, mode=mode)
    P.check(case, r, ref, mode=mode, label=f"split ns={ns} {kind}", check_mse=False)


def test_split_invariants():
    """What is unique regardless of the split layout (pins for the unpinned
    split-KV path): mode-0 output, row_max and row_sum."""
    B, Hq, Hkv, Lq, Lk, d = 1, 4, 1, 2, 2048, 128
    q, k, v = W.sink_qkv(B, Hq, Hkv, Lq, Lk, d, 10.0, seed=4)
    case = P.make_case(q, k, v, "bf16")
    base = P.run_gpu(case, causal=False, S=256.0, order=1, mode=0, block_n=128, num_splits=1)
    for ns in (2, 5, 16):
        for order in (0, 1):
            r = P.run_gpu(case, causal=False, S=256.0, order=order, mode=0, block_n=128, num_splits=ns)
            assert torch.allclose(r.o, base.o, rtol=1e-5, atol=1e-6)
            assert torch.allclose(r.row_max, base.row_max, rtol=0, atol=1e-6)
            assert torch.allclose(r.row_sum, base.row_sum, rtol=1e-5, atol=0)
            r1 = P.run_gpu(case, causal=False, S=256.0, order=order, mode=1, block_n=128, num_splits=ns)
            assert torch.allclose(r1.row_max, base.row_max, rtol=0, atol=1e-6)
            assert torch.allclose(r1.row_sum, base.row_sum, rtol=1e-5, atol=0)


# ------------------------------------------------------------------ host-buffer entry point
def test_fwd_host_equals_fwd():
    f = P.fa()
    q, k, v = W.sink_qkv(1, 4, 2, 200, 264, 128, 7.0, seed=8)
    case = P.make_case(q, k, v, "e4m3")
    r = P.run_gpu(case, causal=True, S=256.0, order=1, mode=2)
    sc = {n: torch.from_numpy(a) for n, a in case.scales.items()}
    pin = lambda a: torch.from_numpy(a).pin_memory()
    rh = f.fwd_host(pin(case.q), pin(case.k), pin(case.v), causal=True, S=256.0, kv_order=1, mode=2,
                    want_stats=True, **sc)
    assert not rh.o.is_cuda
    assert torch.equal(rh.o, r.o.cpu())
    assert torch.equal(rh.row_max, r.row_max.cpu()) and torch.equal(rh.row_sum, r.row_sum.cpu())
    assert torch.equal(rh.underflow, r.underflow.cpu())


@pytest.mark.parametrize("shape", [(2, 8, 2, 4096, 4096), (12, 2, 1, 2048, 2048)])
def test_fwd_host_pipelined_pieces_equal_fwd(shape):
    """Calls above 32 MB of host traffic are cut into (batch, kv-head group) pieces whose copies and kernels
    overlap (csrc/fp8attn.cu, fp8attn_fwd_host): 2 x 2 pieces for the first shape, 8 batch ranges for the second.
    The pieces are independent, so the result equals the one-call result bit for bit."""
    f = P.fa()
    B, Hq, Hkv, Lq, Lk = shape
    q, k, v = W.sink_qkv(B, Hq, Hkv, Lq, Lk, 128, 7.0, seed=11)
    case = P.make_case(q, k, v, "e4m3")
    r = P.run_gpu(case, causal=True, S=256.0, order=1, mode=2, underflow=False)
    assert r.kernel_id == 2
    sc = {n: torch.from_numpy(a) for n, a in case.scales.items()}
    pin = lambda a: torch.from_numpy(a).pin_memory()
    rh = f.fwd_host(pin(case.q), pin(case.k), pin(case.v), causal=True, S=256.0, kv_order=1, mode=2,
                    want_stats=True, want_underflow=False, **sc)
    assert rh.kernel_id == 2 and rh.n_launches > 1
    assert torch.equal(rh.o, r.o.cpu())
    assert torch.equal(rh.row_max, r.row_max.cpu()) and torch.equal(rh.row_sum, r.row_sum.cpu())
