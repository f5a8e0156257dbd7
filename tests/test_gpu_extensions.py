"""GPU parity of the SURVEY.md 8(f) extensions against the oracle: the dynamic per-(row, block) power-of-two P scale
(reading R26), sink keys at arbitrary positions with the sink-blocks-last order (reading
R27), and the BF16 output option (the output format of the kernel the paper simulates)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_06521_b200 import workloads as W
import parity as P

pytestmark = pytest.mark.gpu


def _compare(case, r, ref, refc, mode, bn, label, dynamic, rows_codes=None, uf_exact_slack=None):
    P.check(case, r, ref, mode=mode, label=label, check_uf=False)
    if r.p_codes is not None:
        g = r.p_codes.cpu().numpy()
        _, n_flip, n_kflip = P.check_codes(g, refc.p_codes, mode, bn, exponent_flips=dynamic, label=label)
    else:
        n_flip = n_kflip = 0
    if r.underflow is not None:
        uf = r.underflow.cpu().numpy()
        slack = max(4, int((2e-4 if mode == 1 else 2e-3) * ref.n_nonsink_visible)) + 128 * n_kflip
        assert abs(int(uf[0]) - ref.uf_sink_block) <= slack, f"{label}: sink-block underflow {uf} vs {ref.uf_sink_block}"
        assert abs(int(uf[1]) - ref.uf_other_blocks) <= slack, f"{label}: other-block underflow {uf} vs {ref.uf_other_blocks}"


# ------------------------------------------------------------------ dynamic per-block scale
@pytest.mark.parametrize("kind,mode,kernel,bn,shape", [
    ("f32", 1, 1, 64, (1, 1, 1, 512, 512, 64, False)),            # config 1 shape, general kernel, FP32 planes
    ("bf16", 1, 1, 128, (1, 2, 1, 300, 700, 128, True)),
    ("e4m3", 2, 1, 64, (2, 2, 2, 200, 520, 128, True)),
    ("bf16", 1, 2, 128, (1, 2, 1, 600, 1000, 128, False)),        # prefill kernel (max warps carry the exponent)
    ("e4m3", 2, 2, 128, (1, 2, 2, 384, 1700, 128, True)),
    ("e4m3", 2, 2, 128, (1, 1, 1, 1280, 1280, 128, True)),
    ("e4m3", 2, 2, 64, (1, 2, 2, 384, 1700, 128, True)),          # Bn = 64 prefill kernel: the exponent travels with the max
    ("bf16", 1, 2, 64, (1, 2, 1, 600, 1000, 128, False)),
])
@pytest.mark.parametrize("order", [0, 1])
def test_dynamic_scale_matches_oracle(kind, mode, kernel, bn, shape, order):
    B, Hq, Hkv, Lq, Lk, d, causal = shape
    q, k, v = W.sink_qkv(B, Hq, Hkv, Lq, Lk, d, 10.0, seed=12)
    case = P.make_case(q, k, v, kind)
    b, h = B - 1, Hq - 1
    r = P.run_gpu(case, causal=causal, S=3.0, order=order, mode=mode, block_n=bn, num_splits=1, kernel=kernel,
                  dump_head=(b, h), scale_mode=1)
    assert r.kernel_id == kernel and r.block_n == bn
    ref = P.run_oracle(case, r, causal=causal, S=3.0, order=order, mode=mode, scale_mode=1)
    rows = (b * Hq + h) * Lq + np.arange(Lq)
    refc = P.run_oracle(case, r, causal=causal, S=3.0, order=order, mode=mode, scale_mode=1, rows=rows, want_codes=True)
    _compare(case, r, ref, refc, mode, bn, f"dynamic {kind} kernel {kernel} {shape} order {order}", True)
    # the point of it: in forward order, after the sink block, static 256 loses P values, the dynamic
    # scale does not
    if order == 0 and not causal:
        st = P.run_gpu(case, causal=causal, S=256.0, order=0, mode=mode, block_n=bn, num_splits=1, kernel=kernel)
        assert int(r.underflow[1]) < int(st.underflow[1])


@pytest.mark.parametrize("ns", [1, 3])
@pytest.mark.parametrize("order", [0, 1])
def test_dynamic_scale_decode_kernel(ns, order):
    B, Hq, Hkv, Lq, Lk = 2, 8, 2, 1, 3000
    q, k, v = W.sink_qkv(B, Hq, Hkv, Lq, Lk, 128, 10.0, seed=14)
    case = P.make_case(q, k, v, "decode")
    r = P.run_gpu(case, causal=False, S=256.0, order=order, mode=2, num_splits=ns, kernel=3, dump_head=(1, 5), scale_mode=1)
    assert r.kernel_id == 3 and r.num_splits == ns
    ref = P.run_oracle(case, r, causal=False, S=256.0, order=order, mode=2, scale_mode=1)
    rows = (1 * Hq + 5) * Lq + np.arange(Lq)
    refc = P.run_oracle(case, r, causal=False, S=256.0, order=order, mode=2, scale_mode=1, rows=rows, want_codes=True)
    _compare(case, r, ref, refc, 2, 128, f"dynamic decode ns={ns} order={order}", True)
    g = P.run_gpu(case, causal=False, S=256.0, order=order, mode=2, num_splits=ns, kernel=1, scale_mode=1)
    assert g.kernel_id == 1 and P.rel_l2(r.o.cpu().numpy().astype(np.float64), g.o.cpu().numpy().astype(np.float64)) <= 1e-3


# ------------------------------------------------------------------ sinks anywhere, sink blocks last
LAYOUTS = [[130, 131, 700, 1500], [5, 64, 1000, 1001, 2047], [1024], [0, 1, 2, 3]]


@pytest.mark.parametrize("pos", LAYOUTS)
@pytest.mark.parametrize("kind,mode", [("bf16", 1), ("e4m3", 2)])
@pytest.mark.parametrize("order", [0, 1, 2])
def test_sink_layouts_general_kernel(pos, kind, mode, order):
    Lq, Lk = 256, 2048
    q, k, v = W.sink_qkv(1, 2, 1, Lq, Lk, 128, 11.0, seed=16, sink_positions=pos)
    case = P.make_case(q, k, v, kind)
    r = P.run_gpu(case, causal=False, S=256.0, order=order, mode=mode, block_n=128, kernel=1, dump_head=(0, 1), sink_pos=pos)
    assert r.kernel_id == 1
    ref = P.run_oracle(case, r, causal=False, S=256.0, order=order, mode=mode, sink_pos=pos)
    refc = P.run_oracle(case, r, causal=False, S=256.0, order=order, mode=mode, sink_pos=pos, rows=Lq + np.arange(Lq),
                        want_codes=True)
    _compare(case, r, ref, refc, mode, 128, f"sinks {pos} {kind} order {order}", False)
    if order == 2:
        assert int(r.underflow[1]) == 0 == ref.uf_other_blocks       # Thm 4 per block
    elif min(pos) >= 128:
        assert int(r.underflow[1]) > 0


@pytest.mark.parametrize("pos", LAYOUTS[:3])
@pytest.mark.parametrize("order", [0, 1])
def test_sink_layouts_prefill_kernel_counters(pos, order):
    """The statistics instance of the throughput kernel classifies underflows by the sink list too."""
    Lq, Lk = 384, 2048
    q, k, v = W.sink_qkv(1, 2, 2, Lq, Lk, 128, 11.0, seed=17, sink_positions=pos)
    case = P.make_case(q, k, v, "e4m3")
    for bn in (128, 64):
        r = P.run_gpu(case, causal=True, S=256.0, order=order, mode=2, block_n=bn, kernel=2, dump_head=(0, 0), sink_pos=pos)
        assert r.kernel_id == 2
        ref = P.run_oracle(case, r, causal=True, S=256.0, order=order, mode=2, sink_pos=pos)
        refc = P.run_oracle(case, r, causal=True, S=256.0, order=order, mode=2, sink_pos=pos, rows=np.arange(Lq), want_codes=True)
        _compare(case, r, ref, refc, 2, bn, f"prefill sinks {pos} order {order} bn {bn}", False)
    f = P.fa()
    with pytest.raises(f.Fp8AttnError) as e:        # the sink-blocks-last order is not built into the prefill kernels
        P.run_gpu(case, causal=True, S=256.0, order=2, mode=2, kernel=2, sink_pos=pos)
    assert e.value.code == -5
    r = P.run_gpu(case, causal=True, S=256.0, order=2, mode=2, sink_pos=pos, stats=False)       # automatic: general kernel
    assert r.kernel_id == 1


@pytest.mark.parametrize("pos", LAYOUTS[:3])
@pytest.mark.parametrize("ns", [1, 4])
def test_sink_blocks_last_decode_kernel(pos, ns):
    B, Hq, Hkv, Lk = 2, 8, 2, 2048
    q, k, v = W.sink_qkv(B, Hq, Hkv, 1, Lk, 128, 11.0, seed=18, sink_positions=pos)
    case = P.make_case(q, k, v, "decode")
    r = P.run_gpu(case, causal=False, S=256.0, order=2, mode=2, num_splits=ns, kernel=3, dump_head=(0, 3), sink_pos=pos)
    assert r.kernel_id == 3 and r.num_splits == ns
    ref = P.run_oracle(case, r, causal=False, S=256.0, order=2, mode=2, sink_pos=pos)
    refc = P.run_oracle(case, r, causal=False, S=256.0, order=2, mode=2, sink_pos=pos, rows=np.array([3]), want_codes=True)
    _compare(case, r, ref, refc, 2, 128, f"decode sinks {pos} ns {ns}", False)
    assert int(r.underflow[1]) == 0 == ref.uf_other_blocks


# ------------------------------------------------------------------ BF16 output
@pytest.mark.parametrize("kind,mode,kernel,bn,ns,shape", [
    ("f32", 1, 1, 64, 1, (1, 2, 2, 200, 300, 64, True)),
    ("bf16", 1, 1, 128, 3, (1, 2, 1, 130, 900, 128, False)),       # general kernel + combine
    ("e4m3", 2, 2, 128, 1, (2, 2, 1, 300, 700, 128, True)),        # prefill kernel: BF16 boxes through TMA
    ("bf16", 1, 2, 128, 1, (1, 2, 2, 257, 257, 128, True)),
    ("e4m3", 2, 2, 64, 1, (1, 2, 2, 300, 300, 128, True)),         # Bn = 64 prefill kernel
    ("decode", 2, 3, 128, 1, (2, 8, 2, 1, 1000, 128, False)),
    ("decode", 2, 3, 128, 4, (2, 8, 2, 2, 2000, 128, True)),
])
def test_bf16_output_is_the_rounded_fp32_output(kind, mode, kernel, bn, ns, shape):
    B, Hq, Hkv, Lq, Lk, d, causal = shape
    q, k, v = W.sink_qkv(B, Hq, Hkv, Lq, Lk, d, 7.0, seed=19)
    case = P.make_case(q, k, v, kind)
    kw = dict(causal=causal, S=256.0, order=1, mode=mode, block_n=bn, num_splits=ns, kernel=kernel, underflow=False)
    r32 = P.run_gpu(case, **kw)
    r16 = P.run_gpu(case, out_dtype=torch.bfloat16, **kw)
    assert r16.kernel_id == kernel and r16.o.dtype == torch.bfloat16
    assert torch.equal(r16.o, r32.o.to(torch.bfloat16))            # same values, rounded to nearest even
    assert torch.equal(r16.row_max, r32.row_max) and torch.equal(r16.row_sum, r32.row_sum)
    ref = P.run_oracle(case, r16, causal=causal, S=256.0, order=1, mode=mode)
    o = r16.o.float().cpu().numpy().reshape(-1, d).astype(np.float64)
    assert P.rel_l2(o, ref.out) <= max(P.REL_L2[mode], 4e-3)       # BF16 rounding: 2^-9 relative per element


def test_bf16_output_host_path():
    f = P.fa()
    q, k, v = W.sink_qkv(2, 16, 2, 4096, 4096, 128, 7.0, seed=20)      # 16 MB of q + 4 MB of k, v + 32 MB of o
    case = P.make_case(q, k, v, "e4m3")
    r = P.run_gpu(case, causal=True, S=256.0, order=1, mode=2, underflow=False, out_dtype=torch.bfloat16)
    sc = {n: torch.from_numpy(a) for n, a in case.scales.items()}
    pin = lambda a: torch.from_numpy(a).pin_memory()
    rh = f.fwd_host(pin(case.q), pin(case.k), pin(case.v), causal=True, S=256.0, kv_order=1, mode=2, want_stats=True,
                    want_underflow=False, out_dtype=torch.bfloat16, **sc)
    assert rh.o.dtype == torch.bfloat16 and rh.n_launches > 1 and torch.equal(rh.o, r.o.cpu())
