"""Robustness of the C-ABI boundary on the GPU (csrc/fp8attn.cu): per-call scratch memory (two calls on two
streams share nothing), the piece count of fp8attn_fwd_host for every batch size, more than 65535 (batch, head)
slabs, and the 0xFF fill of the P dump for a direct C caller."""
import ctypes as C

import numpy as np
import pytest
import torch

import oracle
from paper_2606_06521_b200 import workloads as W
import parity as P

pytestmark = pytest.mark.gpu


def test_concurrent_split_kv_calls_on_two_streams():
    """Two split-KV decode calls (each with its own partials and its own quantised q) enqueued on two streams
    give the results of the same calls run one after the other."""
    f = P.fa()
    cases = []
    for seed, Lk in ((1, 16384), (2, 12288)):
        q, k, v = W.sink_qkv(4, 8, 2, 1, Lk, 128, 10.0, seed=seed)
        cases.append(P.make_case(q, k, v, "decode"))
    scs = [{n: torch.from_numpy(a).to(P.dev()) for n, a in c.scales.items()} for c in cases]
    serial = [f.fwd(c.tq, c.tk, c.tv, causal=False, S=256.0, kv_order=1, mode=2, num_splits=8, want_stats=True,
                    want_underflow=False, **sc) for c, sc in zip(cases, scs)]
    torch.cuda.synchronize()
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    for rep in range(20):
        outs = []
        for c, sc, st in zip(cases, scs, streams):
            with torch.cuda.stream(st):
                outs.append(f.fwd(c.tq, c.tk, c.tv, causal=False, S=256.0, kv_order=1, mode=2, num_splits=8,
                                  want_stats=True, want_underflow=False, stream=st, **sc))
        torch.cuda.synchronize()
        for a, b in zip(outs, serial):
            assert a.kernel_id == 3 and a.num_splits == 8
            assert torch.equal(a.o, b.o) and torch.equal(a.row_max, b.row_max) and torch.equal(a.row_sum, b.row_sum)


def test_concurrent_fp32_calls_on_two_streams():
    """The BF16 planes of FP32 inputs are per-call scratch too."""
    f = P.fa()
    cases = [P.make_case(*W.sink_qkv(2, 2, 2, 300, 700, 64, 8.0, seed=s), "f32") for s in (3, 4)]
    serial = [f.fwd(c.tq, c.tk, c.tv, causal=True, S=256.0, kv_order=1, mode=1, block_n=64) for c in cases]
    torch.cuda.synchronize()
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    for rep in range(10):
        outs = []
        for c, st in zip(cases, streams):
            with torch.cuda.stream(st):
                outs.append(f.fwd(c.tq, c.tk, c.tv, causal=True, S=256.0, kv_order=1, mode=1, block_n=64, stream=st))
        torch.cuda.synchronize()
        for a, b in zip(outs, serial):
            assert torch.equal(a.o, b.o)


@pytest.mark.parametrize("B,Hkv,G", [(3, 8, 1), (5, 4, 2), (7, 2, 1), (6, 3, 2), (1, 16, 1)])
def test_fwd_host_piece_count_for_every_batch_size(B, Hkv, G):
    """fp8attn_fwd_host cuts calls above 32 MB into at most 8 pieces whatever B and Hkv are (ADVICE round 1:
    B in {3,5,6,7} with an even Hkv used to give 10-14 pieces against 8 event slots); results equal fp8attn_fwd."""
    f = P.fa()
    Hq, L = Hkv * G, 2048
    q, k, v = W.sink_qkv(B, Hq, Hkv, L, L, 128, 7.0, seed=13)
    case = P.make_case(q, k, v, "bf16")
    nbytes = case.q.nbytes + case.k.nbytes + case.v.nbytes + q.nbytes
    assert nbytes >= 32 << 20
    r = P.run_gpu(case, causal=True, S=256.0, order=1, mode=1, underflow=False)
    pin = lambda a: torch.from_numpy(a).view(torch.bfloat16).pin_memory()
    rh = f.fwd_host(pin(case.q), pin(case.k), pin(case.v), causal=True, S=256.0, kv_order=1, mode=1,
                    want_stats=True, want_underflow=False)
    assert 1 < rh.n_launches <= 8
    assert torch.equal(rh.o, r.o.cpu())
    assert torch.equal(rh.row_max, r.row_max.cpu()) and torch.equal(rh.row_sum, r.row_sum.cpu())


def test_more_than_65535_head_slabs():
    """B * Hq = 70000 slabs (the grids are one-dimensional over slabs): sampled heads against the oracle."""
    B, H, L, d = 70, 1000, 8, 64
    q, k, v = W.sink_qkv(B, H, H, L, L, d, 3.0, seed=21)
    case = P.make_case(q, k, v, "bf16")
    r = P.run_gpu(case, causal=True, S=256.0, order=0, mode=1, block_n=64)
    assert r.kernel_id == 1
    heads = [0, 65535, 65536, 69999]
    rows = np.concatenate([h * L + np.arange(L) for h in heads])
    ref = P.run_oracle(case, r, causal=True, S=256.0, order=0, mode=1, rows=rows)
    P.check(case, r, ref, mode=1, rows=rows, label="70000 slabs", check_mse=False)
    codes, scale = P.fa().quantize_e4m3(torch.from_numpy(q).to(P.dev()))       # 70000 slabs through the quantiser
    rc, rs = oracle.quantize_e4m3(q[-1:, -3:])
    assert np.array_equal(codes[-1, -3:].cpu().numpy(), rc[0]) and np.array_equal(scale[-1, -3:].cpu().numpy(), rs[0])


def test_p_dump_is_filled_by_the_library():
    """A direct C caller hands in an uninitialised p_codes buffer: positions no kernel writes (masked keys,
    blocks a causal tile skips) read 0xFF afterwards (include/fp8attn.h)."""
    f = P.fa()
    q, k, v = W.sink_qkv(1, 2, 2, 300, 300, 128, 7.0, seed=2)
    case = P.make_case(q, k, v, "bf16")
    for kernel in (1, 2):
        o = torch.empty((1, 2, 300, 128), dtype=torch.float32, device=P.dev())
        codes = torch.full((300, 300), 0x80, dtype=torch.uint8, device=P.dev())
        st = f.Stats()
        st.struct_size = C.sizeof(f.Stats)
        st.n_sink, st.kernel = 4, kernel
        st.p_codes, st.p_batch, st.p_head = codes.data_ptr(), 0, 1
        st.stream = torch.cuda.current_stream().cuda_stream
        rc = f.fp8attn_fwd(case.tq.data_ptr(), case.tk.data_ptr(), case.tv.data_ptr(), o.data_ptr(), 1, 2, 2, 300, 300,
                           128, 1, 256.0, 1, 1 | f.DTYPE_BF16, C.byref(st))
        assert rc == 0 and st.kernel_id == kernel
        torch.cuda.synchronize()
        g = codes.cpu().numpy()
        i, j = np.indices(g.shape)
        assert np.all(g[j > i] == 0xFF) and np.all(g[j <= i] < 0x7F)      # P >= 0: codes 0 .. 0x7E
    assert f.fp8attn_trim() == 0
