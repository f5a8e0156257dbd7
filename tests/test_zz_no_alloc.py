"""fp8attn_decode_noalloc (include/fp8attn.h): the split-KV decode path with its scratch -- the quantised q and the
(m_s, l_s, O_s) partials -- in the library's file-scope static device array instead of per-call pool memory, for
callers that must not allocate.  Same kernels and split layout as fp8attn_fwd, so the results are compared with
fp8attn_fwd's on the same inputs: bit for bit (which is inside the tolerance the other GPU tests use, P.REL_L2[2]),
on calls that follow each other on one stream and share the array, in a file pytest collects last."""
import ctypes as C

import numpy as np
import pytest
import torch

from paper_2606_06521_b200 import workloads as W
import parity as P

pytestmark = pytest.mark.gpu

# (B, Hq, Hkv, Lq, Lk, causal, kind, num_splits): different shapes, so that a call finds the other's data in the array
CALLS = [
    (4, 8, 2, 1, 4096, False, "decode", 0),      # BF16 q quantised into the array, automatic split count (> 1)
    (2, 4, 2, 3, 1000, True, "e4m3", 3),         # E4M3 q with its own scale, 3 splits, ragged last block, causal
    (1, 16, 1, 1, 517, False, "decode", 1),      # one split: no partials, only the quantised q
]


def _inputs(spec, seed):
    B, Hq, Hkv, Lq, Lk, causal, kind, ns = spec
    q, k, v = W.sink_qkv(B, Hq, Hkv, Lq, Lk, 128, 10.0, seed=seed)
    case = P.make_case(q, k, v, kind)
    sc = {n: torch.from_numpy(a).to(P.dev()) for n, a in case.scales.items()}
    return case, sc


def _buffers(spec):
    B, Hq, _, Lq = spec[:4]
    dev = P.dev()
    return dict(o=torch.full((B, Hq, Lq, 128), float("nan"), dtype=torch.float32, device=dev),
                row_max=torch.full((B, Hq, Lq), float("nan"), dtype=torch.float32, device=dev),
                row_sum=torch.full((B, Hq, Lq), float("nan"), dtype=torch.float32, device=dev))


def _noalloc(f, spec, case, sc, buf, S=256.0, order=1):
    return f.decode_noalloc(case.tq, case.tk, case.tv, buf["o"], S=S, kv_order=order, causal=spec[5], num_splits=spec[7],
                            row_max=buf["row_max"], row_sum=buf["row_sum"], **sc)


def test_noalloc_equals_fwd_on_calls_in_a_row():
    f = P.fa()
    prepared = [(spec,) + _inputs(spec, seed=30 + i) for i, spec in enumerate(CALLS)]
    # the existing path, one call at a time
    want = [P.run_gpu(case, causal=spec[5], S=256.0, order=1, mode=2, num_splits=spec[7], kernel=3, underflow=False)
            for spec, case, sc in prepared]
    # the new entry point: all calls back to back on the current stream, no synchronisation in between, twice over
    for rep in range(2):
        bufs = [_buffers(spec) for spec, _, _ in prepared]
        got = [_noalloc(f, spec, case, sc, buf) for (spec, case, sc), buf in zip(prepared, bufs)]
        torch.cuda.synchronize()
        for (spec, case, sc), g, w in zip(prepared, got, want):
            assert g.kernel_id == 3 and g.num_splits == w.num_splits and g.split_bounds == w.split_bounds
            assert g.n_launches == w.n_launches
            od, ow = g.o.cpu().numpy().astype(np.float64), w.o.cpu().numpy().astype(np.float64)
            assert P.rel_l2(od, ow) <= P.REL_L2[2]
            assert torch.equal(g.o, w.o), f"{spec} rep {rep}: outputs differ from fp8attn_fwd"
            assert torch.equal(g.row_max, w.row_max) and torch.equal(g.row_sum, w.row_sum)
    assert want[0].num_splits > 1 and want[1].num_splits == 3 and want[2].num_splits == 1
    # and against the oracle, like every other kernel path (same split boundaries, reading R14)
    spec, case, sc = prepared[1]
    ref = P.run_oracle(case, got[1], causal=spec[5], S=256.0, order=1, mode=2)
    P.check(case, got[1], ref, mode=2, label="decode_noalloc", check_mse=False, check_uf=False)


def test_noalloc_statistics_instance_and_forward_order():
    """The underflow counters (caller memory, cleared by the call) and a non-power-of-two S in forward order."""
    f = P.fa()
    spec = CALLS[1]
    case, sc = _inputs(spec, seed=41)
    for S, order in ((448.0, 0), (256.0, 1)):
        w = P.run_gpu(case, causal=spec[5], S=S, order=order, mode=2, num_splits=spec[7], kernel=3, underflow=True)
        buf = _buffers(spec)
        uf = torch.full((2,), 12345, dtype=torch.int64, device=P.dev())
        g = f.decode_noalloc(case.tq, case.tk, case.tv, buf["o"], S=S, kv_order=order, causal=spec[5], num_splits=spec[7],
                             row_max=buf["row_max"], row_sum=buf["row_sum"], underflow=uf, **sc)
        torch.cuda.synchronize()
        assert torch.equal(g.o, w.o) and torch.equal(g.row_max, w.row_max) and torch.equal(g.row_sum, w.row_sum)
        assert torch.equal(uf, w.underflow)


def test_noalloc_takes_no_device_memory():
    """After a warm-up call (kernel images load on first use) the free device memory does not move over further
    calls, with the library's own pool emptied first: the entry point draws on nothing but the static array."""
    f = P.fa()
    spec = CALLS[0]
    case, sc = _inputs(spec, seed=50)
    buf = _buffers(spec)
    _noalloc(f, spec, case, sc, buf)
    torch.cuda.synchronize()
    assert f.fp8attn_trim() == 0
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(5):
        _noalloc(f, spec, case, sc, buf)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0


def _raw_call(f, t, B, Hq, Hkv, Lq, Lk, d, mode, num_splits=0):
    st = f.Stats()
    st.struct_size = C.sizeof(f.Stats)
    st.num_splits = num_splits
    st.k_scale = st.v_scale = st.q_scale = t.data_ptr()
    st.stream = torch.cuda.current_stream().cuda_stream
    p = C.c_void_p(t.data_ptr())
    return f.fp8attn_decode_noalloc(p, p, p, p, B, Hq, Hkv, Lq, Lk, d, 0, 256.0, 1, mode, C.byref(st))


def test_noalloc_rejects_what_it_cannot_hold_or_serve():
    """Sizes beyond the static array: a clear error before anything is launched (the pointers here are never used)."""
    f = P.fa()
    t = torch.zeros(1024, dtype=torch.float32, device=P.dev())
    mode = f.MODE_FP8 | f.DTYPE_BF16Q_E4M3KV
    # B*Hq = 2048 rows x 16 splits x (128 + 2) x 4 B = 17.0 MB of partials > 16 MiB
    need = 2048 * 128 + 2048 * 4 + 16 * 2048 * 130 * 4
    assert need > f.NOALLOC_SCRATCH_BYTES
    rc = _raw_call(f, t, 64, 32, 8, 1, 2048, 128, mode, num_splits=16)
    assert rc == -9
    msg = f._lib.fp8attn_last_cuda_error().decode()
    assert str(need) in msg and str(f.NOALLOC_SCRATCH_BYTES) in msg
    assert "scratch" in f.fp8attn_strerror(rc)
    with pytest.raises(f.Fp8AttnError, match="scratch"):
        f._check(rc)
    # the same call with 8 splits fits (8.5 MB) -- checked by size only: not launched on these pointers
    assert 2048 * 128 + 2048 * 4 + 8 * 2048 * 130 * 4 <= f.NOALLOC_SCRATCH_BYTES
    # not a decode shape / not the FP8 mode / d = 64: unsupported, as documented
    assert _raw_call(f, t, 1, 8, 2, 64, 2048, 128, mode) == -5
    assert _raw_call(f, t, 1, 8, 2, 1, 2048, 128, f.MODE_ISOLATION | f.DTYPE_BF16) == -5
    assert _raw_call(f, t, 1, 8, 2, 1, 2048, 64, mode) == -5
    torch.cuda.synchronize()
