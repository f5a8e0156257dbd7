"""Python binding of libfp8attn.so (include/fp8attn.h).  Argument marshalling only: every step
of the method runs in the CUDA kernels behind the C ABI.  torch is used for device memory and
streams.  There is no CPU path: if the library cannot be loaded, importing this module fails.

The C entry points are exposed under their own names (`fp8attn_fwd`, `fp8attn_fwd_host`,
`fp8attn_decode_noalloc`, `fp8attn_quantize_e4m3`, `fp8attn_debug_gemm`, `fp8attn_strerror`,
`fp8attn_version`) taking raw device pointers, plus the tensor-level wrappers `fwd`, `fwd_host`,
`decode_noalloc`, `quantize_e4m3` and `debug_gemm`.
"""
import ctypes as C
import os
import subprocess
from dataclasses import dataclass
from typing import Optional

import torch

from .build import LIB, build

MODE_NOCAST, MODE_ISOLATION, MODE_FP8 = 0, 1, 2
DTYPE_F32, DTYPE_BF16, DTYPE_E4M3, DTYPE_BF16Q_E4M3KV = 0 << 8, 1 << 8, 2 << 8, 3 << 8
ORDER_FORWARD, ORDER_REVERSE, ORDER_SINK_LAST = 0, 1, 2
SCALE_STATIC, SCALE_DYNAMIC = 0, 1
MAX_SPLITS = 64


class Stats(C.Structure):
    """struct fp8attn_stats"""
    _fields_ = [
        ("struct_size", C.c_int32), ("n_sink", C.c_int32), ("block_n", C.c_int32),
        ("num_splits", C.c_int32), ("kernel", C.c_int32), ("scale_mode", C.c_int32),
        ("q_scale", C.c_void_p), ("k_scale", C.c_void_p), ("v_scale", C.c_void_p),
        ("stream", C.c_void_p), ("p_codes", C.c_void_p),
        ("p_batch", C.c_int32), ("p_head", C.c_int32),
        ("sink_pos", C.c_void_p), ("o_dtype", C.c_int32), ("reserved1", C.c_int32),
        ("seqlens_q", C.c_void_p), ("seqlens_k", C.c_void_p), ("block_table", C.c_void_p),
        ("page_size", C.c_int32), ("max_pages", C.c_int32), ("num_pages", C.c_int32), ("reserved2", C.c_int32),
        ("row_max", C.c_void_p), ("row_sum", C.c_void_p), ("underflow", C.c_void_p),
        ("block_m_used", C.c_int32), ("block_n_used", C.c_int32), ("num_splits_used", C.c_int32),
        ("split_bounds", C.c_int32 * (MAX_SPLITS + 1)),
        ("kernel_id", C.c_int32), ("n_launches", C.c_int32),
    ]


def _load():
    # build() compares modification times and rebuilds a stale library (needs nvcc); without nvcc an
    # existing library is used as it is
    try:
        path = build()
    except (OSError, subprocess.CalledProcessError):
        if not os.path.exists(LIB):
            raise
        path = LIB
    lib = C.CDLL(path)
    lib.fp8attn_fwd.argtypes = [C.c_void_p] * 4 + [C.c_int] * 7 + [C.c_float, C.c_int, C.c_int,
                                                                  C.POINTER(Stats)]
    lib.fp8attn_fwd.restype = C.c_int
    lib.fp8attn_fwd_host.argtypes = lib.fp8attn_fwd.argtypes
    lib.fp8attn_fwd_host.restype = C.c_int
    lib.fp8attn_decode_noalloc.argtypes = lib.fp8attn_fwd.argtypes
    lib.fp8attn_decode_noalloc.restype = C.c_int
    lib.fp8attn_quantize_e4m3.argtypes = [C.c_void_p] * 3 + [C.c_int] * 4 + [C.c_void_p]
    lib.fp8attn_quantize_e4m3.restype = C.c_int
    lib.fp8attn_debug_gemm.argtypes = [C.c_void_p] * 3 + [C.c_int] * 5 + [C.c_void_p]
    lib.fp8attn_debug_gemm.restype = C.c_int
    lib.fp8attn_strerror.argtypes = [C.c_int]
    lib.fp8attn_strerror.restype = C.c_char_p
    lib.fp8attn_last_cuda_error.restype = C.c_char_p
    lib.fp8attn_version.restype = C.c_int
    lib.fp8attn_trim.restype = C.c_int
    return lib


_lib = _load()
LIB_PATH = _lib._name

fp8attn_fwd = _lib.fp8attn_fwd
fp8attn_fwd_host = _lib.fp8attn_fwd_host
fp8attn_decode_noalloc = _lib.fp8attn_decode_noalloc
NOALLOC_SCRATCH_BYTES = 16 << 20        # FP8ATTN_NOALLOC_SCRATCH_BYTES
fp8attn_quantize_e4m3 = _lib.fp8attn_quantize_e4m3
fp8attn_debug_gemm = _lib.fp8attn_debug_gemm
fp8attn_version = _lib.fp8attn_version
fp8attn_trim = _lib.fp8attn_trim


def fp8attn_strerror(code: int) -> str:
    return _lib.fp8attn_strerror(code).decode()


class Fp8AttnError(RuntimeError):
    def __init__(self, code):
        self.code = code
        detail = _lib.fp8attn_last_cuda_error().decode() if code in (-6, -7, -9) else ""
        super().__init__(f"fp8attn error {code}: {fp8attn_strerror(code)}" + (f" [{detail}]" if detail else ""))


def _check(rc):
    if rc != 0:
        raise Fp8AttnError(rc)


def _stream_ptr(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _ptr(t: Optional[torch.Tensor]):
    return None if t is None else C.c_void_p(t.data_ptr())


def _set_sinks(st, sink_pos, keep):
    """sink_pos (host list of ascending key indices) -> st.sink_pos / st.n_sink."""
    if sink_pos is None:
        return
    arr = (C.c_int32 * len(sink_pos))(*[int(x) for x in sink_pos])
    keep.append(arr)
    st.sink_pos = C.cast(arr, C.c_void_p)
    st.n_sink = len(sink_pos)


@dataclass
class FwdResult:
    o: torch.Tensor                       # [B,Hq,Lq,d] float32
    row_max: Optional[torch.Tensor]       # [B,Hq,Lq] float32
    row_sum: Optional[torch.Tensor]       # [B,Hq,Lq] float32
    underflow: Optional[torch.Tensor]     # [2] int64 (sink block, other blocks)
    p_codes: Optional[torch.Tensor]       # [Lq,Lk] uint8 of head (p_batch, p_head); 0xFF = masked
    block_m: int
    block_n: int
    num_splits: int
    split_bounds: list
    kernel_id: int
    n_launches: int


def _dtype_code(q, k):
    if q.dtype == torch.float32 and k.dtype == torch.float32:
        return DTYPE_F32
    if q.dtype == torch.bfloat16 and k.dtype == torch.bfloat16:
        return DTYPE_BF16
    e4 = (torch.uint8, torch.float8_e4m3fn)
    if q.dtype in e4 and k.dtype in e4:
        return DTYPE_E4M3
    if q.dtype == torch.bfloat16 and k.dtype in e4:
        return DTYPE_BF16Q_E4M3KV
    raise TypeError(f"unsupported q/k dtypes {q.dtype}/{k.dtype}")


def fwd(q, k, v, *, causal: bool, S: float, kv_order: int, mode: int, n_sink: int = 4,
        block_n: int = 0, num_splits: int = 0, kernel: int = 0, q_scale=None, k_scale=None, v_scale=None,
        want_stats: bool = False, want_underflow: Optional[bool] = None, dump_head=None, out=None,
        stream=None, scale_mode: int = 0, sink_pos=None, out_dtype=None, seqlens_q=None, seqlens_k=None,
        block_table=None, Lk=None) -> FwdResult:
    """fp8attn_fwd on CUDA tensors q [B,Hq,Lq,d], k/v [B,Hkv,Lk,d] (contiguous).  `mode` is the
    P mode (0 no-cast, 1 isolation, 2 FP8); the input dtype bits are derived from the tensors.
    `dump_head=(b,h)` returns the E4M3 code of every P of that head.  `kernel` requests a kernel
    family (0 automatic, 1 general, 2 prefill, 3 decode).  `scale_mode=1`: dynamic per-(row, block) 2^k scale;
    `sink_pos`: ascending key indices of the sink keys (replaces n_sink); `out_dtype=torch.bfloat16`: BF16 output.
    `seqlens_q` / `seqlens_k`: int32 CUDA tensors [B] (variable-length sequences in the padded layout).
    `block_table`: int32 CUDA tensor [B, max_pages]; k, v are then page pools [num_pages, Hkv, page_size, d] and
    `Lk` (the longest sequence, default max_pages * page_size) must be given."""
    for t in (q, k, v):
        if not (t.is_cuda and t.is_contiguous() and t.dim() == 4):
            raise ValueError("q, k, v must be contiguous 4-D CUDA tensors")
    B, Hq, Lq, d = q.shape
    if block_table is not None:
        n_pages, Hkv, page_size, dk = k.shape
        max_pages = block_table.shape[1]
        Lk = max_pages * page_size if Lk is None else int(Lk)
        if dk != d or v.shape != k.shape or block_table.shape[0] != B or block_table.dtype != torch.int32:
            raise ValueError("paged k, v must be [num_pages, Hkv, page_size, d] and block_table int32 [B, max_pages]")
    else:
        Bk, Hkv, Lk, dk = k.shape
        if (Bk, dk) != (B, d) or v.shape != k.shape:
            raise ValueError("shape mismatch between q, k, v")
    if out is not None:
        out_dtype = out.dtype
    out_dtype = torch.float32 if out_dtype is None else out_dtype
    if out_dtype not in (torch.float32, torch.bfloat16):
        raise TypeError("o must be float32 or bfloat16")
    o = out if out is not None else torch.empty((B, Hq, Lq, d), dtype=out_dtype, device=q.device)
    st = Stats()
    st.struct_size = C.sizeof(Stats)
    st.n_sink, st.block_n, st.num_splits, st.kernel = n_sink, block_n, num_splits, kernel
    st.scale_mode = int(scale_mode)
    st.o_dtype = 1 if out_dtype == torch.bfloat16 else 0
    st.stream = _stream_ptr(stream)
    keep = []
    _set_sinks(st, sink_pos, keep)
    for name, t in (("seqlens_q", seqlens_q), ("seqlens_k", seqlens_k), ("block_table", block_table)):
        if t is not None:
            t = t.to(device=q.device, dtype=torch.int32).contiguous()
            keep.append(t)
            setattr(st, name, t.data_ptr())
    if block_table is not None:
        st.page_size, st.max_pages, st.num_pages = int(page_size), int(max_pages), int(n_pages)
    for name, t in (("q_scale", q_scale), ("k_scale", k_scale), ("v_scale", v_scale)):
        if t is not None:
            t = t.to(device=q.device, dtype=torch.float32).contiguous()
            keep.append(t)
            setattr(st, name, t.data_ptr())
    row_max = row_sum = underflow = codes = None
    if want_stats:
        row_max = torch.empty((B, Hq, Lq), dtype=torch.float32, device=q.device)
        row_sum = torch.empty((B, Hq, Lq), dtype=torch.float32, device=q.device)
        st.row_max, st.row_sum = row_max.data_ptr(), row_sum.data_ptr()
    if want_stats if want_underflow is None else want_underflow:
        underflow = torch.zeros(2, dtype=torch.int64, device=q.device)
        st.underflow = underflow.data_ptr()
    if dump_head is not None:
        codes = torch.full((Lq, Lk), 0xFF, dtype=torch.uint8, device=q.device)
        st.p_codes = codes.data_ptr()
        st.p_batch, st.p_head = int(dump_head[0]), int(dump_head[1])
    with torch.cuda.device(q.device):
        rc = fp8attn_fwd(_ptr(q), _ptr(k), _ptr(v), _ptr(o), B, Hq, Hkv, Lq, Lk, d, int(bool(causal)),
                         float(S), int(kv_order), int(mode) | _dtype_code(q, k), C.byref(st))
    _check(rc)
    ns = st.num_splits_used
    return FwdResult(o, row_max, row_sum, underflow, codes, st.block_m_used, st.block_n_used, ns,
                     [st.split_bounds[i] for i in range(ns + 1)], st.kernel_id, st.n_launches)


def decode_noalloc(q, k, v, o, *, S: float, kv_order: int, k_scale, v_scale, q_scale=None, causal: bool = False,
                   n_sink: int = 4, num_splits: int = 0, row_max=None, row_sum=None, underflow=None, stream=None,
                   scale_mode: int = 0) -> FwdResult:
    """fp8attn_decode_noalloc: the split-KV decode path with its scratch in the library's static device array -- no
    allocation in the library (include/fp8attn.h) and none here: every buffer, `o` and the optional statistics
    (`row_max`, `row_sum` float32 [B,Hq,Lq]; `underflow` int64 [2]) included, is the caller's.  q is BF16 (quantised
    per slab by the library) or E4M3 codes with `q_scale`; k, v are E4M3 codes with float32 CUDA scales [B,Hkv].
    Calls that overlap on the GPU race on the scratch: keep them on one stream."""
    for t in (q, k, v, o):
        if not (t.is_cuda and t.is_contiguous() and t.dim() == 4):
            raise ValueError("q, k, v, o must be contiguous 4-D CUDA tensors")
    B, Hq, Lq, d = q.shape
    Bk, Hkv, Lk, dk = k.shape
    if (Bk, dk) != (B, d) or v.shape != k.shape or o.shape != q.shape:
        raise ValueError("shape mismatch between q, k, v, o")
    if o.dtype not in (torch.float32, torch.bfloat16):
        raise TypeError("o must be float32 or bfloat16")
    st = Stats()
    st.struct_size = C.sizeof(Stats)
    st.n_sink, st.num_splits, st.scale_mode = int(n_sink), int(num_splits), int(scale_mode)
    st.o_dtype = 1 if o.dtype == torch.bfloat16 else 0
    st.stream = _stream_ptr(stream)
    for name, t in (("q_scale", q_scale), ("k_scale", k_scale), ("v_scale", v_scale), ("row_max", row_max),
                    ("row_sum", row_sum)):
        if t is not None:
            if not (t.is_cuda and t.is_contiguous() and t.dtype == torch.float32):
                raise TypeError(f"{name} must be a contiguous float32 CUDA tensor")
            setattr(st, name, t.data_ptr())
    if underflow is not None:
        if not (underflow.is_cuda and underflow.dtype == torch.int64 and underflow.numel() == 2):
            raise TypeError("underflow must be an int64 CUDA tensor of 2 elements")
        st.underflow = underflow.data_ptr()
    with torch.cuda.device(q.device):
        rc = fp8attn_decode_noalloc(_ptr(q), _ptr(k), _ptr(v), _ptr(o), B, Hq, Hkv, Lq, Lk, d, int(bool(causal)), float(S),
                                    int(kv_order), MODE_FP8 | _dtype_code(q, k), C.byref(st))
    _check(rc)
    ns = st.num_splits_used
    return FwdResult(o, row_max, row_sum, underflow, None, st.block_m_used, st.block_n_used, ns,
                     [st.split_bounds[i] for i in range(ns + 1)], st.kernel_id, st.n_launches)


def fwd_host(q, k, v, *, causal: bool, S: float, kv_order: int, mode: int, n_sink: int = 4,
             block_n: int = 0, num_splits: int = 0, kernel: int = 0, q_scale=None, k_scale=None, v_scale=None,
             want_stats: bool = False, want_underflow: Optional[bool] = None, out=None, stream=None,
             device=None, scale_mode: int = 0, sink_pos=None, out_dtype=None) -> FwdResult:
    """fp8attn_fwd_host on HOST tensors (CPU, ideally pinned): the library copies them to the
    device, runs the kernels, copies `o` (and statistics) back and synchronises the stream."""
    for t in (q, k, v):
        if t.is_cuda or not t.is_contiguous() or t.dim() != 4:
            raise ValueError("q, k, v must be contiguous 4-D CPU tensors")
    B, Hq, Lq, d = q.shape
    Bk, Hkv, Lk, dk = k.shape
    if (Bk, dk) != (B, d) or v.shape != k.shape:
        raise ValueError("shape mismatch between q, k, v")
    if out is not None:
        out_dtype = out.dtype
    out_dtype = torch.float32 if out_dtype is None else out_dtype
    o = out if out is not None else torch.empty((B, Hq, Lq, d), dtype=out_dtype, pin_memory=True)
    st = Stats()
    st.struct_size = C.sizeof(Stats)
    st.n_sink, st.block_n, st.num_splits, st.kernel = n_sink, block_n, num_splits, kernel
    st.scale_mode = int(scale_mode)
    st.o_dtype = 1 if out_dtype == torch.bfloat16 else 0
    keep = []
    _set_sinks(st, sink_pos, keep)
    for name, t in (("q_scale", q_scale), ("k_scale", k_scale), ("v_scale", v_scale)):
        if t is not None:
            t = t.to(device="cpu", dtype=torch.float32).contiguous()
            keep.append(t)
            setattr(st, name, t.data_ptr())
    row_max = row_sum = underflow = None
    if want_stats:
        row_max = torch.empty((B, Hq, Lq), dtype=torch.float32, pin_memory=True)
        row_sum = torch.empty((B, Hq, Lq), dtype=torch.float32, pin_memory=True)
        st.row_max, st.row_sum = row_max.data_ptr(), row_sum.data_ptr()
    if want_stats if want_underflow is None else want_underflow:
        underflow = torch.zeros(2, dtype=torch.int64, pin_memory=True)
        st.underflow = underflow.data_ptr()
    dev = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
    with torch.cuda.device(dev):
        st.stream = _stream_ptr(stream)
        rc = fp8attn_fwd_host(_ptr(q), _ptr(k), _ptr(v), _ptr(o), B, Hq, Hkv, Lq, Lk, d, int(bool(causal)),
                              float(S), int(kv_order), int(mode) | _dtype_code(q, k), C.byref(st))
    _check(rc)
    ns = st.num_splits_used
    return FwdResult(o, row_max, row_sum, underflow, None, st.block_m_used, st.block_n_used, ns,
                     [st.split_bounds[i] for i in range(ns + 1)], st.kernel_id, st.n_launches)


def quantize_e4m3(x: torch.Tensor, stream=None):
    """Per-(b,h) absmax/448 quantisation of float32 [B,H,L,d] -> (uint8 codes, float32 [B,H] scale)."""
    if not (x.is_cuda and x.is_contiguous() and x.dim() == 4 and x.dtype == torch.float32):
        raise ValueError("x must be a contiguous 4-D float32 CUDA tensor")
    B, H, L, d = x.shape
    codes = torch.empty(x.shape, dtype=torch.uint8, device=x.device)
    scale = torch.empty((B, H), dtype=torch.float32, device=x.device)
    with torch.cuda.device(x.device):
        _check(fp8attn_quantize_e4m3(_ptr(x), _ptr(codes), _ptr(scale), B, H, L, d, _stream_ptr(stream)))
    return codes, scale


def debug_gemm(A: torch.Tensor, Bm: torch.Tensor, a_in_tmem: bool, b_mn_major: bool, stream=None):
    """D[128,N] = A[128,K] . B on one tcgen05 tile; A, B are bfloat16 or uint8 (E4M3 codes).
    B is [N,K] when b_mn_major is False, [K,N] when True."""
    eb = 2 if A.dtype == torch.bfloat16 else 1
    K = A.shape[1]
    N = Bm.shape[1] if b_mn_major else Bm.shape[0]
    D = torch.empty((128, N), dtype=torch.float32, device=A.device)
    with torch.cuda.device(A.device):
        _check(fp8attn_debug_gemm(_ptr(A), _ptr(Bm), _ptr(D), N, K, eb, int(a_in_tmem), int(b_mn_major),
                                  _stream_ptr(stream)))
    return D
