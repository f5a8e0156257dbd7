"""ctypes front end of oracle/fp8attn_oracle.c (test infrastructure, not the product).

Argument marshalling only; every step of the method is in the C file, which cites the
paper passage each step follows.
"""
import ctypes as C
from dataclasses import dataclass
from typing import Optional, Sequence

import numpy as np

from .build import build as _build

DT_F32, DT_BF16, DT_E4M3, DT_BF16Q_E4M3KV = 0, 1, 2, 3


class _Opts(C.Structure):
    _fields_ = [
        ("in_dtype", C.c_int32), ("block_n", C.c_int32), ("n_sink", C.c_int32),
        ("num_splits", C.c_int32), ("split_bounds", C.c_void_p),
        ("q_scale", C.c_void_p), ("k_scale", C.c_void_p), ("v_scale", C.c_void_p),
        ("n_rows", C.c_int64), ("rows", C.c_void_p),
        ("ref_out", C.c_void_p), ("row_max", C.c_void_p), ("row_sum", C.c_void_p),
        ("p_codes", C.c_void_p), ("row_uf_sink", C.c_void_p), ("row_uf_other", C.c_void_p),
        ("uf_sink_block", C.c_uint64), ("uf_other_blocks", C.c_uint64),
        ("n_nonsink_visible", C.c_uint64), ("n_threads", C.c_int32),
        ("scale_mode", C.c_int32), ("sink_pos", C.c_void_p),
    ]


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(_build())
        lib.fp8attn_oracle_e4m3_table.argtypes = [C.c_void_p]
        lib.fp8attn_oracle_e4m3_value.argtypes = [C.c_uint8]
        lib.fp8attn_oracle_e4m3_value.restype = C.c_double
        lib.fp8attn_oracle_round_e4m3.argtypes = [C.c_float]
        lib.fp8attn_oracle_round_e4m3.restype = C.c_uint8
        lib.fp8attn_oracle_dp.argtypes = [C.c_double]
        lib.fp8attn_oracle_dp.restype = C.c_double
        lib.fp8attn_oracle_quantize_e4m3.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p,
                                                     C.c_int64, C.c_int64]
        lib.fp8attn_oracle_quantize_e4m3.restype = None
        lib.fp8attn_oracle_fwd.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p] + \
            [C.c_int] * 7 + [C.c_float, C.c_int, C.c_int, C.POINTER(_Opts)]
        lib.fp8attn_oracle_fwd.restype = C.c_int
        lib.fp8attn_oracle_opts_size.restype = C.c_int
        assert lib.fp8attn_oracle_opts_size() == C.sizeof(_Opts)
        _lib = lib
    return _lib


def e4m3_table() -> np.ndarray:
    """The 126 positive E4M3 values, code order 0x01..0x7E."""
    out = np.empty(126, dtype=np.float64)
    _load().fp8attn_oracle_e4m3_table(out.ctypes.data)
    return out


def e4m3_value(code: int) -> float:
    return float(_load().fp8attn_oracle_e4m3_value(int(code) & 0xFF))


def round_e4m3(x: float) -> int:
    """RNE (ties to even code), saturating cast of one FP32 value to an E4M3 code."""
    return int(_load().fp8attn_oracle_round_e4m3(float(np.float32(x))))


def dp(S: float) -> float:
    """Normalised maximum quantisation step dp(S) (Eq. 17-18)."""
    return float(_load().fp8attn_oracle_dp(float(S)))


def quantize_e4m3(x: np.ndarray, slab_ndim: int = 2):
    """Per-slab absmax/448 quantisation; a slab is the trailing `slab_ndim` dims."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    lead = x.shape[:x.ndim - slab_ndim]
    n_slabs = int(np.prod(lead)) if lead else 1
    slab = int(np.prod(x.shape[x.ndim - slab_ndim:]))
    codes = np.empty(x.shape, dtype=np.uint8)
    scales = np.empty(lead if lead else (1,), dtype=np.float32)
    _load().fp8attn_oracle_quantize_e4m3(x.ctypes.data, codes.ctypes.data, scales.ctypes.data,
                                         n_slabs, slab)
    return codes, scales


@dataclass
class OracleResult:
    out: np.ndarray                 # [n, d] float64  cast-P attention output
    ref: np.ndarray                 # [n, d] float64  unquantised FP64 attention
    row_max: np.ndarray             # [n] float32
    row_sum: np.ndarray             # [n] float64
    p_codes: Optional[np.ndarray]   # [n, Lk] uint8 (0xFF = masked) or None
    row_uf_sink: np.ndarray         # [n] uint32
    row_uf_other: np.ndarray        # [n] uint32
    uf_sink_block: int
    uf_other_blocks: int
    n_nonsink_visible: int
    n_threads: int
    rows: np.ndarray                # [n] int64 flat row ids

    @property
    def mse(self) -> float:
        """Per-dimension MSE against the unquantised reference."""
        return float(np.mean((self.out - self.ref) ** 2))

    @property
    def underflow_fraction(self) -> float:
        return (self.uf_sink_block + self.uf_other_blocks) / max(1, self.n_nonsink_visible)


def _as_input(a: np.ndarray, dtype_code: int, is_q: bool) -> np.ndarray:
    if dtype_code == DT_BF16Q_E4M3KV:
        dtype_code = DT_BF16 if is_q else DT_E4M3
    want = {DT_F32: np.float32, DT_BF16: np.uint16, DT_E4M3: np.uint8}[dtype_code]
    if a.dtype != want:
        raise TypeError(f"expected {want} array for dtype code {dtype_code}, got {a.dtype}")
    return np.ascontiguousarray(a)


def attention_fwd(q, k, v, *, causal: bool, S: float, kv_order: int, mode: int,
                  in_dtype: int = DT_F32, block_n: int = 64, n_sink: int = 4,
                  split_bounds: Optional[Sequence[int]] = None,
                  q_scale=None, k_scale=None, v_scale=None,
                  rows: Optional[Sequence[int]] = None, want_codes: bool = False,
                  n_threads: int = 0, scale_mode: int = 0,
                  sink_pos: Optional[Sequence[int]] = None) -> OracleResult:
    """q [B,Hq,Lq,d], k/v [B,Hkv,Lk,d] numpy arrays (float32, uint16 = BF16 bits, uint8 =
    E4M3 codes).  Returns the cast-P output and statistics for the selected rows.
    kv_order 0 forward, 1 reverse, 2 sink blocks last; scale_mode 1 = dynamic per-(row, block) 2^k scale (S unused);
    sink_pos = key indices of the sink keys (default: the first n_sink keys)."""
    q = _as_input(q, in_dtype, True)
    k = _as_input(k, in_dtype, False)
    v = _as_input(v, in_dtype, False)
    B, Hq, Lq, d = q.shape
    Bk, Hkv, Lk, dk = k.shape
    assert (Bk, dk) == (B, d) and v.shape == k.shape
    total = B * Hq * Lq
    rows_arr = np.arange(total, dtype=np.int64) if rows is None else \
        np.ascontiguousarray(rows, dtype=np.int64)
    n = rows_arr.size
    o = _Opts()
    o.in_dtype, o.block_n, o.n_sink = in_dtype, block_n, n_sink
    keep = []
    if split_bounds is not None and len(split_bounds) > 2:
        sb = np.ascontiguousarray(split_bounds, dtype=np.int32)
        nb = (Lk + block_n - 1) // block_n
        assert sb[0] == 0 and sb[-1] == nb and np.all(np.diff(sb) >= 0)
        keep.append(sb)
        o.num_splits, o.split_bounds = len(sb) - 1, sb.ctypes.data
    else:
        o.num_splits, o.split_bounds = 1, None
    for name, arr, cnt in (("q_scale", q_scale, B * Hq), ("k_scale", k_scale, B * Hkv),
                           ("v_scale", v_scale, B * Hkv)):
        if arr is not None:
            a = np.ascontiguousarray(arr, dtype=np.float32).reshape(-1)
            assert a.size == cnt, name
            keep.append(a)
            setattr(o, name, a.ctypes.data)
    o.n_rows, o.rows = n, rows_arr.ctypes.data
    out = np.zeros((n, d), dtype=np.float64)
    ref = np.zeros((n, d), dtype=np.float64)
    row_max = np.zeros(n, dtype=np.float32)
    row_sum = np.zeros(n, dtype=np.float64)
    codes = np.zeros((n, Lk), dtype=np.uint8) if want_codes else None
    ufs = np.zeros(n, dtype=np.uint32)
    ufo = np.zeros(n, dtype=np.uint32)
    o.ref_out, o.row_max, o.row_sum = ref.ctypes.data, row_max.ctypes.data, row_sum.ctypes.data
    o.p_codes = codes.ctypes.data if want_codes else None
    o.row_uf_sink, o.row_uf_other = ufs.ctypes.data, ufo.ctypes.data
    o.n_threads = n_threads
    o.scale_mode = scale_mode
    if sink_pos is not None:
        sp = np.ascontiguousarray(sorted(int(x) for x in sink_pos), dtype=np.int32)
        assert sp.size >= 1 and sp[0] >= 0 and sp[-1] < Lk and np.all(np.diff(sp) > 0)
        keep.append(sp)
        o.n_sink, o.sink_pos = int(sp.size), sp.ctypes.data
    rc = _load().fp8attn_oracle_fwd(q.ctypes.data, k.ctypes.data, v.ctypes.data, out.ctypes.data,
                                    B, Hq, Hkv, Lq, Lk, d, int(bool(causal)), float(S),
                                    int(kv_order), int(mode), C.byref(o))
    if rc != 0:
        raise ValueError(f"fp8attn_oracle_fwd returned {rc}")
    return OracleResult(out, ref, row_max, row_sum, codes, ufs, ufo, int(o.uf_sink_block),
                        int(o.uf_other_blocks), int(o.n_nonsink_visible), int(o.n_threads),
                        rows_arr)
