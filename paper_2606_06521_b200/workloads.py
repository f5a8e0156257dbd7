"""Seeded synthetic inputs with the paper's attention-sink structure.

This module serves BOTH the CUDA path's tests/bench and the CPU oracle's tests.  It holds
none of the method's arithmetic: it only draws numbers and lays them out.

Recipe (BASELINE.json configs):
NumPy default_rng(seed) (PCG64), standard_normal(float32), draw order Q, K, V, shapes
[B,H,L,d]; then Q[..., d-1] = 1, K[..., :n_sink, d-1] = Delta*sqrt(d), K[..., n_sink:, d-1] = 0.
The logit of a sink key is then Delta + N(0, ~1) and of any other key N(0, ~1).
"""
from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class Config:
    name: str
    B: int
    Hq: int
    Hkv: int
    Lq: int
    Lk: int
    d: int
    causal: bool
    delta: float
    n_sink: int = 4

    @property
    def flops(self) -> float:
        """4*B*Hq*Lq*Lk*d, halved for causal."""
        f = 4.0 * self.B * self.Hq * self.Lq * self.Lk * self.d
        return f / 2 if self.causal else f


# BASELINE.json `configs`, in order.
CONFIGS = {
    "cfg1": Config("cfg1", 1, 1, 1, 512, 512, 64, False, 8.0),
    "cfg2": Config("cfg2", 1, 8, 8, 2048, 2048, 128, False, 7.0),
    "cfg3": Config("cfg3", 4, 32, 32, 8192, 8192, 128, True, 7.0),
    "cfg4": Config("cfg4", 2, 64, 8, 16384, 16384, 128, True, 9.0),
    "cfg5": Config("cfg5", 64, 32, 8, 1, 32768, 128, False, 10.0),
}


def sink_qkv(B, Hq, Hkv, Lq, Lk, d, delta, n_sink=4, seed=0, sink_positions=None):
    """FP32 Q [B,Hq,Lq,d], K, V [B,Hkv,Lk,d] with the sink construction.  `sink_positions` puts the sink keys at
    the given key indices instead of the first n_sink (multi-sink / distributed-sink layouts); the
    random draws do not depend on it."""
    rng = np.random.default_rng(seed)
    q = rng.standard_normal((B, Hq, Lq, d), dtype=np.float32)
    k = rng.standard_normal((B, Hkv, Lk, d), dtype=np.float32)
    v = rng.standard_normal((B, Hkv, Lk, d), dtype=np.float32)
    q[..., d - 1] = 1.0
    k[..., d - 1] = 0.0
    pos = list(range(n_sink)) if sink_positions is None else [int(x) for x in sink_positions]
    k[..., pos, d - 1] = np.float32(delta * np.sqrt(d))
    return q, k, v


def set_delta(k, delta, n_sink=4):
    """Overwrite the sink entries of K in place (only these change with Delta)."""
    d = k.shape[-1]
    k[..., :n_sink, d - 1] = np.float32(delta * np.sqrt(d))
    return k


def config_qkv(cfg: Config, seed=0, delta=None):
    return sink_qkv(cfg.B, cfg.Hq, cfg.Hkv, cfg.Lq, cfg.Lk, cfg.d,
                    cfg.delta if delta is None else delta, cfg.n_sink, seed)


def to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """Round FP32 to BF16 (round-to-nearest-even), returned as uint16 bit patterns."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    bias = ((u >> 16) & 1) + np.uint32(0x7FFF)
    return ((u + bias) >> 16).astype(np.uint16)


def bf16_bits_to_f32(h: np.ndarray) -> np.ndarray:
    return (h.astype(np.uint32) << 16).view(np.float32)


def sample_rows(B, Hq, Lq, n_per_head, seed=0, heads=None):
    """Flat row ids ((b*Hq+h)*Lq+i) of n_per_head rows from each (b,h), always including
    the first and last row of the head."""
    rng = np.random.default_rng(seed + 7919)
    out = []
    bh_list = range(B * Hq) if heads is None else heads
    for bh in bh_list:
        if n_per_head >= Lq:
            idx = np.arange(Lq)
        else:
            idx = rng.choice(Lq, size=n_per_head, replace=False)
            idx[0], idx[-1] = 0, Lq - 1
            idx = np.unique(idx)
        out.append(bh * Lq + idx)
    return np.concatenate(out).astype(np.int64)


def batch_qkv(cfg: Config, b: int, seed=0, delta=None):
    """Batch element `b` of a large config (cfg3..cfg5), drawn on its own from
    default_rng([seed, b]) so that bench and tests can build the workload piece by piece:
    Q [Hq,Lq,d], K, V [Hkv,Lk,d] (FP32, sink construction as in sink_qkv)."""
    rng = np.random.default_rng([seed, b])
    d = cfg.d
    q = rng.standard_normal((cfg.Hq, cfg.Lq, d), dtype=np.float32)
    k = rng.standard_normal((cfg.Hkv, cfg.Lk, d), dtype=np.float32)
    v = rng.standard_normal((cfg.Hkv, cfg.Lk, d), dtype=np.float32)
    q[..., d - 1] = 1.0
    k[..., d - 1] = 0.0
    k[..., :cfg.n_sink, d - 1] = np.float32((cfg.delta if delta is None else delta) * np.sqrt(d))
    return q, k, v
