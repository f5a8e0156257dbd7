"""Multi-GPU sharding of the attention forward.

Every (batch element, kv head) pair -- a kv head together with the Hq/Hkv query heads that read it -- is an
independent unit of Alg. 1: no value crosses from one unit to another.  The units are split into `world`
contiguous, balanced ranges, one per rank; each rank runs `fp8attn_fwd` on views of its own range and writes
its own rows of `o`.  There is NO data-path collective; the only communication is the barrier and the
max-over-ranks reduction of the timing in bench.py.  Host logic only: nothing here touches CUDA.
"""
from dataclasses import dataclass
from typing import List


@dataclass(frozen=True)
class Shard:
    """Units [lo, hi) of the flattened (b, kv head) index u = b * Hkv + kvh, and the calls that cover them:
    one `Piece` per batch element the range touches."""
    rank: int
    lo: int
    hi: int
    pieces: tuple


@dataclass(frozen=True)
class Piece:
    b: int            # batch element
    kvh_lo: int       # kv heads [kvh_lo, kvh_hi) of that batch element
    kvh_hi: int
    hq_lo: int        # the query heads that read them: [hq_lo, hq_hi) = [kvh_lo * G, kvh_hi * G)
    hq_hi: int


def unit_range(rank: int, world: int, n_units: int):
    """Balanced contiguous split: the first n_units % world ranks get one unit more."""
    if not (0 <= rank < world) or n_units < 0:
        raise ValueError("bad rank / world / n_units")
    base, extra = divmod(n_units, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def shard(rank: int, world: int, B: int, Hq: int, Hkv: int) -> Shard:
    if Hq % Hkv:
        raise ValueError("Hq must be a multiple of Hkv")
    g = Hq // Hkv
    lo, hi = unit_range(rank, world, B * Hkv)
    pieces: List[Piece] = []
    u = lo
    while u < hi:
        b, k0 = divmod(u, Hkv)
        k1 = min(Hkv, k0 + (hi - u))
        pieces.append(Piece(b, k0, k1, k0 * g, k1 * g))
        u += k1 - k0
    return Shard(rank, lo, hi, tuple(pieces))


def run_sharded(fwd, q, k, v, o, rank: int, world: int, **kw):
    """Run `fwd(q_view, k_view, v_view, out=o_view, **kw)` on every piece of this rank's shard.  q, o:
    [B,Hq,Lq,d]; k, v: [B,Hkv,Lk,d] (any array type with numpy-style slicing; the views of one piece are
    contiguous in memory when the piece covers whole batch elements, otherwise the caller's `fwd` must accept
    strided heads or copy).  Per-head scale arrays in `kw` named q_scale / k_scale / v_scale are sliced too."""
    B, Hq = q.shape[0], q.shape[1]
    Hkv = k.shape[1]
    out = []
    for pc in shard(rank, world, B, Hq, Hkv).pieces:
        kw_p = dict(kw)
        for name, lo_, hi_ in (("q_scale", pc.hq_lo, pc.hq_hi), ("k_scale", pc.kvh_lo, pc.kvh_hi),
                               ("v_scale", pc.kvh_lo, pc.kvh_hi)):
            if kw_p.get(name) is not None:
                kw_p[name] = kw_p[name][pc.b:pc.b + 1, lo_:hi_]
        out.append(fwd(q[pc.b:pc.b + 1, pc.hq_lo:pc.hq_hi], k[pc.b:pc.b + 1, pc.kvh_lo:pc.kvh_hi],
                       v[pc.b:pc.b + 1, pc.kvh_lo:pc.kvh_hi], out=o[pc.b:pc.b + 1, pc.hq_lo:pc.hq_hi], **kw_p))
    return out
