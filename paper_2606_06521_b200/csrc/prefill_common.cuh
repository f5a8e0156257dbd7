// prefill_common.cuh -- building blocks shared by the warp-specialised prefill kernels (attn_prefill.cuh, Bn = 128;
// attn_prefill64.cuh, Bn = 64): operand geometry, the exp / sum / cast pass of Alg. 1 lines 7-9
// on one 32-column chunk, the FMA-pipe exp2, row max / mask helpers, the P hand-off and the O rescale warp.
#pragma once
#include "common.cuh"

namespace fp8attn {

template <int EB>
struct PrefillCfg {
    static constexpr int D = 128, BN = 128;
    static constexpr int CH = 128 / EB;              // elements per 128-byte swizzle row
    static constexpr int NCH = D / CH;               // 128-byte chunks per operand row
    static constexpr int TILE = NCH * 128 * 128;     // bytes of one 128-row operand tile (Q, K_j or V_j)
    static constexpr int NS = (EB == 1) ? 4 : 2;     // K ring depth = V ring depth
    static constexpr int KSTEP = 32 / EB;            // contraction elements per MMA
    static constexpr int P_COLS = BN * EB / 4;       // TMEM columns of P
    static constexpr int TM_S = 0, TM_O = 256;
    static constexpr uint32_t KIND = (EB == 1) ? ptx::KIND_F8F6F4 : ptx::KIND_F16;
    static constexpr uint32_t FMT = (EB == 1) ? ptx::FMT_E4M3 : ptx::FMT_BF16;
};

// exact E4M3 pair -> BF16 pair: the code shifted left by 4 is the BF16 bit pattern of value * 2^-120
// (subnormal codes map to BF16 subnormals), and the packed multiply by 2^120 is exact.
__device__ __forceinline__ uint32_t e4m3x2_to_bf16x2(uint32_t pair) {
    const uint32_t spread = ((pair & 0xFF00u) << 12) | ((pair & 0xFFu) << 4);
    uint32_t r;
    asm("mul.rn.bf16x2 %0, %1, %2;" : "=r"(r) : "r"(spread), "r"(0x7B807B80u));   // 2^120 in both halves
    return r;
}

// 2^x for a packed pair on the FMA pipe (the MUFU pipe is the busy one in the exp pass): x = n + f with
// n = round(x) taken from the low mantissa bits of x + 1.5 * 2^23, f in [-0.5, 0.5], a degree-5 polynomial for
// 2^f (near-minimax, Chebyshev nodes; max relative error 2.3e-7 in FP32 Horner form, the same order as
// ex2.approx), and n added to the exponent field.  x is clamped at -125 (2^-125 casts to E4M3 zero and adds
// nothing to a row sum that holds at least one term equal to S).
__device__ __forceinline__ void exp2_poly2(uint64_t x2, float& r0, float& r1) {
    constexpr float MAGIC = 12582912.0f;
    float x0, x1;
    ptx::unpack2(x2, x0, x1);
    x0 = fmaxf(x0, -125.0f);
    x1 = fmaxf(x1, -125.0f);
    const uint64_t xc = ptx::pack2(x0, x1);
    const uint64_t t2 = ptx::add2(xc, ptx::pack2(MAGIC, MAGIC));
    const uint64_t n2 = ptx::add2(t2, ptx::pack2(-MAGIC, -MAGIC));
    const uint64_t f2 = ptx::fma2(n2, ptx::pack2(-1.0f, -1.0f), xc);
    uint64_t p2 = ptx::fma2(ptx::pack2(0.00134004f, 0.00134004f), f2, ptx::pack2(0.00967604f, 0.00967604f));
    p2 = ptx::fma2(p2, f2, ptx::pack2(0.05550327f, 0.05550327f));
    p2 = ptx::fma2(p2, f2, ptx::pack2(0.24022107f, 0.24022107f));
    p2 = ptx::fma2(p2, f2, ptx::pack2(0.6931472f, 0.6931472f));
    p2 = ptx::fma2(p2, f2, ptx::pack2(1.0000001f, 1.0000001f));
    float p0, p1, t0, t1;
    ptx::unpack2(p2, p0, p1);
    ptx::unpack2(t2, t0, t1);
    r0 = __int_as_float(__float_as_int(p0) + (__float_as_int(t0) << 23));
    r1 = __int_as_float(__float_as_int(p1) + (__float_as_int(t1) << 23));
}

// ---- one 32-column chunk of the exp pass (Alg. 1 lines 7-9) -------------------------------------
// v: raw logits of 32 keys.  Returns P codes / BF16 values in w (P_COLS/4 words) and adds the FP32
// pre-cast P (times S when the scale is folded into the exponent) to the two packed sums.
// NPOLY: bit i set = element pair i of the 16 pairs of the chunk takes exp2_poly2 instead of ex2.approx
// (0: all on the MUFU pipe).
// The two halves of exp_chunk: exp_part is line 7 (P = exp2 of the scaled, shifted logit; FP32), cast_part lines 8-9
// (row sum from the pre-cast P, the cast, the packing).  The exp warps of attn_prefill.cuh run the exp_part of BOTH
// their quarters first and the cast_part + hand-off of each afterwards, so that the MUFU pipe works on the second
// quarter while the first one is cast, stored and handed over.
template <bool MASK, int NPOLY>
__device__ __forceinline__ void exp_part(const uint32_t* v, float* pr, int j_first, int jlim, uint64_t cl2_2,
                                         uint64_t negm_2) {
#pragma unroll
    for (int e = 0; e < 32; e += 2) {
        uint32_t a = v[e], b = v[e + 1];
        if constexpr (MASK) {
            if (j_first + e > jlim) a = 0xFF800000u;       // -inf
            if (j_first + e + 1 > jlim) b = 0xFF800000u;
        }
        const uint64_t x = ptx::fma2(ptx::pack2u(a, b), cl2_2, negm_2);
        if ((NPOLY >> (e >> 1)) & 1) {
            exp2_poly2(x, pr[e], pr[e + 1]);
        } else {
            float x0, x1;
            ptx::unpack2(x, x0, x1);
            pr[e] = ptx::ex2_approx(x0);
            pr[e + 1] = ptx::ex2_approx(x1);
        }
    }
}
template <int EB, bool FOLD>
__device__ __forceinline__ void cast_part(const float* pr, uint32_t* w, uint64_t s_2, uint64_t& sum_a, uint64_t& sum_b) {
    uint32_t pair[16];
#pragma unroll
    for (int e = 0; e < 32; e += 4) {
        const uint64_t p0 = ptx::pack2(pr[e], pr[e + 1]), p1 = ptx::pack2(pr[e + 2], pr[e + 3]);
        sum_a = ptx::add2(sum_a, p0);
        sum_b = ptx::add2(sum_b, p1);
    }
    if constexpr (!FOLD) {
#pragma unroll
        for (int e = 0; e < 32; e += 2) {
            float y0, y1;
            ptx::unpack2(ptx::mul2(ptx::pack2(pr[e], pr[e + 1]), s_2), y0, y1);
            pair[e / 2] = ptx::cvt_e4m3x2(y0, y1);
        }
    } else {
#pragma unroll
        for (int e = 0; e < 32; e += 2) pair[e / 2] = ptx::cvt_e4m3x2(pr[e], pr[e + 1]);
    }
    if constexpr (EB == 1) {
#pragma unroll
        for (int e = 0; e < 8; ++e) w[e] = pair[2 * e] | (pair[2 * e + 1] << 16);
    } else {
#pragma unroll
        for (int e = 0; e < 16; ++e) w[e] = e4m3x2_to_bf16x2(pair[e]);
    }
}
template <int EB, bool FOLD, bool MASK, int NPOLY = 0>
__device__ __forceinline__ void exp_chunk(const uint32_t* v, uint32_t* w, int j_first, int jlim, uint64_t cl2_2,
                                          uint64_t negm_2, uint64_t s_2, uint64_t& sum_a, uint64_t& sum_b) {
    float pr[32];
    exp_part<MASK, NPOLY>(v, pr, j_first, jlim, cl2_2, negm_2);
    cast_part<EB, FOLD>(pr, w, s_2, sum_a, sum_b);
}

// max over 32 (masked) raw logits folded into m
__device__ __forceinline__ float max32(const uint32_t* v, float m) {
    float m0 = m, m1 = -INFINITY;
#pragma unroll
    for (int e = 0; e < 32; e += 4) {
        m0 = fmaxf(fmaxf(m0, __uint_as_float(v[e])), __uint_as_float(v[e + 1]));
        m1 = fmaxf(fmaxf(m1, __uint_as_float(v[e + 2])), __uint_as_float(v[e + 3]));
    }
    return fmaxf(m0, m1);
}
__device__ __forceinline__ void mask32(uint32_t* v, int j_first, int jlim) {
#pragma unroll
    for (int e = 0; e < 32; ++e)
        if (j_first + e > jlim) v[e] = 0xFF800000u;   // -inf
}


// Statistics of one 32-key chunk of P (statistics instances only): the E4M3 codes of the visible keys go to
// dump_row (this query row of the P dump of fp8attn_stats, or null) and the zero codes among the visible
// non-sink keys are counted and returned (Prop. 1; `count` false = not counted, 0).  w holds the
// chunk as exp_chunk leaves it; BF16 mode recovers a code from its exact BF16 value: times 2^-120, shifted right by 4.
// The general case (a dump, a sink key in the chunk, a masked key) is a function call: it runs for a few chunks per
// row, and inlined four times it doubles the size of the loop the exp warps live in.
template <int EB>
struct ChunkWords {
    uint32_t w[8 * EB];
};
template <int EB>
__device__ __noinline__ uint32_t chunk_statistics_general(ChunkWords<EB> cw, int jq, int jlim, uint8_t* dump_row,
                                                          uint32_t sinks) {
    uint32_t zeros = 0;
#pragma unroll
    for (int e = 0; e < 32; ++e) {
        uint32_t code;
        if constexpr (EB == 1) {
            code = (cw.w[e >> 2] >> (8 * (e & 3))) & 0xFFu;
        } else {
            uint32_t back;
            asm("mul.rn.bf16x2 %0, %1, %2;" : "=r"(back) : "r"(cw.w[e >> 1]), "r"(0x03800380u));   // 2^-120
            code = (back >> (16 * (e & 1) + 4)) & 0xFFu;
        }
        const bool vis = jq + e <= jlim;
        if (vis && dump_row != nullptr) dump_row[jq + e] = (uint8_t)code;
        if (vis && code == 0 && !((sinks >> e) & 1u)) ++zeros;
    }
    return zeros;
}
template <int EB>
__device__ __forceinline__ uint32_t chunk_statistics(const uint32_t* w, int jq, int jlim, uint8_t* dump_row, bool count,
                                                     const FwdParams& p, bool sink_blk) {
    constexpr int NW = 8 * EB;      // words of the chunk
    if (dump_row == nullptr && !count) return 0u;
    // which keys of the chunk are sink keys (sink_blk: the KV block of the chunk holds one at all)
    const uint32_t sinks = sink_blk ? sink_mask32(p, jq) : 0u;
    if (dump_row == nullptr && sinks == 0u && jq + 31 <= jlim) {
        // every key of the chunk is visible and none is a sink: count the NON-zero codes a word at a time.  P >= 0,
        // so a code is at most 0x7E (a BF16 value at most 0x7FFF) and adding 0x7F.. sets the top bit of exactly the
        // non-zero lanes without a carry between them; no popc (it shares the MUFU pipe with ex2)
        uint32_t nz = 0;
#pragma unroll
        for (int i = 0; i < NW; ++i) {
            if constexpr (EB == 1) nz = __dp4a((w[i] + 0x7F7F7F7Fu) & 0x80808080u, 0x01010101u, nz);   // += 128 per code
            else nz += ((w[i] + 0x7FFF7FFFu) >> 15) & 0x00010001u;
        }
        return 32u - ((EB == 1) ? (nz >> 7) : ((nz & 0xFFFFu) + (nz >> 16)));
    }
    ChunkWords<EB> cw;
#pragma unroll
    for (int i = 0; i < NW; ++i) cw.w[i] = w[i];
    const uint32_t zeros = chunk_statistics_general<EB>(cw, jq, jlim, dump_row, sinks);
    return count ? zeros : 0u;
}

}  // namespace fp8attn
