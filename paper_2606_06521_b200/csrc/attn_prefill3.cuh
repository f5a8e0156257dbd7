// attn_prefill3.cuh -- prefill kernel, third structure: correction warpgroups + boustrophedon quarters.
//
// Same arithmetic as attn_prefill.cuh (Alg. 1: exact running max after every block, l from
// the FP32 pre-cast P, cvt.rn.satfinite.e4m3x2.f32 of P*S, epilogue O / (S l)); d = 128, Bn = 128, two
// 128-row query tiles per CTA.  What changes is who does what and in which order, to shorten the serial
// chain between the exp pass of block c and the exp pass of block c+1 of a tile:
//   * O <- alpha O (Alg. 1 line 10, first half) is done by a correction warpgroup per tile, in parallel with
//     the exp pass of the softmax warpgroup; the MMA issuer waits for it before the first P.V of the block.
//   * The four 32-key quarters of a block are processed in the order 0,1,2,3 on even blocks and 3,2,1,0 on
//     odd blocks.  QK^T of block c+1 is issued in two halves: the half whose P quarters were consumed first
//     ("early", right after the second P.V of block c) and the other one ("late", after the fourth P.V).
//     The softmax warps take the max of the early half while the tensor pipe is still finishing block c,
//     then load the late half ONCE, keep it in registers through the max and start the exp pass on it, so
//     between the last P quarter of block c and the first ex2 of block c+1 there is one P.V quarter, one
//     N = 64 QK^T group, one 64-column TMEM load and 32 FMNMX3.
// Roles (640 threads, register budgets moved with setmaxnreg):
//   warps 0-3 / 4-7    softmax of tile 0 / 1 (one query row per thread = TMEM lane)        144 registers
//   warps 8-11 / 12-15 correction of tile 0 / 1                                            72 registers
//   warps 16, 17       tcgen05.mma issuers of tile 0 / 1;  warp 18 TMA producer;  19 idle  40 registers
// TMEM (512 columns): S0 [0,128) S1 [128,256) O0 [256,384) O1 [384,512); P over the head of each S quarter.
#pragma once
#include "attn_prefill.cuh"

namespace fp8attn {

// Development aid (off in the product build): -DFP8ATTN_TRACE records clock64 stamps of warps 0 and 4 of
// CTA (0,0) into g_trace3[tile][block][16], read back with fp8attn_debug_trace.
#ifdef FP8ATTN_TRACE
__device__ long long g_trace3[2 * 80 * 16];
#define FP8ATTN_STAMP3(k)                                                                          \
    do {                                                                                           \
        if (blockIdx.x == 0 && blockIdx.y == 0 && (threadIdx.x & 127) == 0 && c < 80)              \
            g_trace3[((threadIdx.x >> 7) * 80 + c) * 16 + (k)] = clock64();                        \
    } while (0)
#else
#define FP8ATTN_STAMP3(k) do { } while (0)
#endif

template <int EB>
struct Prefill3Cfg {
    using P = PrefillCfg<EB>;
    static constexpr int THREADS = 640;
    // q_full[2] k_full/k_empty/v_full/v_empty[NS] s_full[2][2] p_full[2][4] a_full[2][4] o_ready[2] o_done[2]
    static constexpr int N_BARS = 2 + 4 * P::NS + 4 + 8 + 8 + 2 + 2 + 8;   // + tok[2][4]
    static constexpr int SMEM_BYTES = (2 + 2 * P::NS) * P::TILE + 1024 /*align*/ + N_BARS * 8 + 16 + 2 * 128 * 4;
    static constexpr int REG_SOFTMAX = 144, REG_CORR = 72, REG_MISC = 40;   // 256 (144 + 72) + 128 * 40 <= 640 * 96, the pool the launch allocates
};

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

// State a softmax thread carries from block to block.
struct SoftmaxState {
    uint32_t r[64];      // raw logits of the late half of the current block (masked), quarters ord[0], ord[1]
    float m_early;       // max over the early half of the current block (masked)
    float m_run, l_run;  // Alg. 1 running max (raw logit units) and row sum (times S when folded)
};

// Loads block n (direction DN = n & 1) into the state: max of the early half, late half resident.
// Early half of a block of direction DN is H1 for DN = 0 and H0 for DN = 1 (see the file header).
__device__ __forceinline__ void load_block(SoftmaxState& s, uint32_t tS, uint64_t* s_full, int n, int j0, bool mask,
                                           int jlim) {
    const int DN = n & 1;                                // direction: only TMEM column offsets depend on it
    const int EH = DN ? 0 : 1;                           // early half
    const int Q0 = DN ? 3 : 0, Q1 = DN ? 2 : 1;          // first two quarters of the block's order (late half)
    ptx::mbar_wait(s_full + 0, n & 1);
    ptx::tc_fence_after();
    ptx::tmem_ld_x32(tS + EH * 64, s.r);
    ptx::tmem_ld_x32(tS + EH * 64 + 32, s.r + 32);
    ptx::tmem_wait_ld();
    if (mask) {
        mask32(s.r, j0 + EH * 64, jlim);
        mask32(s.r + 32, j0 + EH * 64 + 32, jlim);
    }
    s.m_early = fmaxf(max32(s.r, -INFINITY), max32(s.r + 32, -INFINITY));
    ptx::mbar_wait(s_full + 1, n & 1);
    ptx::tc_fence_after();
    ptx::tmem_ld_x32(tS + Q0 * 32, s.r);
    ptx::tmem_ld_x32(tS + Q1 * 32, s.r + 32);
    ptx::tmem_wait_ld();
    if (mask) {
        mask32(s.r, j0 + Q0 * 32, jlim);
        mask32(s.r + 32, j0 + Q1 * 32, jlim);
    }
}

// One P quarter: exp / sum / cast (exp_chunk), P over the head of its S quarter, hand-off to the issuer.
// AUX (statistics instance): the E4M3 codes of the visible keys also go to dump_row (row of the P dump of
// fp8attn_stats) and the zero codes among the visible non-sink keys are counted into *uf (Prop. 1,
// PAPER.md:147-155).  BF16 mode recovers a code from its exact BF16 value: times 2^-120, shifted right by 4.
template <int EB, bool FOLD, int NPOLY = 0, bool AUX = false>
__device__ __forceinline__ void p_quarter(const uint32_t* v, bool mask, uint32_t tS, int quarter, int j0, int jlim,
                                          uint64_t cl2_2, uint64_t negm_2, uint64_t s_2, uint64_t& sum_a,
                                          uint64_t& sum_b, uint64_t* bar, int lane, uint8_t* dump_row = nullptr,
                                          uint32_t* uf = nullptr, int n_sink = 0) {
    using C = PrefillCfg<EB>;
    uint32_t w[C::P_COLS / 4];
    if (mask) exp_chunk<EB, FOLD, true>(v, w, j0 + quarter * 32, jlim, cl2_2, negm_2, s_2, sum_a, sum_b);
    else exp_chunk<EB, FOLD, false, NPOLY>(v, w, j0 + quarter * 32, jlim, cl2_2, negm_2, s_2, sum_a, sum_b);
    if constexpr (AUX) {
        const int jq = j0 + quarter * 32;
        if (dump_row == nullptr && uf != nullptr && jq >= n_sink && jq + 31 <= jlim) {
            // every key of the quarter is visible and none is a sink: count the zero codes a word at a time
            uint32_t zeros = 0;
#pragma unroll
            for (int i = 0; i < C::P_COLS / 4; ++i)
                zeros += (EB == 1) ? (__popc(__vcmpeq4(w[i], 0u)) >> 3) : (__popc(__vcmpeq2(w[i], 0u)) >> 4);
            *uf += zeros;
        } else if (dump_row != nullptr || uf != nullptr) {
            uint32_t zeros = 0;
#pragma unroll
            for (int e = 0; e < 32; ++e) {
                uint32_t code;
                if constexpr (EB == 1) {
                    code = (w[e >> 2] >> (8 * (e & 3))) & 0xFFu;
                } else {
                    uint32_t back;
                    asm("mul.rn.bf16x2 %0, %1, %2;" : "=r"(back) : "r"(w[e >> 1]), "r"(0x03800380u));   // 2^-120
                    code = (back >> (16 * (e & 1) + 4)) & 0xFFu;
                }
                const bool vis = jq + e <= jlim;
                if (vis && dump_row != nullptr) dump_row[jq + e] = (uint8_t)code;
                if (vis && jq + e >= n_sink && code == 0) ++zeros;
            }
            if (uf != nullptr) *uf += zeros;
        }
    }
    if constexpr (EB == 1) ptx::tmem_st_x8(tS + quarter * 32, w);
    else ptx::tmem_st_x16(tS + quarter * 32, w);
    ptx::tmem_wait_st();
    ptx::tc_fence_before();
    __syncwarp();
    if (lane == 0) ptx::mbar_arrive(bar);
}

// Geometry of block n of a tile: first key index and whether some row of the warp needs the mask.
struct BlockGeo {
    int j0;
    bool mask;
};
__device__ __forceinline__ BlockGeo block_geo(const FwdParams& p, int n, int n_t, long long warp_vis) {
    const int blk = (p.kv_order == 0) ? n : n_t - 1 - n;
    BlockGeo g;
    g.j0 = blk * 128;
    g.mask = (g.j0 + 127 > warp_vis) || (g.j0 + 128 > p.Lk);
    return g;
}

// Alg. 1 lines 4-9 for block c (direction D = c & 1), then the loads of block c+1.
template <int EB, bool FOLD>
__device__ __forceinline__ void softmax_block(SoftmaxState& s, const FwdParams& p, int c, int n_t, uint32_t tS,
                                              uint64_t* s_full, uint64_t* p_full, uint64_t* a_full_w,
                                              float* alpha_slot, int lane, float cl2, float log2S, uint64_t cl2_2,
                                              uint64_t s_2, int jlim, long long warp_vis, uint64_t* tok_take,
                                              int take_idx, uint64_t* tok_give) {
    const int D = c & 1;
    const int Q0 = D ? 3 : 0, Q1 = D ? 2 : 1, Q2 = D ? 1 : 2, Q3 = D ? 0 : 3;
    const BlockGeo g = block_geo(p, c, n_t, warp_vis);
    FP8ATTN_STAMP3(0);
    // ---- lines 4-6: block max, running max, alpha; alpha goes to the correction warp of these rows ----
    const float mloc = fmaxf(s.m_early, fmaxf(max32(s.r, -INFINITY), max32(s.r + 32, -INFINITY)));
    const float m_new = fmaxf(s.m_run, mloc);
    const float m_used = (m_new == -INFINITY) ? 0.0f : m_new;
    const float alpha = ptx::ex2_approx((s.m_run - m_used) * cl2);   // 0 when m_run = -inf
    const float negm = fmaf(-m_used, cl2, log2S);
    const uint64_t negm_2 = ptx::pack2(negm, negm);
    *alpha_slot = alpha;
    __syncwarp();
    if (lane == 0) ptx::mbar_arrive(a_full_w);
    // the two tiles take turns on the MUFU pipe: wait until the partner warp of the other tile (same
    // scheduler) has issued the exps of the block that precedes this one in the interleaved order
    if (take_idx >= 0) ptx::mbar_wait(tok_take, take_idx & 1);
    FP8ATTN_STAMP3(1);

    // ---- lines 7-9: four P quarters; the first two come from the resident half ----
    uint64_t sum_a = ptx::pack2(0.f, 0.f), sum_b = sum_a;
    uint32_t x[32];
    ptx::tmem_ld_x32(tS + Q2 * 32, x);            // in flight during the first two quarters
    p_quarter<EB, FOLD>(s.r, false, tS, Q0, g.j0, jlim, cl2_2, negm_2, s_2, sum_a, sum_b, p_full + 0, lane);
    FP8ATTN_STAMP3(2);
    p_quarter<EB, FOLD>(s.r + 32, false, tS, Q1, g.j0, jlim, cl2_2, negm_2, s_2, sum_a, sum_b, p_full + 1, lane);
    FP8ATTN_STAMP3(3);
    ptx::tmem_wait_ld();
    ptx::tmem_ld_x32(tS + Q3 * 32, s.r);          // in flight during the third quarter
    p_quarter<EB, FOLD>(x, g.mask, tS, Q2, g.j0, jlim, cl2_2, negm_2, s_2, sum_a, sum_b, p_full + 2, lane);
    FP8ATTN_STAMP3(4);
    ptx::tmem_wait_ld();
    p_quarter<EB, FOLD>(s.r, g.mask, tS, Q3, g.j0, jlim, cl2_2, negm_2, s_2, sum_a, sum_b, p_full + 3, lane);
    FP8ATTN_STAMP3(5);
    // the MUFU pipe of this scheduler goes to the partner warp of the other tile
    if (tok_give) {
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(tok_give);
    }

    // ---- block c+1: early-half max while the tensor pipe finishes block c, then the late half ----
    if (c + 1 < n_t) {
        const BlockGeo gn = block_geo(p, c + 1, n_t, warp_vis);
        load_block(s, tS, s_full, c + 1, gn.j0, gn.mask, jlim);
    }
    float sa, sb, sc, sd;
    ptx::unpack2(sum_a, sa, sb);
    ptx::unpack2(sum_b, sc, sd);
    s.l_run = alpha * s.l_run + ((sa + sb) + (sc + sd));   // line 8
    s.m_run = m_new;
}

// ---- softmax warpgroup of one tile ----------------------------------------------------------------
template <int EB, bool FOLD>
__device__ __forceinline__ void prefill3_softmax(const FwdParams& p, int t, int wq, int lane, uint32_t tbase,
                                                 uint64_t* s_full, uint64_t* p_full, uint64_t* a_full_w,
                                                 float* alpha_slot, uint64_t* o_done, int n_t, int row0, int bh,
                                                 int kvh, uint64_t* tok_take, uint64_t* tok_give, int first,
                                                 int first_other, int n_other) {
    using C = PrefillCfg<EB>;
    const uint32_t tlane = tbase + (static_cast<uint32_t>(wq * 32) << 16);
    const uint32_t tS = tlane + C::TM_S + t * 128, tO = tlane + C::TM_O + t * 128;
    const int qrow = row0 + wq * 32 + lane;
    const int off = p.Lk - p.Lq;
    long long jl = p.causal ? (long long)qrow + off : (long long)p.Lk - 1;
    if (jl > p.Lk - 1) jl = p.Lk - 1;
    const int jlim = (int)jl;
    const int warp_first_row = row0 + wq * 32;
    const long long warp_vis = p.causal ? (long long)warp_first_row + off : (long long)p.Lk - 1;

    float c_nat = p.sm_scale, vs = 1.0f;
    if constexpr (EB == 1) {
        c_nat *= p.q_scale[bh] * p.k_scale[kvh];
        vs = p.v_scale[kvh];
    }
    const float cl2 = c_nat * LOG2E;
    const float log2S = FOLD ? log2f(p.S) : 0.0f;   // exact for S = 2^k
    const uint64_t cl2_2 = ptx::pack2(cl2, cl2), s_2 = ptx::pack2(p.S, p.S);

    SoftmaxState s;
    s.m_run = -INFINITY;
    s.l_run = 0.0f;
    s.m_early = -INFINITY;
    if (n_t > 0) {
        const BlockGeo g0 = block_geo(p, 0, n_t, warp_vis);
        load_block(s, tS, s_full, 0, g0.j0, g0.mask, jlim);
    }
    // Interleaved order of the exp passes: ... (it, tile 1), (it, tile 0), (it + 1, tile 1) ...  (it = K/V ring
    // iteration = c + first).  tok[1]: tile 1 gives and tile 0 takes on the iterations both tiles take part in;
    // tok[0]: tile 0 gives on iteration j and tile 1 takes on j + 1 where both exist.  Gives and takes pair
    // one to one in order, so the parity of a phase is the parity of its index in the range.  The tokens only
    // order the use of the MUFU pipe, no value depends on them.
    const int f0 = (t == 0) ? first : first_other, f1 = (t == 0) ? first_other : first;
    const int e0 = f0 + ((t == 0) ? n_t : n_other), e1 = f1 + ((t == 0) ? n_other : n_t);
    const int loA = max(f0, f1), hiA = min(e0, e1);
    const int loB = max(f0, f1 - 1), hiB = min(e0, e1 - 1);
    auto take = [&](int c) {
        if (tok_take == nullptr) return -1;
        const int it = c + first;
        if (t == 0) return (it >= loA && it < hiA) ? it - loA : -1;
        return (it - 1 >= loB && it - 1 < hiB) ? it - 1 - loB : -1;
    };
    auto give = [&](int c) {
        const int it = c + first;
        const bool g = (t == 0) ? (it >= loB && it < hiB) : (it >= loA && it < hiA);
        return g ? tok_give : nullptr;
    };
#pragma unroll 1
    for (int c = 0; c < n_t; ++c)
        softmax_block<EB, FOLD>(s, p, c, n_t, tS, s_full, p_full, a_full_w, alpha_slot, lane, cl2, log2S, cl2_2, s_2,
                                jlim, warp_vis, tok_take, take(c), give(c));
    const float m_run = s.m_run, l_run = s.l_run;

    // ---- line 12: O / (S l), statistics ----
    const long long grow = (long long)bh * p.Lq + qrow;
    const float l_true = FOLD ? l_run / p.S : l_run;
    if (qrow < p.Lq) {
        if (p.row_max) p.row_max[grow] = (m_run == -INFINITY) ? -INFINITY : m_run * c_nat;
        if (p.row_sum) p.row_sum[grow] = l_true;
    }
    const float inv = (l_run > 0.0f) ? (FOLD ? vs / l_run : vs / (p.S * l_run)) : 0.0f;
    if (n_t > 0) {
        ptx::mbar_wait(o_done, 0);
        ptx::tc_fence_after();
    }
    float* dst = p.o + grow * C::D;
#pragma unroll 1
    for (int cb = 0; cb < 4; ++cb) {
        uint32_t v[32];
        if (n_t > 0) {
            ptx::tmem_ld_x32(tO + cb * 32, v);
            ptx::tmem_wait_ld();
        } else {
#pragma unroll
            for (int e = 0; e < 32; ++e) v[e] = 0u;
        }
        if (qrow < p.Lq) {
#pragma unroll
            for (int e = 0; e < 32; e += 4) {
                float4 o4 = make_float4(__uint_as_float(v[e]) * inv, __uint_as_float(v[e + 1]) * inv,
                                        __uint_as_float(v[e + 2]) * inv, __uint_as_float(v[e + 3]) * inv);
                if (l_run <= 0.0f) o4 = make_float4(0.f, 0.f, 0.f, 0.f);
                *reinterpret_cast<float4*>(dst + cb * 32 + e) = o4;
            }
        }
    }
}

// ---- correction warp: O <- alpha O for its 32 rows, once per block ---------------------------------
__device__ __forceinline__ void prefill3_correction(int t, int wq, int lane, uint32_t tbase, uint64_t* a_full_w,
                                                    const float* alpha_slot, uint64_t* o_ready, int n_t) {
    const uint32_t tO = tbase + (static_cast<uint32_t>(wq * 32) << 16) + 256 + t * 128;
    for (int c = 0; c < n_t; ++c) {
        ptx::mbar_wait(a_full_w, c & 1);
        const float alpha = *alpha_slot;
        // alpha(c) is published after S(c) is complete, which implies P.V(c-1) is complete (in-order pipe)
        if (c > 0 && __any_sync(0xFFFFFFFFu, alpha != 1.0f)) {
            ptx::tc_fence_after();
            const uint64_t a2 = ptx::pack2(alpha, alpha);
            uint32_t va[16], vb[16];
            ptx::tmem_ld_x16(tO, va);
#pragma unroll
            for (int cb = 0; cb < 8; ++cb) {
                uint32_t* cur = (cb & 1) ? vb : va;
                uint32_t* nxt = (cb & 1) ? va : vb;
                ptx::tmem_wait_ld();
                if (cb < 7) ptx::tmem_ld_x16(tO + (cb + 1) * 16, nxt);
#pragma unroll
                for (int e = 0; e < 16; e += 2) {
                    float y0, y1;
                    ptx::unpack2(ptx::mul2(ptx::pack2u(cur[e], cur[e + 1]), a2), y0, y1);
                    cur[e] = __float_as_uint(y0);
                    cur[e + 1] = __float_as_uint(y1);
                }
                ptx::tmem_st_x16(tO + cb * 16, cur);
            }
            ptx::tmem_wait_st();
        }
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(o_ready);
    }
}

// ---- the kernel ---------------------------------------------------------------------------------
// grid = (ceil(Lq / 256), B*Hq).  Causal launches the heaviest tile pairs first.
template <int EB, bool FOLD>
__global__ void __launch_bounds__(640, 1)
attn_prefill3_kernel(const __grid_constant__ CUtensorMap mapQ, const __grid_constant__ CUtensorMap mapK,
                     const __grid_constant__ CUtensorMap mapV, const FwdParams p) {
    using C = PrefillCfg<EB>;
    using C3 = Prefill3Cfg<EB>;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint8_t* sQ = smem;                           // 2 tiles
    uint8_t* sK = sQ + 2 * C::TILE;               // NS tiles
    uint8_t* sV = sK + C::NS * C::TILE;           // NS tiles
    uint64_t* bars = reinterpret_cast<uint64_t*>(sV + C::NS * C::TILE);
    uint64_t* q_full = bars;                      // [2]
    uint64_t* k_full = bars + 2;                  // [NS]
    uint64_t* k_empty = k_full + C::NS;
    uint64_t* v_full = k_empty + C::NS;
    uint64_t* v_empty = v_full + C::NS;
    uint64_t* s_full = v_empty + C::NS;           // [2 tiles][early, late]      MMA -> softmax
    uint64_t* p_full = s_full + 4;                // [2 tiles][4 steps]          softmax (4 warps) -> MMA
    uint64_t* a_full = p_full + 8;                // [2 tiles][4 warps]          softmax warp -> correction warp
    uint64_t* o_ready = a_full + 8;               // [2]                         correction (4 warps) -> MMA
    uint64_t* o_done = o_ready + 2;               // [2]
    uint64_t* tok = o_done + 2;                   // [2][4]  tok[t][wq]: tile t has issued the exps of a block
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tok + 8);
    float* alpha_s = reinterpret_cast<float*>(tmem_slot + 4);   // [2 tiles][128 rows]

    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xFFFFFFFFu, tid >> 5, 0);   // provably warp-uniform
    const int pair = p.causal ? (int)(gridDim.x - 1 - blockIdx.x) : (int)blockIdx.x;
    const int bh = blockIdx.y;
    const int b = bh / p.Hq, h = bh % p.Hq;
    const int kvh = b * p.Hkv + h / (p.Hq / p.Hkv);

    // visible block count of each tile (bottom-right causal, reading R15)
    int n_tile[2];
#pragma unroll
    for (int t = 0; t < 2; ++t) {
        const long long r0 = (long long)(pair * 2 + t) * BM;
        int n = 0;
        if (r0 < p.Lq) {
            n = p.nb;
            if (p.causal) {
                long long kmax = r0 + (BM - 1) + (p.Lk - p.Lq);
                if (kmax > p.Lk - 1) kmax = p.Lk - 1;
                n = kmax < 0 ? 0 : (int)(kmax / C::BN) + 1;
            }
        }
        n_tile[t] = n;
    }
    const int n_it = n_tile[0] > n_tile[1] ? n_tile[0] : n_tile[1];

    if (tid == 0) {
        ptx::prefetch_tmap(&mapQ);
        ptx::prefetch_tmap(&mapK);
        ptx::prefetch_tmap(&mapV);
        for (int i = 0; i < 2; ++i) ptx::mbar_init(q_full + i, 1);
        for (int i = 0; i < C::NS; ++i) {
            ptx::mbar_init(k_full + i, 1);
            ptx::mbar_init(v_full + i, 1);
            ptx::mbar_init(k_empty + i, 2);   // one arrival per tile
            ptx::mbar_init(v_empty + i, 2);
        }
        for (int i = 0; i < 4; ++i) ptx::mbar_init(s_full + i, 1);
        for (int i = 0; i < 8; ++i) {
            ptx::mbar_init(p_full + i, 4);
            ptx::mbar_init(a_full + i, 1);
            ptx::mbar_init(tok + i, 1);
        }
        for (int i = 0; i < 2; ++i) {
            ptx::mbar_init(o_ready + i, 4);
            ptx::mbar_init(o_done + i, 1);
        }
        ptx::fence_mbar_init();
    }
    if (warp == 16) {
        __syncwarp();
        ptx::tmem_alloc(tmem_slot, 512);
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tbase = *tmem_slot;

    if (warp < 8) {
        ptx::setmaxnreg_inc<C3::REG_SOFTMAX>();
        const int t = warp >> 2, wq = warp & 3;
        prefill3_softmax<EB, FOLD>(p, t, wq, lane, tbase, s_full + 2 * t, p_full + 4 * t, a_full + 4 * t + wq,
                                   alpha_s + t * 128 + wq * 32 + lane, o_done + t, n_tile[t], (pair * 2 + t) * BM, bh,
                                   kvh, p.alternate ? tok + 4 * (t ^ 1) + wq : nullptr,
                                   p.alternate ? tok + 4 * t + wq : nullptr, (p.kv_order == 0) ? 0 : n_it - n_tile[t],
                                   (p.kv_order == 0) ? 0 : n_it - n_tile[t ^ 1], n_tile[t ^ 1]);
    } else if (warp < 16) {
        ptx::setmaxnreg_dec<C3::REG_CORR>();
        const int t = (warp - 8) >> 2, wq = warp & 3;
        prefill3_correction(t, wq, lane, tbase, a_full + 4 * t + wq, alpha_s + t * 128 + wq * 32 + lane, o_ready + t,
                            n_tile[t]);
    } else {
        ptx::setmaxnreg_dec<C3::REG_MISC>();
        if (warp == 18) {
            // ================= TMA producer =================
            if (lane == 0 && n_it > 0) {
                for (int t = 0; t < 2; ++t) {
                    if (n_tile[t] == 0) continue;
                    ptx::mbar_arrive_expect_tx(q_full + t, C::TILE);
                    for (int c = 0; c < C::NCH; ++c)
                        ptx::tma_load_3d(sQ + t * C::TILE + c * (128 * 128), &mapQ, q_full + t, c * C::CH,
                                         (pair * 2 + t) * BM, bh);
                }
                for (int it = 0; it < n_it; ++it) {
                    const int blk = (p.kv_order == 0) ? it : n_it - 1 - it;
                    const int st = it % C::NS;
                    const uint32_t ph = (it / C::NS) & 1;
                    ptx::mbar_wait(k_empty + st, ph ^ 1);
                    ptx::mbar_arrive_expect_tx(k_full + st, C::TILE);
                    for (int c = 0; c < C::NCH; ++c)
                        ptx::tma_load_3d(sK + st * C::TILE + c * (128 * 128), &mapK, k_full + st, c * C::CH,
                                         blk * C::BN, kvh);
                    ptx::mbar_wait(v_empty + st, ph ^ 1);
                    ptx::mbar_arrive_expect_tx(v_full + st, C::TILE);
                    for (int c = 0; c < C::NCH; ++c)
                        ptx::tma_load_3d(sV + st * C::TILE + c * (128 * 128), &mapV, v_full + st, c * C::CH,
                                         blk * C::BN, kvh);
                }
            }
        } else if (warp < 18 && n_tile[warp - 16] > 0) {
            // ================= MMA issuer of tile t = warp - 16 =================
            // Block c of tile t uses K/V ring iteration it = c + first (in reverse order the tile with fewer
            // visible blocks joins later).  A ring slot is released by two arrivals, one per tile; on
            // iterations that only one tile uses, that tile arrives twice.
            const int t = warp - 16;
            const int n_t = n_tile[t];
            const bool leader = ptx::elect_one();
            constexpr uint32_t idesc_qk = ptx::make_idesc(C::FMT, C::FMT, ptx::MAJOR_K, ptx::MAJOR_K, BM, 64);
            constexpr uint32_t idesc_pv = ptx::make_idesc(C::FMT, C::FMT, ptx::MAJOR_K, ptx::MAJOR_MN, BM, C::D);
            constexpr uint32_t desc_hi = ptx::smem_desc_hi(1024);
            const uint32_t q_lo = ptx::smem_desc_lo(ptx::smem_u32(sQ + t * C::TILE), 16);
            const uint32_t k_lo = ptx::smem_desc_lo(ptx::smem_u32(sK), 16);
            const uint32_t v_lo = ptx::smem_desc_lo(ptx::smem_u32(sV), C::BN * 128);
            const uint32_t tS = tbase + C::TM_S + t * 128, tO = tbase + C::TM_O + t * 128;
            const int first = (p.kv_order == 0) ? 0 : n_it - n_t;
            const int n_other = n_tile[t ^ 1];
            const int first_other = (p.kv_order == 0) ? 0 : n_it - n_other;
            uint64_t* const sf = s_full + 2 * t;
            uint64_t* const pf = p_full + 4 * t;

            // S_t[:, 64 half .. 64 half + 64) = Q_t K[64 half .. 64 half + 64, :]^T on ring iteration it;
            // which = 0: early half of its block (waits for the K tile), 1: late half (releases the K tile)
            auto qk_half = [&](const int half, const int it, const int which) {
                const int st = it % C::NS;
                if (which == 0) {
                    ptx::mbar_wait(k_full + st, (it / C::NS) & 1);
                    ptx::tc_fence_after();
                }
                if (leader) {
                    const uint32_t b0 = k_lo + st * (C::TILE >> 4) + half * ((64 * 128) >> 4);
#pragma unroll
                    for (int ks = 0; ks < C::D / C::KSTEP; ++ks) {
                        const uint32_t o = (((ks * 32) / 128) * (128 * 128) + (ks * 32) % 128) >> 4;
                        ptx::mma_ss<C::KIND>(tS + half * 64, ptx::pack2u(q_lo + o, desc_hi),
                                             ptx::pack2u(b0 + o, desc_hi), idesc_qk, ks > 0 ? 1u : 0u);
                    }
                    ptx::tc_commit(sf + which);
                    if (which == 1) {
                        ptx::tc_commit(k_empty + st);
                        if (it < first_other || it >= first_other + n_other) ptx::tc_commit(k_empty + st);
                    }
                }
            };
            // O_t += P_t[:, 32q .. 32q+32) V[32q .. 32q+32, :]
            auto pv_quarter = [&](const int q, const int it, const uint32_t acc0, const bool last_of_tile,
                                  const bool release) {
                const int st = it % C::NS;
                if (leader) {
                    const uint32_t b0 = v_lo + st * (C::TILE >> 4) + q * ((32 * 128) >> 4);
                    uint32_t acc = acc0;
#pragma unroll
                    for (int ks = 0; ks < 32 / C::KSTEP; ++ks) {
                        ptx::mma_ts<C::KIND>(tO, tS + q * 32 + ks * 8,
                                             ptx::pack2u(b0 + ks * ((C::KSTEP * 128) >> 4), desc_hi), idesc_pv, acc);
                        acc = 1;
                    }
                    if (last_of_tile) ptx::tc_commit(o_done + t);
                    if (release) {
                        ptx::tc_commit(v_empty + st);
                        if (it < first_other || it >= first_other + n_other) ptx::tc_commit(v_empty + st);
                    }
                }
            };

            ptx::mbar_wait(q_full + t, 0);
            ptx::tc_fence_after();
            qk_half(1, first, 0);      // block 0 has direction 0: early half H1, late half H0
            qk_half(0, first, 1);
            for (int c = 0; c < n_t; ++c) {
                const int it = c + first;
                const int dir = c & 1;
                const bool has_next = c + 1 < n_t;
                ptx::mbar_wait(v_full + it % C::NS, (it / C::NS) & 1);
                ptx::mbar_wait(o_ready + t, c & 1);
#pragma unroll
                for (int s = 0; s < 4; ++s) {
                    const int q = dir ? 3 - s : s;
                    ptx::mbar_wait(pf + s, c & 1);
                    ptx::tc_fence_after();
                    pv_quarter(q, it, (c > 0 || s > 0) ? 1u : 0u, !has_next && s == 3, s == 3);
                    if (has_next && s == 1) qk_half(dir ? 1 : 0, it + 1, 0);
                    if (has_next && s == 3) qk_half(dir ? 0 : 1, it + 1, 1);
                }
            }
        }
    }

    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 16) ptx::tmem_dealloc(tbase, 512);
}

}  // namespace fp8attn
