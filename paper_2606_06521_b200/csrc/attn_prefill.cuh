// attn_prefill.cuh -- warp-specialised throughput kernel for Alg. 1, d = 128, Bn = 128.
//
// One CTA = two 128-row query tiles (256 consecutive query rows) of one (batch, q head).  Roles:
//   warps 0-3  softmax of tile 0      warps 4-7  softmax of tile 1   (one query row per thread = TMEM lane)
//   warps 8, 9 tcgen05.mma issuers of tile 0 / tile 1     warp 10  TMA producer
// TMEM (512 columns): S0 [0,128) S1 [128,256) O0 [256,384) O1 [384,512); P_t is written over the first
// head of each 32-column quarter of S_t (8 columns E4M3 / 16 BF16) and read from there as the A operand
// of O_t += P_t V.  S and P move in quarters: QK^T is issued as four N = 32 MMAs groups, P.V as four K = 32
// groups, each with its own mbarrier, so the tensor pipe works on quarter q while the softmax warps are
// still on quarter q+1 and the serial chain exp -> P.V -> QK^T -> max shrinks to one quarter.
// The tensor pipe executes in issue order: ... PV_0(j), QK_0(j+1), PV_1(j), QK_1(j+1) ..., so while the
// softmax warps of tile 0 work on S_0(j+1) the tensor core runs tile 1 and vice versa; the two softmax
// groups share the MUFU pipe, which is the binding unit (16 ex2 / clk / SM against 16384 FP8 FLOP / clk).
// Semantics are exactly those of attn_general.cuh: the running max is exact after every block (no lazy
// rescale -- it would change which E4M3 code a P value gets), l is summed from the FP32 pre-cast P
// (Alg. 1 line 8), P*S is cast with cvt.rn.satfinite.e4m3x2.f32 (line 9), the epilogue divides by S l
// (line 12).  For S = 2^k the factor is folded into the exponent (exact).
// No P dump and no underflow counters here: calls that ask for them take the general kernel.
#pragma once
#include "attn_general.cuh"

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
    static constexpr int N_BARS = 2 + 4 * NS + 8 + 8 + 2;
    static constexpr int SMEM_BYTES = (2 + 2 * NS) * TILE + 1024 /*align*/ + N_BARS * 8 + 16;
    static constexpr uint32_t KIND = (EB == 1) ? ptx::KIND_F8F6F4 : ptx::KIND_F16;
    static constexpr uint32_t FMT = (EB == 1) ? ptx::FMT_E4M3 : ptx::FMT_BF16;
    static constexpr int THREADS = 352;
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
template <int EB, bool FOLD, bool MASK, int NPOLY = 0>
__device__ __forceinline__ void exp_chunk(const uint32_t* v, uint32_t* w, int j_first, int jlim, uint64_t cl2_2,
                                          uint64_t negm_2, uint64_t s_2, uint64_t& sum_a, uint64_t& sum_b) {
    float pr[32];
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

// ---- softmax warpgroup: all of Alg. 1 lines 4-9 and 12 for one 128-row tile ----------------------
template <int EB, bool FOLD, int QKG>
__device__ __forceinline__ void prefill_softmax(const FwdParams& p, int t, int wq, int lane, uint32_t tbase,
                                                uint64_t* s_full, uint64_t* p_full, uint64_t* o_done, int n_t,
                                                int row0, int bh, int kvh) {
    using C = PrefillCfg<EB>;
    const uint32_t tlane = tbase + (static_cast<uint32_t>(wq * 32) << 16);
    const uint32_t tS = tlane + C::TM_S + t * 128, tO = tlane + C::TM_O + t * 128;
    const int qrow = row0 + wq * 32 + lane;
    const int off = p.Lk - p.Lq;
    long long jl = p.causal ? (long long)qrow + off : (long long)p.Lk - 1;
    if (jl > p.Lk - 1) jl = p.Lk - 1;
    const int jlim = (int)jl;
    // first key index that some row of this warp cannot see (blocks reaching it need the masked path)
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

    float m_run = -INFINITY, l_run = 0.0f;   // l_run carries the factor S when FOLD
    for (int c = 0; c < n_t; ++c) {
        const int blk = (p.kv_order == 0) ? c : n_t - 1 - c;
        const int j0 = blk * C::BN;
        const bool mask = (j0 + C::BN - 1 > warp_vis) || (j0 + C::BN > p.Lk);
        // ---- lines 4-5: block max, running max.  S arrives in four 32-column quarters ----
        float mloc = -INFINITY;
        {
            uint32_t va[32], vb[32];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                if constexpr (QKG == 4) {
                    ptx::mbar_wait(s_full + 2 * h, c & 1);
                    ptx::tc_fence_after();
                    ptx::tmem_ld_x32(tS + h * 64, va);
                    ptx::mbar_wait(s_full + 2 * h + 1, c & 1);
                    ptx::tc_fence_after();
                } else {
                    if (QKG == 2 || h == 0) {
                        ptx::mbar_wait(s_full + (QKG == 2 ? h : 0), c & 1);
                        ptx::tc_fence_after();
                    }
                    ptx::tmem_ld_x32(tS + h * 64, va);
                }
                ptx::tmem_ld_x32(tS + h * 64 + 32, vb);
                ptx::tmem_wait_ld();
                if (mask) {
#pragma unroll
                    for (int e = 0; e < 32; ++e) {
                        if (j0 + h * 64 + e > jlim) va[e] = 0xFF800000u;
                        if (j0 + h * 64 + 32 + e > jlim) vb[e] = 0xFF800000u;
                    }
                }
                float m0 = mloc, m1 = -INFINITY;
#pragma unroll
                for (int e = 0; e < 32; e += 2) {
                    m0 = fmaxf(fmaxf(m0, __uint_as_float(va[e])), __uint_as_float(va[e + 1]));
                    m1 = fmaxf(fmaxf(m1, __uint_as_float(vb[e])), __uint_as_float(vb[e + 1]));
                }
                mloc = fmaxf(m0, m1);
            }
        }
        const float m_new = fmaxf(m_run, mloc);
        const float m_used = (m_new == -INFINITY) ? 0.0f : m_new;
        const float alpha = ptx::ex2_approx((m_run - m_used) * cl2);   // line 6 (0 when m_run = -inf)
        const float negm = fmaf(-m_used, cl2, log2S);
        const uint64_t negm_2 = ptx::pack2(negm, negm);

        // ---- line 10, first half: O <- alpha O.  S(c) complete implies PV(c-1) complete (in-order pipe) ----
        if (c > 0 && __any_sync(0xFFFFFFFFu, alpha != 1.0f)) {
            const uint64_t a2 = ptx::pack2(alpha, alpha);
#pragma unroll 1
            for (int hb = 0; hb < 2; ++hb) {
                uint32_t v[64];
                ptx::tmem_ld_x32(tO + hb * 64, v);
                ptx::tmem_ld_x32(tO + hb * 64 + 32, v + 32);
                ptx::tmem_wait_ld();
#pragma unroll
                for (int e = 0; e < 64; e += 2) {
                    float y0, y1;
                    ptx::unpack2(ptx::mul2(ptx::pack2u(v[e], v[e + 1]), a2), y0, y1);
                    v[e] = __float_as_uint(y0);
                    v[e + 1] = __float_as_uint(y1);
                }
                ptx::tmem_st_x32(tO + hb * 64, v);
                ptx::tmem_st_x32(tO + hb * 64 + 32, v + 32);
            }
        }

        // ---- lines 7-9: P = exp(Z - m), l from the pre-cast P, cast, P -> TMEM over S ----
        uint64_t sum_a = ptx::pack2(0.f, 0.f), sum_b = sum_a;
        {
            uint32_t va[32], vb[32], w[C::P_COLS / 4];
            ptx::tmem_ld_x32(tS, va);
            ptx::tmem_wait_ld();
#pragma unroll
            for (int cb = 0; cb < 4; ++cb) {
                uint32_t* cur = (cb & 1) ? vb : va;
                uint32_t* nxt = (cb & 1) ? va : vb;
                if (cb < 3) ptx::tmem_ld_x32(tS + (cb + 1) * 32, nxt);
                if (mask)
                    exp_chunk<EB, FOLD, true>(cur, w, j0 + cb * 32, jlim, cl2_2, negm_2, s_2, sum_a, sum_b);
                else
                    exp_chunk<EB, FOLD, false>(cur, w, j0 + cb * 32, jlim, cl2_2, negm_2, s_2, sum_a, sum_b);
                // P quarter over the head of its own S quarter; the P.V of this quarter can start at once
                if constexpr (EB == 1) ptx::tmem_st_x8(tS + cb * 32, w);
                else ptx::tmem_st_x16(tS + cb * 32, w);
                ptx::tmem_wait_st();       // (also covers the O rescale stores before the first quarter)
                ptx::tc_fence_before();
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(p_full + cb);
                if (cb < 3) ptx::tmem_wait_ld();
            }
        }
        float sa, sb, sc, sd;
        ptx::unpack2(sum_a, sa, sb);
        ptx::unpack2(sum_b, sc, sd);
        l_run = alpha * l_run + ((sa + sb) + (sc + sd));   // line 8
        m_run = m_new;
    }

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

// ---- the kernel ---------------------------------------------------------------------------------
// grid = (ceil(Lq / 256), B*Hq).  Causal launches the heaviest tile pairs first.
template <int EB, bool FOLD, int QKG>
__global__ void __launch_bounds__(352, 1)
attn_prefill_kernel(const __grid_constant__ CUtensorMap mapQ, const __grid_constant__ CUtensorMap mapK,
                    const __grid_constant__ CUtensorMap mapV, const FwdParams p) {
    using C = PrefillCfg<EB>;
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
    uint64_t* s_full = v_empty + C::NS;           // [2 tiles][4 quarters]  MMA -> softmax
    uint64_t* p_full = s_full + 8;                // [2 tiles][4 quarters]  softmax (4 warps) -> MMA
    uint64_t* o_done = p_full + 8;                // [2]
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(o_done + 2);

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
        for (int i = 0; i < 8; ++i) {
            ptx::mbar_init(s_full + i, 1);
            ptx::mbar_init(p_full + i, 4);
        }
        ptx::mbar_init(o_done + 0, 1);
        ptx::mbar_init(o_done + 1, 1);
        ptx::fence_mbar_init();
    }
    if (warp == 8) {
        __syncwarp();
        ptx::tmem_alloc(tmem_slot, 512);
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tbase = *tmem_slot;

    if (warp < 8) {
        const int t = warp >> 2;
        prefill_softmax<EB, FOLD, QKG>(p, t, warp & 3, lane, tbase, s_full + 4 * t, p_full + 4 * t, o_done + t,
                                  n_tile[t], (pair * 2 + t) * BM, bh, kvh);
    } else if (warp == 10) {
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
    } else if (n_tile[warp - 8] > 0) {
        // ================= MMA issuer of tile t = warp - 8 =================
        // One issuer warp per tile, each blocking only on its own tile's barriers and on the K/V ring, so
        // neither tile can hold up the other.  The whole warp runs the loop (warp-uniform control flow keeps
        // descriptors and counters in uniform registers); one elected lane issues the MMAs and commits.
        // Block c of tile t uses K/V ring iteration it = c + first (in reverse order the tile with fewer
        // visible blocks joins later).  A ring slot is released by two arrivals, one per tile; on iterations
        // that only one tile uses, that tile arrives twice.
        const int t = warp - 8;
        const int n_t = n_tile[t];
        const bool leader = ptx::elect_one();
        constexpr int NG = 128 / QKG;          // keys per QK^T group
        constexpr int QPG = 4 / QKG;           // P quarters per QK^T group
        constexpr uint32_t idesc_qk = ptx::make_idesc(C::FMT, C::FMT, ptx::MAJOR_K, ptx::MAJOR_K, BM, NG);
        constexpr uint32_t idesc_pv = ptx::make_idesc(C::FMT, C::FMT, ptx::MAJOR_K, ptx::MAJOR_MN, BM, C::D);
        constexpr uint32_t desc_hi = ptx::smem_desc_hi(1024);
        const uint32_t q_lo = ptx::smem_desc_lo(ptx::smem_u32(sQ + t * C::TILE), 16);
        const uint32_t k_lo = ptx::smem_desc_lo(ptx::smem_u32(sK), 16);
        const uint32_t v_lo = ptx::smem_desc_lo(ptx::smem_u32(sV), C::BN * 128);
        const uint32_t tS = tbase + C::TM_S + t * 128, tO = tbase + C::TM_O + t * 128;
        const int first = (p.kv_order == 0) ? 0 : n_it - n_t;
        const int n_other = n_tile[t ^ 1];
        const int first_other = (p.kv_order == 0) ? 0 : n_it - n_other;
        uint64_t* const sf = s_full + 4 * t;
        uint64_t* const pf = p_full + 4 * t;

        // S_t[:, NG g .. NG (g+1)) = Q_t K[NG g .. NG (g+1), :]^T on ring iteration it
        auto qk_group = [&](const int g, const int it) {
            const int st = it % C::NS;
            if (g == 0) {
                ptx::mbar_wait(k_full + st, (it / C::NS) & 1);
                ptx::tc_fence_after();
            }
            if (leader) {
                const uint32_t b0 = k_lo + st * (C::TILE >> 4) + g * ((NG * 128) >> 4);
#pragma unroll
                for (int ks = 0; ks < C::D / C::KSTEP; ++ks) {
                    const uint32_t o = (((ks * 32) / 128) * (128 * 128) + (ks * 32) % 128) >> 4;
                    ptx::mma_ss<C::KIND>(tS + g * NG, ptx::pack2u(q_lo + o, desc_hi), ptx::pack2u(b0 + o, desc_hi),
                                         idesc_qk, ks > 0 ? 1u : 0u);
                }
                ptx::tc_commit(sf + g);
                if (g == QKG - 1) {
                    ptx::tc_commit(k_empty + st);
                    if (it < first_other || it >= first_other + n_other) ptx::tc_commit(k_empty + st);
                }
            }
        };
        // O_t += P_t[:, 32q .. 32q+32) V[32q .. 32q+32, :]
        auto pv_group = [&](const int q, const int it, const uint32_t acc0, const bool last_of_tile) {
            const int st = it % C::NS;
            if (q == 0) {
                ptx::mbar_wait(v_full + st, (it / C::NS) & 1);
                ptx::tc_fence_after();
            }
            if (leader) {
                const uint32_t b0 = v_lo + st * (C::TILE >> 4) + q * ((32 * 128) >> 4);
                uint32_t acc = acc0;
#pragma unroll
                for (int ks = 0; ks < 32 / C::KSTEP; ++ks) {
                    ptx::mma_ts<C::KIND>(tO, tS + q * 32 + ks * 8, ptx::pack2u(b0 + ks * ((C::KSTEP * 128) >> 4), desc_hi),
                                         idesc_pv, acc);
                    acc = 1;
                }
                if (last_of_tile) ptx::tc_commit(o_done + t);
                if (q == 3) {
                    ptx::tc_commit(v_empty + st);
                    if (it < first_other || it >= first_other + n_other) ptx::tc_commit(v_empty + st);
                }
            }
        };

        ptx::mbar_wait(q_full + t, 0);
        ptx::tc_fence_after();
#pragma unroll
        for (int g = 0; g < QKG; ++g) qk_group(g, first);
        for (int c = 0; c < n_t; ++c) {
            const int it = c + first;
            const bool has_next = c + 1 < n_t;
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                ptx::mbar_wait(pf + q, c & 1);
                ptx::tc_fence_after();
                pv_group(q, it, (c > 0 || q > 0) ? 1u : 0u, !has_next && q == 3);
                if (has_next && (q + 1) % QPG == 0) qk_group(q / QPG, it + 1);
            }
        }
    }

    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 8) ptx::tmem_dealloc(tbase, 512);
}

}  // namespace fp8attn
