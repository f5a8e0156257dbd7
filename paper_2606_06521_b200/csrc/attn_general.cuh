// attn_general.cuh -- the general (all modes, all statistics) sm_100a attention forward kernel.
//
// One CTA = one 128-row query tile of one (batch, q head) and one KV split.  Per KV block, in
// the order Alg. 1 line 2 selects:
//   TMA K tile -> tcgen05.mma S = Q K^T into TMEM (line 3) -> every thread owns one query row:
//   tcgen05.ld S, mask, block max / running max (lines 4-5), alpha (line 6), P = exp (line 7),
//   l from the FP32 pre-cast P (line 8), P*S -> cvt.rn.satfinite.e4m3x2 (line 9), P written back
//   to TMEM as the A operand, O rescaled by alpha in TMEM -> tcgen05.mma O += P V (line 10).
// Epilogue: O / (S l) (line 12).  The steps of one block are serialised (no overlap): this is
// the reference-grade kernel that carries every feature (FP32 inputs as three BF16 planes,
// no-cast mode, P-code dump, underflow counters, split-KV partials); the throughput kernels
// live in attn_prefill.cuh / attn_prefill64.cuh / attn_decode.cuh.
#pragma once
#include <cuda_bf16.h>
#include "common.cuh"

namespace fp8attn {

// MODE 0: no cast (P kept as three BF16 planes h+m+l = FP32 P exactly)
// MODE 1: isolation (P -> E4M3 -> exact BF16), MODE 2: production FP8 (P E4M3 into kind::f8f6f4)
// EB: operand element bytes (2 = BF16 planes, 1 = E4M3).  NPL: planes per operand (3 for FP32 inputs).
template <int D, int BN, int EB, int NPL, int MODE>
struct GeneralCfg {
    static constexpr int CH = 128 / EB;            // elements per 128-byte swizzle row
    static constexpr int NCH = D / CH;             // 128-byte chunks per operand row
    static constexpr int KSTEP = 32 / EB;          // contraction elements per MMA
    static constexpr int Q_PLANE = NCH * BM * 128; // bytes
    static constexpr int KV_PLANE = NCH * BN * 128;
    static constexpr int PEB = (MODE == 2) ? 1 : 2;      // P element bytes
    static constexpr int NPP = (MODE == 0) ? 3 : 1;      // P planes
    static constexpr int P_PLANE_COLS = BN * PEB / 4;    // TMEM columns per P plane
    static constexpr int PKSTEP = 32 / PEB;
    static constexpr int TM_S = 0, TM_O = 128, TM_P = 256;
    static constexpr int SMEM_BYTES = NPL * (Q_PLANE + 2 * KV_PLANE) + 1024 /*align*/ + 64 /*barriers*/;
    static constexpr uint32_t KIND = (EB == 1) ? ptx::KIND_F8F6F4 : ptx::KIND_F16;
    static constexpr uint32_t FMT = (EB == 1) ? ptx::FMT_E4M3 : ptx::FMT_BF16;
    static_assert(D == 64 || D == 128, "d");
    static_assert(BN == 64 || BN == 128, "Bn");
    static_assert(TM_P + NPP * P_PLANE_COLS <= 512, "TMEM");
    static_assert((MODE == 2) == (EB == 1), "mode 2 <=> E4M3 operands");
};

template <int D, int BN, int EB, int NPL, int MODE>
__global__ void __launch_bounds__(128, 1)
attn_general_kernel(const __grid_constant__ CUtensorMap mapQ, const __grid_constant__ CUtensorMap mapK,
                    const __grid_constant__ CUtensorMap mapV, const FwdParams p) {
    using C = GeneralCfg<D, BN, EB, NPL, MODE>;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint8_t* sQ = smem;
    uint8_t* sK = sQ + NPL * C::Q_PLANE;
    uint8_t* sV = sK + NPL * C::KV_PLANE;
    uint64_t* bars = reinterpret_cast<uint64_t*>(sV + NPL * C::KV_PLANE);
    uint64_t* bar_q = bars + 0;
    uint64_t* bar_k = bars + 1;
    uint64_t* bar_v = bars + 2;
    uint64_t* bar_s = bars + 3;
    uint64_t* bar_o = bars + 4;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 6);

    const int tid = threadIdx.x, warp = tid >> 5;
    // grid = (query tiles x (batch, q head) slabs, 1, KV splits)
    const int n_qtiles = (p.Lq + BM - 1) / BM;
    const int qtile = (int)(blockIdx.x % n_qtiles), bh = (int)(blockIdx.x / n_qtiles), split = blockIdx.z;
    const int b = bh / p.Hq, h = bh % p.Hq;
    const int kvh = b * p.Hkv + h / (p.Hq / p.Hkv);
    const int qrow = qtile * BM + tid;
    const long long grow = (long long)bh * p.Lq + qrow;

    if (tid == 0) {
        ptx::prefetch_tmap(&mapQ);
        ptx::prefetch_tmap(&mapK);
        ptx::prefetch_tmap(&mapV);
        for (int i = 0; i < 5; ++i) ptx::mbar_init(bars + i, 1);
        ptx::fence_mbar_init();
    }
    if (warp == 0) {
        __syncwarp();
        ptx::tmem_alloc(tmem_slot, 512);
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tbase = *tmem_slot;
    const uint32_t tlane = tbase + (static_cast<uint32_t>(warp * 32) << 16);   // this warp's 32 lanes

    // ---- block range of this CTA: split range, clipped by the causal diagonal of the tile ----
    const Seq sq = seq_of(p, b, BN);       // this batch element's lengths (variable-length sequences)
    const int sb0 = (int)(((long long)split * sq.nb) / p.num_splits);
    const int sb1 = (int)(((long long)(split + 1) * sq.nb) / p.num_splits);
    int blk_hi = sb1;
    if (p.causal) {
        long long kmax = (long long)qtile * BM + (BM - 1) + (sq.Lk - sq.Lq);   // last key any row of the tile sees
        if (kmax > sq.Lk - 1) kmax = sq.Lk - 1;
        int lim = kmax < 0 ? 0 : (int)(kmax / BN) + 1;
        if (lim < blk_hi) blk_hi = lim;
    }
    if (qtile * BM >= sq.Lq) blk_hi = sb0;                 // no row of this tile exists in this batch element
    const int n_iter = blk_hi > sb0 ? blk_hi - sb0 : 0;
    const int jlim = last_visible_key(p, sq, qrow);        // may be negative: row sees nothing

    // softmax scale folded with the dequantisation scales and log2(e)
    float c_nat = p.sm_scale;
    float vs = 1.0f;
    if constexpr (MODE == 2) {
        c_nat *= p.q_scale[bh] * p.k_scale[kvh];
        vs = p.v_scale[kvh];
    }
    const float cl2 = c_nat * LOG2E;
    const float S_eff = (MODE == 0) ? 1.0f : p.S;

    if (n_iter > 0 && tid == 0) {
        ptx::mbar_arrive_expect_tx(bar_q, NPL * C::Q_PLANE);
        for (int pl = 0; pl < NPL; ++pl)
            for (int c = 0; c < C::NCH; ++c)
                ptx::tma_load_3d(sQ + pl * C::Q_PLANE + c * (BM * 128), &mapQ, bar_q, c * C::CH, qtile * BM,
                                 pl * p.q_slabs + bh);
    }

    float m_run = -INFINITY, l_run = 0.0f;
    int k_run = 0;            // dynamic scale: O in TMEM carries 2^k_run (the exponent of the last block)
    const bool dynamic = (MODE != 0) && p.scale_mode == 1;
    unsigned int uf_sink = 0, uf_other = 0;
    const bool dump = (MODE != 0) && p.p_codes != nullptr && bh == p.p_bh && qrow < sq.Lq;
    const bool count = (MODE != 0) && p.underflow != nullptr && qrow < sq.Lq;

    constexpr uint32_t idesc_qk = ptx::make_idesc(C::FMT, C::FMT, ptx::MAJOR_K, ptx::MAJOR_K, BM, BN);
    constexpr uint32_t pfmt = (MODE == 2) ? ptx::FMT_E4M3 : ptx::FMT_BF16;
    constexpr uint32_t idesc_pv = ptx::make_idesc(pfmt, C::FMT, ptx::MAJOR_K, ptx::MAJOR_MN, BM, D);

    for (int it = 0; it < n_iter; ++it) {
        const int blk = block_at(p, sb0, blk_hi, it, BN);
        const int j0 = blk * BN;
        const uint32_t ph = it & 1;

        if (tid == 0) {
            // K and V tiles of this block (their previous readers finished: bar_s / bar_o were waited on)
            int kv_row, kv_slab;
            kv_coords(p, b, h / (p.Hq / p.Hkv), kvh, blk, BN, kv_row, kv_slab);
            ptx::mbar_arrive_expect_tx(bar_k, NPL * C::KV_PLANE);
            for (int pl = 0; pl < NPL; ++pl)
                for (int c = 0; c < C::NCH; ++c)
                    ptx::tma_load_3d(sK + pl * C::KV_PLANE + c * (BN * 128), &mapK, bar_k, c * C::CH, kv_row,
                                     pl * p.kv_slabs + kv_slab);
            ptx::mbar_arrive_expect_tx(bar_v, NPL * C::KV_PLANE);
            for (int pl = 0; pl < NPL; ++pl)
                for (int c = 0; c < C::NCH; ++c)
                    ptx::tma_load_3d(sV + pl * C::KV_PLANE + c * (BN * 128), &mapV, bar_v, c * C::CH, kv_row,
                                     pl * p.kv_slabs + kv_slab);
            if (it == 0) ptx::mbar_wait(bar_q, 0);
            ptx::mbar_wait(bar_k, ph);
            ptx::tc_fence_after();
            // S = Q K^T  (Alg. 1 line 3).  FP32 inputs: six BF16 plane products, smallest terms first so
            // the FP32 accumulator is small while the low-order terms are added.
            constexpr int NT = (NPL == 3) ? 6 : 1;
            const int qa[6] = {2, 1, 0, 1, 0, 0};
            const int kb[6] = {0, 1, 2, 0, 1, 0};
            uint32_t acc = 0;
            for (int t = 0; t < NT; ++t) {
                const int pa = (NPL == 3) ? qa[t] : 0, pb = (NPL == 3) ? kb[t] : 0;
                for (int ks = 0; ks < D / C::KSTEP; ++ks) {
                    const int c = (ks * 32) / 128, w = (ks * 32) % 128;
                    const uint64_t da = ptx::make_smem_desc(ptx::smem_u32(sQ + pa * C::Q_PLANE + c * (BM * 128) + w), 16, 1024);
                    const uint64_t db = ptx::make_smem_desc(ptx::smem_u32(sK + pb * C::KV_PLANE + c * (BN * 128) + w), 16, 1024);
                    ptx::mma_ss<C::KIND>(tbase + C::TM_S, da, db, idesc_qk, acc);
                    acc = 1;
                }
            }
            ptx::tc_commit(bar_s);
        }
        __syncwarp();
        ptx::mbar_wait(bar_s, ph);
        ptx::tc_fence_after();

        // ---- lines 4-5: block max over the visible keys of this row, running max ----
        float mloc = -INFINITY;
#pragma unroll 1
        for (int cb = 0; cb < BN / 32; ++cb) {
            uint32_t v[32];
            ptx::tmem_ld_x32(tlane + C::TM_S + cb * 32, v);
            ptx::tmem_wait_ld();
#pragma unroll
            for (int e = 0; e < 32; ++e) {
                const float s = (j0 + cb * 32 + e <= jlim) ? __uint_as_float(v[e]) : -INFINITY;
                mloc = fmaxf(mloc, s);
            }
        }
        const float m_new = fmaxf(m_run, mloc);
        const float m_used = (m_new == -INFINITY) ? 0.0f : m_new;
        const float alpha = ptx::ex2_approx((m_run - m_used) * cl2);   // line 6 (0 when m_run = -inf)
        const float neg_ml2 = -m_used * cl2;
        const bool sink_blk = sink_in_range(p, j0, BN);
        // scale of this block: S, or (reading R26) the largest 2^k that keeps the block maximum at or below 448
        float S_blk = S_eff, o_factor = alpha;          // o_factor: what O (carrying the previous scale) is multiplied by
        if (dynamic) {
            const int k_new = (mloc == -INFINITY) ? k_run : dyn_exponent((m_new - mloc) * cl2);
            S_blk = exp2f((float)k_new);
            o_factor = alpha * exp2f((float)(k_new - k_run));
            k_run = k_new;
        }

        // ---- lines 7-9: P, row sum from the pre-cast P, cast, P -> TMEM ----
        float psum = 0.0f;
#pragma unroll 1
        for (int cb = 0; cb < BN / 32; ++cb) {
            uint32_t v[32];
            ptx::tmem_ld_x32(tlane + C::TM_S + cb * 32, v);
            ptx::tmem_wait_ld();
            float pr[32];
#pragma unroll
            for (int e = 0; e < 32; ++e) {
                const float s = (j0 + cb * 32 + e <= jlim) ? __uint_as_float(v[e]) : -INFINITY;
                pr[e] = ptx::ex2_approx(fmaf(s, cl2, neg_ml2));
                psum += pr[e];
            }
            if constexpr (MODE == 0) {
                uint32_t wh[16], wm[16], wl[16];
#pragma unroll
                for (int e = 0; e < 32; e += 2) {
                    const uint32_t hh = ptx::cvt_bf16x2(pr[e], pr[e + 1]);
                    const float r0 = pr[e] - ptx::bf16_lo_to_f32(hh), r1 = pr[e + 1] - ptx::bf16_hi_to_f32(hh);
                    const uint32_t mm = ptx::cvt_bf16x2(r0, r1);
                    const float s0 = r0 - ptx::bf16_lo_to_f32(mm), s1 = r1 - ptx::bf16_hi_to_f32(mm);
                    wh[e / 2] = hh;
                    wm[e / 2] = mm;
                    wl[e / 2] = ptx::cvt_bf16x2(s0, s1);
                }
                ptx::tmem_st_x16(tlane + C::TM_P + 0 * C::P_PLANE_COLS + cb * 16, wh);
                ptx::tmem_st_x16(tlane + C::TM_P + 1 * C::P_PLANE_COLS + cb * 16, wm);
                ptx::tmem_st_x16(tlane + C::TM_P + 2 * C::P_PLANE_COLS + cb * 16, wl);
            } else {
                uint32_t pair[16];
#pragma unroll
                for (int e = 0; e < 32; e += 2)
                    pair[e / 2] = ptx::cvt_e4m3x2(pr[e] * S_blk, pr[e + 1] * S_blk);   // line 9
                if (count || dump) {
                    const uint32_t sinks = sink_mask32(p, j0 + cb * 32);
#pragma unroll
                    for (int e = 0; e < 32; ++e) {
                        const int j = j0 + cb * 32 + e;
                        const uint32_t code = (pair[e / 2] >> ((e & 1) * 8)) & 0xFFu;
                        const bool vis = j <= jlim;
                        if (count && vis && code == 0 && !((sinks >> e) & 1u)) {
                            if (sink_blk) ++uf_sink; else ++uf_other;
                        }
                        if (dump && j < p.Lk) p.p_codes[(size_t)qrow * p.Lk + j] = vis ? (uint8_t)code : (uint8_t)0xFF;
                    }
                }
                if constexpr (MODE == 2) {
                    uint32_t w[8];
#pragma unroll
                    for (int e = 0; e < 8; ++e) w[e] = pair[2 * e] | (pair[2 * e + 1] << 16);
                    ptx::tmem_st_x8(tlane + C::TM_P + cb * 8, w);
                } else {
                    uint32_t w[16];
#pragma unroll
                    for (int e = 0; e < 16; ++e) {
                        const uint32_t h2 = ptx::cvt_e4m3x2_to_f16x2(pair[e]);
                        const float lo = __half2float(__ushort_as_half((unsigned short)(h2 & 0xFFFFu)));
                        const float hi = __half2float(__ushort_as_half((unsigned short)(h2 >> 16)));
                        w[e] = ptx::cvt_bf16x2(lo, hi);   // exact: E4M3 values are BF16-representable
                    }
                    ptx::tmem_st_x16(tlane + C::TM_P + cb * 16, w);
                }
            }
        }
        l_run = alpha * l_run + psum;   // line 8
        m_run = m_new;

        // ---- line 10, first half: O <- alpha O (in TMEM) ----
        if (it > 0) {
#pragma unroll 1
            for (int cb = 0; cb < D / 32; ++cb) {
                uint32_t v[32];
                ptx::tmem_ld_x32(tlane + C::TM_O + cb * 32, v);
                ptx::tmem_wait_ld();
#pragma unroll
                for (int e = 0; e < 32; ++e) v[e] = __float_as_uint(__uint_as_float(v[e]) * o_factor);
                ptx::tmem_st_x32(tlane + C::TM_O + cb * 32, v);
            }
        }
        ptx::tmem_wait_st();
        ptx::tc_fence_before();
        __syncthreads();

        // ---- line 10, second half: O += P V ----
        if (tid == 0) {
            ptx::tc_fence_after();
            ptx::mbar_wait(bar_v, ph);
            ptx::tc_fence_after();
            constexpr int NT = (MODE == 0) ? ((NPL == 3) ? 6 : 3) : NPL;
            // (P plane, V plane) products, smallest first
            const int pa6[6] = {2, 1, 0, 1, 0, 0}, vb6[6] = {0, 1, 2, 0, 1, 0};
            uint32_t acc = (it > 0) ? 1u : 0u;
            for (int t = 0; t < NT; ++t) {
                int pa, vb;
                if constexpr (MODE == 0) {
                    pa = (NPL == 3) ? pa6[t] : 2 - t;
                    vb = (NPL == 3) ? vb6[t] : 0;
                } else {
                    pa = 0;
                    vb = NPL - 1 - t;
                }
                for (int ks = 0; ks < BN / C::PKSTEP; ++ks) {
                    const uint32_t ta = tbase + C::TM_P + pa * C::P_PLANE_COLS + ks * 8;
                    const uint64_t db = ptx::make_smem_desc(
                        ptx::smem_u32(sV + vb * C::KV_PLANE + ks * (C::PKSTEP * 128)), BN * 128, 1024);
                    ptx::mma_ts<C::KIND>(tbase + C::TM_O, ta, db, idesc_pv, acc);
                    acc = 1;
                }
            }
            ptx::tc_commit(bar_o);
        }
        __syncwarp();
        ptx::mbar_wait(bar_o, ph);
        ptx::tc_fence_after();
    }

    // ---- line 12: O / (S l); statistics ----
    const long long R = (long long)p.B * p.Hq * p.Lq;
    if (qrow < p.Lq) {
        const float m_nat = (m_run == -INFINITY) ? -INFINITY : m_run * c_nat;
        if (p.num_splits == 1) {
            if (p.row_max) p.row_max[grow] = m_nat;
            if (p.row_sum) p.row_sum[grow] = l_run;
        } else {
            p.part_ml[((long long)split * R + grow) * 2 + 0] = m_nat;
            p.part_ml[((long long)split * R + grow) * 2 + 1] = l_run;
        }
    }
    // (dynamic scale: O carries 2^k_run; partials of a split are written in true units, the combine divides by 1)
    const float S_fin = dynamic ? exp2f((float)k_run) : S_eff;
    const float inv = (p.num_splits == 1) ? ((l_run > 0.0f) ? vs / (S_fin * l_run) : 0.0f) : (dynamic ? 1.0f / S_fin : 1.0f);
    float* const dst_part = p.part_o + ((long long)split * R + grow) * D;
#pragma unroll 1
    for (int cb = 0; cb < D / 32; ++cb) {
        uint32_t v[32];
        if (n_iter > 0) {
            ptx::tmem_ld_x32(tlane + C::TM_O + cb * 32, v);
            ptx::tmem_wait_ld();
        } else {
#pragma unroll
            for (int e = 0; e < 32; ++e) v[e] = 0u;
        }
        if (qrow < p.Lq) {
#pragma unroll
            for (int e = 0; e < 32; e += 4) {
                float4 o4;
                o4.x = __uint_as_float(v[e + 0]) * inv;
                o4.y = __uint_as_float(v[e + 1]) * inv;
                o4.z = __uint_as_float(v[e + 2]) * inv;
                o4.w = __uint_as_float(v[e + 3]) * inv;
                if (l_run <= 0.0f) o4 = make_float4(0.f, 0.f, 0.f, 0.f);
                if (p.num_splits == 1) store_o4(p, grow * D + cb * 32 + e, o4.x, o4.y, o4.z, o4.w);
                else *reinterpret_cast<float4*>(dst_part + cb * 32 + e) = o4;
            }
        }
    }
    if (p.underflow != nullptr && MODE != 0) {
        uf_sink = __reduce_add_sync(0xFFFFFFFFu, uf_sink);
        uf_other = __reduce_add_sync(0xFFFFFFFFu, uf_other);
        if ((tid & 31) == 0) {
            if (uf_sink) atomicAdd(p.underflow + 0, (unsigned long long)uf_sink);
            if (uf_other) atomicAdd(p.underflow + 1, (unsigned long long)uf_other);
        }
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 0) ptx::tmem_dealloc(tbase, 512);
}

// ---------------------------------------------------------------------------------------------
// Combine of split-KV partials: m = max_s m_s; w_s = exp(m_s - m);
// O = sum_s w_s O_s / (S sum_s w_s l_s) (x v_scale in mode 2).  One warp per row.
__global__ void combine_kernel(const float* __restrict__ part_o, const float* __restrict__ part_ml, void* __restrict__ o,
                               float* __restrict__ row_max, float* __restrict__ row_sum, const float* __restrict__ v_scale,
                               long long R, int d, int ns, float S_eff, int Hq, int Hkv, int Lq, int o_bf16) {
    const long long row = (long long)blockIdx.x * (blockDim.x / 32) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (row >= R) return;
    float m = -INFINITY;
    for (int s = 0; s < ns; ++s) m = fmaxf(m, part_ml[((long long)s * R + row) * 2]);
    float l = 0.0f;
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
    for (int s = 0; s < ns; ++s) {
        const float ms = part_ml[((long long)s * R + row) * 2];
        if (ms == -INFINITY) continue;
        const float w = ptx::ex2_approx((ms - m) * LOG2E);
        l += w * part_ml[((long long)s * R + row) * 2 + 1];
        const float* po = part_o + ((long long)s * R + row) * d;
        for (int t = lane, i = 0; t < d; t += 32, ++i) acc[i] += w * po[t];
    }
    float vs = 1.0f;
    if (v_scale) {
        const long long bh = row / Lq;
        vs = v_scale[(bh / Hq) * Hkv + (bh % Hq) / (Hq / Hkv)];
    }
    const float inv = l > 0.0f ? vs / (S_eff * l) : 0.0f;
    for (int t = lane, i = 0; t < d; t += 32, ++i) {
        if (o_bf16) static_cast<__nv_bfloat16*>(o)[row * d + t] = __float2bfloat16_rn(acc[i] * inv);
        else static_cast<float*>(o)[row * d + t] = acc[i] * inv;
    }
    if (lane == 0) {
        if (row_max) row_max[row] = m;
        if (row_sum) row_sum[row] = l;
    }
}

}  // namespace fp8attn
