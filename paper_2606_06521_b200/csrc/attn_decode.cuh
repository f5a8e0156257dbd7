// attn_decode.cuh -- split-KV decode kernel (reading R14): Alg. 1
// for a handful of query rows per kv head against a long E4M3 KV cache.  HBM-bound: every K and V byte is read
// once, so the kernel is built around keeping the TMA ring full.
//
// One CTA = one (batch, kv head, KV split).  The NV = (Hq/Hkv) * Lq <= 16 query rows that share the kv head are
// the N side of both matmuls, the streamed tile is the M side (operands swapped w.r.t. the prefill kernel):
//   S^T = K_j Q^T          M = 128 keys (TMEM lanes), N = 16 query rows, contraction over d = 128
//   O^T += V_j^T P_j^T     M = d = 128 (TMEM lanes),  N = 16 query rows, contraction over the 128 keys;
//                          A = the V tile as it lands (MN-major), B = P^T written to shared memory
// so a thread owns one key and NV logits: NV exps per thread and block instead of 128, and the MMAs cost a few
// cycles.  Block max: redux over the warp on order-preserving integer keys + a 4-warp exchange in shared memory.
// The row sum l is kept per thread (its own key) and reduced once at the end; all 128 threads carry the same
// running max, so alpha is warp-uniform.  Semantics as in attn_general.cuh: exact running max after every
// block, l from the FP32 pre-cast P, P*S cast with cvt.rn.satfinite.e4m3x2.f32, O / (S l) at the end (or in the
// combine kernel when the KV range is split).
#pragma once
#include <cuda_bf16.h>
#include "common.cuh"

namespace fp8attn {

struct DecodeCfg {
    static constexpr int D = 128, BN = 128, NQ = 16;   // NQ: N of both MMAs (query rows, padded)
    static constexpr int TILE = 128 * 128;             // bytes of one K or V tile (E4M3)
    static constexpr int NS = 3;                       // K ring depth = V ring depth (2 CTAs per SM)
    static constexpr int Q_BYTES = NQ * 128, P_BYTES = NQ * 128;
    static constexpr int N_BARS = 1 + 4 * NS + 2 + 2 + 2 + 2 + 1;
    static constexpr int SMEM_BYTES = 2 * NS * TILE + Q_BYTES + 2 * P_BYTES + 1024 /*align*/ + N_BARS * 8 + 16 +
                                      2 * 4 * 16 * 4 /*warp maxima*/ + 4 * 16 * 4 /*warp sums*/;
    static constexpr int TM_S = 0, TM_O = 32, TM_COLS = 64;
    static constexpr int THREADS = 192;
};

// order-preserving float -> int map (so that redux.sync.max.s32 gives the float max), and back
__device__ __forceinline__ int float_to_ordered(float f) {
    const int i = __float_as_int(f);
    return i >= 0 ? i : i ^ 0x7FFFFFFF;
}
__device__ __forceinline__ float ordered_to_float(int i) { return __int_as_float(i >= 0 ? i : i ^ 0x7FFFFFFF); }

// NVT: compile-time bound on the query rows handled (4, 8 or 16); nv <= NVT of them are real.
// AUX: the statistics instance -- same schedule, plus the E4M3 code of every visible P of head (p_batch, p_head)
// written to fp8attn_stats.p_codes and the zero codes among the visible non-sink keys counted (Prop. 1,
// PAPER.md:147-155), split into blocks that hold a sink key / all other blocks.
template <int NVT, bool FOLD, bool AUX = false>
__global__ void __launch_bounds__(192, 2)
attn_decode_kernel(const __grid_constant__ CUtensorMap mapQ, const __grid_constant__ CUtensorMap mapK,
                   const __grid_constant__ CUtensorMap mapV, const FwdParams p) {
    using C = DecodeCfg;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint8_t* sK = smem;
    uint8_t* sV = sK + C::NS * C::TILE;
    uint8_t* sP = sV + C::NS * C::TILE;            // 2 buffers of P^T [16 rows][128 keys], 128-byte swizzle
    uint8_t* sQ = sP + 2 * C::P_BYTES;             // Q^T operand [16 rows][128 B]
    uint64_t* bars = reinterpret_cast<uint64_t*>(sQ + C::Q_BYTES);
    uint64_t* q_full = bars;
    uint64_t* k_full = bars + 1;
    uint64_t* k_empty = k_full + C::NS;
    uint64_t* v_full = k_empty + C::NS;
    uint64_t* v_empty = v_full + C::NS;
    uint64_t* s_full = v_empty + C::NS;            // [2]  MMA -> softmax
    uint64_t* s_empty = s_full + 2;                // [2]  softmax (4 warps) -> MMA
    uint64_t* p_full = s_empty + 2;                // [2]  softmax (4 warps) -> MMA
    uint64_t* pv_done = p_full + 2;                // [2]  MMA -> softmax: P.V of that buffer finished
    uint64_t* o_done = pv_done + 2;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(o_done + 1);
    int* wmax = reinterpret_cast<int*>(tmem_slot + 4);            // [2][4 warps][16]
    float* wsum = reinterpret_cast<float*>(wmax + 2 * 4 * 16);    // [4 warps][16]

    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xFFFFFFFFu, tid >> 5, 0);
    const int G = p.Hq / p.Hkv, nv = G * p.Lq;
    const int kvslab = blockIdx.x;                  // b * Hkv + kv head
    const int split = blockIdx.y;
    const int b = kvslab / p.Hkv, kvh_in_b = kvslab % p.Hkv;
    const long long row0 = ((long long)b * p.Hq + (long long)kvh_in_b * G) * p.Lq;   // first of the nv output rows
    const Seq sq = seq_of(p, b, DecodeCfg::BN);      // this batch element's lengths (variable-length sequences)
    const int sb0 = (int)(((long long)split * sq.nb) / p.num_splits);
    const int sb1 = (int)(((long long)(split + 1) * sq.nb) / p.num_splits);
    const int n_it = sb1 - sb0;

    if (tid == 0) {
        ptx::prefetch_tmap(&mapQ);
        ptx::prefetch_tmap(&mapK);
        ptx::prefetch_tmap(&mapV);
        ptx::mbar_init(q_full, 1);
        for (int i = 0; i < C::NS; ++i) {
            ptx::mbar_init(k_full + i, 1);
            ptx::mbar_init(k_empty + i, 1);
            ptx::mbar_init(v_full + i, 1);
            ptx::mbar_init(v_empty + i, 1);
        }
        for (int i = 0; i < 2; ++i) {
            ptx::mbar_init(s_full + i, 1);
            ptx::mbar_init(s_empty + i, 4);
            ptx::mbar_init(p_full + i, 4);
            ptx::mbar_init(pv_done + i, 1);
        }
        ptx::mbar_init(o_done, 1);
        ptx::fence_mbar_init();
    }
    // rows of P^T that no thread ever writes (query rows >= NVT) must be finite: zero both buffers once
    for (int i = tid; i < 2 * C::P_BYTES / 4; i += C::THREADS) reinterpret_cast<uint32_t*>(sP)[i] = 0u;
    ptx::fence_proxy_async_smem();
    if (warp == 4) {
        __syncwarp();
        ptx::tmem_alloc(tmem_slot, C::TM_COLS);
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tbase = *tmem_slot;

    if (warp == 5) {
        // ================= TMA producer =================
        if (lane == 0 && n_it > 0) {
            const uint64_t stream_once = ptx::policy_evict_first();
            ptx::mbar_arrive_expect_tx(q_full, C::Q_BYTES);
            ptx::tma_load_3d(sQ, &mapQ, q_full, 0, (int)row0, 0);
            for (int it = 0; it < n_it; ++it) {
                const int blk = block_at(p, sb0, sb1, it, C::BN);
                const int st = it % C::NS;
                const uint32_t ph = (it / C::NS) & 1;
                int kv_row, kv_slab;                         // (paged cache: one block-table entry per block)
                kv_coords(p, b, kvh_in_b, kvslab, blk, C::BN, kv_row, kv_slab);
                ptx::mbar_wait(k_empty + st, ph ^ 1);
                ptx::mbar_arrive_expect_tx(k_full + st, C::TILE);
                ptx::tma_load_3d_hint(sK + st * C::TILE, &mapK, k_full + st, 0, kv_row, kv_slab, stream_once);
                ptx::mbar_wait(v_empty + st, ph ^ 1);
                ptx::mbar_arrive_expect_tx(v_full + st, C::TILE);
                ptx::tma_load_3d_hint(sV + st * C::TILE, &mapV, v_full + st, 0, kv_row, kv_slab, stream_once);
            }
        }
    } else if (warp == 4) {
        // ================= MMA issuer (warp-uniform loop, one elected lane issues) =================
        if (n_it > 0) {
            const bool leader = ptx::elect_one();
            constexpr uint32_t idesc_qk =
                ptx::make_idesc(ptx::FMT_E4M3, ptx::FMT_E4M3, ptx::MAJOR_K, ptx::MAJOR_K, 128, C::NQ);
            constexpr uint32_t idesc_pv =
                ptx::make_idesc(ptx::FMT_E4M3, ptx::FMT_E4M3, ptx::MAJOR_MN, ptx::MAJOR_K, 128, C::NQ);
            constexpr uint32_t desc_hi = ptx::smem_desc_hi(1024);
            const uint32_t q_lo = ptx::smem_desc_lo(ptx::smem_u32(sQ), 16);
            const uint32_t k_lo = ptx::smem_desc_lo(ptx::smem_u32(sK), 16);
            const uint32_t v_lo = ptx::smem_desc_lo(ptx::smem_u32(sV), C::BN * 128);
            const uint32_t p_lo = ptx::smem_desc_lo(ptx::smem_u32(sP), 16);
            // O^T += V_j^T P_j^T for block j (ring slot j % NS, P / S buffer j & 1)
            auto issue_pv = [&](int j) {
                const int st = j % C::NS, buf = j & 1;
                ptx::mbar_wait(p_full + buf, (j >> 1) & 1);
                ptx::mbar_wait(v_full + st, (j / C::NS) & 1);
                ptx::tc_fence_after();
                if (leader) {
#pragma unroll
                    for (int ks = 0; ks < 4; ++ks)      // 32 keys per MMA
                        ptx::mma_ss<ptx::KIND_F8F6F4>(tbase + C::TM_O,
                                                      ptx::pack2u(v_lo + st * (C::TILE >> 4) + ks * ((32 * 128) >> 4), desc_hi),
                                                      ptx::pack2u(p_lo + buf * (C::P_BYTES >> 4) + ks * (32 >> 4), desc_hi),
                                                      idesc_pv, (j > 0 || ks > 0) ? 1u : 0u);
                    ptx::tc_commit(v_empty + st);
                    ptx::tc_commit(pv_done + buf);
                    if (j == n_it - 1) ptx::tc_commit(o_done);
                }
            };
            ptx::mbar_wait(q_full, 0);
            for (int j = 0; j < n_it; ++j) {
                const int st = j % C::NS, buf = j & 1;
                // S^T(j) = K_j Q^T into S buffer j & 1 (free once the softmax warps have read block j-2)
                ptx::mbar_wait(k_full + st, (j / C::NS) & 1);
                ptx::mbar_wait(s_empty + buf, ((j >> 1) & 1) ^ 1);
                ptx::tc_fence_after();
                if (leader) {
#pragma unroll
                    for (int ks = 0; ks < 4; ++ks)      // 32 elements of d per MMA
                        ptx::mma_ss<ptx::KIND_F8F6F4>(tbase + C::TM_S + buf * 16,
                                                      ptx::pack2u(k_lo + st * (C::TILE >> 4) + ks * (32 >> 4), desc_hi),
                                                      ptx::pack2u(q_lo + ks * (32 >> 4), desc_hi), idesc_qk, ks > 0 ? 1u : 0u);
                    ptx::tc_commit(s_full + buf);
                    ptx::tc_commit(k_empty + st);
                }
                if (j > 0) issue_pv(j - 1);
            }
            issue_pv(n_it - 1);
        }
    } else {
        // ================= softmax: thread = key within the block (S^T lane), later = d index (O^T lane) ======
        const uint32_t tlane = tbase + (static_cast<uint32_t>(warp * 32) << 16);
        const float c_nat = p.sm_scale * p.k_scale[kvslab];     // times q_scale[row] below (per query head)
        float cl2[NVT], m_run[NVT], l_t[NVT];
        int jlim[NVT];
        int k_run[NVT];                  // dynamic scale: O^T column n and l_t[n] carry 2^k_run[n]
        const bool dynamic = p.scale_mode == 1;
#pragma unroll
        for (int n = 0; n < NVT; ++n) {
            const int g = n / p.Lq, lq = n % p.Lq;
            const float qs = (n < nv) ? p.q_scale[(long long)b * p.Hq + kvh_in_b * G + g] : 1.0f;
            cl2[n] = c_nat * qs * LOG2E;
            m_run[n] = -INFINITY;
            l_t[n] = 0.0f;
            k_run[n] = 0;
            jlim[n] = (n < nv) ? last_visible_key(p, sq, lq) : -1;
        }
        const float log2S = FOLD ? log2f(p.S) : 0.0f;
        // AUX: which query row (if any) belongs to the dumped head; Lq rows of one q head are consecutive n
        uint32_t uf_sink = 0, uf_other = 0;
        int dump_n0 = -1;                      // first n of the dumped head, or -1
        if constexpr (AUX) {
            if (p.p_codes != nullptr) {
                const int g = p.p_bh - (b * p.Hq + kvh_in_b * G);
                if (g >= 0 && g < G) dump_n0 = g * p.Lq;
            }
        }

        for (int j = 0; j < n_it; ++j) {
            const int blk = block_at(p, sb0, sb1, j, C::BN);
            const int key = blk * C::BN + tid;
            const int buf = j & 1;
            ptx::mbar_wait(s_full + buf, (j >> 1) & 1);
            ptx::tc_fence_after();
            uint32_t sv[NVT];
            if constexpr (NVT == 4) ptx::tmem_ld_x4(tlane + C::TM_S + buf * 16, sv);
            else if constexpr (NVT == 8) ptx::tmem_ld_x8(tlane + C::TM_S + buf * 16, sv);
            else ptx::tmem_ld_x16(tlane + C::TM_S + buf * 16, sv);
            ptx::tmem_wait_ld();
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(s_empty + buf);
            // ---- lines 4-5: block max of every query row over the 128 keys ----
            float s[NVT];
            int wm[NVT];
#pragma unroll
            for (int n = 0; n < NVT; ++n) {
                s[n] = (key <= jlim[n]) ? __uint_as_float(sv[n]) : -INFINITY;
                wm[n] = __reduce_max_sync(0xFFFFFFFFu, float_to_ordered(s[n]));
            }
            if (lane < NVT) {
                int mine = wm[0];
#pragma unroll
                for (int n = 1; n < NVT; ++n) mine = (lane == n) ? wm[n] : mine;
                wmax[(buf * 4 + warp) * 16 + lane] = mine;
            }
            asm volatile("bar.sync 1, 128;" ::: "memory");
            bool any_rescale = false;
            float alpha[NVT], negm[NVT];
#pragma unroll
            for (int n = 0; n < NVT; ++n) {
                const int* w = wmax + buf * 64 + n;
                const int mi = max(max(w[0], w[16]), max(w[32], w[48]));
                const float m_loc = ordered_to_float(mi);
                const float m_new = fmaxf(m_run[n], m_loc);
                const float m_used = (m_new == -INFINITY) ? 0.0f : m_new;
                alpha[n] = ptx::ex2_approx((m_run[n] - m_used) * cl2[n]);    // line 6
                negm[n] = fmaf(-m_used, cl2[n], log2S);
                if (dynamic) {
                    // reading R26: this block's scale 2^k goes into the exponent of P, and what O^T and l carry
                    // (the previous block's scale) is brought to it together with alpha
                    const int k_new = (m_loc == -INFINITY) ? k_run[n] : dyn_exponent((m_new - m_loc) * cl2[n]);
                    negm[n] = fmaf(-m_used, cl2[n], (float)k_new);
                    alpha[n] *= exp2f((float)(k_new - k_run[n]));
                    k_run[n] = k_new;
                }
                any_rescale |= (n < nv) && (alpha[n] != 1.0f);
                m_run[n] = m_new;
            }
            // ---- lines 7-9: P, l from the pre-cast P, cast; P^T -> shared memory (B operand of P.V) ----
            if (j >= 2) ptx::mbar_wait(pv_done + buf, ((j - 2) >> 1) & 1);     // P buffer free again
            uint8_t* prow = sP + buf * C::P_BYTES + (tid & 15);
            const int chunk = tid >> 4;
#pragma unroll
            for (int n = 0; n < NVT; n += 2) {
                const float p0 = ptx::ex2_approx(fmaf(s[n], cl2[n], negm[n]));
                const float p1 = ptx::ex2_approx(fmaf(s[n + 1], cl2[n + 1], negm[n + 1]));
                l_t[n] = alpha[n] * l_t[n] + p0;                              // line 8
                l_t[n + 1] = alpha[n + 1] * l_t[n + 1] + p1;
                const uint32_t pair = (FOLD || dynamic) ? ptx::cvt_e4m3x2(p0, p1) : ptx::cvt_e4m3x2(p0 * p.S, p1 * p.S);   // line 9
                prow[n * 128 + ((chunk ^ (n & 7)) << 4)] = (uint8_t)(pair & 0xFFu);
                prow[(n + 1) * 128 + ((chunk ^ ((n + 1) & 7)) << 4)] = (uint8_t)(pair >> 8);
                if constexpr (AUX) {
                    // the same two codes that feed P.V: dump (coalesced over the keys of the block) and count
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        const int nn = n + e;
                        const uint32_t code = e ? (pair >> 8) & 0xFFu : pair & 0xFFu;
                        const bool vis = key <= jlim[nn];        // jlim = -1 for the padding rows nn >= nv
                        if (vis && dump_n0 >= 0 && nn >= dump_n0 && nn < dump_n0 + p.Lq)
                            p.p_codes[(size_t)(nn - dump_n0) * p.Lk + key] = (uint8_t)code;
                        if (vis && code == 0u && !is_sink_key(p, key)) {
                            if (sink_in_range(p, blk * C::BN, C::BN)) ++uf_sink; else ++uf_other;
                        }
                    }
                }
            }
            ptx::fence_proxy_async_smem();
            // ---- line 10, first half: O^T <- O^T * alpha (column n by alpha[n]); needs P.V(j-1) finished ----
            if (j > 0 && any_rescale) {
                ptx::mbar_wait(pv_done + (buf ^ 1), ((j - 1) >> 1) & 1);
                ptx::tc_fence_after();
                uint32_t ov[NVT];
                if constexpr (NVT == 4) ptx::tmem_ld_x4(tlane + C::TM_O, ov);
                else if constexpr (NVT == 8) ptx::tmem_ld_x8(tlane + C::TM_O, ov);
                else ptx::tmem_ld_x16(tlane + C::TM_O, ov);
                ptx::tmem_wait_ld();
#pragma unroll
                for (int n = 0; n < NVT; ++n) ov[n] = __float_as_uint(__uint_as_float(ov[n]) * alpha[n]);
                if constexpr (NVT == 4) ptx::tmem_st_x4(tlane + C::TM_O, ov);
                else if constexpr (NVT == 8) ptx::tmem_st_x8(tlane + C::TM_O, ov);
                else ptx::tmem_st_x16(tlane + C::TM_O, ov);
                ptx::tmem_wait_st();
            }
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(p_full + buf);
        }

        if constexpr (AUX) {
            if (p.underflow != nullptr) {       // one atomic per warp and counter
                const uint32_t a = __reduce_add_sync(0xFFFFFFFFu, uf_sink), b2 = __reduce_add_sync(0xFFFFFFFFu, uf_other);
                if (lane == 0) {
                    if (a) atomicAdd(p.underflow + 0, (unsigned long long)a);
                    if (b2) atomicAdd(p.underflow + 1, (unsigned long long)b2);
                }
            }
        }
        // ---- row sums over the 128 keys; line 12 or the partial result of this split ----
#pragma unroll
        for (int n = 0; n < NVT; ++n) {
            float v = l_t[n];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
            l_t[n] = v;
        }
        if (lane < NVT) {
            float mine = l_t[0];
#pragma unroll
            for (int n = 1; n < NVT; ++n) mine = (lane == n) ? l_t[n] : mine;
            wsum[warp * 16 + lane] = mine;
        }
        asm volatile("bar.sync 1, 128;" ::: "memory");
        if (n_it > 0) {
            ptx::mbar_wait(o_done, 0);
            ptx::tc_fence_after();
        }
        uint32_t ov[NVT];
        if (n_it > 0) {
            if constexpr (NVT == 4) ptx::tmem_ld_x4(tlane + C::TM_O, ov);
            else if constexpr (NVT == 8) ptx::tmem_ld_x8(tlane + C::TM_O, ov);
            else ptx::tmem_ld_x16(tlane + C::TM_O, ov);
            ptx::tmem_wait_ld();
        } else {
#pragma unroll
            for (int n = 0; n < NVT; ++n) ov[n] = 0u;
        }
        const float vs = p.v_scale[kvslab];
        const long long R = (long long)p.B * p.Hq * p.Lq;
#pragma unroll
        for (int n = 0; n < NVT; ++n) {
            if (n >= nv) break;
            const float l = (wsum[n] + wsum[16 + n]) + (wsum[32 + n] + wsum[48 + n]);   // carries S when FOLD / dynamic
            const float carried = dynamic ? exp2f((float)k_run[n]) : (FOLD ? p.S : 1.0f);    // what l and O^T carry
            const float l_true = l / carried;
            const float m_nat = (m_run[n] == -INFINITY) ? -INFINITY : m_run[n] * (cl2[n] / LOG2E);
            const long long grow = row0 + n;
            if (p.num_splits == 1) {
                const float inv = (l > 0.0f) ? ((FOLD || dynamic) ? vs / l : vs / (p.S * l)) : 0.0f;
                const float val = (l > 0.0f) ? __uint_as_float(ov[n]) * inv : 0.0f;
                if (p.o_bf16) static_cast<__nv_bfloat16*>(p.o)[grow * C::D + tid] = __float2bfloat16_rn(val);
                else static_cast<float*>(p.o)[grow * C::D + tid] = val;
                if (tid == 0) {
                    if (p.row_max) p.row_max[grow] = m_nat;
                    if (p.row_sum) p.row_sum[grow] = l_true;
                }
            } else {
                // unnormalised partial: O carrying S like the general kernel's partials (dynamic: true units), m, l
                p.part_o[((long long)split * R + grow) * C::D + tid] =
                    dynamic ? __uint_as_float(ov[n]) / carried : __uint_as_float(ov[n]);
                if (tid == 0) {
                    p.part_ml[((long long)split * R + grow) * 2 + 0] = m_nat;
                    p.part_ml[((long long)split * R + grow) * 2 + 1] = l_true;
                }
            }
        }
    }

    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 4) ptx::tmem_dealloc(tbase, C::TM_COLS);
}

}  // namespace fp8attn
