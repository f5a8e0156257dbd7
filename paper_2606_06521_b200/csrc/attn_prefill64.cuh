// attn_prefill64.cuh -- warp-specialised throughput kernel for Alg. 1 with KV blocks of
// Bn = 64 keys (the block size of the paper's experiments) and the S tile of every query tile
// double-buffered in TMEM.
//
// Two 128-row query tiles per CTA; warps 0-7 / 8-15 softmax of tile 0 / 1 (one query row per thread, two warps
// per 32 rows taking alternate blocks); warps 16 / 17 tcgen05.mma issuers; warp 18 TMA producer.  TMEM:
//   S0a S0b S1a S1b   64 columns each  [0,256)      O0 O1   128 columns each  [256,512)
// Block j of a tile uses S buffer j & 1; P(j) is written over the head of that buffer (16 columns E4M3, 32
// BF16) and read from there as the A operand of O += P(j) V(j).  QK^T of block j+2 is issued right after
// P.V of block j, into the buffer that P.V has just released, so S(j+1) is complete long before the softmax
// warps finish block j: they never wait for the tensor pipe in steady state, and the serial chain
// exp -> P.V -> QK^T -> max of the Bn = 128 kernel is gone.  A softmax thread reads its 64 logits once, keeps
// them in registers for the max pass and the exp pass.  The O rescale needs P.V(j-1) complete; it waits for
// that barrier only when some row of the warp has a new maximum.
// Semantics as everywhere: exact running max after every block, l from the FP32 pre-cast P (line 8), P*S
// cast with cvt.rn.satfinite.e4m3x2.f32 (line 9), O / (S l) at the end (line 12).
#pragma once
#include "prefill_common.cuh"

namespace fp8attn {

template <int EB>
struct Prefill64Cfg {
    static constexpr int D = 128, BN = 64;
    static constexpr int CH = 128 / EB;              // elements per 128-byte swizzle row
    static constexpr int NCH = D / CH;               // 128-byte chunks per operand row
    static constexpr int QTILE = NCH * 128 * 128;    // bytes of one 128-row Q tile
    static constexpr int TILE = NCH * BN * 128;      // bytes of one 64-key K or V tile
    static constexpr int NS = (EB == 1) ? 8 : 4;     // K ring depth = V ring depth
    static constexpr int KSTEP = 32 / EB;            // contraction elements per MMA
    static constexpr int TM_S = 0, TM_O = 256;
    static constexpr int N_BARS = 2 + 4 * NS + 4 + 4 + 2 + 2 + 16;
    static constexpr int SMEM_BYTES = 2 * QTILE + 2 * NS * TILE + 1024 /*align*/ + N_BARS * 8 + 16 + 8192 /*Softmax64Shared*/;
    static constexpr uint32_t KIND = (EB == 1) ? ptx::KIND_F8F6F4 : ptx::KIND_F16;
    static constexpr uint32_t FMT = (EB == 1) ? ptx::FMT_E4M3 : ptx::FMT_BF16;
    static constexpr int THREADS = 608;
};

// ---- softmax warps ------------------------------------------------------------------------------------
// Each 128-row tile has eight softmax warps, two per 32 rows (TMEM lane quarter wq): warp (wq, par) handles the
// blocks c with c & 1 == par of those rows, i.e. always the same S buffer.  The only value block c needs from
// block c-1 is the running max m(c-1), which its partner publishes (shared memory + mbarrier) right after its
// max pass, long before its exp pass ends: the exp passes of consecutive blocks overlap, and each scheduler
// has four independent softmax warps to keep the MUFU pipe busy.  Each warp keeps the partial row sum of its
// own blocks, rescaled against the max it used last; the two partials are merged at the end.  O is rescaled
// by the warp of block c after its exp pass (P does not depend on O), once P.V(c-1) has finished.
struct Softmax64Shared {
    float m[2][2][128];         // [tile][block parity][row]  running max after that block
    float l[2][2][128];         // [tile][par][row]           final partial row sums
    float mlast[2][2][128];     // [tile][par][row]           the max each partial sum is relative to
    int kexp[2][2][128];        // [tile][block parity][row]  dynamic scale: exponent of that block (what O carries)
};
static_assert(sizeof(Softmax64Shared) == 8192, "SMEM_BYTES accounts for 8192 bytes");

template <int EB, bool FOLD, bool AUX>
__device__ __forceinline__ void prefill64_softmax(const FwdParams& p, int t, int par, int wq, int lane, uint32_t tbase,
                                                  uint64_t* s_full, uint64_t* p_full, uint64_t* pv_done,
                                                  uint64_t* o_done, uint64_t* m_full, int n_t, int row0, int bh,
                                                  int kvh, Softmax64Shared* sh) {
    using C = Prefill64Cfg<EB>;
    const uint32_t tlane = tbase + (static_cast<uint32_t>(wq * 32) << 16);
    const uint32_t tS = tlane + C::TM_S + t * 128 + par * 64, tO = tlane + C::TM_O + t * 128;
    const int r = wq * 32 + lane;
    const int qrow = row0 + r;
    const Seq sq = seq_of(p, bh / p.Hq, C::BN);      // this batch element's lengths (variable-length sequences)
    const int off = sq.Lk - sq.Lq;
    const int jlim = last_visible_key(p, sq, qrow);
    // last key that every row of this warp sees (blocks reaching past it need the masked path); a warp with a row
    // past the end of its sequence always masks
    const long long warp_vis = (row0 + wq * 32 + 31 >= sq.Lq) ? -1
                               : (p.causal ? (long long)(row0 + wq * 32) + off : (long long)sq.Lk - 1);
    const bool dynamic = p.scale_mode == 1;          // reading R26 (the host launches the FOLD instance for it)
    const int bar_id = 1 + t * 4 + wq;            // named barrier of the two warps of these 32 rows

    float c_nat = p.sm_scale, vs = 1.0f;
    if constexpr (EB == 1) {
        c_nat *= p.q_scale[bh] * p.k_scale[kvh];
        vs = p.v_scale[kvh];
    }
    const float cl2 = c_nat * LOG2E;
    const float log2S = (FOLD && !dynamic) ? log2f(p.S) : 0.0f;   // exact for S = 2^k
    const uint64_t cl2_2 = ptx::pack2(cl2, cl2), s_2 = ptx::pack2(p.S, p.S);

    float m_own = -INFINITY, l_own = 0.0f;   // partial sum of this warp's blocks, relative to m_own; carries S when FOLD
    int k_own = 0;                           // dynamic: the exponent l_own carries (this warp's last block)
    // statistics instance: this row of the P dump, and the zero codes among visible non-sink keys
    uint8_t* const dump_row = (AUX && p.p_codes != nullptr && bh == p.p_bh && qrow < sq.Lq)
                                  ? p.p_codes + (size_t)qrow * p.Lk : nullptr;
    const bool count = AUX && p.underflow != nullptr && qrow < sq.Lq;
    uint32_t uf_sink = 0, uf_other = 0;
    for (int c = par; c < n_t; c += 2) {
        const int blk = (p.kv_order == 0) ? c : n_t - 1 - c;
        const int j0 = blk * C::BN;
        const bool mask = (j0 + C::BN - 1 > warp_vis) || (j0 + C::BN > sq.Lk);
        const bool sink_blk = AUX && sink_in_range(p, j0, C::BN);
        ptx::mbar_wait(s_full + par, (c >> 1) & 1);
        ptx::tc_fence_after();
        // ---- lines 4-5: block max, running max ----
        float mloc;
        {
            uint32_t va[32], vb[32];
            ptx::tmem_ld_x32(tS, va);
            ptx::tmem_ld_x32(tS + 32, vb);
            ptx::tmem_wait_ld();
            if (mask) {
#pragma unroll
                for (int e = 0; e < 32; ++e) {
                    if (j0 + e > jlim) va[e] = 0xFF800000u;          // -inf
                    if (j0 + 32 + e > jlim) vb[e] = 0xFF800000u;
                }
            }
            float m0 = -INFINITY, m1 = -INFINITY, m2 = -INFINITY, m3 = -INFINITY;
#pragma unroll
            for (int e = 0; e < 32; e += 4) {
                m0 = fmaxf(fmaxf(m0, __uint_as_float(va[e])), __uint_as_float(va[e + 1]));
                m1 = fmaxf(fmaxf(m1, __uint_as_float(va[e + 2])), __uint_as_float(va[e + 3]));
                m2 = fmaxf(fmaxf(m2, __uint_as_float(vb[e])), __uint_as_float(vb[e + 1]));
                m3 = fmaxf(fmaxf(m3, __uint_as_float(vb[e + 2])), __uint_as_float(vb[e + 3]));
            }
            mloc = fmaxf(fmaxf(m0, m1), fmaxf(m2, m3));
        }
        float m_prev = -INFINITY;                 // running max after block c-1, from the partner warp
        int k_prev = 0;                           // dynamic: the exponent O carries after block c-1
        if (c > 0) {
            ptx::mbar_wait(m_full + (par ^ 1), ((c - 1) >> 1) & 1);
            m_prev = sh->m[t][par ^ 1][r];
            k_prev = sh->kexp[t][par ^ 1][r];
        }
        const float m_new = fmaxf(m_prev, mloc);
        const int k_new = !dynamic ? 0 : ((mloc == -INFINITY) ? k_prev : dyn_exponent((m_new - mloc) * cl2));
        sh->m[t][par][r] = m_new;
        sh->kexp[t][par][r] = k_new;
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(m_full + par);
        const float m_used = (m_new == -INFINITY) ? 0.0f : m_new;
        float alpha_o = ptx::ex2_approx((m_prev - m_used) * cl2);   // line 6: what O (state after c-1) is scaled by
        float alpha_l = ptx::ex2_approx((m_own - m_used) * cl2);    // the same for this warp's partial sum
        float negm = fmaf(-m_used, cl2, log2S);
        if (dynamic) {        // 2^k of this block in the exponent of P; O and l are brought from their scales to it
            negm = fmaf(-m_used, cl2, (float)k_new);
            alpha_o *= exp2f((float)(k_new - k_prev));
            alpha_l *= exp2f((float)(k_new - k_own));
            k_own = k_new;
        }
        const uint64_t negm_2 = ptx::pack2(negm, negm);

        // ---- lines 7-9: P = exp(Z - m), l from the pre-cast P, cast, P -> TMEM over the head of S ----
        uint64_t sum_a = ptx::pack2(0.f, 0.f), sum_b = sum_a;
#pragma unroll
        for (int cb = 0; cb < 2; ++cb) {
            uint32_t v[32], w[8 * EB];
            ptx::tmem_ld_x32(tS + cb * 32, v);
            ptx::tmem_wait_ld();
            if (mask) exp_chunk<EB, FOLD, true>(v, w, j0 + cb * 32, jlim, cl2_2, negm_2, s_2, sum_a, sum_b);
            else exp_chunk<EB, FOLD, false>(v, w, j0 + cb * 32, jlim, cl2_2, negm_2, s_2, sum_a, sum_b);
            if constexpr (AUX) {
                const uint32_t zeros = chunk_statistics<EB>(w, j0 + cb * 32, jlim, dump_row, count, p, sink_blk);
                if (sink_blk) uf_sink += zeros;
                else uf_other += zeros;
            }
            // (P of chunk cb lands on columns of chunk 0, whose logits are already in registers)
            if constexpr (EB == 1) ptx::tmem_st_x8(tS + cb * 8, w);
            else ptx::tmem_st_x16(tS + cb * 16, w);
        }
        float sa, sb, sc, sd;
        ptx::unpack2(sum_a, sa, sb);
        ptx::unpack2(sum_b, sc, sd);
        l_own = alpha_l * l_own + ((sa + sb) + (sc + sd));   // line 8
        m_own = m_new;

        // ---- line 10, first half: O <- alpha O, after P.V(c-1) has finished ----
        if (c > 0 && __any_sync(0xFFFFFFFFu, alpha_o != 1.0f)) {
            ptx::mbar_wait(pv_done, (c - 1) & 1);
            ptx::tc_fence_after();
            const uint64_t a2 = ptx::pack2(alpha_o, alpha_o);
#pragma unroll 1
            for (int cb = 0; cb < 4; ++cb) {
                uint32_t v[32];
                ptx::tmem_ld_x32(tO + cb * 32, v);
                ptx::tmem_wait_ld();
#pragma unroll
                for (int e = 0; e < 32; e += 2) {
                    float y0, y1;
                    ptx::unpack2(ptx::mul2(ptx::pack2u(v[e], v[e + 1]), a2), y0, y1);
                    v[e] = __float_as_uint(y0);
                    v[e + 1] = __float_as_uint(y1);
                }
                ptx::tmem_st_x32(tO + cb * 32, v);
            }
        }
        ptx::tmem_wait_st();
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(p_full + par);
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
    // ---- merge the two partial row sums; line 12: O / (S l), statistics ----
    // (dynamic scale: each partial sum is first brought to true units, 2^-k_own; O carries the exponent of the last
    // block, which the warp of that block published)
    const float own_true = dynamic ? l_own * exp2f((float)-k_own) : l_own;
    sh->l[t][par][r] = own_true;
    sh->mlast[t][par][r] = m_own;
    asm volatile("bar.sync %0, 64;" ::"r"(bar_id) : "memory");
    const float m_oth = sh->mlast[t][par ^ 1][r], l_oth = sh->l[t][par ^ 1][r];
    const float m_fin = fmaxf(m_own, m_oth);
    const float m_fu = (m_fin == -INFINITY) ? 0.0f : m_fin;
    const float l_all = own_true * ptx::ex2_approx((m_own - m_fu) * cl2) + l_oth * ptx::ex2_approx((m_oth - m_fu) * cl2);
    const float o_carries = (dynamic && n_t > 0) ? exp2f((float)sh->kexp[t][(n_t - 1) & 1][r]) : 1.0f;
    const long long grow = (long long)bh * p.Lq + qrow;
    if (qrow < p.Lq && par == 0) {
        if (p.row_max) p.row_max[grow] = (m_fin == -INFINITY) ? -INFINITY : m_fin * c_nat;
        if (p.row_sum) p.row_sum[grow] = (FOLD && !dynamic) ? l_all / p.S : l_all;
    }
    const float inv = (l_all > 0.0f) ? (dynamic ? vs / (o_carries * l_all) : (FOLD ? vs / l_all : vs / (p.S * l_all))) : 0.0f;
    if (n_t > 0) {
        ptx::mbar_wait(o_done, 0);
        ptx::tc_fence_after();
    }
    const long long dst = grow * C::D + par * 64;  // this warp stores columns 64 par .. 64 par + 63
#pragma unroll 1
    for (int cb = 0; cb < 2; ++cb) {
        uint32_t v[32];
        if (n_t > 0) {
            ptx::tmem_ld_x32(tO + par * 64 + cb * 32, v);
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
                if (l_all <= 0.0f) o4 = make_float4(0.f, 0.f, 0.f, 0.f);
                store_o4(p, dst + cb * 32 + e, o4.x, o4.y, o4.z, o4.w);
            }
        }
    }
}

// ---- the kernel ---------------------------------------------------------------------------------
// grid = ceil(Lq / 256) * B*Hq CTAs in one dimension, tile pair fastest.  Causal launches the heaviest tile pairs
// first.  AUX: the statistics instance (P dump, underflow counters), same schedule.
template <int EB, bool FOLD, bool AUX = false>
__global__ void __launch_bounds__(608, 1)
attn_prefill64_kernel(const __grid_constant__ CUtensorMap mapQ, const __grid_constant__ CUtensorMap mapK,
                      const __grid_constant__ CUtensorMap mapV, const FwdParams p) {
    using C = Prefill64Cfg<EB>;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint8_t* sQ = smem;                           // 2 tiles of 128 rows
    uint8_t* sK = sQ + 2 * C::QTILE;              // NS tiles of 64 keys
    uint8_t* sV = sK + C::NS * C::TILE;           // NS tiles of 64 keys
    uint64_t* bars = reinterpret_cast<uint64_t*>(sV + C::NS * C::TILE);
    uint64_t* q_full = bars;                      // [2]
    uint64_t* k_full = bars + 2;                  // [NS]
    uint64_t* k_empty = k_full + C::NS;           //        two arrivals: one per tile
    uint64_t* v_full = k_empty + C::NS;
    uint64_t* v_empty = v_full + C::NS;
    uint64_t* s_full = v_empty + C::NS;           // [2 tiles][2 buffers]  MMA -> softmax
    uint64_t* p_full = s_full + 4;                // [2 tiles][2 buffers]  softmax (4 warps) -> MMA
    uint64_t* pv_done = p_full + 4;               // [2 tiles]  P.V of a block finished
    uint64_t* o_done = pv_done + 2;               // [2 tiles]
    uint64_t* m_full = o_done + 2;                // [2 tiles][4 lane quarters][2 block parities]  running max published
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(m_full + 16);
    Softmax64Shared* sh = reinterpret_cast<Softmax64Shared*>(tmem_slot + 4);

    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xFFFFFFFFu, tid >> 5, 0);   // provably warp-uniform
    const int n_pairs = (p.Lq + 2 * BM - 1) / (2 * BM);
    const int pair_idx = (int)(blockIdx.x % n_pairs);
    const int pair = p.causal ? n_pairs - 1 - pair_idx : pair_idx;
    const int bh = (int)(blockIdx.x / n_pairs);
    const int b = bh / p.Hq, h = bh % p.Hq;
    const int kvh = b * p.Hkv + h / (p.Hq / p.Hkv);

    // visible block count of each tile (bottom-right causal, reading R15; this batch element's lengths)
    const Seq sq = seq_of(p, b, C::BN);
    int n_tile[2];
#pragma unroll
    for (int t = 0; t < 2; ++t) {
        const long long r0 = (long long)(pair * 2 + t) * BM;
        int n = 0;
        if (r0 < sq.Lq) {
            n = sq.nb;
            if (p.causal) {
                long long kmax = r0 + (BM - 1) + (sq.Lk - sq.Lq);
                if (kmax > sq.Lk - 1) kmax = sq.Lk - 1;
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
            ptx::mbar_init(k_empty + i, 2);
            ptx::mbar_init(v_empty + i, 2);
        }
        for (int i = 0; i < 4; ++i) {
            ptx::mbar_init(s_full + i, 1);
            ptx::mbar_init(p_full + i, 4);
        }
        for (int i = 0; i < 2; ++i) {
            ptx::mbar_init(pv_done + i, 1);
            ptx::mbar_init(o_done + i, 1);
        }
        for (int i = 0; i < 16; ++i) ptx::mbar_init(m_full + i, 1);
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

    if (warp < 16) {
        const int t = warp >> 3, wq = warp & 3;
        prefill64_softmax<EB, FOLD, AUX>(p, t, (warp >> 2) & 1, wq, lane, tbase, s_full + 2 * t, p_full + 2 * t, pv_done + t,
                                    o_done + t, m_full + (t * 4 + wq) * 2, n_tile[t], (pair * 2 + t) * BM, bh, kvh, sh);
    } else if (warp == 18) {
        // ================= TMA producer =================
        if (lane == 0 && n_it > 0) {
            for (int t = 0; t < 2; ++t) {
                if (n_tile[t] == 0) continue;
                ptx::mbar_arrive_expect_tx(q_full + t, C::QTILE);
                for (int c = 0; c < C::NCH; ++c)
                    ptx::tma_load_3d(sQ + t * C::QTILE + c * (128 * 128), &mapQ, q_full + t, c * C::CH,
                                     (pair * 2 + t) * BM, bh);
            }
            for (int it = 0; it < n_it; ++it) {
                const int blk = (p.kv_order == 0) ? it : n_it - 1 - it;
                const int st = it % C::NS;
                const uint32_t ph = (it / C::NS) & 1;
                int kv_row, kv_slab;                         // (paged cache: one block-table entry per block)
                kv_coords(p, b, h / (p.Hq / p.Hkv), kvh, blk, C::BN, kv_row, kv_slab);
                ptx::mbar_wait(k_empty + st, ph ^ 1);
                ptx::mbar_arrive_expect_tx(k_full + st, C::TILE);
                for (int c = 0; c < C::NCH; ++c)
                    ptx::tma_load_3d(sK + st * C::TILE + c * (C::BN * 128), &mapK, k_full + st, c * C::CH,
                                     kv_row, kv_slab);
                ptx::mbar_wait(v_empty + st, ph ^ 1);
                ptx::mbar_arrive_expect_tx(v_full + st, C::TILE);
                for (int c = 0; c < C::NCH; ++c)
                    ptx::tma_load_3d(sV + st * C::TILE + c * (C::BN * 128), &mapV, v_full + st, c * C::CH,
                                     kv_row, kv_slab);
            }
        }
    } else if (n_tile[warp - 16] > 0) {
        // ================= MMA issuer of tile t = warp - 8 (warp-uniform loop, one elected lane issues) ======
        // Block c of tile t uses K/V ring iteration it = c + first (in reverse order the tile with fewer visible
        // blocks joins later).  A ring slot is released by two arrivals, one per tile; on iterations that
        // only one tile uses, that tile arrives twice.
        const int t = warp - 16;
        const int n_t = n_tile[t];
        const bool leader = ptx::elect_one();
        constexpr uint32_t idesc_qk = ptx::make_idesc(C::FMT, C::FMT, ptx::MAJOR_K, ptx::MAJOR_K, BM, C::BN);
        constexpr uint32_t idesc_pv = ptx::make_idesc(C::FMT, C::FMT, ptx::MAJOR_K, ptx::MAJOR_MN, BM, C::D);
        constexpr uint32_t desc_hi = ptx::smem_desc_hi(1024);
        const uint32_t q_lo = ptx::smem_desc_lo(ptx::smem_u32(sQ + t * C::QTILE), 16);
        const uint32_t k_lo = ptx::smem_desc_lo(ptx::smem_u32(sK), 16);
        const uint32_t v_lo = ptx::smem_desc_lo(ptx::smem_u32(sV), C::BN * 128);
        const uint32_t tS = tbase + C::TM_S + t * 128, tO = tbase + C::TM_O + t * 128;
        const int first = (p.kv_order == 0) ? 0 : n_it - n_t;
        const int n_other = n_tile[t ^ 1];
        const int first_other = (p.kv_order == 0) ? 0 : n_it - n_other;
        uint64_t* const sf = s_full + 2 * t;
        uint64_t* const pf = p_full + 2 * t;

        // S_t(c) = Q_t K(it)^T into S buffer c & 1
        auto issue_qk = [&](const int c) {
            const int it = c + first, st = it % C::NS;
            ptx::mbar_wait(k_full + st, (it / C::NS) & 1);
            ptx::tc_fence_after();
            if (leader) {
                const uint32_t b0 = k_lo + st * (C::TILE >> 4);
#pragma unroll
                for (int ks = 0; ks < C::D / C::KSTEP; ++ks) {
                    const uint32_t oq = (((ks * 32) / 128) * (128 * 128) + (ks * 32) % 128) >> 4;
                    const uint32_t ok = (((ks * 32) / 128) * (C::BN * 128) + (ks * 32) % 128) >> 4;
                    ptx::mma_ss<C::KIND>(tS + (c & 1) * 64, ptx::pack2u(q_lo + oq, desc_hi), ptx::pack2u(b0 + ok, desc_hi),
                                         idesc_qk, ks > 0 ? 1u : 0u);
                }
                ptx::tc_commit(sf + (c & 1));
                ptx::tc_commit(k_empty + st);
                if (it < first_other || it >= first_other + n_other) ptx::tc_commit(k_empty + st);
            }
        };
        ptx::mbar_wait(q_full + t, 0);
        issue_qk(0);
        if (n_t > 1) issue_qk(1);
        for (int c = 0; c < n_t; ++c) {
            const int it = c + first, st = it % C::NS;
            ptx::mbar_wait(pf + (c & 1), (c >> 1) & 1);
            ptx::mbar_wait(v_full + st, (it / C::NS) & 1);
            ptx::tc_fence_after();
            if (leader) {
                // O_t += P_t(c) V(it): P in the head of S buffer c & 1
                const uint32_t b0 = v_lo + st * (C::TILE >> 4);
#pragma unroll
                for (int ks = 0; ks < C::BN / C::KSTEP; ++ks)
                    ptx::mma_ts<C::KIND>(tO, tS + (c & 1) * 64 + ks * 8, ptx::pack2u(b0 + ks * ((C::KSTEP * 128) >> 4), desc_hi),
                                         idesc_pv, (c > 0 || ks > 0) ? 1u : 0u);
                ptx::tc_commit(pv_done + t);
                if (c == n_t - 1) ptx::tc_commit(o_done + t);
                ptx::tc_commit(v_empty + st);
                if (it < first_other || it >= first_other + n_other) ptx::tc_commit(v_empty + st);
            }
            if (c + 2 < n_t) issue_qk(c + 2);      // into the buffer this P.V has just released
        }
    }

    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 16) ptx::tmem_dealloc(tbase, 512);
}

}  // namespace fp8attn
