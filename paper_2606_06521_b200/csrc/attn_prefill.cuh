// attn_prefill.cuh -- warp-specialised prefill kernel, d = 128, Bn = 128, two 128-row query tiles per CTA.
//
// Arithmetic as in attn_general.cuh (Alg. 1: exact running max after every block, l from the
// FP32 pre-cast P, cvt.rn.satfinite.e4m3x2.f32 of P*S, epilogue O / (S l)).  Who does what:
//   warps 0-3 / 4-7    "exp" warps, key-column half 0 / 1: lane = query row (TMEM lane) of BOTH tiles; Alg. 1
//                      lines 7-9 (P = exp, row sum from the pre-cast P, cast, P -> TMEM) and line 12
//   warps 8-11 / 12-15 "max" warps of tile 0 / 1: lines 4-6 (block max over all 128 columns, running max, alpha),
//                      published to the exp warps through shared memory, then O <- alpha O in TMEM (line 10)
//   warps 16, 17       tcgen05.mma issuers of tile 0 / 1;  warp 18 TMA producer;  19 idle
// Why: the exp pass is the MUFU-bound part of the kernel (16 ex2 / clk / SM against 16384 FP8 FLOP / clk), so the
// warps that run it do nothing else.  An exp warp alternates between the two tiles -- (it, tile 1), (it, tile 0),
// (it + 1, tile 1) ... -- and while it is in the exp pass of one tile, the tensor pipe turns the other tile
// around (P.V, QK^T of the next block) and the max warp of that tile reduces the new S.  The row maximum needs
// all 128 columns of a row, the exp pass splits them between two warps: with the maximum computed by a third
// warp there is no exchange between the two (round 1 swapped 64-column maxima through a named barrier).
// TMEM (512 columns): S0 [0,128) S1 [128,256) O0 [256,384) O1 [384,512); P over the head of each S quarter.
#pragma once
#include "prefill_common.cuh"

namespace fp8attn {

template <int EB>
struct PrefillKCfg {
    using P = PrefillCfg<EB>;
    static constexpr int THREADS = 640;
    static constexpr int HEAD_GROUP = 16;      // (batch, q head) slabs whose CTAs are launched together
    // which of the 16 element pairs of a P quarter take the FMA-pipe exp2.  BF16 operands: none (measured: the
    // BF16 mode has twice the tensor time and the extra code-to-BF16 conversion, the polynomial costs 6 % there)
    static constexpr int NPOLY = (EB == 1) ? 0x8080 : 0;
    // q_full[2] k_full/k_empty/v_full/v_empty[NS] s_full[2] p_full[2][2] m_full[2][4] o_ready[2] o_done[2]
    static constexpr int N_BARS = 2 + 4 * P::NS + 2 + 4 + 8 + 2 + 2;
    // + mstat[2 tiles][2 block parities][128 rows] float2 + lsum[2 tiles][2 halves][128 rows] float
    // + lscale[2 tiles][128 rows] float
    static constexpr int SMEM_BYTES = (2 + 2 * P::NS) * P::TILE + 1024 /*align*/ + N_BARS * 8 + 16 + 2 * 2 * 128 * 8 +
                                      2 * 2 * 128 * 4 + 2 * 128 * 4;
    static constexpr int REG_EXP = 128, REG_MAX = 80, REG_MISC = 56;   // 256 (128 + 80) + 128 * 56 <= 640 * 96
};

// Which blocks of a tile need the mask for some row of the 32-row group `wq`: blocks whose first key index
// exceeds the returned value (bottom-right causal diagonal, tail of the sequence, rows past the end of a
// variable-length sequence; reading R15).
__device__ __forceinline__ int mask_threshold(const FwdParams& p, const Seq& s, int row0, int wq) {
    if (row0 + wq * 32 + 31 >= s.Lq) return -(1 << 30);        // some row of the group does not exist: always mask
    const long long wvis = p.causal ? (long long)row0 + wq * 32 + (s.Lk - s.Lq) : (long long)s.Lk - 1;
    long long thr = wvis - 127 < (long long)s.Lk - 128 ? wvis - 127 : (long long)s.Lk - 128;
    if (thr < -(1ll << 30)) thr = -(1ll << 30);
    return (int)thr;
}

// What a max warp publishes per (tile, block, row) for the exp warps: the exponent offset of line 7,
// -m_new c log2(e) (+ log2 S when the scale is folded), and alpha of line 6.
struct RowStat {
    float negm, alpha;
};

// ---- max warp (t, wq): Alg. 1 lines 4-6 for rows 32 wq .. 32 wq + 31 of tile t, then O <- alpha O ----
// ---- line 12 for one (tile, column half): O / (S l) of 32 rows x 64 columns, written as 32-row x 128-byte boxes
// (128-byte swizzle; FP32: two boxes of 32 floats, BF16: one box of 64) into the K / V ring -- no MMA reads it any
// more once both tiles are done -- and stored with TMA (rows >= Lq are clipped by the map).  The four warps that can
// read a 32-lane quarter of TMEM (two exp warps, the max warps of both tiles) take one (tile, half) each.
template <int EB, bool FOLD, typename OB>
__device__ __forceinline__ void prefill_store_half(const FwdParams& p, int t, int half, int wq, int lane, uint32_t tbase,
                                                   const float* lsum, const float* lscale, OB o_done, bool has_blocks,
                                                   bool other_has_blocks,
                                                   int row0, int bh, float vs, const CUtensorMap* mapO, uint8_t* stage,
                                                   bool write_row_sum) {
    using C = PrefillCfg<EB>;
    const int rl = wq * 32 + lane;
    // both tiles must be done: the staging area is the K / V ring, which the other tile's MMAs may still read
    if (has_blocks) ptx::mbar_wait(o_done + t, 0);
    if (other_has_blocks) ptx::mbar_wait(o_done + (t ^ 1), 0);
    ptx::tc_fence_after();
    const float l_all = lsum[(t * 2) * 128 + rl] + lsum[(t * 2 + 1) * 128 + rl];
    // l_all and O carry the same factor: S when the static scale is folded into the exponent, the last block's 2^k
    // under the dynamic scale (published by the max warp), 1 otherwise
    const float carried = has_blocks ? lscale[t * 128 + rl] : 1.0f;
    if (write_row_sum && row0 + rl < p.Lq && p.row_sum != nullptr) p.row_sum[(long long)bh * p.Lq + row0 + rl] = l_all / carried;
    const float inv = (l_all > 0.0f) ? (FOLD ? vs / l_all : vs / (p.S * l_all)) : 0.0f;
    if (row0 >= p.Lq) return;                   // no row of this tile exists (warp-uniform)
    const uint32_t tO = tbase + (static_cast<uint32_t>(wq * 32) << 16) + C::TM_O + t * 128 + half * 64;
#pragma unroll 1
    for (int cb = 0; cb < 2; ++cb) {
        const int ch = half * 2 + cb;           // 32-column chunk of the output row
        uint32_t v[32];
        if (has_blocks) {
            ptx::tmem_ld_x32(tO + cb * 32, v);
            ptx::tmem_wait_ld();
        } else {
#pragma unroll
            for (int e = 0; e < 32; ++e) v[e] = 0u;
        }
        if (p.o_bf16) {
            uint8_t* box = stage + (half * 8 + wq) * 4096;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                uint4 w4;
                w4.x = ptx::cvt_bf16x2(__uint_as_float(v[8 * j]) * inv, __uint_as_float(v[8 * j + 1]) * inv);
                w4.y = ptx::cvt_bf16x2(__uint_as_float(v[8 * j + 2]) * inv, __uint_as_float(v[8 * j + 3]) * inv);
                w4.z = ptx::cvt_bf16x2(__uint_as_float(v[8 * j + 4]) * inv, __uint_as_float(v[8 * j + 5]) * inv);
                w4.w = ptx::cvt_bf16x2(__uint_as_float(v[8 * j + 6]) * inv, __uint_as_float(v[8 * j + 7]) * inv);
                *reinterpret_cast<uint4*>(box + lane * 128 + (((cb * 4 + j) ^ (lane & 7)) << 4)) = w4;
            }
            if (cb == 1) {
                ptx::fence_proxy_async_smem();
                __syncwarp();
                if (lane == 0) ptx::tma_store_3d(mapO, box, half * 64, row0 + wq * 32, bh);
            }
            continue;
        }
        uint8_t* box = stage + (ch * 4 + wq) * 4096;
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const float4 o4 = make_float4(__uint_as_float(v[4 * j]) * inv, __uint_as_float(v[4 * j + 1]) * inv,
                                          __uint_as_float(v[4 * j + 2]) * inv, __uint_as_float(v[4 * j + 3]) * inv);
            *reinterpret_cast<float4*>(box + lane * 128 + ((j ^ (lane & 7)) << 4)) = o4;
        }
        ptx::fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) ptx::tma_store_3d(mapO, box, ch * 32, row0 + wq * 32, bh);
    }
    if (lane == 0) {
        ptx::bulk_commit_group();
        ptx::bulk_wait_group_read0();
    }
}

// EXT: the instance that carries the extensions (dynamic P scale, variable-length sequences, paged KV); the plain
// instance has none of that code (measured: 1.3 % of cfg3).
template <int EB, bool FOLD, bool EXT>
__device__ __forceinline__ void prefill_max_warp(const FwdParams& p, int t, int wq, int lane, uint32_t tbase,
                                                 ptx::SPtr<uint64_t> s_full_t, ptx::SPtr<uint64_t> m_full_w,
                                                 ptx::SPtr<RowStat> mstat_t, float* lscale_t, ptx::SPtr<uint64_t> o_ready_t,
                                                 int n_t, int row0, int bh, int kvh, const float* lsum,
                                                 ptx::SPtr<uint64_t> o_done, int n_other, const CUtensorMap* mapO,
                                                 uint8_t* stage) {
    using C = PrefillCfg<EB>;
    const uint32_t tlane = tbase + (static_cast<uint32_t>(wq * 32) << 16);
    const uint32_t tS = tlane + C::TM_S + t * 128, tO = tlane + C::TM_O + t * 128;
    const int rl = wq * 32 + lane;
    const Seq sq = EXT ? seq_of(p, bh / p.Hq, 128) : Seq{p.Lq, p.Lk, p.nb};
    const int jlim = last_visible_key(p, sq, row0 + rl);
    const int mask_from = mask_threshold(p, sq, row0, wq);
    float c_nat = p.sm_scale;
    if constexpr (EB == 1) c_nat *= p.q_scale[bh] * p.k_scale[kvh];
    const float cl2 = c_nat * LOG2E;
    const bool dynamic = EXT && p.scale_mode == 1;  // reading R26 (the host launches the FOLD instance for it)
    const float log2S = (FOLD && !dynamic) ? log2f(p.S) : 0.0f;   // exact for S = 2^k
    float m_run = -INFINITY;
    int k_run = 0;            // dynamic: the exponent O and the row sums carry

#pragma unroll 1
    for (int c = 0; c < n_t; ++c) {
        const int blk = (p.kv_order == 0) ? c : n_t - 1 - c;
        const int j0 = blk * 128;
        const bool mask = j0 > mask_from;
        ptx::mbar_wait(s_full_t, c & 1);
        ptx::tc_fence_after();
        // ---- line 4: block max over the 128 columns of the row.  A TMEM load takes ~300 cycles to come back while
        // the tensor pipe is busy and tcgen05.wait::ld waits for every load in flight: two round trips of 64 columns ----
        float m0 = -INFINITY, m1 = -INFINITY;
#pragma unroll
        for (int hb = 0; hb < 2; ++hb) {
            uint32_t v[64];
            ptx::tmem_ld_x32(tS + hb * 64, v);
            ptx::tmem_ld_x32(tS + hb * 64 + 32, v + 32);
            ptx::tmem_wait_ld();
            if (mask) {
                mask32(v, j0 + hb * 64, jlim);
                mask32(v + 32, j0 + hb * 64 + 32, jlim);
            }
#pragma unroll
            for (int e = 0; e < 64; e += 4) {
                m0 = fmaxf(fmaxf(m0, __uint_as_float(v[e])), __uint_as_float(v[e + 1]));
                m1 = fmaxf(fmaxf(m1, __uint_as_float(v[e + 2])), __uint_as_float(v[e + 3]));
            }
        }
        // ---- lines 5-6 ----
        const float m_loc = fmaxf(m0, m1);
        const float m_new = fmaxf(m_run, m_loc);
        const float m_used = (m_new == -INFINITY) ? 0.0f : m_new;
        float alpha = ptx::ex2_approx((m_run - m_used) * cl2);             // 0 when m_run = -inf
        float negm = fmaf(-m_used, cl2, log2S);
        m_run = m_new;
        if (dynamic) {
            // this block's scale 2^k goes into the exponent of P; what O and the row sums carry (the previous
            // block's scale) is brought to it together with alpha -- exact, a power of two (Prop. 5)
            const int k_new = (m_loc == -INFINITY) ? k_run : dyn_exponent((m_new - m_loc) * cl2);
            negm = fmaf(-m_used, cl2, (float)k_new);
            alpha *= exp2f((float)(k_new - k_run));
            k_run = k_new;
        }
        if (c == n_t - 1) lscale_t[rl] = dynamic ? exp2f((float)k_run) : (FOLD ? p.S : 1.0f);   // read after o_done
        ptx::st_shared_v2(mstat_t + (c & 1) * 128 + rl, negm, alpha);
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(m_full_w);
        // ---- line 10, first half: O <- alpha O.  S(c) complete implies P.V(c-1) complete (in-order pipe) ----
        if (c > 0 && __any_sync(0xFFFFFFFFu, alpha != 1.0f)) {
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
        if (lane == 0) ptx::mbar_arrive(o_ready_t);
    }
    // statistics: the final running max (natural-log units of the scaled logit)
    const int qrow = row0 + rl;
    if (p.row_max != nullptr && qrow < p.Lq)
        p.row_max[(long long)bh * p.Lq + qrow] = (m_run == -INFINITY) ? -INFINITY : m_run * c_nat;
    // this warp's share of the epilogue: (tile t, the column half the exp warps do not store)
    float vs = 1.0f;
    if constexpr (EB == 1) vs = p.v_scale[kvh];
    ptx::named_bar_sync(1 + wq, 128);           // the row sums of the exp warps are in shared memory
    prefill_store_half<EB, FOLD>(p, t, 1 - t, wq, lane, tbase, lsum, lscale_t - t * 128, o_done, n_t > 0, n_other > 0, row0,
                                 bh, vs, mapO, stage, false);
}

// One P quarter: exp / sum / cast (exp_chunk), statistics (AUX), P over the head of its S quarter in TMEM (the A
// operand of P.V), arrival on the issuer's barrier.
template <int EB, bool FOLD, int NPOLY, bool AUX, typename BAR>
__device__ __forceinline__ void p_quarter(const uint32_t* v, uint32_t tS, int quarter, int j0, int jlim, uint64_t cl2_2,
                                          uint64_t negm_2, uint64_t s_2, uint64_t& sum_a, uint64_t& sum_b, BAR bar,
                                          int lane, uint8_t* dump_row, bool count, uint32_t& zeros, const FwdParams& p,
                                          bool sink_blk) {
    using C = PrefillCfg<EB>;
    uint32_t w[C::P_COLS / 4];
    exp_chunk<EB, FOLD, false, NPOLY>(v, w, j0 + quarter * 32, jlim, cl2_2, negm_2, s_2, sum_a, sum_b);
    if constexpr (EB == 1) ptx::tmem_st_x8(tS + quarter * 32, w);
    else ptx::tmem_st_x16(tS + quarter * 32, w);
    ptx::tmem_wait_st();
    ptx::tc_fence_before();
    __syncwarp();
    if (lane == 0) ptx::mbar_arrive(bar);
    // (after the hand-off: the statistics are not on the path the tensor pipe waits for)
    if constexpr (AUX) zeros += chunk_statistics<EB>(w, j0 + quarter * 32, jlim, dump_row, count, p, sink_blk);
}

// Lines 8-9 of one P quarter whose exp_part is done: sum / cast (cast_part), P over the head of its S quarter in TMEM,
// arrival on the issuer's barrier, then the statistics (AUX).
template <int EB, bool FOLD, bool AUX, typename BAR>
__device__ __forceinline__ void p_quarter_finish(const float* pr, uint32_t tS, int quarter, int j0, int jlim, uint64_t s_2,
                                                 uint64_t& sum_a, uint64_t& sum_b, BAR bar, int lane,
                                                 uint8_t* dump_row, bool count, uint32_t& zeros, const FwdParams& p,
                                                 bool sink_blk) {
    using C = PrefillCfg<EB>;
    uint32_t w[C::P_COLS / 4];
    cast_part<EB, FOLD>(pr, w, s_2, sum_a, sum_b);
    if constexpr (EB == 1) ptx::tmem_st_x8(tS + quarter * 32, w);
    else ptx::tmem_st_x16(tS + quarter * 32, w);
    ptx::tmem_wait_st();
    ptx::tc_fence_before();
    __syncwarp();
    if (lane == 0) ptx::mbar_arrive(bar);
    if constexpr (AUX) zeros += chunk_statistics<EB>(w, j0 + quarter * 32, jlim, dump_row, count, p, sink_blk);
}

// ---- exp warp (wq, half): Alg. 1 lines 7-9 and 12 for its rows of both tiles, its 64 key columns ----
template <int EB, bool FOLD, bool AUX, bool EXT>
__device__ __forceinline__ void prefill_exp_warp(const FwdParams& p, int wq, int half, int lane, uint32_t tbase,
                                                 ptx::SPtr<uint64_t> m_full, ptx::SPtr<uint64_t> p_full,
                                                 ptx::SPtr<RowStat> mstat, float* lsum, const float* lscale,
                                                 ptx::SPtr<uint64_t> o_done, const int* n_tile, int n_it, int pair, int bh,
                                                 int kvh, const CUtensorMap* mapO, uint8_t* stage0, uint8_t* stage1) {
    using C = PrefillCfg<EB>;
    using CK = PrefillKCfg<EB>;
    const uint32_t tlane = tbase + (static_cast<uint32_t>(wq * 32) << 16);
    const int rl = wq * 32 + lane;              // row within the tile = TMEM lane

    float c_nat = p.sm_scale, vs = 1.0f;
    if constexpr (EB == 1) {
        c_nat *= p.q_scale[bh] * p.k_scale[kvh];
        vs = p.v_scale[kvh];
    }
    const float cl2 = c_nat * LOG2E;
    const uint64_t cl2_2 = ptx::pack2(cl2, cl2), s_2 = ptx::pack2(p.S, p.S);

    const Seq sq = EXT ? seq_of(p, bh / p.Hq, 128) : Seq{p.Lq, p.Lk, p.nb};
    int jlim[2], first[2], mask_from[2];
    bool count_row[2];        // AUX: this row exists and its zero codes are counted
    uint8_t* dump_row[2];     // AUX: this row of the P dump (fp8attn_stats.p_codes), else null
    uint32_t uf_sink = 0, uf_other = 0;   // AUX: zero codes among visible non-sink keys (sink block / other blocks)
    float l_run[2] = {0.0f, 0.0f};
#pragma unroll
    for (int t = 0; t < 2; ++t) {
        const int row0 = (pair * 2 + t) * BM;
        jlim[t] = last_visible_key(p, sq, row0 + rl);
        mask_from[t] = mask_threshold(p, sq, row0, wq);
        first[t] = (p.kv_order == 0) ? 0 : n_it - n_tile[t];
        count_row[t] = AUX && p.underflow != nullptr && row0 + rl < sq.Lq;
        dump_row[t] = (AUX && p.p_codes != nullptr && bh == p.p_bh && row0 + rl < sq.Lq)
                          ? p.p_codes + (size_t)(row0 + rl) * p.Lk
                          : nullptr;
    }

    // A successful mbarrier wait takes ~100 cycles to report.  When the next block belongs to the other tile its
    // running max has been ready for a while, so that barrier is probed before the second P quarter of the
    // current block and the answer is read when the next block starts (probed_tile >= 0: a probe is pending).
    FP8ATTN_DECL_PROBE_PRED();
    int probed_tile = -1;
#pragma unroll 1
    for (int it = 0; it < n_it; ++it) {
#pragma unroll
        for (int tt = 0; tt < 2; ++tt) {
            const int t = 1 - tt;               // tile 1 first: under a causal mask it has the extra block
            const int c = it - first[t];
            if (c < 0 || c >= n_tile[t]) continue;
            // the block after this one, if it is a block of the other tile
            const int it_o = it + tt;           // tile 1 -> (it, tile 0);  tile 0 -> (it + 1, tile 1)
            const int c_o = it_o - first[t ^ 1];
            const bool probe_next = c_o >= 0 && c_o < n_tile[t ^ 1];
            const int blk = (p.kv_order == 0) ? c : n_tile[t] - 1 - c;
            const int j0 = blk * 128;
            const bool mask = j0 > mask_from[t];
            const uint32_t tS = tlane + C::TM_S + t * 128;
            // ---- the running max of block c is published (which implies S(c) is complete): this warp's 64
            // logits of the row, loaded once.  (Waiting for S first, loading, then waiting for the max -- two
            // barrier round trips -- measured 8 % slower than this single wait.) ----
            uint32_t r[64];
            if (probed_tile != t || !ptx::mbar_probe_result()) ptx::mbar_wait(m_full + 4 * t + wq, c & 1);
            probed_tile = -1;
            ptx::tc_fence_after();
            ptx::tmem_ld_x32(tS + half * 64, r);
            ptx::tmem_ld_x32(tS + half * 64 + 32, r + 32);
            const float2 ms = ptx::ld_shared_v2(mstat + (t * 2 + (c & 1)) * 128 + rl);   // (negm, alpha)
            const uint64_t negm_2 = ptx::pack2(ms.x, ms.x);
            ptx::tmem_wait_ld();
            if (mask) {
                mask32(r, j0 + half * 64, jlim[t]);
                mask32(r + 32, j0 + half * 64 + 32, jlim[t]);
            }
            // ---- lines 7-9: two P quarters ----
            uint64_t sum_a = ptx::pack2(0.f, 0.f), sum_b = sum_a;
            // (a masked logit is -inf: exp2_poly2 turns it into 2^-125, which casts to the E4M3 code 0 and is
            // far below one ulp of a row sum that holds a visible key; rows without any visible key are set to
            // l = 0 in the epilogue)
            // AUX: the counter this block adds to (blocks that hold a sink key / all others); rows >= Lq do not
            // exist and are not counted
            const bool sink_blk = AUX && sink_in_range(p, j0, 128);
            uint32_t zeros = 0;
            // line 7 of both quarters first (in place: the logits become P), then lines 8-9 and the hand-off of each:
            // the MUFU pipe works on the second quarter while the first one is cast, stored and handed over
            float* const pr = reinterpret_cast<float*>(r);
            exp_part<false, CK::NPOLY>(r, pr, j0 + half * 64, jlim[t], cl2_2, negm_2);
            exp_part<false, CK::NPOLY>(r + 32, pr + 32, j0 + half * 64 + 32, jlim[t], cl2_2, negm_2);
            p_quarter_finish<EB, FOLD, AUX>(pr, tS, 2 * half, j0, jlim[t], s_2, sum_a, sum_b, p_full + 2 * t + 0, lane,
                                            dump_row[t], count_row[t], zeros, p, sink_blk);
            if (probe_next) {
                ptx::mbar_probe(m_full + 4 * (t ^ 1) + wq, c_o & 1);
                probed_tile = t ^ 1;
            }
            p_quarter_finish<EB, FOLD, AUX>(pr + 32, tS, 2 * half + 1, j0, jlim[t], s_2, sum_a, sum_b, p_full + 2 * t + 1,
                                            lane, dump_row[t], count_row[t], zeros, p, sink_blk);
            if constexpr (AUX) {
                if (sink_blk) uf_sink += zeros;
                else uf_other += zeros;
            }
            float sa, sb, sc, sd;
            ptx::unpack2(sum_a, sa, sb);
            ptx::unpack2(sum_b, sc, sd);
            l_run[t] = ms.y * l_run[t] + ((sa + sb) + (sc + sd));   // line 8 (this warp's columns)
        }
    }

    if constexpr (AUX) {
        if (p.underflow != nullptr) {       // one atomic per warp and counter (ballot / popc style reduction)
            const uint32_t a = __reduce_add_sync(0xFFFFFFFFu, uf_sink), b2 = __reduce_add_sync(0xFFFFFFFFu, uf_other);
            if (lane == 0) {
                if (a) atomicAdd(p.underflow + 0, (unsigned long long)a);
                if (b2) atomicAdd(p.underflow + 1, (unsigned long long)b2);
            }
        }
    }
    // ---- line 12: O / (S l), row sum.  The two warps of a row add their partial sums (same running max, so they
    // just add); then this warp stores (tile `half`, column half `half`), see prefill_store_half ----
#pragma unroll
    for (int t = 0; t < 2; ++t)
        lsum[(t * 2 + half) * 128 + rl] = (jlim[t] < 0) ? 0.0f : l_run[t];     // no visible key: l = 0 exactly
    ptx::named_bar_sync(1 + wq, 128);           // the four warps of this 32-row group (2 exp + 2 max)
    if (half == 0 && p.row_sum != nullptr) {    // the row sum of the tile this warp does not store
        const int row1 = (pair * 2 + 1) * BM + rl;
        const float l1 = lsum[2 * 128 + rl] + lsum[3 * 128 + rl];
        if (row1 < p.Lq) p.row_sum[(long long)bh * p.Lq + row1] = l1 / ((n_tile[1] > 0) ? lscale[128 + rl] : 1.0f);
    }
    prefill_store_half<EB, FOLD>(p, half, half, wq, lane, tbase, lsum, lscale, o_done, n_tile[half] > 0,
                                 n_tile[half ^ 1] > 0, (pair * 2 + half) * BM, bh, vs, mapO, half ? stage1 : stage0, half == 0);
}
// ---- the kernel ---------------------------------------------------------------------------------
// grid = ceil(Lq / 256) * B*Hq CTAs in one dimension (order: see below).
template <int EB, bool FOLD, bool AUX = false, bool EXT = false>
__global__ void __launch_bounds__(640, 1)
attn_prefill_kernel(const __grid_constant__ CUtensorMap mapQ, const __grid_constant__ CUtensorMap mapK,
                     const __grid_constant__ CUtensorMap mapV, const __grid_constant__ CUtensorMap mapO,
                     const FwdParams p) {
    using C = PrefillCfg<EB>;
    using C4 = PrefillKCfg<EB>;
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
    uint64_t* s_full = v_empty + C::NS;           // [2 tiles]                   MMA -> max warps
    uint64_t* p_full = s_full + 2;                // [2 tiles][2 steps]          exp warps (8) -> MMA
    uint64_t* m_full = p_full + 4;                // [2 tiles][4 row groups]     max warp -> its two exp warps
    uint64_t* o_ready = m_full + 8;               // [2]                         max warps (4) -> MMA
    uint64_t* o_done = o_ready + 2;               // [2]
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(o_done + 2);
    RowStat* mstat = reinterpret_cast<RowStat*>(tmem_slot + 4);   // [2 tiles][2 block parities][128 rows]
    float* lsum = reinterpret_cast<float*>(mstat + 2 * 2 * 128);  // [2 tiles][2 halves][128 rows]
    float* lscale = lsum + 2 * 2 * 128;                           // [2 tiles][128 rows]  factor the row sums carry

    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xFFFFFFFFu, tid >> 5, 0);   // provably warp-uniform
    // 1-D grid, launch order = longest work first within groups of HEAD_GROUP (batch, q head) slabs: a group's
    // K and V (2 x Lk x 128 B per kv head) stay in L2 while its CTAs run, and only the last group's lightest CTAs
    // are left for the tail of the kernel.
    const int n_pairs = (p.Lq + 2 * BM - 1) / (2 * BM), n_heads = p.B * p.Hq;
    const int grp = (int)blockIdx.x / (C4::HEAD_GROUP * n_pairs);
    const int rem = (int)blockIdx.x - grp * C4::HEAD_GROUP * n_pairs;
    const int grp_size = min(C4::HEAD_GROUP, n_heads - grp * C4::HEAD_GROUP);
    const int pair_idx = rem / grp_size;
    const int pair = p.causal ? n_pairs - 1 - pair_idx : pair_idx;
    const int bh = grp * C4::HEAD_GROUP + rem % grp_size;
    const int b = bh / p.Hq, h = bh % p.Hq;
    const int kvh = b * p.Hkv + h / (p.Hq / p.Hkv);

    // visible block count of each tile (bottom-right causal, reading R15; this batch element's lengths)
    const Seq sq = EXT ? seq_of(p, b, C::BN) : Seq{p.Lq, p.Lk, p.nb};
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
        ptx::prefetch_tmap(&mapO);
        for (int i = 0; i < 2; ++i) ptx::mbar_init(q_full + i, 1);
        for (int i = 0; i < C::NS; ++i) {
            ptx::mbar_init(k_full + i, 1);
            ptx::mbar_init(v_full + i, 1);
            ptx::mbar_init(k_empty + i, 2);   // one arrival per tile
            ptx::mbar_init(v_empty + i, 2);
        }
        for (int i = 0; i < 2; ++i) {
            ptx::mbar_init(s_full + i, 1);
            ptx::mbar_init(o_ready + i, 4);
            ptx::mbar_init(o_done + i, 1);
        }
        for (int i = 0; i < 4; ++i) ptx::mbar_init(p_full + i, 8);
        for (int i = 0; i < 8; ++i) ptx::mbar_init(m_full + i, 1);
        ptx::fence_mbar_init();
    }
    if (warp == 16) {
        __syncwarp();
        ptx::tmem_alloc(tmem_slot, 512);
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    // Every role reads the TMEM base address itself and builds its own 32-bit shared addresses from one opaque base
    // register, after its setmaxnreg: a value defined up here is spilled by the register budget of the smallest
    // role and reloaded from local memory at every use, and generic pointers into the aligned dynamic shared
    // memory are rematerialised (S2UR window + align) at every barrier operation.
    constexpr uint32_t OFF_BARS = (2 + 2 * C::NS) * C::TILE;
    constexpr uint32_t OFF_MSTAT = OFF_BARS + C4::N_BARS * 8 + 16;
    const auto shared_base = [&]() { return ptx::opaque_u32((ptx::smem_u32(smem_raw) + 1023u) & ~1023u); };
    if (warp < 8) {
        ptx::setmaxnreg_inc<C4::REG_EXP>();
        const uint32_t tbase = ptx::ld_shared_u32(tmem_slot);
        const ptx::SPtr<uint64_t> sbar{shared_base() + OFF_BARS};
        const ptx::SPtr<RowStat> smstat{sbar.a + (OFF_MSTAT - OFF_BARS)};
        prefill_exp_warp<EB, FOLD, AUX, EXT>(p, warp & 3, warp >> 2, lane, tbase, sbar + (8 + 4 * C::NS), sbar + (4 + 4 * C::NS),
                                             smstat, lsum, lscale, sbar + (18 + 4 * C::NS), n_tile, n_it, pair, bh, kvh, &mapO,
                                             sK, sV);
    } else if (warp < 16) {
        ptx::setmaxnreg_dec<C4::REG_MAX>();
        const uint32_t tbase = ptx::ld_shared_u32(tmem_slot);
        const ptx::SPtr<uint64_t> sbar{shared_base() + OFF_BARS};
        const ptx::SPtr<RowStat> smstat{sbar.a + (OFF_MSTAT - OFF_BARS)};
        const int t = (warp - 8) >> 2, wq = warp & 3;
        prefill_max_warp<EB, FOLD, EXT>(p, t, wq, lane, tbase, sbar + (2 + 4 * C::NS + t), sbar + (8 + 4 * C::NS + 4 * t + wq),
                                        smstat + t * 2 * 128, lscale + t * 128, sbar + (16 + 4 * C::NS + t), n_tile[t],
                                        (pair * 2 + t) * BM, bh, kvh, lsum, sbar + (18 + 4 * C::NS), n_tile[t ^ 1], &mapO,
                                        t ? sV : sK);
    } else {
        ptx::setmaxnreg_dec<C4::REG_MISC>();
        // the same barriers and tiles as 32-bit shared addresses (these names shadow the generic pointers above)
        const uint32_t sb = shared_base();
        const ptx::SPtr<uint8_t> sQ{sb}, sK{sb + 2 * C::TILE}, sV{sb + (2 + C::NS) * C::TILE};
        const ptx::SPtr<uint64_t> q_full{sb + OFF_BARS};
        const ptx::SPtr<uint64_t> k_full = q_full + 2, k_empty = k_full + C::NS, v_full = k_empty + C::NS,
                                  v_empty = v_full + C::NS, s_full = v_empty + C::NS, p_full = s_full + 2,
                                  o_ready = p_full + 12, o_done = o_ready + 2;
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
                    int kv_row = blk * C::BN, kv_slab = kvh;
                    if constexpr (EXT) kv_coords(p, b, h / (p.Hq / p.Hkv), kvh, blk, C::BN, kv_row, kv_slab);   // paged cache
                    ptx::mbar_wait(k_empty + st, ph ^ 1);
                    ptx::mbar_arrive_expect_tx(k_full + st, C::TILE);
                    for (int c = 0; c < C::NCH; ++c)
                        ptx::tma_load_3d(sK + st * C::TILE + c * (128 * 128), &mapK, k_full + st, c * C::CH,
                                         kv_row, kv_slab);
                    ptx::mbar_wait(v_empty + st, ph ^ 1);
                    ptx::mbar_arrive_expect_tx(v_full + st, C::TILE);
                    for (int c = 0; c < C::NCH; ++c)
                        ptx::tma_load_3d(sV + st * C::TILE + c * (128 * 128), &mapV, v_full + st, c * C::CH,
                                         kv_row, kv_slab);
                }
            }
        } else if (warp < 18 && n_tile[warp - 16] > 0) {
            // ================= MMA issuer of tile t = warp - 16 =================
            // Block c of tile t uses K/V ring iteration it = c + first.  A ring slot is released by two
            // arrivals, one per tile; on iterations that only one tile uses, that tile arrives twice.
            const int t = warp - 16;
            const int n_t = n_tile[t];
            const bool leader = ptx::elect_one();
            constexpr uint32_t idesc_qk = ptx::make_idesc(C::FMT, C::FMT, ptx::MAJOR_K, ptx::MAJOR_K, BM, C::BN);
            constexpr uint32_t idesc_pv = ptx::make_idesc(C::FMT, C::FMT, ptx::MAJOR_K, ptx::MAJOR_MN, BM, C::D);
            constexpr uint32_t desc_hi = ptx::smem_desc_hi(1024);
            const uint32_t q_lo = ptx::smem_desc_lo(ptx::smem_u32(sQ + t * C::TILE), 16);
            const uint32_t k_lo = ptx::smem_desc_lo(ptx::smem_u32(sK), 16);
            const uint32_t v_lo = ptx::smem_desc_lo(ptx::smem_u32(sV), C::BN * 128);
            const uint32_t tbase = ptx::ld_shared_u32(tmem_slot);
            const uint32_t tS = tbase + C::TM_S + t * 128, tO = tbase + C::TM_O + t * 128;
            const int first = (p.kv_order == 0) ? 0 : n_it - n_t;
            const int n_other = n_tile[t ^ 1];
            const int first_other = (p.kv_order == 0) ? 0 : n_it - n_other;
            const ptx::SPtr<uint64_t> pf = p_full + 2 * t;

            // S_t = Q_t K^T on ring iteration it
            // (the caller has waited for the K tile of ring iteration it: k_full)
            auto qk_block = [&](const int it) {
                const int st = it % C::NS;
                if (leader) {
                    const uint32_t b0 = k_lo + st * (C::TILE >> 4);
#pragma unroll
                    for (int ks = 0; ks < C::D / C::KSTEP; ++ks) {
                        const uint32_t o = (((ks * 32) / 128) * (128 * 128) + (ks * 32) % 128) >> 4;
                        ptx::mma_ss<C::KIND>(tS, ptx::pack2u(q_lo + o, desc_hi), ptx::pack2u(b0 + o, desc_hi), idesc_qk,
                                             ks > 0 ? 1u : 0u);
                    }
                    ptx::tc_commit(s_full + t);
                    ptx::tc_commit(k_empty + st);
                    if (it < first_other || it >= first_other + n_other) ptx::tc_commit(k_empty + st);
                }
            };
            // O_t += P_t[:, 32q .. 32q+32) V[32q .. 32q+32, :]
            auto pv_quarter = [&](const int q, const int it, const uint32_t acc0) {
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
                }
            };

            ptx::mbar_wait(q_full + t, 0);
            ptx::tc_fence_after();
            ptx::mbar_wait(k_full + first % C::NS, (first / C::NS) & 1);
            ptx::tc_fence_after();
            qk_block(first);
            for (int c = 0; c < n_t; ++c) {
                const int it = c + first;
                const int st = it % C::NS;
                const bool has_next = c + 1 < n_t;
                ptx::mbar_wait(v_full + st, (it / C::NS) & 1);
                ptx::mbar_wait(o_ready + t, c & 1);
                // first quarter of each column half, then the second one (the order the softmax warps write them)
                ptx::mbar_wait(pf + 0, c & 1);
                ptx::tc_fence_after();
                pv_quarter(0, it, c > 0 ? 1u : 0u);
                pv_quarter(2, it, 1u);
                // everything between the last P quarter and S(c+1) is on the chain the exp warps wait for (an mbarrier
                // wait costs 150-300 cycles even when the phase is complete): the next K tile is waited for here
                if (has_next) ptx::mbar_wait(k_full + (it + 1) % C::NS, ((it + 1) / C::NS) & 1);
                ptx::mbar_wait(pf + 1, c & 1);
                ptx::tc_fence_after();
                pv_quarter(1, it, 1u);
                pv_quarter(3, it, 1u);
                if (leader) {
                    if (!has_next) ptx::tc_commit(o_done + t);
                    ptx::tc_commit(v_empty + st);
                    if (it < first_other || it >= first_other + n_other) ptx::tc_commit(v_empty + st);
                }
                if (has_next) qk_block(it + 1);
            }
        }
    }

    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 16) ptx::tmem_dealloc(ptx::ld_shared_u32(tmem_slot), 512);
}

}  // namespace fp8attn
