// common.cuh -- constants and the kernel parameter block shared by every attention kernel of libfp8attn.so.
#pragma once
#include <cuda_fp16.h>
#include "ptx.cuh"

namespace fp8attn {

constexpr int BM = 128;   // query rows per tile = UMMA M = TMEM lanes
constexpr float LOG2E = 1.4426950408889634f;

constexpr int MAX_SINKS = 32;          // FP8ATTN_MAX_SINKS
constexpr int DYN_K_MAX = 30;          // largest exponent of the dynamic P scale (reading R26)
constexpr float LOG2_448 = 8.80735492205760410744f;

struct FwdParams {
    void* o;          // float32, or bfloat16 when o_bf16
    float* row_max;
    float* row_sum;
    unsigned long long* underflow;
    uint8_t* p_codes;
    int p_bh;
    const float* q_scale;
    const float* k_scale;
    const float* v_scale;
    float* part_o;    // [ns][rows][d]   unnormalised O of each split
    float* part_ml;   // [ns][rows][2]   (m in natural-log units of the scaled logit, l)
    int B, Hq, Hkv, Lq, Lk, causal, kv_order, n_sink, num_splits, nb;
    int q_slabs, kv_slabs;   // B*Hq, B*Hkv: plane stride of the staged operands, in slabs
    float S, sm_scale;
    int scale_mode;          // 1: dynamic per-(row, block) power-of-two scale
    int o_bf16;
    int n_sinkpos;           // -1: the sink keys are the first n_sink keys; else sink_pos[0 .. n_sinkpos) (ascending)
    int sink_pos[MAX_SINKS];
    const int* seqlens_q;    // [B] or null
    const int* seqlens_k;    // [B] or null
    const int* block_table;  // [B, max_pages] or null: k, v are page pools [num_pages, Hkv, page_size, d]
    int page_size, max_pages;
};

// ---- per-batch-element geometry (variable-length sequences) and the address of a KV block (paged cache) ----
struct Seq {
    int Lq, Lk, nb;          // query rows, keys and KV blocks of this batch element
};
__device__ __forceinline__ Seq seq_of(const FwdParams& p, int b, int bn) {
    Seq s{p.Lq, p.Lk, p.nb};
    if (p.seqlens_q != nullptr) s.Lq = min(p.Lq, max(0, p.seqlens_q[b]));
    if (p.seqlens_k != nullptr) {
        s.Lk = min(p.Lk, max(0, p.seqlens_k[b]));
        s.nb = (s.Lk + bn - 1) / bn;
    }
    return s;
}
// Last key row `qrow` sees (bottom-right aligned causal mask, reading R15); negative: it sees no key.
__device__ __forceinline__ int last_visible_key(const FwdParams& p, const Seq& s, int qrow) {
    if (qrow >= s.Lq) return -1;
    long long jl = p.causal ? (long long)qrow + (s.Lk - s.Lq) : (long long)s.Lk - 1;
    if (jl > s.Lk - 1) jl = s.Lk - 1;
    return jl < -1 ? -1 : (int)jl;
}
// TMA coordinates (row, slab) of KV block `blk` of kv head `kvh_in_b` of batch element b (kvslab = b * Hkv + kvh_in_b)
__device__ __forceinline__ void kv_coords(const FwdParams& p, int b, int kvh_in_b, int kvslab, int blk, int bn, int& row,
                                          int& slab) {
    if (p.block_table == nullptr) {
        row = blk * bn;
        slab = kvslab;
    } else {
        const int key0 = blk * bn;
        const int page = p.block_table[(long long)b * p.max_pages + key0 / p.page_size];
        row = key0 % p.page_size;
        slab = page * p.Hkv + kvh_in_b;
    }
}

// ---- sink keys (underflow classification, Prop. 1 / PAPER.md:443) and the block order (Alg. 1 line 2) ----
__device__ __forceinline__ bool sink_in_range(const FwdParams& p, int j0, int n) {     // a sink key in [j0, j0 + n)?
    if (p.n_sinkpos < 0) return j0 < p.n_sink;
    bool any = false;
#pragma unroll 1
    for (int s = 0; s < p.n_sinkpos; ++s) any |= (p.sink_pos[s] >= j0 && p.sink_pos[s] < j0 + n);
    return any;
}
__device__ __forceinline__ bool is_sink_key(const FwdParams& p, int j) { return sink_in_range(p, j, 1); }
// bit e set = key j0 + e is a sink key (e < 32)
__device__ __forceinline__ uint32_t sink_mask32(const FwdParams& p, int j0) {
    if (p.n_sinkpos < 0) {
        const int n = p.n_sink - j0;
        return n <= 0 ? 0u : (n >= 32 ? 0xFFFFFFFFu : ((1u << n) - 1u));
    }
    uint32_t m = 0;
#pragma unroll 1
    for (int s = 0; s < p.n_sinkpos; ++s) {
        const int e = p.sink_pos[s] - j0;
        if (e >= 0 && e < 32) m |= 1u << e;
    }
    return m;
}
// Block visited at step `step` of the block range [b0, b1): forward, reverse, or sink blocks last (the blocks
// without a sink key in descending order, then those with one, in descending order; reading R27).
__device__ __forceinline__ int block_at(const FwdParams& p, int b0, int b1, int step, int bn) {
    if (p.kv_order == 0) return b0 + step;
    if (p.kv_order == 1) return b1 - 1 - step;
    int seen = 0;
    for (int pass = 0; pass < 2; ++pass)
        for (int b = b1 - 1; b >= b0; --b)
            if ((int)sink_in_range(p, b * bn, bn) == pass) {
                if (seen == step) return b;
                ++seen;
            }
    return b0;
}
// Exponent of the dynamic scale of a block: the largest k <= DYN_K_MAX with 2^k * 2^(-g2) <= 448, where
// g2 = (m_new - m_loc) in base-2 units of the scaled logit (>= 0); both in FP32 (reading R26).
__device__ __forceinline__ int dyn_exponent(float g2) {
    const int k = (int)floorf(g2 + LOG2_448);
    return k > DYN_K_MAX ? DYN_K_MAX : k;
}
// o element stores
__device__ __forceinline__ void store_o4(const FwdParams& p, long long idx, float a, float b, float c, float d) {
    if (p.o_bf16) {
        uint2 w = make_uint2(ptx::cvt_bf16x2(a, b), ptx::cvt_bf16x2(c, d));
        *reinterpret_cast<uint2*>(static_cast<uint16_t*>(p.o) + idx) = w;
    } else {
        *reinterpret_cast<float4*>(static_cast<float*>(p.o) + idx) = make_float4(a, b, c, d);
    }
}

}  // namespace fp8attn
