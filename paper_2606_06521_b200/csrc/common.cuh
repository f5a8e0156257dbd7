// common.cuh -- constants and the kernel parameter block shared by every attention kernel of libfp8attn.so.
#pragma once
#include <cuda_fp16.h>
#include "ptx.cuh"

namespace fp8attn {

constexpr int BM = 128;   // query rows per tile = UMMA M = TMEM lanes
constexpr float LOG2E = 1.4426950408889634f;

struct FwdParams {
    float* o;
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
};

}  // namespace fp8attn
