// prep.cuh -- operand staging kernels: FP32 -> three BF16 planes, per-slab E4M3 quantisation.
#pragma once
#include <cuda_bf16.h>
#include "ptx.cuh"

namespace fp8attn {

// x = h + m + l exactly (up to the last FP32 bit), each a BF16: h = rn(x), m = rn(x - h),
// l = rn(x - h - m).  Products of BF16 planes are exact in the tensor core's FP32 accumulator,
// which is how FP32 Q, K, V reach FP32-accurate logits on tcgen05 (hard part 1).
__global__ void split_planes_kernel(const float* __restrict__ x, uint16_t* __restrict__ planes, long long n) {
    const long long stride = (long long)gridDim.x * blockDim.x * 4;
    for (long long i = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * 4; i < n; i += stride) {
        float v[4];
        if (i + 3 < n) {
            const float4 f = *reinterpret_cast<const float4*>(x + i);
            v[0] = f.x; v[1] = f.y; v[2] = f.z; v[3] = f.w;
        } else {
            for (int e = 0; e < 4; ++e) v[e] = (i + e < n) ? x[i + e] : 0.0f;
        }
        uint16_t hh[4], mm[4], ll[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const __nv_bfloat16 h = __float2bfloat16_rn(v[e]);
            const float r1 = v[e] - __bfloat162float(h);
            const __nv_bfloat16 m = __float2bfloat16_rn(r1);
            const float r2 = r1 - __bfloat162float(m);
            const __nv_bfloat16 l = __float2bfloat16_rn(r2);
            hh[e] = __bfloat16_as_ushort(h);
            mm[e] = __bfloat16_as_ushort(m);
            ll[e] = __bfloat16_as_ushort(l);
        }
        if (i + 3 < n) {
            *reinterpret_cast<uint2*>(planes + i) = make_uint2(hh[0] | (hh[1] << 16), hh[2] | (hh[3] << 16));
            *reinterpret_cast<uint2*>(planes + n + i) = make_uint2(mm[0] | (mm[1] << 16), mm[2] | (mm[3] << 16));
            *reinterpret_cast<uint2*>(planes + 2 * n + i) = make_uint2(ll[0] | (ll[1] << 16), ll[2] | (ll[3] << 16));
        } else {
            for (int e = 0; e < 4 && i + e < n; ++e) {
                planes[i + e] = hh[e];
                planes[n + i + e] = mm[e];
                planes[2 * n + i + e] = ll[e];
            }
        }
    }
}

template <typename T>
__device__ __forceinline__ float load_as_f32(const T* p, long long i);
template <>
__device__ __forceinline__ float load_as_f32<float>(const float* p, long long i) { return p[i]; }
template <>
__device__ __forceinline__ float load_as_f32<__nv_bfloat16>(const __nv_bfloat16* p, long long i) {
    return __bfloat162float(p[i]);
}

// amax_bits[slab] = bit pattern of max |x| over the slab (non-negative floats order like uints)
template <typename T>
__global__ void absmax_kernel(const T* __restrict__ x, unsigned int* __restrict__ amax_bits, long long slab_elems) {
    const long long slab = blockIdx.x;            // grid = (slabs, chunks of the slab)
    const T* xs = x + slab * slab_elems;
    float m = 0.0f;
    for (long long i = (long long)blockIdx.y * blockDim.x + threadIdx.x; i < slab_elems;
         i += (long long)gridDim.y * blockDim.x)
        m = fmaxf(m, fabsf(load_as_f32<T>(xs, i)));
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xFFFFFFFFu, m, o));
    if ((threadIdx.x & 31) == 0) atomicMax(amax_bits + slab, __float_as_uint(m));
}

// code = cvt.rn.satfinite.e4m3(x * (448/absmax)); x*inv is one FP32 multiply
template <typename T>
__global__ void quantize_kernel(const T* __restrict__ x, const unsigned int* __restrict__ amax_bits,
                                uint8_t* __restrict__ codes, long long slab_elems) {
    const long long slab = blockIdx.x;
    const float amax = __uint_as_float(amax_bits[slab]);
    const float inv = amax > 0.0f ? __fdiv_rn(448.0f, amax) : 1.0f;
    const T* xs = x + slab * slab_elems;
    uint8_t* cs = codes + slab * slab_elems;
    for (long long i = ((long long)blockIdx.y * blockDim.x + threadIdx.x) * 2; i < slab_elems;
         i += (long long)gridDim.y * blockDim.x * 2) {
        const float a = __fmul_rn(load_as_f32<T>(xs, i), inv);
        const float b = (i + 1 < slab_elems) ? __fmul_rn(load_as_f32<T>(xs, i + 1), inv) : 0.0f;
        const uint32_t pr = ptx::cvt_e4m3x2(a, b);
        cs[i] = (uint8_t)(pr & 0xFF);
        if (i + 1 < slab_elems) cs[i + 1] = (uint8_t)(pr >> 8);
    }
}

// The three steps above in one launch for small slabs (the BF16 q of a decode call: Lq * d elements per slab):
// one warp per slab, same arithmetic in the same order, so codes and scales are bit-identical.
template <typename T>
__global__ void quantize_small_slabs_kernel(const T* __restrict__ x, uint8_t* __restrict__ codes,
                                            float* __restrict__ scale, int slab_elems, int n_slabs) {
    const int slab = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (slab >= n_slabs) return;
    const T* xs = x + (long long)slab * slab_elems;
    uint8_t* cs = codes + (long long)slab * slab_elems;
    float m = 0.0f;
    for (int i = lane; i < slab_elems; i += 32) m = fmaxf(m, fabsf(load_as_f32<T>(xs, i)));
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xFFFFFFFFu, m, o));
    const float inv = m > 0.0f ? __fdiv_rn(448.0f, m) : 1.0f;
    for (int i = lane * 2; i < slab_elems; i += 64) {
        const float a = __fmul_rn(load_as_f32<T>(xs, i), inv);
        const float b = (i + 1 < slab_elems) ? __fmul_rn(load_as_f32<T>(xs, i + 1), inv) : 0.0f;
        const uint32_t pr = ptx::cvt_e4m3x2(a, b);
        cs[i] = (uint8_t)(pr & 0xFF);
        if (i + 1 < slab_elems) cs[i + 1] = (uint8_t)(pr >> 8);
    }
    if (lane == 0) scale[slab] = m > 0.0f ? __fdiv_rn(m, 448.0f) : 1.0f;
}

__global__ void finalize_scale_kernel(const unsigned int* __restrict__ amax_bits, float* __restrict__ scale, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) {
        const float amax = __uint_as_float(amax_bits[i]);
        scale[i] = amax > 0.0f ? __fdiv_rn(amax, 448.0f) : 1.0f;
    }
}

}  // namespace fp8attn
