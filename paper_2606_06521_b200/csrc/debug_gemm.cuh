// debug_gemm.cuh -- one-tile GEMM through the TMA / UMMA-descriptor / TMEM helpers of the attention
// kernels (fp8attn_debug_gemm in include/fp8attn.h).  D[128,N] = A[128,K] . B with
//   A from 128-byte-swizzled shared memory (the Q path) or staged in TMEM (the P path),
//   B K-major [N,K] (the K-tile path) or MN-major [K,N] (the V-tile path).
#pragma once
#include "ptx.cuh"

namespace fp8attn {

template <int EB>
__global__ void __launch_bounds__(128, 1)
debug_gemm_kernel(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapB,
                  const uint8_t* __restrict__ A_gl, float* __restrict__ Dg, int N, int K, int a_in_tmem,
                  int b_mn_major) {
    constexpr int CH = 128 / EB;
    constexpr int KSTEP = 32 / EB;
    constexpr uint32_t KIND = (EB == 1) ? ptx::KIND_F8F6F4 : ptx::KIND_F16;
    constexpr uint32_t FMT = (EB == 1) ? ptx::FMT_E4M3 : ptx::FMT_BF16;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    const int nchK = K / CH;            // 128-byte chunks along K
    const int nchN = N / CH;            // 128-byte chunks along N (MN-major B)
    uint8_t* sA = smem;                                   // nchK x [128 rows x 128 B]
    uint8_t* sB = sA + nchK * 128 * 128;                  // K-major: nchK x [N x 128 B]; MN-major: nchN x [K x 128 B]
    const int b_bytes = b_mn_major ? nchN * K * 128 : nchK * N * 128;
    uint64_t* bars = reinterpret_cast<uint64_t*>(sB + b_bytes);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2);
    const int tid = threadIdx.x, warp = tid >> 5;

    if (tid == 0) {
        ptx::mbar_init(bars + 0, 1);
        ptx::mbar_init(bars + 1, 1);
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
    const uint32_t tlane = tbase + (static_cast<uint32_t>(warp * 32) << 16);
    constexpr int TM_D = 0, TM_A = 256;

    if (tid == 0) {
        ptx::mbar_arrive_expect_tx(bars + 0, nchK * 128 * 128 + b_bytes);
        for (int c = 0; c < nchK; ++c) ptx::tma_load_3d(sA + c * 128 * 128, &mapA, bars + 0, c * CH, 0, 0);
        if (b_mn_major)
            for (int c = 0; c < nchN; ++c) ptx::tma_load_3d(sB + c * K * 128, &mapB, bars + 0, c * CH, 0, 0);
        else
            for (int c = 0; c < nchK; ++c) ptx::tma_load_3d(sB + c * N * 128, &mapB, bars + 0, c * CH, 0, 0);
    }
    if (a_in_tmem) {
        // row tid of A, packed little-endian into 32-bit columns: K*EB/4 columns
        const uint32_t* arow = reinterpret_cast<const uint32_t*>(A_gl + (size_t)tid * K * EB);
        for (int c0 = 0; c0 < K * EB / 4; c0 += 8) {
            uint32_t w[8];
            for (int e = 0; e < 8; ++e) w[e] = arow[c0 + e];
            ptx::tmem_st_x8(tlane + TM_A + c0, w);
        }
        ptx::tmem_wait_st();
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (tid == 0) {
        ptx::tc_fence_after();
        ptx::mbar_wait(bars + 0, 0);
        ptx::tc_fence_after();
        const uint32_t idesc = ptx::make_idesc(FMT, FMT, ptx::MAJOR_K, b_mn_major ? ptx::MAJOR_MN : ptx::MAJOR_K, 128, N);
        for (int ks = 0; ks < K / KSTEP; ++ks) {
            const int c = (ks * 32) / 128, w = (ks * 32) % 128;
            uint64_t db;
            if (b_mn_major)
                db = ptx::make_smem_desc(ptx::smem_u32(sB + ks * KSTEP * 128), K * 128, 1024);
            else
                db = ptx::make_smem_desc(ptx::smem_u32(sB + c * N * 128 + w), 16, 1024);
            if (a_in_tmem) {
                ptx::mma_ts<KIND>(tbase + TM_D, tbase + TM_A + ks * 8, db, idesc, ks > 0);
            } else {
                const uint64_t da = ptx::make_smem_desc(ptx::smem_u32(sA + c * 128 * 128 + w), 16, 1024);
                ptx::mma_ss<KIND>(tbase + TM_D, da, db, idesc, ks > 0);
            }
        }
        ptx::tc_commit(bars + 1);
    }
    __syncwarp();
    ptx::mbar_wait(bars + 1, 0);
    ptx::tc_fence_after();
    for (int cb = 0; cb < N / 32; ++cb) {
        uint32_t v[32];
        ptx::tmem_ld_x32(tlane + TM_D + cb * 32, v);
        ptx::tmem_wait_ld();
        for (int e = 0; e < 32; ++e) Dg[(size_t)tid * N + cb * 32 + e] = __uint_as_float(v[e]);
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 0) ptx::tmem_dealloc(tbase, 512);
}

}  // namespace fp8attn
