// fp8attn.cu -- the C ABI of libfp8attn.so (include/fp8attn.h): argument checks, tensor maps,
// library-owned scratch memory, kernel selection and launch.  No step of the method runs on
// the host and there is no CPU fallback: without a compute-capability-10 device every entry
// point that computes returns FP8ATTN_E_DEVICE.
#include <cmath>
#include <cstdarg>
#include <cstdlib>
#include <cstring>
#include <mutex>

#include "../../include/fp8attn.h"
#include <atomic>

#include "attn_general.cuh"
#include "attn_prefill.cuh"
#include "attn_prefill64.cuh"
#include "attn_decode.cuh"
#include "debug_gemm.cuh"
#include "prep.cuh"

namespace {

using namespace fp8attn;

thread_local char g_err[512] = "";

void set_err(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
}

#define CU_TRY(expr)                                                                              \
    do {                                                                                          \
        cudaError_t e__ = (expr);                                                                 \
        if (e__ != cudaSuccess) {                                                                 \
            set_err("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__), __FILE__, __LINE__); \
            return FP8ATTN_E_CUDA;                                                                \
        }                                                                                         \
    } while (0)

// ---------------------------------------------------------------------------- device check
int check_device() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        cudaGetLastError();
        set_err("no CUDA device");
        return FP8ATTN_E_DEVICE;
    }
    static std::mutex mu;
    static int cached_dev = -1, cached_rc = 0;
    std::lock_guard<std::mutex> lock(mu);
    static int cached_major = 0;
    if (dev == cached_dev) {
        // (the message is per thread: write it again for a caller that did not make the first query)
        if (cached_rc) set_err("device %d has compute capability %d.x; sm_100 is required", dev, cached_major);
        return cached_rc;
    }
    int major = 0;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) {
        cudaGetLastError();
        set_err("cannot query the device");
        return FP8ATTN_E_DEVICE;
    }
    cached_dev = dev;
    cached_major = major;
    cached_rc = (major == 10) ? FP8ATTN_OK : FP8ATTN_E_DEVICE;
    if (cached_rc) set_err("device %d has compute capability %d.x; sm_100 is required", dev, major);
    return cached_rc;
}

// ---------------------------------------------------------------------------- tensor maps
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = [] {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess) p = nullptr;
        return reinterpret_cast<EncodeTiledFn>(p);
    }();
    return fn;
}

// [slabs, rows, cols] row-major, element size eb; box = one 128-byte chunk of `box_rows` rows, 128-byte swizzle.
// Rows past `rows` read as zero.
int make_map(CUtensorMap* m, const void* base, int eb, long long slabs, long long rows, int cols, int box_rows) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) {
        set_err("cuTensorMapEncodeTiled not available from the driver");
        return FP8ATTN_E_CUDA;
    }
    const cuuint64_t gdim[3] = {(cuuint64_t)cols, (cuuint64_t)rows, (cuuint64_t)slabs};
    const cuuint64_t gstr[2] = {(cuuint64_t)cols * eb, (cuuint64_t)cols * eb * (cuuint64_t)rows};
    const cuuint32_t box[3] = {(cuuint32_t)(128 / eb), (cuuint32_t)box_rows, 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    const CUtensorMapDataType dt = (eb == 4)   ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32
                                   : (eb == 2) ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16
                                               : CU_TENSOR_MAP_DATA_TYPE_UINT8;
    CUresult r = fn(m, dt, 3, const_cast<void*>(base), gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                    CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        set_err("cuTensorMapEncodeTiled failed with CUresult %d (base %p eb %d slabs %lld rows %lld cols %d box %d)",
                (int)r, base, eb, slabs, rows, cols, box_rows);
        return FP8ATTN_E_CUDA;
    }
    return FP8ATTN_OK;
}

// ---------------------------------------------------------------------------- per-device state, scratch memory
// Scratch (split-KV partials, BF16 planes of FP32 inputs, the quantised q of a decode call, the staging of
// fp8attn_fwd_host) is allocated PER CALL from a library-owned stream-ordered memory pool of the current device,
// on the caller's stream, and freed on that stream once the call's kernels are enqueued.  Two calls therefore
// never share scratch, whatever streams or devices they run on, and nothing is freed while a kernel that uses it
// is pending.  The pool keeps freed memory (release threshold = max), so steady-state calls do not reach the OS.
constexpr int MAX_DEVICES = 64;
struct DeviceState {
    std::mutex mu;           // guards `pool`
    cudaMemPool_t pool = nullptr;
    // fp8attn_fwd_host: two copy streams and the events that chain the pieces; host calls on one device take
    // turns (host_mu), each synchronises its stream before it returns anyway
    std::mutex host_mu;
    cudaStream_t s_in = nullptr, s_out = nullptr;
    cudaEvent_t ev_start = nullptr, ev_in[8] = {}, ev_done[8] = {};
};
DeviceState g_dev[MAX_DEVICES];

int current_device(int* dev) {
    if (cudaGetDevice(dev) != cudaSuccess || *dev < 0 || *dev >= MAX_DEVICES) {
        cudaGetLastError();
        set_err("no usable CUDA device");
        return FP8ATTN_E_DEVICE;
    }
    return FP8ATTN_OK;
}

int device_pool(cudaMemPool_t* out) {
    int dev = 0;
    if (int rc = current_device(&dev)) return rc;
    DeviceState& d = g_dev[dev];
    std::lock_guard<std::mutex> lock(d.mu);
    if (!d.pool) {
        cudaMemPoolProps props;
        memset(&props, 0, sizeof props);
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        CU_TRY(cudaMemPoolCreate(&d.pool, &props));
        unsigned long long keep = ~0ull;
        CU_TRY(cudaMemPoolSetAttribute(d.pool, cudaMemPoolAttrReleaseThreshold, &keep));
    }
    *out = d.pool;
    return FP8ATTN_OK;
}

// One allocation, returned to the pool on `st` when the lease goes out of scope.
struct Lease {
    void* ptr = nullptr;
    cudaStream_t st = nullptr;
    Lease() = default;
    Lease(const Lease&) = delete;
    Lease& operator=(const Lease&) = delete;
    ~Lease() {
        if (ptr) cudaFreeAsync(ptr, st);
    }
    int get(size_t bytes, cudaStream_t stream) {
        cudaMemPool_t pool;
        if (int rc = device_pool(&pool)) return rc;
        st = stream;
        CU_TRY(cudaMallocFromPoolAsync(&ptr, bytes < 256 ? 256 : bytes, pool, stream));
        return FP8ATTN_OK;
    }
};

// Opt a kernel in to more than 48 KB of dynamic shared memory: the attribute is per device, `done` holds one
// bit per device (one static mask per kernel instance).
template <typename K>
int ensure_smem(K kern, int bytes, std::atomic<unsigned long long>& done) {
    int dev = 0;
    if (int rc = current_device(&dev)) return rc;
    const unsigned long long bit = 1ull << dev;
    if (!(done.load(std::memory_order_acquire) & bit)) {
        CU_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
        done.fetch_or(bit, std::memory_order_release);
    }
    return FP8ATTN_OK;
}

// ---------------------------------------------------------------------------- general kernel launch
template <int D, int BN, int EB, int NPL, int MODE>
int launch_general(const CUtensorMap& mq, const CUtensorMap& mk, const CUtensorMap& mv, const FwdParams& p,
                   dim3 grid, cudaStream_t st) {
    using C = GeneralCfg<D, BN, EB, NPL, MODE>;
    auto kern = attn_general_kernel<D, BN, EB, NPL, MODE>;
    static std::atomic<unsigned long long> done{0};
    if (int rc = ensure_smem(kern, C::SMEM_BYTES, done)) return rc;
    kern<<<grid, 128, C::SMEM_BYTES, st>>>(mq, mk, mv, p);
    CU_TRY(cudaGetLastError());
    return FP8ATTN_OK;
}

template <int EB, int NPL, int MODE>
int dispatch_general(int d, int bn, const CUtensorMap& mq, const CUtensorMap& mk, const CUtensorMap& mv,
                     const FwdParams& p, dim3 grid, cudaStream_t st) {
    if constexpr (NPL == 3) {   // FP32 inputs: Bn = 64 only (three planes of Q, K, V must fit in shared memory)
        if (d == 64 && bn == 64) return launch_general<64, 64, EB, NPL, MODE>(mq, mk, mv, p, grid, st);
        if (d == 128 && bn == 64) return launch_general<128, 64, EB, NPL, MODE>(mq, mk, mv, p, grid, st);
    } else if constexpr (EB == 1) {   // E4M3: d = 128 only (a 64-byte operand row does not fill a 128-byte swizzle row)
        if (d == 128 && bn == 64) return launch_general<128, 64, EB, NPL, MODE>(mq, mk, mv, p, grid, st);
        if (d == 128 && bn == 128) return launch_general<128, 128, EB, NPL, MODE>(mq, mk, mv, p, grid, st);
    } else {
        if (d == 64 && bn == 64) return launch_general<64, 64, EB, NPL, MODE>(mq, mk, mv, p, grid, st);
        if (d == 64 && bn == 128) return launch_general<64, 128, EB, NPL, MODE>(mq, mk, mv, p, grid, st);
        if (d == 128 && bn == 64) return launch_general<128, 64, EB, NPL, MODE>(mq, mk, mv, p, grid, st);
        if (d == 128 && bn == 128) return launch_general<128, 128, EB, NPL, MODE>(mq, mk, mv, p, grid, st);
    }
    set_err("no kernel instance for d=%d block_n=%d", d, bn);
    return FP8ATTN_E_UNSUPPORTED;
}

// ---------------------------------------------------------------------------- prefill kernel launch (Bn = 128)
template <int EB, bool FOLD>
int launch_prefill(const CUtensorMap& mq, const CUtensorMap& mk, const CUtensorMap& mv, const FwdParams& p,
                   cudaStream_t st) {
    using C = PrefillKCfg<EB>;
    // the statistics instance (P dump, underflow counters of fp8attn_stats) has the same schedule; the plain
    // instance carries none of that code
    const bool aux = p.p_codes || p.underflow;
    // o as [B*Hq, Lq, d]: boxes of 32 rows x 128 bytes (32 floats / 64 bfloat16), stored by TMA from the epilogue
    CUtensorMap mo;
    if (int rc = make_map(&mo, p.o, p.o_bf16 ? 2 : 4, (long long)p.B * p.Hq, p.Lq, 128, 32)) return rc;
    const dim3 grid((unsigned)(((p.Lq + 2 * BM - 1) / (2 * BM)) * (p.B * p.Hq)));
    // the extensions (dynamic scale, variable-length sequences, paged KV) live in their own instance, like the
    // statistics: the plain instance is the headline path and carries no code it does not need
    const bool ext = p.scale_mode == 1 || p.seqlens_q || p.seqlens_k || p.block_table;
    if (aux && ext) {
        auto kern = attn_prefill_kernel<EB, FOLD, true, true>;
        static std::atomic<unsigned long long> done{0};
        if (int rc = ensure_smem(kern, C::SMEM_BYTES, done)) return rc;
        kern<<<grid, C::THREADS, C::SMEM_BYTES, st>>>(mq, mk, mv, mo, p);
    } else if (aux) {
        auto kern = attn_prefill_kernel<EB, FOLD, true, false>;
        static std::atomic<unsigned long long> done{0};
        if (int rc = ensure_smem(kern, C::SMEM_BYTES, done)) return rc;
        kern<<<grid, C::THREADS, C::SMEM_BYTES, st>>>(mq, mk, mv, mo, p);
    } else if (ext) {
        auto kern = attn_prefill_kernel<EB, FOLD, false, true>;
        static std::atomic<unsigned long long> done{0};
        if (int rc = ensure_smem(kern, C::SMEM_BYTES, done)) return rc;
        kern<<<grid, C::THREADS, C::SMEM_BYTES, st>>>(mq, mk, mv, mo, p);
    } else {
        auto kern = attn_prefill_kernel<EB, FOLD, false, false>;
        static std::atomic<unsigned long long> done{0};
        if (int rc = ensure_smem(kern, C::SMEM_BYTES, done)) return rc;
        kern<<<grid, C::THREADS, C::SMEM_BYTES, st>>>(mq, mk, mv, mo, p);
    }
    CU_TRY(cudaGetLastError());
    return FP8ATTN_OK;
}

// ---------------------------------------------------------------------------- Bn = 64 prefill kernel launch
template <int EB, bool FOLD>
int launch_prefill64(const CUtensorMap& mq, const CUtensorMap& mk, const CUtensorMap& mv, const FwdParams& p,
                     cudaStream_t st) {
    using C = Prefill64Cfg<EB>;
    const bool aux = p.p_codes || p.underflow;
    const dim3 grid((unsigned)(((p.Lq + 2 * BM - 1) / (2 * BM)) * (p.B * p.Hq)));
    if (aux) {
        auto kern = attn_prefill64_kernel<EB, FOLD, true>;
        static std::atomic<unsigned long long> done{0};
        if (int rc = ensure_smem(kern, C::SMEM_BYTES, done)) return rc;
        kern<<<grid, C::THREADS, C::SMEM_BYTES, st>>>(mq, mk, mv, p);
    } else {
        auto kern = attn_prefill64_kernel<EB, FOLD, false>;
        static std::atomic<unsigned long long> done{0};
        if (int rc = ensure_smem(kern, C::SMEM_BYTES, done)) return rc;
        kern<<<grid, C::THREADS, C::SMEM_BYTES, st>>>(mq, mk, mv, p);
    }
    CU_TRY(cudaGetLastError());
    return FP8ATTN_OK;
}

// ---------------------------------------------------------------------------- decode kernel launch
template <int NVT, bool FOLD, bool AUX>
int launch_decode_t(const CUtensorMap& mq, const CUtensorMap& mk, const CUtensorMap& mv, const FwdParams& p,
                    cudaStream_t st) {
    auto kern = attn_decode_kernel<NVT, FOLD, AUX>;
    static std::atomic<unsigned long long> done{0};
    if (int rc = ensure_smem(kern, DecodeCfg::SMEM_BYTES, done)) return rc;
    const dim3 grid((unsigned)(p.B * p.Hkv), (unsigned)p.num_splits);
    kern<<<grid, DecodeCfg::THREADS, DecodeCfg::SMEM_BYTES, st>>>(mq, mk, mv, p);
    CU_TRY(cudaGetLastError());
    return FP8ATTN_OK;
}
template <bool FOLD>
int launch_decode(int nv, const CUtensorMap& mq, const CUtensorMap& mk, const CUtensorMap& mv, const FwdParams& p,
                  cudaStream_t st) {
    // the statistics instance (P dump, underflow counters) has the same schedule; the plain one carries no such code
    if (p.p_codes || p.underflow) {
        if (nv <= 4) return launch_decode_t<4, FOLD, true>(mq, mk, mv, p, st);
        if (nv <= 8) return launch_decode_t<8, FOLD, true>(mq, mk, mv, p, st);
        return launch_decode_t<16, FOLD, true>(mq, mk, mv, p, st);
    }
    if (nv <= 4) return launch_decode_t<4, FOLD, false>(mq, mk, mv, p, st);
    if (nv <= 8) return launch_decode_t<8, FOLD, false>(mq, mk, mv, p, st);
    return launch_decode_t<16, FOLD, false>(mq, mk, mv, p, st);
}
// Number of KV splits for the decode kernel: enough CTAs to fill 2 x 148 resident slots several times over,
// with a last wave that is nearly full.
int decode_auto_splits(long long kv_slabs, int nb) {
    const long long slots = 2 * 148;
    int best = 1;
    for (int ns = 1; ns <= 16 && ns <= nb; ++ns) {
        const long long ctas = kv_slabs * ns;
        const long long waves = (ctas + slots - 1) / slots;
        best = ns;
        if (ctas >= 4 * slots && (double)ctas / (double)(waves * slots) >= 0.95) break;
        if (nb / ns < 8) break;      // keep at least 8 blocks per split
    }
    return best;
}

// S = 2^k with a comfortable exponent: the factor can be folded into the exponent of P exactly
bool is_pow2_scale(float S) {
    int e = 0;
    return std::frexp(S, &e) == 0.5f && e > -20 && e < 20;
}

// Argument checks shared by fp8attn_fwd and fp8attn_fwd_host: no CUDA call before these pass.
int validate_args(const void* q, const void* k, const void* v, const void* o, int B, int Hq, int Hkv, int Lq, int Lk,
                  int d, float S, int kv_order, int mode, const fp8attn_stats* stats) {
    if (!q || !k || !v || !o) return FP8ATTN_E_NULL;
    if (B < 1 || Hq < 1 || Hkv < 1 || Lq < 1 || Lk < 1) return FP8ATTN_E_SHAPE;
    if (Hq % Hkv != 0 || (d != 64 && d != 128)) return FP8ATTN_E_SHAPE;
    if (!(S > 0.0f) || !std::isfinite(S)) return FP8ATTN_E_SCALE;
    const int pm = mode & 0xFF, dt = (mode >> 8) & 0xF;
    if ((mode & ~0xFFF) || pm > 2 || dt > 3) return FP8ATTN_E_MODE;
    if (kv_order < FP8ATTN_ORDER_FORWARD || kv_order > FP8ATTN_ORDER_SINK_LAST) return FP8ATTN_E_MODE;
    const bool e4m3_kv = (dt == 2 || dt == 3);
    if ((pm == FP8ATTN_MODE_FP8) != e4m3_kv) return FP8ATTN_E_MODE;
    if (stats && stats->struct_size != (int32_t)sizeof(fp8attn_stats)) return FP8ATTN_E_STATS;
    if (e4m3_kv) {
        if (!stats || !stats->k_scale || !stats->v_scale) return FP8ATTN_E_NULL;
        if (dt == 2 && !stats->q_scale) return FP8ATTN_E_NULL;
        if (d != 128) return FP8ATTN_E_UNSUPPORTED;
    }
    const int bn = stats ? stats->block_n : 0;
    if (bn != 0 && bn != 64 && bn != 128) return FP8ATTN_E_UNSUPPORTED;
    if (dt == 0 && bn == 128) return FP8ATTN_E_UNSUPPORTED;
    const int ns = stats ? stats->num_splits : 0;
    if (ns < 0 || ns > FP8ATTN_MAX_SPLITS) return FP8ATTN_E_UNSUPPORTED;
    if (stats && (stats->kernel < 0 || stats->kernel > 3 || stats->reserved1 != 0)) return FP8ATTN_E_MODE;
    if (stats && (stats->scale_mode < 0 || stats->scale_mode > 1 || stats->o_dtype < 0 || stats->o_dtype > 1)) return FP8ATTN_E_MODE;
    if (stats && stats->scale_mode == FP8ATTN_SCALE_DYNAMIC && pm == FP8ATTN_MODE_NOCAST) return FP8ATTN_E_MODE;
    if (stats && stats->reserved2 != 0) return FP8ATTN_E_MODE;
    if (stats && stats->block_table) {
        if (stats->page_size < 1 || stats->max_pages < 1 || stats->num_pages < 1) return FP8ATTN_E_SHAPE;
        if ((long long)stats->max_pages * stats->page_size < Lk) return FP8ATTN_E_SHAPE;
        if (dt == 0) return FP8ATTN_E_UNSUPPORTED;            // FP32 planes of a page pool: not built
    }
    if (stats && stats->n_sink < 0) return FP8ATTN_E_SHAPE;
    if (stats && stats->sink_pos) {
        if (stats->n_sink < 1 || stats->n_sink > FP8ATTN_MAX_SINKS) return FP8ATTN_E_SHAPE;
        for (int i = 0; i < stats->n_sink; ++i)
            if (stats->sink_pos[i] < 0 || stats->sink_pos[i] >= Lk || (i > 0 && stats->sink_pos[i] <= stats->sink_pos[i - 1]))
                return FP8ATTN_E_SHAPE;
    }
    if (stats && stats->p_codes && (stats->p_batch < 0 || stats->p_batch >= B || stats->p_head < 0 || stats->p_head >= Hq))
        return FP8ATTN_E_SHAPE;
    if ((long long)B * Hq * ((Lq + 127) / 128) > 0x7FFFFFFFll) return FP8ATTN_E_UNSUPPORTED;
    return FP8ATTN_OK;
}

}  // namespace

// ---------------------------------------------------------------------------- static scratch (fp8attn_decode_noalloc)
// The scratch of the entry point that allocates nothing.  In HOST code this name is a host-side stand-in, not a
// device address: the address a kernel can use comes from cudaGetSymbolAddress, asked once per device with that
// device current (every device that loads the library has its own copy of the array).
static __device__ __align__(256) unsigned char g_noalloc_scratch[FP8ATTN_NOALLOC_SCRATCH_BYTES];

namespace {

int noalloc_scratch_ptr(unsigned char** out) {
    static std::mutex mu;
    static unsigned char* ptrs[MAX_DEVICES] = {};
    int dev = 0;
    if (int rc = current_device(&dev)) return rc;
    std::lock_guard<std::mutex> lock(mu);
    if (!ptrs[dev]) {
        void* ptr = nullptr;
        CU_TRY(cudaGetSymbolAddress(&ptr, g_noalloc_scratch));
        if (!ptr || (reinterpret_cast<uintptr_t>(ptr) & 255u)) {
            set_err("cudaGetSymbolAddress gave %p for the static scratch of device %d", ptr, dev);
            return FP8ATTN_E_CUDA;
        }
        ptrs[dev] = static_cast<unsigned char*>(ptr);
    }
    *out = ptrs[dev];
    return FP8ATTN_OK;
}

}  // namespace

// =============================================================================================
// C ABI
// =============================================================================================
extern "C" {

int fp8attn_version(void) { return 201; }   // 0.2.1

int fp8attn_trim(void) {
    int dev = 0;
    if (int rc = current_device(&dev)) return rc;
    DeviceState& d = g_dev[dev];
    std::lock_guard<std::mutex> lock(d.mu);
    if (d.pool) CU_TRY(cudaMemPoolTrimTo(d.pool, 0));
    return FP8ATTN_OK;
}

const char* fp8attn_last_cuda_error(void) { return g_err; }

const char* fp8attn_strerror(int code) {
    switch (code) {
        case FP8ATTN_OK: return "success";
        case FP8ATTN_E_NULL: return "a required pointer is NULL";
        case FP8ATTN_E_SHAPE: return "bad shape: sizes must be >= 1, Hq % Hkv == 0, d in {64, 128}";
        case FP8ATTN_E_SCALE: return "S must be a finite float > 0";
        case FP8ATTN_E_MODE: return "unknown or inconsistent mode / dtype / kv_order";
        case FP8ATTN_E_UNSUPPORTED: return "valid request that this build does not support";
        case FP8ATTN_E_DEVICE: return "the current device is not compute capability 10.x";
        case FP8ATTN_E_CUDA: return "a CUDA call failed (see fp8attn_last_cuda_error)";
        case FP8ATTN_E_STATS: return "stats->struct_size does not match this header";
        case FP8ATTN_E_SCRATCH: return "the call needs more scratch than the static array of fp8attn_decode_noalloc holds";
        default: return "unknown error code";
    }
}

int fp8attn_fwd(const void* q, const void* k, const void* v, void* o, int B, int Hq, int Hkv, int Lq, int Lk, int d,
                int causal, float S, int kv_order, int mode, fp8attn_stats* stats) {
    if (int rc = validate_args(q, k, v, o, B, Hq, Hkv, Lq, Lk, d, S, kv_order, mode, stats)) return rc;
    const int pm = mode & 0xFF, dt = (mode >> 8) & 0xF;
    int bn = stats ? stats->block_n : 0;
    if (bn == 0) bn = (dt == 0) ? 64 : 128;
    int ns = stats ? stats->num_splits : 0;
    const long long q_slabs = (long long)B * Hq, kv_slabs = (long long)B * Hkv;
    if (int rc = check_device()) return rc;

    cudaStream_t st = stats ? reinterpret_cast<cudaStream_t>(stats->stream) : nullptr;
    const int nb = (Lk + bn - 1) / bn;
    const int n_qtiles = (Lq + BM - 1) / BM;
    const int want_kernel = stats ? stats->kernel : 0;
    const bool want_aux = stats && (stats->p_codes || stats->underflow);
    // decode shape: a handful of query rows per kv head against an E4M3 KV cache
    const bool decode_ok = pm == 2 && d == 128 && bn == 128 && (long long)(Hq / Hkv) * Lq <= 16;
    if (want_kernel == 3 && !decode_ok) return FP8ATTN_E_UNSUPPORTED;
    const bool use_decode = decode_ok && (want_kernel == 3 || want_kernel == 0);
    if (ns == 0 && use_decode) ns = decode_auto_splits(kv_slabs, nb);
    if (ns == 0) {
        // automatic: split only decode-shaped calls (a handful of query rows per head) whose query
        // tiles alone cannot fill the GPU.  Splitting changes which P values are cast against the
        // sink's running max (reading R14), so prefill is never split behind the caller's back.
        const long long tiles = (long long)n_qtiles * q_slabs;
        ns = 1;
        if (Lq <= 16 && tiles < 2 * 148 && nb > 1) {
            long long want = (4 * 148 + tiles - 1) / tiles;
            ns = (int)(want < nb ? want : nb);
            if (ns > FP8ATTN_MAX_SPLITS) ns = FP8ATTN_MAX_SPLITS;
        }
    }
    if (ns > nb) ns = nb;

    const long long nq = q_slabs * Lq * d, nkv = kv_slabs * Lk * d;
    const void *qs = q, *ks = k, *vs = v;   // staged operands the kernel reads
    const float* q_scale = stats ? stats->q_scale : nullptr;
    int n_launches = 0;
    int eb = 2, npl = 1;
    Lease planes, qquant, amax_buf, partial;     // per-call scratch, returned to the pool on `st` at return
    if (dt == 0) {
        // FP32 -> three BF16 planes each (exact split), so that tcgen05 reproduces FP32 logits
        if (int rc = planes.get((size_t)(nq + 2 * nkv) * 3 * 2, st)) return rc;
        uint16_t* pq = static_cast<uint16_t*>(planes.ptr);
        uint16_t* pk = pq + 3 * nq;
        uint16_t* pv = pk + 3 * nkv;
        const int thr = 256;
        auto blocks = [&](long long n) { long long b = (n / 4 + thr - 1) / thr; return (unsigned)(b < 1 ? 1 : (b > 148 * 16 ? 148 * 16 : b)); };
        split_planes_kernel<<<blocks(nq), thr, 0, st>>>(static_cast<const float*>(q), pq, nq);
        split_planes_kernel<<<blocks(nkv), thr, 0, st>>>(static_cast<const float*>(k), pk, nkv);
        split_planes_kernel<<<blocks(nkv), thr, 0, st>>>(static_cast<const float*>(v), pv, nkv);
        CU_TRY(cudaGetLastError());
        n_launches += 3;
        qs = pq; ks = pk; vs = pv;
        npl = 3;
    } else if (dt == 2) {
        eb = 1;
    } else if (dt == 3) {
        // decode: quantise the BF16 q of every (b, hq) slab to E4M3 (reading R24 in DESIGN.md)
        eb = 1;
        if (int rc = qquant.get((size_t)nq + (size_t)q_slabs * 4 + 16, st)) return rc;
        uint8_t* codes = static_cast<uint8_t*>(qquant.ptr);
        float* qsc = reinterpret_cast<float*>(codes + ((nq + 15) / 16) * 16);
        const long long slab = (long long)Lq * d;
        if (slab <= 4096) {
            // a decode-sized q: one warp per slab does absmax, codes and scale in one launch
            quantize_small_slabs_kernel<__nv_bfloat16><<<(unsigned)((q_slabs + 3) / 4), 128, 0, st>>>(
                static_cast<const __nv_bfloat16*>(q), codes, qsc, (int)slab, (int)q_slabs);
            CU_TRY(cudaGetLastError());
            n_launches += 1;
        } else {
            if (int rc = amax_buf.get((size_t)q_slabs * 4, st)) return rc;
            unsigned int* amax = static_cast<unsigned int*>(amax_buf.ptr);
            CU_TRY(cudaMemsetAsync(amax, 0, (size_t)q_slabs * 4, st));
            unsigned gy = (unsigned)((slab + 255) / 256);
            if (gy > 64) gy = 64;
            absmax_kernel<__nv_bfloat16><<<dim3((unsigned)q_slabs, gy), 256, 0, st>>>(static_cast<const __nv_bfloat16*>(q), amax, slab);
            quantize_kernel<__nv_bfloat16><<<dim3((unsigned)q_slabs, gy), 256, 0, st>>>(static_cast<const __nv_bfloat16*>(q), amax, codes, slab);
            finalize_scale_kernel<<<(unsigned)((q_slabs + 255) / 256), 256, 0, st>>>(amax, qsc, (int)q_slabs);
            CU_TRY(cudaGetLastError());
            n_launches += 3;
        }
        qs = codes;
        q_scale = qsc;
    }

    const bool paged = stats && stats->block_table;
    if (paged && stats->page_size % bn != 0) return FP8ATTN_E_UNSUPPORTED;    // a KV block must not straddle pages
    CUtensorMap mq, mk, mv;
    if (int rc = make_map(&mq, qs, eb, npl * q_slabs, Lq, d, BM)) return rc;
    if (paged) {       // k, v are page pools [num_pages, Hkv, page_size, d]: slab = page * Hkv + kv head
        if (int rc = make_map(&mk, ks, eb, (long long)stats->num_pages * Hkv, stats->page_size, d, bn)) return rc;
        if (int rc = make_map(&mv, vs, eb, (long long)stats->num_pages * Hkv, stats->page_size, d, bn)) return rc;
    } else {
        if (int rc = make_map(&mk, ks, eb, npl * kv_slabs, Lk, d, bn)) return rc;
        if (int rc = make_map(&mv, vs, eb, npl * kv_slabs, Lk, d, bn)) return rc;
    }

    FwdParams p;
    memset(&p, 0, sizeof p);
    p.o = o;
    p.row_max = stats ? stats->row_max : nullptr;
    p.row_sum = stats ? stats->row_sum : nullptr;
    p.underflow = stats ? stats->underflow : nullptr;
    p.p_codes = stats ? stats->p_codes : nullptr;
    p.p_bh = stats ? stats->p_batch * Hq + stats->p_head : 0;
    p.q_scale = q_scale;
    p.k_scale = stats ? stats->k_scale : nullptr;
    p.v_scale = stats ? stats->v_scale : nullptr;
    p.B = B; p.Hq = Hq; p.Hkv = Hkv; p.Lq = Lq; p.Lk = Lk;
    p.causal = causal ? 1 : 0;
    p.kv_order = kv_order;
    p.n_sink = stats ? stats->n_sink : 0;
    p.scale_mode = stats ? stats->scale_mode : 0;
    p.o_bf16 = (stats && stats->o_dtype == FP8ATTN_O_BF16) ? 1 : 0;
    p.n_sinkpos = -1;
    if (stats && stats->sink_pos) {
        p.n_sinkpos = stats->n_sink;
        for (int i = 0; i < stats->n_sink; ++i) p.sink_pos[i] = stats->sink_pos[i];
    }
    const bool dynamic = p.scale_mode == 1;
    p.seqlens_q = stats ? stats->seqlens_q : nullptr;
    p.seqlens_k = stats ? stats->seqlens_k : nullptr;
    p.block_table = paged ? stats->block_table : nullptr;
    p.page_size = paged ? stats->page_size : 0;
    p.max_pages = paged ? stats->max_pages : 0;
    p.num_splits = ns;
    p.nb = nb;
    p.q_slabs = (int)q_slabs;
    p.kv_slabs = (int)kv_slabs;
    p.S = S;
    p.sm_scale = 1.0f / sqrtf((float)d);
    const long long R = q_slabs * Lq;
    if (ns > 1) {
        if (int rc = partial.get((size_t)ns * R * (d + 2) * 4, st)) return rc;
        p.part_o = static_cast<float*>(partial.ptr);
        p.part_ml = p.part_o + (size_t)ns * R * d;
    }
    if (pm == 0) p.p_codes = nullptr;          // the no-cast mode has no codes (and counts nothing)
    if (p.underflow) CU_TRY(cudaMemsetAsync(p.underflow, 0, 2 * sizeof(unsigned long long), st));
    // masked positions of the P dump (and the blocks a causal tile skips) read 0xFF
    if (p.p_codes) CU_TRY(cudaMemsetAsync(p.p_codes, 0xFF, (size_t)Lq * Lk, st));

    // kernel family.  The warp-specialised prefill kernels serve d = 128, one split, BF16 or E4M3 operands,
    // modes 1 and 2 (Bn = 128 and Bn = 64); the decode kernel serves decode shapes with any split count; each
    // has a statistics instance (same schedule + P dump + underflow counters).  Everything else -- FP32
    // inputs, the no-cast mode, d = 64, prefill with splits -- runs on the general kernel.
    // (not built into the prefill kernels: the sink-blocks-last order)
    const bool prefill_ok = d == 128 && ns == 1 && npl == 1 && pm != 0 && dt != 3 && kv_order != FP8ATTN_ORDER_SINK_LAST;
    if (want_kernel == 2 && !prefill_ok) return FP8ATTN_E_UNSUPPORTED;
    // (automatic selection keeps prefill-shaped calls that ask for the P dump or the underflow counters on the
    // general kernel, whose serial schedule is the reference for them; stats->kernel = 2 takes the statistics
    // instance of the throughput kernel)
    const bool use_prefill = !use_decode && prefill_ok && (want_kernel == 2 || (want_kernel == 0 && Lq > 16 && !want_aux));
    int kernel_id = 1;
    int rc;
    if (use_decode) {
        kernel_id = 3;
        // the G*Lq query rows of one kv head are consecutive rows of q: one 16-row box per CTA
        CUtensorMap mq16;
        if (int rc2 = make_map(&mq16, qs, 1, 1, q_slabs * Lq, d, 16)) return rc2;
        const int nv = (Hq / Hkv) * Lq;
        rc = (is_pow2_scale(S) || dynamic) ? launch_decode<true>(nv, mq16, mk, mv, p, st)
                                           : launch_decode<false>(nv, mq16, mk, mv, p, st);
    } else if (use_prefill) {
        kernel_id = 2;
        const bool fold = is_pow2_scale(S) || dynamic;      // the dynamic 2^k goes through the folded-scale instance
        if (bn == 64) {
            if (eb == 1) rc = fold ? launch_prefill64<1, true>(mq, mk, mv, p, st) : launch_prefill64<1, false>(mq, mk, mv, p, st);
            else rc = fold ? launch_prefill64<2, true>(mq, mk, mv, p, st) : launch_prefill64<2, false>(mq, mk, mv, p, st);
        } else if (eb == 1) rc = fold ? launch_prefill<1, true>(mq, mk, mv, p, st) : launch_prefill<1, false>(mq, mk, mv, p, st);
        else rc = fold ? launch_prefill<2, true>(mq, mk, mv, p, st) : launch_prefill<2, false>(mq, mk, mv, p, st);
    } else {
        const dim3 grid((unsigned)(n_qtiles * q_slabs), 1u, (unsigned)ns);
        if (npl == 3)
            rc = (pm == 0) ? dispatch_general<2, 3, 0>(d, bn, mq, mk, mv, p, grid, st)
                           : dispatch_general<2, 3, 1>(d, bn, mq, mk, mv, p, grid, st);
        else if (eb == 2)
            rc = (pm == 0) ? dispatch_general<2, 1, 0>(d, bn, mq, mk, mv, p, grid, st)
                           : dispatch_general<2, 1, 1>(d, bn, mq, mk, mv, p, grid, st);
        else
            rc = dispatch_general<1, 1, 2>(d, bn, mq, mk, mv, p, grid, st);
    }
    if (rc) return rc;
    ++n_launches;
    if (ns > 1) {
        const int rows_per_block = 8;
        combine_kernel<<<(unsigned)((R + rows_per_block - 1) / rows_per_block), rows_per_block * 32, 0, st>>>(
            p.part_o, p.part_ml, p.o, p.row_max, p.row_sum, (pm == 2) ? p.v_scale : nullptr, R, d, ns,
            (pm == 0 || dynamic) ? 1.0f : S, Hq, Hkv, Lq, p.o_bf16);
        CU_TRY(cudaGetLastError());
        ++n_launches;
    }
    if (stats) {
        stats->block_m_used = (kernel_id == 2) ? 2 * BM : BM;
        stats->block_n_used = bn;
        stats->num_splits_used = ns;
        for (int s = 0; s <= ns; ++s) stats->split_bounds[s] = (int)(((long long)s * nb) / ns);
        stats->kernel_id = kernel_id;
        stats->n_launches = n_launches;
    }
    return FP8ATTN_OK;
}

// The decode path of fp8attn_fwd (q quantiser, split-KV decode kernel, combine) with its scratch in the static
// array above: no cudaMalloc, no cudaFree, no pool (include/fp8attn.h).  Same kernels, same launch configuration
// and the same split layout as fp8attn_fwd, so the results are the same bit for bit.
int fp8attn_decode_noalloc(const void* q, const void* k, const void* v, void* o, int B, int Hq, int Hkv, int Lq, int Lk,
                           int d, int causal, float S, int kv_order, int mode, fp8attn_stats* stats) {
    if (int rc = validate_args(q, k, v, o, B, Hq, Hkv, Lq, Lk, d, S, kv_order, mode, stats)) return rc;
    const int pm = mode & 0xFF, dt = (mode >> 8) & 0xF;
    const int bn = 128;
    const int want_kernel = stats ? stats->kernel : 0;
    if (pm != FP8ATTN_MODE_FP8 || d != 128 || (stats && stats->block_n != 0 && stats->block_n != 128) ||
        (long long)(Hq / Hkv) * Lq > 16 || (want_kernel != 0 && want_kernel != 3)) {
        set_err("fp8attn_decode_noalloc serves decode shapes only: FP8 mode, d = 128, block_n 128, (Hq/Hkv)*Lq <= 16");
        return FP8ATTN_E_UNSUPPORTED;
    }
    if (int rc = check_device()) return rc;
    cudaStream_t st = stats ? reinterpret_cast<cudaStream_t>(stats->stream) : nullptr;
    const long long q_slabs = (long long)B * Hq, kv_slabs = (long long)B * Hkv;
    const int nb = (Lk + bn - 1) / bn;
    int ns = stats ? stats->num_splits : 0;
    if (ns == 0) ns = decode_auto_splits(kv_slabs, nb);
    if (ns > nb) ns = nb;
    const long long nq = q_slabs * Lq * d, R = q_slabs * Lq;

    // ---- layout of the call in the static array: [q codes][q scales][partial O][partial (m, l)]
    auto up = [](size_t x) { return (x + 255) & ~size_t(255); };
    size_t off = 0;
    const size_t o_codes = off;  off += (dt == 3) ? up((size_t)nq) : 0;
    const size_t o_qsc = off;    off += (dt == 3) ? up((size_t)q_slabs * 4) : 0;
    const size_t o_part = off;   off += (ns > 1) ? up((size_t)ns * R * (d + 2) * 4) : 0;
    if (off > (size_t)FP8ATTN_NOALLOC_SCRATCH_BYTES) {
        set_err("fp8attn_decode_noalloc: this call needs %zu bytes of scratch (%d splits), the static array holds %u",
                off, ns, (unsigned)FP8ATTN_NOALLOC_SCRATCH_BYTES);
        return FP8ATTN_E_SCRATCH;
    }
    unsigned char* scratch = nullptr;
    if (int rc = noalloc_scratch_ptr(&scratch)) return rc;

    const void* qs = q;
    const float* q_scale = stats ? stats->q_scale : nullptr;
    int n_launches = 0;
    if (dt == 3) {
        // the BF16 q of every (b, hq) slab to E4M3 (reading R24): Lq * d <= 2048 elements per slab, one warp each
        uint8_t* codes = scratch + o_codes;
        float* qsc = reinterpret_cast<float*>(scratch + o_qsc);
        quantize_small_slabs_kernel<__nv_bfloat16><<<(unsigned)((q_slabs + 3) / 4), 128, 0, st>>>(
            static_cast<const __nv_bfloat16*>(q), codes, qsc, Lq * d, (int)q_slabs);
        CU_TRY(cudaGetLastError());
        ++n_launches;
        qs = codes;
        q_scale = qsc;
    }

    const bool paged = stats && stats->block_table;
    if (paged && stats->page_size % bn != 0) return FP8ATTN_E_UNSUPPORTED;
    CUtensorMap mq16, mk, mv;
    // the G*Lq query rows of one kv head are consecutive rows of q: one 16-row box per CTA
    if (int rc = make_map(&mq16, qs, 1, 1, q_slabs * Lq, d, 16)) return rc;
    if (paged) {
        if (int rc = make_map(&mk, k, 1, (long long)stats->num_pages * Hkv, stats->page_size, d, bn)) return rc;
        if (int rc = make_map(&mv, v, 1, (long long)stats->num_pages * Hkv, stats->page_size, d, bn)) return rc;
    } else {
        if (int rc = make_map(&mk, k, 1, kv_slabs, Lk, d, bn)) return rc;
        if (int rc = make_map(&mv, v, 1, kv_slabs, Lk, d, bn)) return rc;
    }
    FwdParams p;
    memset(&p, 0, sizeof p);
    p.o = o;
    p.row_max = stats ? stats->row_max : nullptr;
    p.row_sum = stats ? stats->row_sum : nullptr;
    p.underflow = stats ? stats->underflow : nullptr;
    p.p_codes = stats ? stats->p_codes : nullptr;
    p.p_bh = stats ? stats->p_batch * Hq + stats->p_head : 0;
    p.q_scale = q_scale;
    p.k_scale = stats ? stats->k_scale : nullptr;
    p.v_scale = stats ? stats->v_scale : nullptr;
    p.B = B; p.Hq = Hq; p.Hkv = Hkv; p.Lq = Lq; p.Lk = Lk;
    p.causal = causal ? 1 : 0;
    p.kv_order = kv_order;
    p.n_sink = stats ? stats->n_sink : 0;
    p.scale_mode = stats ? stats->scale_mode : 0;
    p.o_bf16 = (stats && stats->o_dtype == FP8ATTN_O_BF16) ? 1 : 0;
    p.n_sinkpos = -1;
    if (stats && stats->sink_pos) {
        p.n_sinkpos = stats->n_sink;
        for (int i = 0; i < stats->n_sink; ++i) p.sink_pos[i] = stats->sink_pos[i];
    }
    const bool dynamic = p.scale_mode == 1;
    p.seqlens_q = stats ? stats->seqlens_q : nullptr;
    p.seqlens_k = stats ? stats->seqlens_k : nullptr;
    p.block_table = paged ? stats->block_table : nullptr;
    p.page_size = paged ? stats->page_size : 0;
    p.max_pages = paged ? stats->max_pages : 0;
    p.num_splits = ns;
    p.nb = nb;
    p.q_slabs = (int)q_slabs;
    p.kv_slabs = (int)kv_slabs;
    p.S = S;
    p.sm_scale = 1.0f / sqrtf((float)d);
    if (ns > 1) {
        p.part_o = reinterpret_cast<float*>(scratch + o_part);
        p.part_ml = p.part_o + (size_t)ns * R * d;
    }
    // caller buffers that must start clean (cudaMemsetAsync allocates nothing); the scratch needs no clearing:
    // the decode kernel writes every partial the combine kernel reads
    if (p.underflow) CU_TRY(cudaMemsetAsync(p.underflow, 0, 2 * sizeof(unsigned long long), st));
    if (p.p_codes) CU_TRY(cudaMemsetAsync(p.p_codes, 0xFF, (size_t)Lq * Lk, st));

    const int nv = (Hq / Hkv) * Lq;
    const int rc = (is_pow2_scale(S) || dynamic) ? launch_decode<true>(nv, mq16, mk, mv, p, st)
                                                 : launch_decode<false>(nv, mq16, mk, mv, p, st);
    if (rc) return rc;
    ++n_launches;
    if (ns > 1) {
        const int rows_per_block = 8;
        combine_kernel<<<(unsigned)((R + rows_per_block - 1) / rows_per_block), rows_per_block * 32, 0, st>>>(
            p.part_o, p.part_ml, p.o, p.row_max, p.row_sum, p.v_scale, R, d, ns, dynamic ? 1.0f : S, Hq, Hkv, Lq, p.o_bf16);
        CU_TRY(cudaGetLastError());
        ++n_launches;
    }
    if (stats) {
        stats->block_m_used = BM;
        stats->block_n_used = bn;
        stats->num_splits_used = ns;
        for (int s = 0; s <= ns; ++s) stats->split_bounds[s] = (int)(((long long)s * nb) / ns);
        stats->kernel_id = 3;
        stats->n_launches = n_launches;
    }
    return FP8ATTN_OK;
}
int fp8attn_fwd_host(const void* q, const void* k, const void* v, void* o, int B, int Hq, int Hkv, int Lq, int Lk,
                     int d, int causal, float S, int kv_order, int mode, fp8attn_stats* stats) {
    if (int rc = validate_args(q, k, v, o, B, Hq, Hkv, Lq, Lk, d, S, kv_order, mode, stats)) return rc;
    if (stats && (stats->seqlens_q || stats->seqlens_k || stats->block_table)) return FP8ATTN_E_UNSUPPORTED;
    if (int rc = check_device()) return rc;
    const int dt = (mode >> 8) & 0xF;
    const size_t ebq = (dt == 0) ? 4 : (dt == 2 ? 1 : 2);
    const size_t ebkv = (dt == 0) ? 4 : (dt == 1 ? 2 : 1);
    const size_t R = (size_t)B * Hq * Lq;
    const size_t nq = R * d, nkv = (size_t)B * Hkv * Lk * d;
    const size_t nqs = (size_t)B * Hq, nkvs = (size_t)B * Hkv;
    auto up = [](size_t x) { return (x + 255) & ~size_t(255); };
    // device staging layout
    size_t off = 0;
    const size_t o_q = off;   off += up(nq * ebq);
    const size_t o_k = off;   off += up(nkv * ebkv);
    const size_t o_v = off;   off += up(nkv * ebkv);
    const size_t ebo = (stats && stats->o_dtype == FP8ATTN_O_BF16) ? 2 : 4;
    const size_t o_o = off;   off += up(nq * ebo);
    const size_t o_qs = off;  off += up(nqs * 4);
    const size_t o_ks = off;  off += up(nkvs * 4);
    const size_t o_vs = off;  off += up(nkvs * 4);
    const size_t o_rm = off;  off += up(R * 4);
    const size_t o_rs = off;  off += up(R * 4);
    const size_t o_uf = off;  off += up(16);
    const size_t o_pc = off;  off += (stats && stats->p_codes) ? up((size_t)Lq * Lk) : 0;

    cudaStream_t st = stats ? reinterpret_cast<cudaStream_t>(stats->stream) : nullptr;
    int dev_now = 0;
    if (int rc = current_device(&dev_now)) return rc;
    DeviceState& ds_dev = g_dev[dev_now];
    std::lock_guard<std::mutex> lock(ds_dev.host_mu);
    Lease staging;                      // returned to the pool after the final synchronisation below
    if (int rc = staging.get(off, st)) return rc;
    // whatever way this function is left, no copy may still be in flight when the staging memory goes back
    struct Drain {
        DeviceState& d;
        cudaStream_t st;
        ~Drain() {
            if (d.s_in) cudaStreamSynchronize(d.s_in);
            cudaStreamSynchronize(st);
            if (d.s_out) cudaStreamSynchronize(d.s_out);
        }
    } drain{ds_dev, st};
    uint8_t* base = static_cast<uint8_t*>(staging.ptr);
    fp8attn_stats dstats;
    fp8attn_stats* ds = nullptr;
    if (stats) {
        dstats = *stats;
        ds = &dstats;
        if (stats->q_scale) {
            CU_TRY(cudaMemcpyAsync(base + o_qs, stats->q_scale, nqs * 4, cudaMemcpyHostToDevice, st));
            dstats.q_scale = reinterpret_cast<const float*>(base + o_qs);
        }
        if (stats->k_scale) {
            CU_TRY(cudaMemcpyAsync(base + o_ks, stats->k_scale, nkvs * 4, cudaMemcpyHostToDevice, st));
            dstats.k_scale = reinterpret_cast<const float*>(base + o_ks);
        }
        if (stats->v_scale) {
            CU_TRY(cudaMemcpyAsync(base + o_vs, stats->v_scale, nkvs * 4, cudaMemcpyHostToDevice, st));
            dstats.v_scale = reinterpret_cast<const float*>(base + o_vs);
        }
        if (stats->row_max) dstats.row_max = reinterpret_cast<float*>(base + o_rm);
        if (stats->row_sum) dstats.row_sum = reinterpret_cast<float*>(base + o_rs);
        if (stats->underflow) dstats.underflow = reinterpret_cast<unsigned long long*>(base + o_uf);
        if (stats->p_codes) {
            dstats.p_codes = base + o_pc;
        }
    }
    // (batch, kv-head group) slabs are independent and contiguous in q, k, v and o: large
    // calls are cut into up to 8 pieces so that the upload of piece i+1, the kernel of piece i and the download
    // of piece i-1 overlap on three streams (PCIe is full duplex).  The P dump and the underflow counters belong
    // to one whole call and keep the single-piece path.
    int pieces_b = 1, pieces_h = 1;      // pieces along the batch, and along the kv heads of one batch element
    const size_t traffic = nq * ebq + 2 * nkv * ebkv + nq * ebo;
    // (the automatic split count of a decode-shaped call depends on B * Hkv: such a call stays whole unless the
    // caller fixes num_splits, otherwise the pieces would take another split layout than the single call, R14)
    const bool auto_split = (long long)(Hq / Hkv) * Lq <= 16 && !(stats && stats->num_splits > 0);
    if (traffic >= (size_t(32) << 20) && !auto_split && !(stats && (stats->p_codes || stats->underflow))) {
        pieces_b = B < 8 ? B : 8;
        // pieces along the kv heads: the largest power of two that divides Hkv and keeps the total at 8 or less
        while (pieces_b * pieces_h * 2 <= 8 && Hkv % (pieces_h * 2) == 0) pieces_h *= 2;
    }
    const int n_pieces = pieces_b * pieces_h;      // <= 8: the size of the event arrays
    if (n_pieces > 8) return FP8ATTN_E_UNSUPPORTED;
    if (n_pieces == 1) {
        CU_TRY(cudaMemcpyAsync(base + o_q, q, nq * ebq, cudaMemcpyHostToDevice, st));
        CU_TRY(cudaMemcpyAsync(base + o_k, k, nkv * ebkv, cudaMemcpyHostToDevice, st));
        CU_TRY(cudaMemcpyAsync(base + o_v, v, nkv * ebkv, cudaMemcpyHostToDevice, st));
        if (int rc = fp8attn_fwd(base + o_q, base + o_k, base + o_v, base + o_o, B, Hq, Hkv, Lq, Lk, d, causal, S,
                                 kv_order, mode, ds))
            return rc;
        CU_TRY(cudaMemcpyAsync(o, base + o_o, nq * ebo, cudaMemcpyDeviceToHost, st));
        if (stats) {
            if (stats->row_max) CU_TRY(cudaMemcpyAsync(stats->row_max, base + o_rm, R * 4, cudaMemcpyDeviceToHost, st));
            if (stats->row_sum) CU_TRY(cudaMemcpyAsync(stats->row_sum, base + o_rs, R * 4, cudaMemcpyDeviceToHost, st));
            if (stats->underflow) CU_TRY(cudaMemcpyAsync(stats->underflow, base + o_uf, 16, cudaMemcpyDeviceToHost, st));
            if (stats->p_codes)
                CU_TRY(cudaMemcpyAsync(stats->p_codes, base + o_pc, (size_t)Lq * Lk, cudaMemcpyDeviceToHost, st));
        }
    } else {
        // the copy streams and events of this device, created on first use
        cudaStream_t& s_in = ds_dev.s_in;
        cudaStream_t& s_out = ds_dev.s_out;
        cudaEvent_t& ev_start = ds_dev.ev_start;
        cudaEvent_t* const ev_in = ds_dev.ev_in;
        cudaEvent_t* const ev_done = ds_dev.ev_done;
        if (!s_in) {
            CU_TRY(cudaStreamCreateWithFlags(&s_in, cudaStreamNonBlocking));
            CU_TRY(cudaStreamCreateWithFlags(&s_out, cudaStreamNonBlocking));
            CU_TRY(cudaEventCreateWithFlags(&ev_start, cudaEventDisableTiming));
            for (int i = 0; i < 8; ++i) {
                CU_TRY(cudaEventCreateWithFlags(&ev_in[i], cudaEventDisableTiming));
                CU_TRY(cudaEventCreateWithFlags(&ev_done[i], cudaEventDisableTiming));
            }
        }
        CU_TRY(cudaEventRecord(ev_start, st));          // the staging buffer and the scales are ordered on st
        CU_TRY(cudaStreamWaitEvent(s_in, ev_start, 0));
        const uint8_t* hq = static_cast<const uint8_t*>(q);
        const uint8_t* hk = static_cast<const uint8_t*>(k);
        const uint8_t* hv = static_cast<const uint8_t*>(v);
        uint8_t* ho = static_cast<uint8_t*>(o);
        int launches = 0;
        for (int i = 0; i < n_pieces; ++i) {
            // piece i: batch elements [b0, b1), kv heads [h0, h0 + hkv_p) of each (one batch element if pieces_h > 1)
            const int ib = i / pieces_h, ih = i % pieces_h;
            const int b0 = (int)((long long)B * ib / pieces_b), b1 = (int)((long long)B * (ib + 1) / pieces_b);
            const int hkv_p = Hkv / pieces_h, hq_p = Hq / pieces_h;
            const size_t q_slab0 = (size_t)b0 * Hq + (size_t)ih * hq_p, kv_slab0 = (size_t)b0 * Hkv + (size_t)ih * hkv_p;
            const size_t q_el = q_slab0 * Lq * d, kv_el = kv_slab0 * Lk * d;
            const size_t q_n = (size_t)(b1 - b0) * hq_p * Lq * d, kv_n = (size_t)(b1 - b0) * hkv_p * Lk * d;
            CU_TRY(cudaMemcpyAsync(base + o_q + q_el * ebq, hq + q_el * ebq, q_n * ebq, cudaMemcpyHostToDevice, s_in));
            CU_TRY(cudaMemcpyAsync(base + o_k + kv_el * ebkv, hk + kv_el * ebkv, kv_n * ebkv, cudaMemcpyHostToDevice, s_in));
            CU_TRY(cudaMemcpyAsync(base + o_v + kv_el * ebkv, hv + kv_el * ebkv, kv_n * ebkv, cudaMemcpyHostToDevice, s_in));
            CU_TRY(cudaEventRecord(ev_in[i], s_in));
            CU_TRY(cudaStreamWaitEvent(st, ev_in[i], 0));
            fp8attn_stats ps;
            fp8attn_stats* pp = nullptr;
            if (ds) {
                ps = dstats;
                pp = &ps;
                if (ps.q_scale) ps.q_scale += q_slab0;
                if (ps.k_scale) ps.k_scale += kv_slab0;
                if (ps.v_scale) ps.v_scale += kv_slab0;
                if (ps.row_max) ps.row_max += q_slab0 * Lq;
                if (ps.row_sum) ps.row_sum += q_slab0 * Lq;
            }
            if (int rc = fp8attn_fwd(base + o_q + q_el * ebq, base + o_k + kv_el * ebkv, base + o_v + kv_el * ebkv,
                                     base + o_o + q_el * ebo, b1 - b0, pieces_h > 1 ? hq_p : Hq, pieces_h > 1 ? hkv_p : Hkv,
                                     Lq, Lk, d, causal, S, kv_order, mode, pp))
                return rc;
            if (pp) {
                launches += ps.n_launches;
                dstats.block_m_used = ps.block_m_used;
                dstats.block_n_used = ps.block_n_used;
                dstats.num_splits_used = ps.num_splits_used;
                memcpy(dstats.split_bounds, ps.split_bounds, sizeof ps.split_bounds);
                dstats.kernel_id = ps.kernel_id;
                dstats.n_launches = launches;
            }
            CU_TRY(cudaEventRecord(ev_done[i], st));
            CU_TRY(cudaStreamWaitEvent(s_out, ev_done[i], 0));
            CU_TRY(cudaMemcpyAsync(ho + q_el * ebo, base + o_o + q_el * ebo, q_n * ebo, cudaMemcpyDeviceToHost, s_out));
            if (stats && stats->row_max)
                CU_TRY(cudaMemcpyAsync(stats->row_max + q_slab0 * Lq, base + o_rm + q_slab0 * Lq * 4,
                                       (size_t)(b1 - b0) * hq_p * Lq * 4, cudaMemcpyDeviceToHost, s_out));
            if (stats && stats->row_sum)
                CU_TRY(cudaMemcpyAsync(stats->row_sum + q_slab0 * Lq, base + o_rs + q_slab0 * Lq * 4,
                                       (size_t)(b1 - b0) * hq_p * Lq * 4, cudaMemcpyDeviceToHost, s_out));
        }
        CU_TRY(cudaStreamSynchronize(s_out));
    }
    if (stats) {
        stats->block_m_used = dstats.block_m_used;
        stats->block_n_used = dstats.block_n_used;
        stats->num_splits_used = dstats.num_splits_used;
        memcpy(stats->split_bounds, dstats.split_bounds, sizeof dstats.split_bounds);
        stats->kernel_id = dstats.kernel_id;
        stats->n_launches = dstats.n_launches;
    }
    CU_TRY(cudaStreamSynchronize(st));
    return FP8ATTN_OK;
}

int fp8attn_quantize_e4m3(const float* x, uint8_t* out_codes, float* out_scale, int B, int H, int L, int d,
                          void* stream) {
    if (!x || !out_codes || !out_scale) return FP8ATTN_E_NULL;
    if (B < 1 || H < 1 || L < 1 || d < 1) return FP8ATTN_E_SHAPE;
    if (int rc = check_device()) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    const long long slabs = (long long)B * H, slab = (long long)L * d;
    if (slabs > 0x7FFFFFFFll) return FP8ATTN_E_UNSUPPORTED;
    Lease amax_buf;
    if (int rc = amax_buf.get((size_t)slabs * 4, st)) return rc;
    unsigned int* amax = static_cast<unsigned int*>(amax_buf.ptr);
    CU_TRY(cudaMemsetAsync(amax, 0, (size_t)slabs * 4, st));
    unsigned gy = (unsigned)((slab + 1023) / 1024);
    if (gy > 148) gy = 148;
    absmax_kernel<float><<<dim3((unsigned)slabs, gy), 256, 0, st>>>(x, amax, slab);
    quantize_kernel<float><<<dim3((unsigned)slabs, gy), 256, 0, st>>>(x, amax, out_codes, slab);
    finalize_scale_kernel<<<(unsigned)((slabs + 255) / 256), 256, 0, st>>>(amax, out_scale, (int)slabs);
    CU_TRY(cudaGetLastError());
    return FP8ATTN_OK;
}

int fp8attn_debug_gemm(const void* A, const void* Bm, float* D, int N, int K, int elem_bytes, int a_in_tmem,
                       int b_mn_major, void* stream) {
    if (!A || !Bm || !D) return FP8ATTN_E_NULL;
    if ((elem_bytes != 1 && elem_bytes != 2) || (N != 64 && N != 128)) return FP8ATTN_E_SHAPE;
    const int ch = 128 / elem_bytes;
    if (K < ch || K % ch != 0 || K > 256) return FP8ATTN_E_SHAPE;
    if (int rc = check_device()) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    CUtensorMap ma, mb;
    if (int rc = make_map(&ma, A, elem_bytes, 1, 128, K, 128)) return rc;
    if (b_mn_major) {
        if (int rc = make_map(&mb, Bm, elem_bytes, 1, K, N, K)) return rc;     // [K, N]: boxes of K rows x 128 B
    } else {
        if (int rc = make_map(&mb, Bm, elem_bytes, 1, N, K, N)) return rc;     // [N, K]: boxes of N rows x 128 B
    }
    const int smem = (K / ch) * 128 * 128 + (b_mn_major ? (N / ch > 0 ? N / ch : 1) * K * 128 : (K / ch) * N * 128) + 1024 + 64;
    if (b_mn_major && N < ch) return FP8ATTN_E_SHAPE;
    if (elem_bytes == 2) {
        CU_TRY(cudaFuncSetAttribute(debug_gemm_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        debug_gemm_kernel<2><<<1, 128, smem, st>>>(ma, mb, static_cast<const uint8_t*>(A), D, N, K, a_in_tmem, b_mn_major);
    } else {
        CU_TRY(cudaFuncSetAttribute(debug_gemm_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        debug_gemm_kernel<1><<<1, 128, smem, st>>>(ma, mb, static_cast<const uint8_t*>(A), D, N, K, a_in_tmem, b_mn_major);
    }
    CU_TRY(cudaGetLastError());
    return FP8ATTN_OK;
}

}  // extern "C"
