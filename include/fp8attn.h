/*
 * fp8attn.h -- C ABI of libfp8attn.so: B200 (sm_100a) FP8 attention forward with the
 * kernel-faithful P-cast semantics of arxiv/paper_2606_06521.
 *
 * The operation is Algorithm 1 of the paper ("FP8 Online Softmax
 * Attention") with the semantics of its section 6.1:
 *     for each KV block j in BlockOrder:   Z = Q K_j^T / sqrt(d);  m_new = max(m, max Z);
 *         alpha = exp(m - m_new);  P = exp(Z - m_new)  (FP32);
 *         l = alpha l + sum(P)                      (FP32, PRE-cast P);
 *         P8 = cast_E4M3(P * S)                     (round-to-nearest-even, saturating);
 *         O = alpha O + P8 V_j                      (FP32 accumulate)
 *     return O / (S l)
 * BlockOrder is forward (0..nb-1) or reverse (nb-1..0, the block holding the sink keys
 * last).  S is the static P scale (Eq. 16).
 *
 * All entry points return 0 on success or a negative FP8ATTN_E_* code; they never throw,
 * abort or exit.  No entry point allocates or frees caller-visible memory or synchronises
 * the stream.  Work is enqueued on the CUDA stream given in `stats->stream` (the legacy
 * default stream if `stats` is NULL).  Scratch memory (split-KV partials, BF16 planes of
 * FP32 inputs, quantised q for decode, the staging of fp8attn_fwd_host) is allocated per call,
 * on that stream, from a library-owned stream-ordered memory pool of the current device and
 * returned to the pool when the call's work is enqueued: calls on different streams, threads
 * or devices share no scratch and may run concurrently.  The pool keeps what it has been given
 * until fp8attn_trim().  Every entry point works on the CURRENT device (cudaSetDevice).
 */
#ifndef FP8ATTN_H
#define FP8ATTN_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define FP8ATTN_API __attribute__((visibility("default")))

/* ---- `mode` argument: (input dtype << 8) | P mode ------------------------------------ */
#define FP8ATTN_MODE_NOCAST     0   /* reference: P stays FP32, S ignored (treated as 1)        */
#define FP8ATTN_MODE_ISOLATION  1   /* P-cast isolation: Q,K,V FP32/BF16, P cast
                                       to E4M3 and dequantised exactly to BF16 for P.V          */
#define FP8ATTN_MODE_FP8        2   /* production: E4M3 q/k/v with per-(b,h) scales, both
                                       matmuls tcgen05 kind::f8f6f4                            */
#define FP8ATTN_DTYPE_F32          (0 << 8)  /* q,k,v float32                                    */
#define FP8ATTN_DTYPE_BF16         (1 << 8)  /* q,k,v bfloat16                                   */
#define FP8ATTN_DTYPE_E4M3         (2 << 8)  /* q,k,v E4M3 codes; q_scale,k_scale,v_scale needed */
#define FP8ATTN_DTYPE_BF16Q_E4M3KV (3 << 8)  /* decode: q bfloat16 (quantised per (b,hq) slab to
                                                E4M3 by the library), k,v E4M3; k_scale,v_scale  */

/* ---- `kv_order` ---------------------------------------------------------------------- */
#define FP8ATTN_ORDER_FORWARD 0     /* blocks 0 .. nb-1                                          */
#define FP8ATTN_ORDER_REVERSE 1     /* blocks nb-1 .. 0 (sink block last)          */
#define FP8ATTN_ORDER_SINK_LAST 2   /* sink keys anywhere (stats->sink_pos): the blocks that hold no
                                       sink key in descending order, then the blocks that hold one,
                                       in descending order (the per-block view of PAPER.md:443;
                                       DESIGN.md reading R27).  With the sink keys in block 0 this
                                       is FP8ATTN_ORDER_REVERSE.  General and decode kernels.     */

/* ---- stats->scale_mode --------------------------------------------------------------- */
#define FP8ATTN_SCALE_STATIC  0     /* P * S, the static scale of Alg. 1 line 9                  */
#define FP8ATTN_SCALE_DYNAMIC 1     /* per-(row, block) power-of-two scale S_j = 2^k_j, k_j the
                                       largest k <= 30 with 2^k * exp(m_loc - m_new) <= 448, i.e.
                                       k_j = floor(log2 448 + (m_new - m_loc) log2 e) in FP32
                                       ("dynamic per-block scale ... constrained to
                                       2^k"; reading R26).  S is not used.  Modes 1, 2.  */

/* ---- stats->o_dtype ------------------------------------------------------------------ */
#define FP8ATTN_O_F32  0
#define FP8ATTN_O_BF16 1            /* o is bfloat16 (round to nearest even in the epilogue)      */

#define FP8ATTN_MAX_SINKS 32

/* ---- error codes --------------------------------------------------------------------- */
#define FP8ATTN_OK              0
#define FP8ATTN_E_NULL         -1   /* a required pointer is NULL                                */
#define FP8ATTN_E_SHAPE        -2   /* a size is < 1, Hq % Hkv != 0, or d not in {64, 128}       */
#define FP8ATTN_E_SCALE        -3   /* S is not a finite FP32 > 0                                */
#define FP8ATTN_E_MODE         -4   /* unknown mode / dtype / kv_order / scale_mode / o_dtype, or a
                                       combination that is not defined (mode 2 needs E4M3 k,v;
                                       modes 0,1 need FP32/BF16; the dynamic scale needs a cast)  */
#define FP8ATTN_E_UNSUPPORTED  -5   /* valid but not built: E4M3 with d != 128 (a 64-byte operand
                                       row does not fill the 128-byte swizzle row the kernels are
                                       built on), block_n not in {0, 64, 128}, FP32 inputs with
                                       block_n 128, num_splits above FP8ATTN_MAX_SPLITS, a kernel
                                       family that cannot serve the call                        */
#define FP8ATTN_E_DEVICE       -6   /* current device is not compute capability 10.x             */
#define FP8ATTN_E_CUDA         -7   /* a CUDA call failed (allocation, tensor map, launch)       */
#define FP8ATTN_E_STATS        -8   /* stats->struct_size does not match this header             */
#define FP8ATTN_E_SCRATCH      -9   /* fp8attn_decode_noalloc: the call needs more scratch than
                                       FP8ATTN_NOALLOC_SCRATCH_BYTES                              */

#define FP8ATTN_MAX_SPLITS 64

/*
 * Optional controls and statistics.  Zero-initialise, set struct_size = sizeof(fp8attn_stats),
 * fill what is needed.  Device pointers are caller-owned.
 */
typedef struct fp8attn_stats {
    /* ---- inputs ---- */
    int32_t struct_size;       /* sizeof(fp8attn_stats)                                          */
    int32_t n_sink;            /* number of sink keys (k_sink): the first n_sink keys
                                  of the sequence, or the n_sink <= FP8ATTN_MAX_SINKS entries of
                                  sink_pos.  Used to classify underflows and by
                                  FP8ATTN_ORDER_SINK_LAST                                        */
    int32_t block_n;           /* KV block size Bn request: 0 = library default, else 64 or 128
                                  ("typically 64 or 128")                          */
    int32_t num_splits;        /* split-KV request: 0 = automatic, n >= 1 = exactly n contiguous
                                  block ranges                             */
    int32_t kernel;            /* kernel family request: 0 = automatic, 1 = general kernel, 2 = warp-
                                  specialised prefill kernel, 3 = split-KV decode kernel; a family
                                  that cannot serve the call gives FP8ATTN_E_UNSUPPORTED       */
    int32_t scale_mode;        /* FP8ATTN_SCALE_*                                                */
    const float *q_scale;      /* device [B*Hq]  dequantisation scale of E4M3 q (value = code*scale) */
    const float *k_scale;      /* device [B*Hkv]                                                 */
    const float *v_scale;      /* device [B*Hkv]                                                 */
    void *stream;              /* cudaStream_t                                                   */
    uint8_t *p_codes;          /* device [Lq, Lk] or NULL: E4M3 code of every P of head
                                  (p_batch, p_head); the library fills the buffer with 0xFF first,
                                  so masked positions hold 0xFF; mode 0 writes nothing.  p_codes and
                                  underflow are served by every kernel family: the general kernel
                                  (the automatic choice for prefill shapes that ask for either), the
                                  statistics instances of the prefill kernels (kernel = 2; same
                                  schedule as the throughput instance) and of the decode kernel
                                  (the automatic choice for decode shapes)                        */
    int32_t p_batch, p_head;
    const int32_t *sink_pos;   /* HOST pointer or NULL: n_sink key indices, ascending, of the sink
                                  keys (multi-sink / distributed-sink layouts)    */
    int32_t o_dtype;           /* FP8ATTN_O_*                                                    */
    int32_t reserved1;         /* must be 0                                                      */
    /* variable-length and paged KV-cache prefill / decode (the shape of the kernel the paper simulates,
       attention_with_kvcache_prefill_fp8).  All optional.                              */
    const int32_t *seqlens_q;  /* device [B] or NULL: batch element b has seqlens_q[b] <= Lq query rows
                                  (q, o stay padded [B,Hq,Lq,d]); the rows beyond produce 0, like rows
                                  that see no key.  The causal diagonal is bottom-right aligned per
                                  batch element: key j visible to row i iff j <= i + seqlens_k[b] -
                                  seqlens_q[b]                                                   */
    const int32_t *seqlens_k;  /* device [B] or NULL: batch element b has seqlens_k[b] <= Lk keys    */
    const int32_t *block_table;/* device [B, max_pages] or NULL.  Not NULL: k and v are page pools
                                  [num_pages, Hkv, page_size, d]; key j of batch element b is row
                                  j % page_size of page block_table[b][j / page_size].  page_size must
                                  be a multiple of the KV block (block_n_used); BF16 / E4M3 k, v.
                                  Memory of a page beyond the end of its sequence must hold finite
                                  values (it is multiplied by P = 0)                             */
    int32_t page_size, max_pages, num_pages;
    int32_t reserved2;         /* must be 0                                                      */
    /* ---- outputs, device (each may be NULL) ---- */
    float *row_max;            /* [B,Hq,Lq] final running max m (scaled logits, natural log)    */
    float *row_sum;            /* [B,Hq,Lq] final l relative to m; NOT multiplied by S           */
    unsigned long long *underflow; /* [2]: number of visible non-sink P values (key index >=
                                  n_sink) whose E4M3 code is zero (Prop. 1),
                                  [0] in blocks that hold a sink key, [1] in all other blocks.
                                  Zeroed by the library at the start of the call.              */
    /* ---- outputs, host (written before the call returns) ---- */
    int32_t block_m_used;      /* query rows per tile                                            */
    int32_t block_n_used;      /* Bn actually used                                               */
    int32_t num_splits_used;
    int32_t split_bounds[FP8ATTN_MAX_SPLITS + 1]; /* split s covers blocks
                                  [split_bounds[s], split_bounds[s+1])                          */
    int32_t kernel_id;         /* which kernel family ran: 1 = general tcgen05 kernel,
                                  2 = warp-specialised prefill kernel, 3 = split-KV decode kernel */
    int32_t n_launches;        /* kernels launched by this call                                  */
} fp8attn_stats;

/*
 * fp8attn_fwd -- attention forward (Alg. 1).
 *   q, o : device, [B, Hq, Lq, d] contiguous row-major; o is float32 (bfloat16 with stats->o_dtype).
 *   k, v : device, [B, Hkv, Lk, d] (or page pools, see stats->block_table; Lk is then the capacity
 *          max_pages * page_size is checked against); query head h reads kv head h / (Hq / Hkv).
 *   d    : 64 or 128.  Softmax scale is 1/sqrt(d).
 *   causal : nonzero = key j visible to query i iff j <= i + (Lk - Lq) (bottom-right).
 *   S    : static P scale, finite > 0 (values above 448 saturate at 448).
 *   kv_order, mode : see the defines above.
 *   stats : NULL, or controls/statistics as documented in the struct.
 * Rows that see no key produce 0, row_max = -inf, row_sum = 0.
 */
FP8ATTN_API int fp8attn_fwd(const void *q, const void *k, const void *v, void *o,
                            int B, int Hq, int Hkv, int Lq, int Lk, int d,
                            int causal, float S, int kv_order, int mode, fp8attn_stats *stats);

/*
 * fp8attn_fwd_host -- the same operation with HOST buffers (the end-to-end call).
 *   q, k, v, o and, in `stats`, q_scale / k_scale / v_scale / row_max / row_sum / underflow /
 *   p_codes are HOST pointers here (pinned memory makes the copies asynchronous; pageable
 *   memory works).  The library copies q, k, v and the scales to library-owned device scratch
 *   on `stats->stream`, runs fp8attn_fwd there, copies o and the requested statistics back and
 *   synchronises that stream before returning, so the outputs are valid on return.
 *   Element sizes follow the dtype bits of `mode`: FP32 4 B, BF16 2 B, E4M3 1 B.
 *   Calls that move 32 MB or more, ask for neither p_codes nor underflow and do not leave the split
 *   count of a decode shape ((Hq/Hkv)*Lq <= 16) to the library are cut into at most 8
 *   (batch, kv-head group) pieces -- independent units of the operation -- whose uploads, kernels
 *   and downloads overlap on `stats->stream` and two library-owned copy streams; the results are
 *   those of the single call bit for bit, `n_launches` counts every piece.
 * Every step of the method still runs in the CUDA kernels; the host side only copies.
 * seqlens_q / seqlens_k / block_table are not taken here (FP8ATTN_E_UNSUPPORTED): a paged cache lives on the device.
 * Errors as fp8attn_fwd.
 */
FP8ATTN_API int fp8attn_fwd_host(const void *q, const void *k, const void *v, void *o,
                                 int B, int Hq, int Hkv, int Lq, int Lk, int d,
                                 int causal, float S, int kv_order, int mode, fp8attn_stats *stats);

/*
 * fp8attn_decode_noalloc -- the split-KV decode path of fp8attn_fwd for callers that must not allocate
 * (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  Same
 * arguments, same kernels, same split layout and therefore the same results bit for bit as
 * fp8attn_fwd on a decode-shaped call; what differs is where the scratch lives.  fp8attn_fwd takes
 * the quantised q and the split-KV partials (m_s, l_s, O_s, reading R14)
 * from a stream-ordered memory pool per call; this entry point keeps them in ONE file-scope
 * `static __device__` array of FP8ATTN_NOALLOC_SCRATCH_BYTES that every GPU which loads the
 * library holds until the process exits.  It calls no cudaMalloc, cudaFree, pool or other
 * allocating routine (what it does call: cudaGetSymbolAddress once per device, tensor-map encoding
 * on the host, cudaMemsetAsync on caller buffers, kernel launches).
 *   Accepted: mode FP8ATTN_MODE_FP8 with FP8ATTN_DTYPE_BF16Q_E4M3KV or FP8ATTN_DTYPE_E4M3, d = 128,
 *   block_n 0 or 128, (Hq / Hkv) * Lq <= 16 (the decode kernel's shape), stats->kernel 0 or 3;
 *   everything else of fp8attn_stats as in fp8attn_fwd (num_splits 0 = the same automatic count).
 *   Anything else: FP8ATTN_E_UNSUPPORTED.
 *   Scratch needed: B*Hq*Lq*d + 4*B*Hq bytes for the quantised q (BF16 q only) plus, with more than
 *   one split, num_splits * B*Hq*Lq * (d + 2) * 4 bytes of partials, each part rounded up to 256 B
 *   (BASELINE config 5 with 4 splits: 4.5 MB).  A call that needs more than
 *   FP8ATTN_NOALLOC_SCRATCH_BYTES gets FP8ATTN_E_SCRATCH and fp8attn_last_cuda_error() names both
 *   sizes; nothing has been launched then.
 *   Every call on a device shares the array, and the array keeps the contents of the last call.
 *   No word of it has to start at zero: every word a kernel of a call reads has been written by an
 *   earlier kernel of the same call on the same stream (the caller's counters in stats->underflow
 *   are cleared by the call, as in fp8attn_fwd).  Calls that can overlap on the GPU -- two streams,
 *   two host threads on one device -- RACE on the array: the caller serialises them (one stream, or
 *   events).  Calls on different devices do not interact.
 */
#define FP8ATTN_NOALLOC_SCRATCH_BYTES (16u << 20)
FP8ATTN_API int fp8attn_decode_noalloc(const void *q, const void *k, const void *v, void *o,
                                       int B, int Hq, int Hkv, int Lq, int Lk, int d,
                                       int causal, float S, int kv_order, int mode, fp8attn_stats *stats);

/*
 * fp8attn_quantize_e4m3 -- per-(b,h) slab quantisation of FP32 to E4M3 (BASELINE config 3
 * "per-head absmax/448"; the paper treats QKV quantisation as orthogonal).
 *   x : device float32 [B,H,L,d];  out_codes : device uint8 [B,H,L,d];
 *   out_scale : device float32 [B,H] = absmax/448 (1 for an all-zero slab);
 *   code = cvt.rn.satfinite.e4m3(x * (448/absmax)).  stream : cudaStream_t.
 */
FP8ATTN_API int fp8attn_quantize_e4m3(const float *x, uint8_t *out_codes, float *out_scale,
                                      int B, int H, int L, int d, void *stream);

/*
 * fp8attn_debug_gemm -- DIAGNOSTIC, not part of the method: one-tile tcgen05 GEMM through the
 * same TMA / shared-memory-descriptor / TMEM helpers the attention kernels use, so that a test
 * can pin those primitives (operand majors, swizzle, A-from-TMEM) against an FP64 product.
 *   D[128,N] (device float32) = A[128,K] . B, FP32 accumulate.
 *   elem_bytes 2 = BF16 (kind::f16), 1 = E4M3 (kind::f8f6f4).
 *   a_in_tmem : 0 = A read from swizzled shared memory, 1 = A staged in TMEM (the P operand path).
 *   b_mn_major: 0 = B given as [N,K] (K contiguous, the K-tile path), 1 = B given as [K,N]
 *               (N contiguous, the V-tile path).
 *   N in {64,128}; K a multiple of 64 (BF16) / 128 (E4M3), K <= 256.
 */
FP8ATTN_API int fp8attn_debug_gemm(const void *A, const void *Bm, float *D, int N, int K,
                                   int elem_bytes, int a_in_tmem, int b_mn_major, void *stream);

/*
 * fp8attn_trim -- give the scratch memory the library's pool holds on the current device back to
 * the driver (memory still in use by enqueued work stays until that work has run).
 */
FP8ATTN_API int fp8attn_trim(void);

FP8ATTN_API const char *fp8attn_strerror(int code);
FP8ATTN_API const char *fp8attn_last_cuda_error(void);   /* text of the last CUDA failure */
FP8ATTN_API int fp8attn_version(void);                   /* major*10000 + minor*100 + patch */

#ifdef __cplusplus
}
#endif
#endif /* FP8ATTN_H */
