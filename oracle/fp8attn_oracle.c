/*
 * fp8attn_oracle.c -- plain, slow, CPU oracle for FP8 attention with the paper's
 * kernel-faithful P-cast semantics (arxiv/paper_2606_06521).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header, table or constant generator with the CUDA path under
 * paper_2606_06521_b200/csrc/.
 *
 * What it follows (PAPER.md line numbers):
 *   - E4M3 value set, Eq. 1-2 and the threshold table.
 *   - Algorithm 1, FP8 online-softmax attention for one query row,
 *     line order repaired from PAPER.md:80 ("l is line 8, O is line 10").
 *   - Kernel-faithful semantics of section 6.1: l in FP32 from the
 *     pre-cast P, O accumulated from the post-cast P, round-to-nearest E4M3,
 *     epilogue O/(S*l).
 *   - dp(S), Def. 1 / Eq. 17 and its overflow extension Eq. 18.
 *   - Proposition 1: a P value underflows iff its cast is zero.
 *
 * Readings of silent / garbled passages are DESIGN.md section "Readings" (R1..).
 *
 * Parity pins (tests/test_oracle_*.py): E4M3 enumeration, RNE ties, dp(S) App. A
 * values, Prop. 5, no-cast == brute-force softmax, Table 1 / Eq. 7 underflow
 * fractions, Thm 4 zero-underflow.  "Parity unpinned by the paper" (pinned by
 * invariants only): split-KV + combine, per-(b,h) absmax/448 input quantisation,
 * the dynamic per-block power-of-two scale (PAPER.md:435 names it as future work
 * without a rule; reading R26, pinned by: equal to static 256 bit for bit when the
 * exponent is constant, never an underflow that static 256 does not have, an
 * independent offline recomputation), sink keys at arbitrary positions and the
 * "sink blocks last" order (reading R27, pinned by: the prefix
 * layout reproduces the default counters, zero underflow outside the sink blocks
 * for S = 256, an independent offline recomputation).
 *
 * Arithmetic: FP64 everywhere except where Alg. 1 fixes FP32 (the logits Z, the
 * probabilities P, the product P*S and the running max are FP32 values).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_API __attribute__((visibility("default")))

/* ------------------------------------------------------------------------- */
/* E4M3 number line (Eq. 1-2)                                 */
/* ------------------------------------------------------------------------- */

/* Value of the positive code c = (E<<3)|M, c in 0x00..0x7E.  0x7F is NaN.   */
static double e4m3_code_value_eq(int c)
{
    int E = (c >> 3) & 0xF, M = c & 7;
    if (E == 0)
        return ldexp((double)M / 8.0, -6);       /* Eq. 1: 2^(1-b) * M/8, b = 7 */
    return ldexp(1.0 + (double)M / 8.0, E - 7);  /* Eq. 2: 2^(E-b) * (1+M/8)    */
}

/* The table of code values {0} U the 126 positive values, filled once from Eq. 1-2 when the
 * library is loaded; every later use reads the table instead of calling ldexp again. */
static double g_code_value[0x7F];
__attribute__((constructor)) static void fill_code_values(void)
{
    for (int c = 0; c < 0x7F; ++c)
        g_code_value[c] = e4m3_code_value_eq(c);
}
static double e4m3_code_value(int c) { return g_code_value[c]; }

/* The 126 positive values in code order 0x01..0x7E. */
ORACLE_API void fp8attn_oracle_e4m3_table(double out[126])
{
    for (int c = 1; c <= 0x7E; ++c)
        out[c - 1] = e4m3_code_value(c);
}

ORACLE_API double fp8attn_oracle_e4m3_value(uint8_t code)
{
    int c = code & 0x7F;
    if (c == 0x7F)
        return NAN;
    double v = e4m3_code_value(c);
    return (code & 0x80) ? -v : v;
}

/*
 * Round-to-nearest-even onto {0} U table, saturating at 448 (reading R6/R7:
 * ties go to the even code, which is what "round-to-nearest" means on the
 * hardware cast the paper's kernels use; x = 2^-10 is the tie between 0 and
 * 2^-9 and goes to 0; "values below 2^-10 -> 0").
 */
static uint8_t round_e4m3_pos(double x)
{
    if (!(x > 0.0))
        return 0;
    if (x >= 448.0)
        return 0x7E;                              /* satfinite, reading R22 */
    int lo = 0;                                   /* largest code with value <= x */
    for (int c = 1; c <= 0x7E; ++c) {
        if (e4m3_code_value(c) <= x)
            lo = c;
        else
            break;
    }
    int hi = lo + 1;                              /* lo < 0x7E because x < 448 */
    double dlo = x - e4m3_code_value(lo);
    double dhi = e4m3_code_value(hi) - x;
    if (dlo < dhi)
        return (uint8_t)lo;
    if (dhi < dlo)
        return (uint8_t)hi;
    return (uint8_t)((lo & 1) ? hi : lo);         /* tie: even code */
}

ORACLE_API uint8_t fp8attn_oracle_round_e4m3(float x)
{
    if (isnan(x))
        return 0x7F;
    if (signbit(x))
        return (uint8_t)(0x80 | round_e4m3_pos(-(double)x));
    return round_e4m3_pos((double)x);
}

/*
 * dp(S), Def. 1 / Eq. 17 with reading R10: the largest gap between consecutive
 * points a < b of {0} U E4M3+ with a < S, divided by S; for S > 448 Eq. 18.
 */
ORACLE_API double fp8attn_oracle_dp(double S)
{
    if (!(S > 0.0))
        return NAN;
    if (S > 448.0) {
        double a = 32.0 / S, b = 2.0 * (1.0 - 448.0 / S);
        return a > b ? a : b;                     /* Eq. 18 */
    }
    double best = 0.0;
    for (int c = 0; c < 0x7E; ++c) {
        double a = e4m3_code_value(c), b = e4m3_code_value(c + 1);
        if (a < S && b - a > best)
            best = b - a;
    }
    return best / S;
}

/* ------------------------------------------------------------------------- */
/* Input formats                                                              */
/* ------------------------------------------------------------------------- */

enum { DT_F32 = 0, DT_BF16 = 1, DT_E4M3 = 2, DT_BF16Q_E4M3KV = 3 };

static double bf16_value(uint16_t h)
{
    uint32_t u = (uint32_t)h << 16;
    float f;
    memcpy(&f, &u, 4);
    return (double)f;
}

/*
 * Per-(b,h) slab quantisation to E4M3 (reading R16: absmax/448 per batch and
 * head; the paper calls QKV quantisation orthogonal, so this is
 * "parity unpinned by the paper").  inv = fl32(448/absmax); code =
 * RNE_E4M3(fl32(x*inv)); scale = fl32(absmax/448).  An all-zero slab gets
 * scale 1 and zero codes.
 */
ORACLE_API void fp8attn_oracle_quantize_e4m3(const float *x, uint8_t *codes, float *scales,
                                             int64_t n_slabs, int64_t slab_elems)
{
    for (int64_t s = 0; s < n_slabs; ++s) {
        const float *xs = x + s * slab_elems;
        float amax = 0.0f;
        for (int64_t e = 0; e < slab_elems; ++e) {
            float a = fabsf(xs[e]);
            if (a > amax)
                amax = a;
        }
        float inv = 1.0f, scale = 1.0f;
        if (amax > 0.0f) {
            inv = 448.0f / amax;
            scale = amax / 448.0f;
        }
        scales[s] = scale;
#pragma omp parallel for schedule(static)
        for (int64_t e = 0; e < slab_elems; ++e) {
            float y = xs[e] * inv;
            codes[s * slab_elems + e] = fp8attn_oracle_round_e4m3(y);
        }
    }
}

/* ------------------------------------------------------------------------- */
/* Attention forward                                                          */
/* ------------------------------------------------------------------------- */

typedef struct {
    int32_t in_dtype;        /* DT_* */
    int32_t block_n;         /* KV block size Bn ("typically 64 or 128") */
    int32_t n_sink;          /* number of sink keys at the start (k_sink) */
    int32_t num_splits;      /* split-KV: number of contiguous block ranges; <=1 = none */
    const int32_t *split_bounds; /* num_splits+1 block indices, [0]=0, [ns]=nb; NULL = none */
    const float *q_scale;    /* [B*Hq]  (E4M3 q), else NULL */
    const float *k_scale;    /* [B*Hkv] (E4M3 k), else NULL */
    const float *v_scale;    /* [B*Hkv] (E4M3 v), else NULL */
    int64_t n_rows;          /* number of selected rows; 0 = all B*Hq*Lq rows */
    const int64_t *rows;     /* flat row ids ((b*Hq+h)*Lq+i); NULL = all */
    /* outputs, indexed by position in the row selection; any may be NULL */
    double *ref_out;         /* [n,d]  unquantised FP64 softmax attention (reading R17) */
    float *row_max;          /* [n]    final m */
    double *row_sum;         /* [n]    final l (relative to final m, not multiplied by S) */
    uint8_t *p_codes;        /* [n,Lk] E4M3 code of every visible P, 0xFF = masked */
    uint32_t *row_uf_sink;   /* [n]    per-row underflow count, sink block */
    uint32_t *row_uf_other;  /* [n]    per-row underflow count, other blocks */
    uint64_t uf_sink_block;  /* out: total underflows in the block(s) holding sink keys */
    uint64_t uf_other_blocks;/* out: total underflows elsewhere */
    uint64_t n_nonsink_visible; /* out: number of visible non-sink (row,key) pairs */
    int32_t n_threads;       /* 0 = OpenMP default; out: threads used */
    int32_t scale_mode;      /* 0: static S (Alg. 1); 1: per-(row, block) power-of-two scale
                                S_j = 2^k_j (reading R26), S is not used */
    const int32_t *sink_pos; /* n_sink key indices (ascending) of the sink keys, or NULL: the
                                first n_sink keys (reading R27) */
} fp8attn_oracle_opts;

/* Largest exponent the dynamic scale takes (reading R26). */
#define DYN_K_MAX 30

static int is_sink_key(const fp8attn_oracle_opts *o, int j)
{
    if (!o->sink_pos)
        return j < o->n_sink;
    for (int s = 0; s < o->n_sink; ++s)
        if (o->sink_pos[s] == j)
            return 1;
    return 0;
}

/* Does block [j0, j0 + Bn) hold a sink key? */
static int is_sink_block(const fp8attn_oracle_opts *o, int j0, int Bn)
{
    if (!o->sink_pos)
        return j0 < o->n_sink;
    for (int s = 0; s < o->n_sink; ++s)
        if (o->sink_pos[s] >= j0 && o->sink_pos[s] < j0 + Bn)
            return 1;
    return 0;
}

/*
 * Block visited at step `step` of the range [b0, b1) (Alg. 1 line 2).
 *   order 0: forward b0 .. b1-1.   order 1: reverse b1-1 .. b0.
 *   order 2: "sink blocks last" (reading R27): the blocks that hold no sink
 *            key in descending order, then the blocks that hold one, in descending order.
 *            With the sink keys in block 0 this is order 1.
 */
static int block_at(const fp8attn_oracle_opts *o, int order, int b0, int b1, int step, int Bn)
{
    if (order == 0)
        return b0 + step;
    if (order == 1)
        return b1 - 1 - step;
    int seen = 0;
    for (int pass = 0; pass < 2; ++pass)          /* pass 0: non-sink blocks, pass 1: sink blocks */
        for (int b = b1 - 1; b >= b0; --b)
            if (is_sink_block(o, b * Bn, Bn) == pass) {
                if (seen == step)
                    return b;
                ++seen;
            }
    return -1;
}

typedef struct {
    const void *q, *k, *v;
    int B, Hq, Hkv, Lq, Lk, d, causal, kv_order, mode;
    float S;
    const fp8attn_oracle_opts *o;
} problem;

static void load_row(const problem *P, const void *base, int dtype_is_q, int64_t slab,
                     int64_t row, int64_t L, double *dst)
{
    const int d = P->d;
    int dt = P->o->in_dtype;
    int64_t off = (slab * L + row) * d;
    if (dt == DT_BF16Q_E4M3KV)
        dt = dtype_is_q ? DT_BF16 : DT_E4M3;
    if (dt == DT_F32) {
        const float *p = (const float *)base + off;
        for (int t = 0; t < d; ++t) dst[t] = (double)p[t];
    } else if (dt == DT_BF16) {
        const uint16_t *p = (const uint16_t *)base + off;
        for (int t = 0; t < d; ++t) dst[t] = bf16_value(p[t]);
    } else {
        const uint8_t *p = (const uint8_t *)base + off;
        for (int t = 0; t < d; ++t) dst[t] = fp8attn_oracle_e4m3_value(p[t]);
    }
}

/* One query row: Alg. 1 over the blocks of each split, then the combine. */
static void attend_row(const problem *P, int64_t rid, int64_t sel,
                       const double *Kd, const double *Vd, /* dequantised K,V of this kv head: [Lk,d] */
                       double *out, uint64_t *uf_sink, uint64_t *uf_other, uint64_t *n_vis)
{
    const fp8attn_oracle_opts *o = P->o;
    const int d = P->d, Lk = P->Lk, Lq = P->Lq, Bn = o->block_n;
    const int i = (int)(rid % Lq);
    const int64_t bh = rid / Lq;                   /* b*Hq + h */
    const int nb = (Lk + Bn - 1) / Bn;
    const float Sf = (P->mode == 0) ? 1.0f : P->S; /* mode 0: no cast, S ignored */
    const double Sd = (double)Sf;
    const double rsd = 1.0 / sqrt((double)d);

    double *qv = (double *)malloc(sizeof(double) * d);
    load_row(P, P->q, 1, bh, i, Lq, qv);
    if (o->in_dtype == DT_E4M3) {
        for (int t = 0; t < d; ++t) qv[t] *= (double)o->q_scale[bh];
    } else if (o->in_dtype == DT_BF16Q_E4M3KV) {
        /* decode: q is BF16 in memory and is quantised to E4M3 per (b,hq) slab
         * before use (reading R24 / DESIGN.md); the input VALUES of the method are
         * the post-quantisation ones. */
        float *qf = (float *)malloc(sizeof(float) * (size_t)Lq * d);
        uint8_t *qc = (uint8_t *)malloc((size_t)Lq * d);
        float qs;
        double *tmp = (double *)malloc(sizeof(double) * d);
        for (int r = 0; r < Lq; ++r) {
            load_row(P, P->q, 1, bh, r, Lq, tmp);
            for (int t = 0; t < d; ++t) qf[(size_t)r * d + t] = (float)tmp[t];
        }
        fp8attn_oracle_quantize_e4m3(qf, qc, &qs, 1, (int64_t)Lq * d);
        for (int t = 0; t < d; ++t)
            qv[t] = fp8attn_oracle_e4m3_value(qc[(size_t)i * d + t]) * (double)qs;
        free(qf); free(qc); free(tmp);
    }

    /* visible keys: j <= jmax (reading R15: bottom-right aligned causal mask) */
    int jmax = Lk - 1;
    if (P->causal) {
        int64_t lim = (int64_t)i + (int64_t)Lk - (int64_t)Lq;
        jmax = lim < Lk - 1 ? (int)lim : Lk - 1;
    }

    uint8_t *codes_out = o->p_codes ? o->p_codes + (size_t)sel * Lk : NULL;
    if (codes_out) memset(codes_out, 0xFF, (size_t)Lk);

    /* logits of every visible key, FP64 then FP32 (Alg. 1 line 3) */
    double *z64 = (double *)malloc(sizeof(double) * (size_t)(jmax + 1 > 0 ? jmax + 1 : 1));
    float *z = (float *)malloc(sizeof(float) * (size_t)(jmax + 1 > 0 ? jmax + 1 : 1));
    for (int j = 0; j <= jmax; ++j) {
        const double *kr = Kd + (size_t)j * d;
        double acc = 0.0;
        for (int t = 0; t < d; ++t) acc += qv[t] * kr[t];
        z64[j] = acc * rsd;
        z[j] = (float)z64[j];
    }

    /* unquantised FP64 reference: plain softmax(z64) . V (reading R17) */
    if (o->ref_out) {
        double *ref = o->ref_out + (size_t)sel * d;
        for (int t = 0; t < d; ++t) ref[t] = 0.0;
        if (jmax >= 0) {
            double mx = z64[0];
            for (int j = 1; j <= jmax; ++j) if (z64[j] > mx) mx = z64[j];
            double den = 0.0;
            for (int j = 0; j <= jmax; ++j) {
                double e = exp(z64[j] - mx);
                den += e;
                const double *vr = Vd + (size_t)j * d;
                for (int t = 0; t < d; ++t) ref[t] += e * vr[t];
            }
            for (int t = 0; t < d; ++t) ref[t] /= den;
        }
    }

    int ns = (o->num_splits > 1 && o->split_bounds) ? o->num_splits : 1;
    float *ms = (float *)malloc(sizeof(float) * ns);
    double *ls = (double *)malloc(sizeof(double) * ns);
    double *Os = (double *)calloc((size_t)ns * d, sizeof(double));
    uint32_t my_sink = 0, my_other = 0;
    uint64_t my_vis = 0;

    for (int s = 0; s < ns; ++s) {
        int b0 = (ns > 1) ? o->split_bounds[s] : 0;
        int b1 = (ns > 1) ? o->split_bounds[s + 1] : nb;
        float m = -INFINITY;                       /* Alg. 1 line 1 */
        double l = 0.0;
        double *O = Os + (size_t)s * d;
        for (int step = 0; step < b1 - b0; ++step) {
            int blk = block_at(o, P->kv_order, b0, b1, step, Bn);       /* line 2 */
            int j0 = blk * Bn;
            int j1 = j0 + Bn < Lk ? j0 + Bn : Lk;
            if (j1 - 1 > jmax) j1 = jmax + 1;
            if (j0 >= j1) continue;                /* block fully masked for this row */
            float m_loc = z[j0];                   /* line 4 */
            for (int j = j0 + 1; j < j1; ++j) if (z[j] > m_loc) m_loc = z[j];
            float m_new = m > m_loc ? m : m_loc;   /* line 5 */
            double alpha = isinf(m) ? 0.0 : exp((double)m - (double)m_new);   /* line 6 */
            double psum = 0.0;
            for (int t = 0; t < d; ++t) O[t] *= alpha;
            int sink_blk = is_sink_block(o, j0, Bn);
            /* scale of this block.  Static: S.  Dynamic (reading R26): the largest power of two
             * 2^k with 2^k * max_j p_j <= 448, where max_j p_j = exp(m_loc - m_new); taken in FP32
             * in base-2 units, k = floor(log2(448) + (m_new - m_loc) log2(e)), capped at DYN_K_MAX.
             * O then holds true (unscaled) values: each block's contribution is divided by its own
             * 2^k, which is exact (Prop. 5). */
            float Sblk = Sf;
            if (o->scale_mode == 1 && P->mode != 0) {
                float g2 = (m_new - m_loc) * 1.44269504088896340736f;
                int kexp = (int)floorf(g2 + 8.80735492205760410744f);
                if (kexp > DYN_K_MAX) kexp = DYN_K_MAX;
                Sblk = ldexpf(1.0f, kexp);
            }
            const double Sblk_d = (o->scale_mode == 1 && P->mode != 0) ? (double)Sblk : 1.0;
            for (int j = j0; j < j1; ++j) {
                float p = (float)exp((double)z[j] - (double)m_new);           /* line 7 */
                psum += (double)p;
                double pq;
                if (P->mode == 0) {
                    pq = (double)p;                /* no-cast reference */
                } else {
                    float x = p * Sblk;            /* line 9: xS in FP32 */
                    uint8_t c = fp8attn_oracle_round_e4m3(x);
                    pq = e4m3_code_value(c) / Sblk_d;
                    if (codes_out) codes_out[j] = c;
                    if (!is_sink_key(o, j)) {
                        ++my_vis;
                        if (c == 0) { if (sink_blk) ++my_sink; else ++my_other; }
                    }
                }
                const double *vr = Vd + (size_t)j * d;
                for (int t = 0; t < d; ++t) O[t] += pq * vr[t];              /* line 10 */
            }
            l = alpha * l + psum;                  /* line 8: pre-cast P */
            m = m_new;
        }
        ms[s] = m;
        ls[s] = l;
    }

    /* combine over splits (log-sum-exp merge; reading R14), then line 12 */
    float mfin = -INFINITY;
    for (int s = 0; s < ns; ++s) if (ms[s] > mfin) mfin = ms[s];
    double lfin = 0.0;
    for (int t = 0; t < d; ++t) out[t] = 0.0;
    for (int s = 0; s < ns; ++s) {
        if (isinf(ms[s])) continue;
        double w = exp((double)ms[s] - (double)mfin);
        lfin += w * ls[s];
        for (int t = 0; t < d; ++t) out[t] += w * Os[(size_t)s * d + t];
    }
    if (lfin > 0.0)
        for (int t = 0; t < d; ++t) out[t] /= ((o->scale_mode == 1 ? 1.0 : Sd) * lfin);
    if (o->row_max) o->row_max[sel] = mfin;
    if (o->row_sum) o->row_sum[sel] = lfin;
    if (o->row_uf_sink) o->row_uf_sink[sel] = my_sink;
    if (o->row_uf_other) o->row_uf_other[sel] = my_other;
    *uf_sink += my_sink;
    *uf_other += my_other;
    *n_vis += my_vis;

    free(qv); free(z64); free(z); free(ms); free(ls); free(Os);
}

/*
 * fp8attn_oracle_fwd: q,o [B,Hq,Lq,d]; k,v [B,Hkv,Lk,d]; host pointers; out is FP64
 * [n,d] over the row selection.  mode 0 = no-cast, 1 = P-cast isolation, 2 = production
 * FP8 (same arithmetic as mode 1 on dequantised inputs).  kv_order 0 = forward, 1 = reverse.
 * Returns 0, or a negative code on a bad argument.
 */
ORACLE_API int fp8attn_oracle_fwd(const void *q, const void *k, const void *v, double *out,
                                  int B, int Hq, int Hkv, int Lq, int Lk, int d, int causal,
                                  float S, int kv_order, int mode, fp8attn_oracle_opts *opts)
{
    if (!q || !k || !v || !out || !opts) return -1;
    if (B < 1 || Hq < 1 || Hkv < 1 || Lq < 1 || Lk < 1 || d < 1) return -2;
    if (Hq % Hkv) return -3;
    if (!(S > 0.0f) || isinf(S)) return -4;
    if (mode < 0 || mode > 2 || kv_order < 0 || kv_order > 2) return -5;
    if (opts->scale_mode != 0 && opts->scale_mode != 1) return -5;
    if (opts->block_n < 1 || opts->in_dtype < 0 || opts->in_dtype > 3) return -6;
    if ((opts->in_dtype == DT_E4M3 && (!opts->q_scale || !opts->k_scale || !opts->v_scale)) ||
        (opts->in_dtype == DT_BF16Q_E4M3KV && (!opts->k_scale || !opts->v_scale)))
        return -7;

    problem P = { q, k, v, B, Hq, Hkv, Lq, Lk, d, causal, kv_order, mode, S, opts };
    const int64_t total = (int64_t)B * Hq * Lq;
    const int64_t n = (opts->rows && opts->n_rows > 0) ? opts->n_rows : total;
    const int group = Hq / Hkv;
    const int kv_e4m3 = (opts->in_dtype == DT_E4M3 || opts->in_dtype == DT_BF16Q_E4M3KV);

    /* group the selected rows by kv head */
    const int64_t n_kvh = (int64_t)B * Hkv;
    int64_t *head_cnt = (int64_t *)calloc((size_t)n_kvh + 1, sizeof(int64_t));
    int64_t *order = (int64_t *)malloc(sizeof(int64_t) * (size_t)n);
    for (int64_t r = 0; r < n; ++r) {
        int64_t rid = opts->rows ? opts->rows[r] : r;
        if (rid < 0 || rid >= total) { free(head_cnt); free(order); return -8; }
        int64_t bh = rid / Lq;
        head_cnt[(bh / Hq) * Hkv + (bh % Hq) / group + 1]++;
    }
    int64_t n_active = 0;
    for (int64_t h = 0; h < n_kvh; ++h) {
        if (head_cnt[h + 1]) ++n_active;
        head_cnt[h + 1] += head_cnt[h];
    }
    {
        int64_t *fill = (int64_t *)malloc(sizeof(int64_t) * (size_t)n_kvh);
        memcpy(fill, head_cnt, sizeof(int64_t) * (size_t)n_kvh);
        for (int64_t r = 0; r < n; ++r) {
            int64_t rid = opts->rows ? opts->rows[r] : r;
            int64_t bh = rid / Lq;
            order[fill[(bh / Hq) * Hkv + (bh % Hq) / group]++] = r;
        }
        free(fill);
    }
    int nthreads = 1;
#ifdef _OPENMP
    if (opts->n_threads > 0) omp_set_num_threads(opts->n_threads);
    nthreads = omp_get_max_threads();
#endif
    /* many heads: one thread per kv head; few heads: threads share a head's rows */
    const int par_heads = (n_active >= nthreads);
    uint64_t tot_sink = 0, tot_other = 0, tot_vis = 0;
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : tot_sink, tot_other, tot_vis) if (par_heads)
    for (int64_t kvh = 0; kvh < n_kvh; ++kvh) {
        const int64_t r0 = head_cnt[kvh], r1 = head_cnt[kvh + 1];
        if (r0 == r1) continue;
        /* dequantised K, V of this kv head (values only, none of the method's arithmetic) */
        double *Kd = (double *)malloc(sizeof(double) * (size_t)Lk * d);
        double *Vd = (double *)malloc(sizeof(double) * (size_t)Lk * d);
#pragma omp parallel for schedule(static) if (!par_heads)
        for (int j = 0; j < Lk; ++j) {
            load_row(&P, k, 0, kvh, j, Lk, Kd + (size_t)j * d);
            load_row(&P, v, 0, kvh, j, Lk, Vd + (size_t)j * d);
            if (kv_e4m3) {
                for (int t = 0; t < d; ++t) {
                    Kd[(size_t)j * d + t] *= (double)opts->k_scale[kvh];
                    Vd[(size_t)j * d + t] *= (double)opts->v_scale[kvh];
                }
            }
        }
        uint64_t hs = 0, ho = 0, hv = 0;
#pragma omp parallel for schedule(dynamic, 4) reduction(+ : hs, ho, hv) if (!par_heads)
        for (int64_t x = r0; x < r1; ++x) {
            int64_t r = order[x];
            int64_t rid = opts->rows ? opts->rows[r] : r;
            uint64_t a = 0, b = 0, c = 0;
            attend_row(&P, rid, r, Kd, Vd, out + (size_t)r * d, &a, &b, &c);
            hs += a; ho += b; hv += c;
        }
        tot_sink += hs; tot_other += ho; tot_vis += hv;
        free(Kd); free(Vd);
    }
    free(head_cnt); free(order);
    opts->uf_sink_block = tot_sink;
    opts->uf_other_blocks = tot_other;
    opts->n_nonsink_visible = tot_vis;
    opts->n_threads = nthreads;
    return 0;
}

ORACLE_API int fp8attn_oracle_opts_size(void) { return (int)sizeof(fp8attn_oracle_opts); }
