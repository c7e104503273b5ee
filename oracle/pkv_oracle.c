/*
 * pkv_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, FP64 CPU oracle for single-query GQA decode attention over a paged KV cache
 * (arxiv/paper_2606_26666, "PersistentKV").  It shares no code with the CUDA path under
 * paper_2606_26666_b200/ and must never be imported, linked or executed by it.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 *
 * What it computes, written out as the paper's definition (no blocking, no online softmax,
 * no reordering):
 *
 *   pkv_oracle_attention      PAPER.md:39 Eq. (1) with the GQA map of PAPER.md:42 (reading A2:
 *                             KV head g serves query heads [g*G, (g+1)*G), G = Hq/Hkv) and the
 *                             block-table gather of PAPER.md:46-50 (token j of row i lives in
 *                             physical page block_table[i][j / P], slot j % P).  Two-pass softmax:
 *                             all scores, their max, the sum of exponentials, the weighted sum.
 *   pkv_oracle_split_states   PAPER.md:56: per split, m_s = max_j x_j, l_s = sum_j exp(x_j - m_s),
 *                             a_s = sum_j exp(x_j - m_s) v_j over the split's token range;
 *                             an empty range gives the neutral state (-inf, 0, 0).
 *   pkv_oracle_merge          PAPER.md:60-61: m = max_s m_s, l = sum_s exp(m_s - m) l_s,
 *                             a = sum_s exp(m_s - m) a_s, O = a / l.
 *
 * Readings: A1 layout via explicit element strides (page, token, head; d is
 * unit-stride); A4 the scale is passed in (the tests pass (double)(float)(1/sqrt(d)));
 * A9 a row with N_i = 0 gives O = 0 and LSE = -inf; A10 tokens >= N_i and block-table entries
 * past ceil(N_i / P) are never read.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): brute-force dense numpy attention on tiny
 * inputs, page-pool permutation invariance, split-count invariance, K = 0 => mean(V),
 * dominant key => V of that token, N = 1 and N = 2 closed forms.
 *
 * FP16 is decoded by the bit decoder below (no cuda_fp16.h, no compiler half type).
 *
 * One-byte KV ("dequantization-aware paged decode", PAPER.md:271 future work; DESIGN.md
 * reading A28): pkv_oracle_attention_q8 is Eq. (1) on k_j = k_scale[g] * dec(K bytes),
 * v_j = v_scale[g] * dec(V bytes), one scale per KV head; dec = OCP FP8 E4M3 ("fn": no infinities,
 * S.1111.111 = NaN, largest finite 448) or two's-complement INT8.  The byte decoder is pinned on all 256 patterns against
 * torch.float8_e4m3fn and against closed forms (tests/test_oracle_pins.py).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* IEEE 754 binary16 -> double, exact. */
static double half_bits_to_double(uint16_t h)
{
    int sign = (h >> 15) & 1;
    int expo = (h >> 10) & 0x1f;
    int mant = h & 0x3ff;
    double v;
    if (expo == 0) {
        v = ldexp((double)mant, -24);               /* subnormal or zero */
    } else if (expo == 31) {
        v = mant ? NAN : INFINITY;
    } else {
        v = ldexp((double)(mant + 1024), expo - 25); /* (1 + mant/1024) * 2^(expo-15) */
    }
    return sign ? -v : v;
}

/* OCP FP8 E4M3 (fn) -> double, exact: 1 sign, 4 exponent (bias 7), 3 mantissa bits. */
static double e4m3_bits_to_double(uint8_t b)
{
    int sign = (b >> 7) & 1;
    int expo = (b >> 3) & 0xf;
    int mant = b & 0x7;
    double v;
    if (expo == 0) {
        v = ldexp((double)mant, -9);                 /* subnormal or zero: mant/8 * 2^-6 */
    } else if (expo == 15 && mant == 7) {
        v = NAN;                                     /* the only non-finite code */
    } else {
        v = ldexp((double)(mant + 8), expo - 10);    /* (1 + mant/8) * 2^(expo-7) */
    }
    return sign ? -v : v;
}

typedef struct {
    int B, Hq, Hkv, d, page_size, max_pages;
    int64_t stride_page, stride_token, stride_head;
    const uint16_t *q, *k_cache, *v_cache;
    const int32_t *block_table, *seq_lens;
    double scale;
    /* one-byte caches (NULL: FP16 caches above are used) and their per-KV-head scales */
    const uint8_t *k8, *v8;
    const double *k_scale, *v_scale;
    int kv_kind;   /* 1: OCP FP8 E4M3 bytes, 2: two's-complement INT8 bytes */
} oracle_problem;

static double byte_to_double(int kv_kind, uint8_t b)
{
    return kv_kind == 2 ? (double)(int8_t)b : e4m3_bits_to_double(b);
}

/* channel c of the K (V) row at element offset off, KV head g, as a real number */
static double k_elem(const oracle_problem *p, int64_t off, int c, int g)
{
    if (p->k8) return p->k_scale[g] * byte_to_double(p->kv_kind, p->k8[off + c]);
    return half_bits_to_double(p->k_cache[off + c]);
}
static double v_elem(const oracle_problem *p, int64_t off, int c, int g)
{
    if (p->v8) return p->v_scale[g] * byte_to_double(p->kv_kind, p->v8[off + c]);
    return half_bits_to_double(p->v_cache[off + c]);
}

/* address (in elements) of token j of row i, KV head g: the page accessor of PAPER.md:50 */
static int64_t token_offset(const oracle_problem *p, int i, int64_t j, int g)
{
    int64_t logical_page = j / p->page_size;
    int64_t slot = j % p->page_size;
    int64_t physical_page = p->block_table[(int64_t)i * p->max_pages + logical_page];
    return physical_page * p->stride_page + slot * p->stride_token + (int64_t)g * p->stride_head;
}

/* scores x_j = scale * <q_{i,h}, k_{i,j}> for j in [j0, j1) into x[0 .. j1-j0) */
static void scores_range(const oracle_problem *p, int i, int h, int64_t j0, int64_t j1, double *x)
{
    int G = p->Hq / p->Hkv;
    int g = h / G;
    const uint16_t *qv = p->q + ((int64_t)i * p->Hq + h) * p->d;
    for (int64_t j = j0; j < j1; ++j) {
        int64_t off = token_offset(p, i, j, g);
        double dot = 0.0;
        for (int c = 0; c < p->d; ++c)
            dot += half_bits_to_double(qv[c]) * k_elem(p, off, c, g);
        x[j - j0] = p->scale * dot;
    }
}

/* state of the token range [j0, j1): m, l, a[d] exactly as PAPER.md:56 (two passes) */
static void range_state(const oracle_problem *p, int i, int h, int64_t j0, int64_t j1,
                        double *x_scratch, double *m_out, double *l_out, double *a_out)
{
    int G = p->Hq / p->Hkv;
    int g = h / G;
    int d = p->d;
    for (int c = 0; c < d; ++c) a_out[c] = 0.0;
    if (j1 <= j0) { *m_out = -INFINITY; *l_out = 0.0; return; }   /* neutral state */
    scores_range(p, i, h, j0, j1, x_scratch);
    double m = -INFINITY;
    for (int64_t j = j0; j < j1; ++j) if (x_scratch[j - j0] > m) m = x_scratch[j - j0];
    double l = 0.0;
    for (int64_t j = j0; j < j1; ++j) {
        double w = exp(x_scratch[j - j0] - m);
        l += w;
        int64_t off = token_offset(p, i, j, g);
        for (int c = 0; c < d; ++c) a_out[c] += w * v_elem(p, off, c, g);
    }
    *m_out = m; *l_out = l;
}

static int attention_impl(const oracle_problem *pp, double *out, double *lse, int num_threads);

/* Eq. (1).  out [B,Hq,d] f64, lse [B,Hq] f64 (may be NULL).  Returns 0, or -1 on bad arguments. */
int pkv_oracle_attention(int B, int Hq, int Hkv, int d, int page_size, int max_pages,
                         int64_t stride_page, int64_t stride_token, int64_t stride_head,
                         const uint16_t *q, const uint16_t *k_cache, const uint16_t *v_cache,
                         const int32_t *block_table, const int32_t *seq_lens, double scale,
                         double *out, double *lse, int num_threads)
{
    if (B < 0 || Hkv <= 0 || Hq % Hkv || d <= 0 || page_size <= 0) return -1;
    oracle_problem p = { B, Hq, Hkv, d, page_size, max_pages, stride_page, stride_token, stride_head,
                         q, k_cache, v_cache, block_table, seq_lens, scale, NULL, NULL, NULL, NULL, 0 };
    return attention_impl(&p, out, lse, num_threads);
}

/* The same on one-byte caches with one scale per KV head (reading A28): kv_kind 1 = FP8 E4M3,
 * 2 = INT8; strides in elements = bytes. */
int pkv_oracle_attention_q8(int B, int Hq, int Hkv, int d, int page_size, int max_pages,
                            int64_t stride_page, int64_t stride_token, int64_t stride_head,
                            const uint16_t *q, const uint8_t *k8, const uint8_t *v8,
                            const double *k_scale, const double *v_scale, int kv_kind,
                            const int32_t *block_table, const int32_t *seq_lens, double scale,
                            double *out, double *lse, int num_threads)
{
    if (B < 0 || Hkv <= 0 || Hq % Hkv || d <= 0 || page_size <= 0 || !k8 || !v8 || !k_scale || !v_scale) return -1;
    if (kv_kind != 1 && kv_kind != 2) return -1;
    oracle_problem p = { B, Hq, Hkv, d, page_size, max_pages, stride_page, stride_token, stride_head,
                         q, NULL, NULL, block_table, seq_lens, scale, k8, v8, k_scale, v_scale, kv_kind };
    return attention_impl(&p, out, lse, num_threads);
}

static int attention_impl(const oracle_problem *pp, double *out, double *lse, int num_threads)
{
    oracle_problem p = *pp;
    int B = p.B, Hq = p.Hq, Hkv = p.Hkv, d = p.d;
    const int32_t *seq_lens = p.seq_lens;
    int G = Hq / Hkv;
    int units = B * Hkv;
    int failed = 0;
#ifdef _OPENMP
    if (num_threads > 0) omp_set_num_threads(num_threads);
#else
    (void)num_threads;
#endif
    #pragma omp parallel for schedule(dynamic, 1)
    for (int u = 0; u < units; ++u) {
        int i = u / Hkv, g = u % Hkv;
        int64_t N = seq_lens[i];
        double *x = (double *)malloc(sizeof(double) * (size_t)(N > 0 ? N : 1));
        if (!x) { failed = 1; continue; }
        for (int hh = 0; hh < G; ++hh) {
            int h = g * G + hh;
            double *o = out + ((int64_t)i * Hq + h) * d;
            double m, l;
            range_state(&p, i, h, 0, N, x, &m, &l, o);
            if (N <= 0) {                                       /* reading A9 */
                for (int c = 0; c < d; ++c) o[c] = 0.0;
                if (lse) lse[(int64_t)i * Hq + h] = -INFINITY;
            } else {
                for (int c = 0; c < d; ++c) o[c] /= l;
                if (lse) lse[(int64_t)i * Hq + h] = m + log(l);
            }
        }
        free(x);
    }
    return failed ? -2 : 0;
}

/* PAPER.md:56 for a list of tasks (row, kvh, split, t_begin, t_end), t_* in tiles of tile_tokens
 * tokens; token range = [t_begin*Tt, min(t_end*Tt, N_row)).  Outputs per task and per head of
 * the group: m [num_tasks][G], l [num_tasks][G], a [num_tasks][G][d]. */
int pkv_oracle_split_states(int B, int Hq, int Hkv, int d, int page_size, int max_pages,
                            int64_t stride_page, int64_t stride_token, int64_t stride_head,
                            const uint16_t *q, const uint16_t *k_cache, const uint16_t *v_cache,
                            const int32_t *block_table, const int32_t *seq_lens, double scale,
                            const int32_t *tasks, int num_tasks, int tile_tokens,
                            double *m_out, double *l_out, double *a_out, int num_threads)
{
    if (B < 0 || Hkv <= 0 || Hq % Hkv || d <= 0 || page_size <= 0 || tile_tokens <= 0) return -1;
    oracle_problem p = { B, Hq, Hkv, d, page_size, max_pages, stride_page, stride_token, stride_head,
                         q, k_cache, v_cache, block_table, seq_lens, scale, NULL, NULL, NULL, NULL, 0 };
    int G = Hq / Hkv;
    int failed = 0;
#ifdef _OPENMP
    if (num_threads > 0) omp_set_num_threads(num_threads);
#else
    (void)num_threads;
#endif
    #pragma omp parallel for schedule(dynamic, 1)
    for (int t = 0; t < num_tasks; ++t) {
        const int32_t *task = tasks + (int64_t)t * 5;
        int i = task[0], g = task[1];
        int64_t N = seq_lens[i];
        int64_t j0 = (int64_t)task[3] * tile_tokens;
        int64_t j1 = (int64_t)task[4] * tile_tokens;
        if (j1 > N) j1 = N;
        if (j0 > j1) j0 = j1;
        double *x = (double *)malloc(sizeof(double) * (size_t)(j1 - j0 > 0 ? j1 - j0 : 1));
        if (!x) { failed = 1; continue; }
        for (int hh = 0; hh < G; ++hh) {
            int h = g * G + hh;
            range_state(&p, i, h, j0, j1, x, m_out + (int64_t)t * G + hh, l_out + (int64_t)t * G + hh,
                        a_out + ((int64_t)t * G + hh) * d);
        }
        free(x);
    }
    return failed ? -2 : 0;
}

/* PAPER.md:60-61 for one (row, query head): n split states -> O[d], LSE.
 * All-neutral input (m = -inf everywhere) gives O = 0, LSE = -inf (reading A9). */
int pkv_oracle_merge(int n, int d, const double *m_s, const double *l_s, const double *a_s,
                     double *out, double *lse)
{
    double m = -INFINITY;
    for (int s = 0; s < n; ++s) if (m_s[s] > m) m = m_s[s];
    for (int c = 0; c < d; ++c) out[c] = 0.0;
    if (n <= 0 || m == -INFINITY) { if (lse) *lse = -INFINITY; return 0; }
    double l = 0.0;
    for (int s = 0; s < n; ++s) {
        if (m_s[s] == -INFINITY) continue;          /* exp(-inf) = 0: neutral states drop out */
        double w = exp(m_s[s] - m);
        l += w * l_s[s];
        for (int c = 0; c < d; ++c) out[c] += w * a_s[(int64_t)s * d + c];
    }
    for (int c = 0; c < d; ++c) out[c] /= l;
    if (lse) *lse = m + log(l);
    return 0;
}

int pkv_oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* exposed so a test can pin the FP16 decoder against numpy's float16 on all 65536 patterns */
double pkv_oracle_half_to_double(uint16_t h) { return half_bits_to_double(h); }
/* ... and the E4M3 decoder against torch.float8_e4m3fn on all 256 */
double pkv_oracle_e4m3_to_double(uint8_t b) { return e4m3_bits_to_double(b); }
