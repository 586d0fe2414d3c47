/*
 * oracle/decode_attn_oracle.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of what the decode-attention hot path
 * computes.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this.  It shares no code, header, table or
 * helper with paper_2605_30842_b200/csrc/ (the CUDA path) and never imports it.
 *
 * What it states (citations are /root/reference/PAPER.md lines, "P:Lnn"):
 *   - P:L49 (§2.2): Q in R^{l x h_q x d_h}, K,V in R^{l x h_kv x d_h}; GQA
 *     (fn. 1): h_q query heads share h_kv KV heads.
 *   - P:L61 (§2.2): at decode step t the cache is [K_cache^(t-1); K^(t)],
 *     [V_cache^(t-1); V^(t)] (typo in the paper's first bracket corrected,
 *     DESIGN.md reading R3) and the one new query attends the WHOLE cache.
 *   - The attention function itself is never written in the paper; it is the
 *     standard scaled-dot-product softmax (reading R1):
 *         s_t   = softmax_scale * sum_d q[d] * k_t[d]
 *         out   = sum_t softmax(s)_t * v_t,   lse = log sum_t exp(s_t)
 *   - Paged cache (PagedAttention is only named): token t of sequence b
 *     lives in physical page block_table[b][t / page_size], slot t % page_size
 *     (reading R5 fixes the layout [page, slot, kv_head, d]).
 *   - GQA map: query head h reads KV head h / (h_q / h_kv) (reading R4).
 *
 * Structure on purpose unlike the GPU path: two passes (max, then sums),
 * logical-order traversal, no tiling, no online rescale, no splits, fp64
 * everywhere; bf16 inputs are widened exactly.  OpenMP only across independent
 * (b, h) rows, so 1-thread and N-thread results are bit-identical.
 *
 * Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): O1..O16 of
 * L=1 returns V; identical keys give mean(V); two-key logistic;
 * constant V; linearity in V; key-shift invariance; +80 logit one-hot; page
 * permutation bit-identity; GQA convention; split/LSE-merge invariance (pins
 * oracle_lse_merge and oracle_decode_attn_partial); tail-poison independence;
 * brute-force dense numpy fp64; torch CPU fp64 SDPA; lse closed form.
 * oracle_decode_attn_window: W1..W5 (window >= L is the full result bit for bit; window 1 returns
 * the last V; equals full attention over a cache compacted to the kept tokens; masked tokens'
 * contents are irrelevant; brute-force dense masked softmax).
 * oracle_decode_attn_fp8 / oracle_e4m3_decode: F1..F6 (tests/test_oracle_fp8_pins.py: the 256-entry
 * decode table vs the format's published values and vs torch's float8_e4m3fn cast; equals the pinned
 * bf16 oracle on a cache whose values both formats hold exactly; L = 1 closed form; scale
 * linearity; tail / unused-page poison independence; brute-force dense numpy fp64).
 * oracle_e4m3_encode / oracle_kv_append_fp8: E1..E4, A1 (same file: inverse of the decode table; torch's cast on
 * random values and on every tie; saturation; hand-computed ties; placement, untouched bytes, page crossing, HND).
 * F7: the HND layout is a relayout of NHD (bit-identical).
 * oracle_prefill_attn: PF1..PF5 (tests/test_oracle_prefill_pins.py: q_len 1 is the decode oracle; every row equals
 * the decode oracle on the cache truncated at its position; torch causal SDPA fp64; chunked == full; brute force).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* bf16 (raw uint16 bits) -> double, exact: bf16 is the top half of an fp32. */
static double bf16_to_double(uint16_t bits)
{
    uint32_t w = ((uint32_t)bits) << 16;
    float f;
    memcpy(&f, &w, sizeof f);
    return (double)f;
}

/* Address of row (token t, kv head kvh) of sequence b in a paged pool
 * laid out [num_pages][page_size][num_kv_heads][head_dim]. */
static const uint16_t *paged_row(const uint16_t *pages, const int32_t *block_table_row,
                                 int64_t t, int kvh, int num_kv_heads, int head_dim,
                                 int page_size)
{
    int64_t pid = (int64_t)block_table_row[t / page_size];
    int64_t slot = t % page_size;
    return pages + ((pid * page_size + slot) * num_kv_heads + kvh) * (int64_t)head_dim;
}

int oracle_version(void) { return 1; }

int oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/*
 * Full decode attention.  One output row per (b, h) pair.
 *   pairs == NULL : rows are all (b, h), b-major; out is [batch*Hq][D],
 *                   lse is [batch*Hq].
 *   pairs != NULL : int32 [num_pairs][2] = (b, h); out is [num_pairs][D].
 * seq_len == 0 -> out row = +0.0, lse = -inf (reading R9).
 * Returns 0, or 1 on an invalid argument.
 */
int oracle_decode_attn(const uint16_t *q,           /* bf16 [batch][Hq][D] */
                       const uint16_t *k_pages,     /* bf16 [P][ps][Hkv][D] */
                       const uint16_t *v_pages,     /* bf16 [P][ps][Hkv][D] */
                       const int32_t *block_table,  /* [batch][max_pages_per_seq] */
                       const int32_t *seq_lens,     /* [batch] */
                       int num_q_heads, int num_kv_heads, int head_dim, int page_size,
                       float softmax_scale, double *out, double *lse, int batch,
                       int max_pages_per_seq, const int32_t *pairs, int64_t num_pairs,
                       int num_threads)
{
    if (!q || !k_pages || !v_pages || !block_table || !seq_lens || !out) return 1;
    if (num_q_heads <= 0 || num_kv_heads <= 0 || num_q_heads % num_kv_heads) return 1;
    if (head_dim <= 0 || page_size <= 0 || batch <= 0) return 1;
    const int G = num_q_heads / num_kv_heads;
    const int D = head_dim;
    const int64_t rows = pairs ? num_pairs : (int64_t)batch * num_q_heads;
    const double scale = (double)softmax_scale; /* the fp32 argument, widened (R7) */
#ifdef _OPENMP
    if (num_threads <= 0) num_threads = omp_get_max_threads();
#else
    (void)num_threads;
#endif

#pragma omp parallel for schedule(dynamic, 1) num_threads(num_threads)
    for (int64_t r = 0; r < rows; ++r) {
        const int b = pairs ? pairs[2 * r] : (int)(r / num_q_heads);
        const int h = pairs ? pairs[2 * r + 1] : (int)(r % num_q_heads);
        const int kvh = h / G;
        const int64_t L = seq_lens[b];
        const int32_t *bt = block_table + (int64_t)b * max_pages_per_seq;
        double *o = out + r * D;
        for (int d = 0; d < D; ++d) o[d] = 0.0;
        if (L <= 0) {
            if (lse) lse[r] = -INFINITY;
            continue;
        }
        double *qd = (double *)malloc(sizeof(double) * D);
        double *s = (double *)malloc(sizeof(double) * (size_t)L);
        const uint16_t *qrow = q + ((int64_t)b * num_q_heads + h) * D;
        for (int d = 0; d < D; ++d) qd[d] = bf16_to_double(qrow[d]);

        /* pass 1: logits and their maximum */
        double m = -INFINITY;
        for (int64_t t = 0; t < L; ++t) {
            const uint16_t *krow = paged_row(k_pages, bt, t, kvh, num_kv_heads, D, page_size);
            double dot = 0.0;
            for (int d = 0; d < D; ++d) dot += qd[d] * bf16_to_double(krow[d]);
            s[t] = scale * dot;
            if (s[t] > m) m = s[t];
        }
        /* pass 2: normaliser and weighted sum of values */
        double Z = 0.0;
        for (int64_t t = 0; t < L; ++t) {
            const double w = exp(s[t] - m);
            const uint16_t *vrow = paged_row(v_pages, bt, t, kvh, num_kv_heads, D, page_size);
            Z += w;
            for (int d = 0; d < D; ++d) o[d] += w * bf16_to_double(vrow[d]);
        }
        for (int d = 0; d < D; ++d) o[d] /= Z;
        if (lse) lse[r] = m + log(Z);
        free(s);
        free(qd);
    }
    return 0;
}

/*
 * Sliding-window + attention-sink variant (the paper names sliding windows and
 * attention sinks as orthogonal byte-reducing approaches; it gives no formula, so the
 * reading is DESIGN.md R17): the one query, which sits at position L-1, attends the kept set
 *     K = { t in [0, L) : t < sink_tokens  or  t >= L - window }
 * and out = softmax over K only.  window >= L (or window <= 0, "no window") keeps everything and is
 * oracle_decode_attn.  Same two-pass fp64 statement, masked positions simply absent.
 */
int oracle_decode_attn_window(const uint16_t *q, const uint16_t *k_pages, const uint16_t *v_pages,
                              const int32_t *block_table, const int32_t *seq_lens, int num_q_heads,
                              int num_kv_heads, int head_dim, int page_size, float softmax_scale,
                              int window, int sink_tokens, double *out, double *lse, int batch,
                              int max_pages_per_seq, int num_threads)
{
    if (!q || !k_pages || !v_pages || !block_table || !seq_lens || !out) return 1;
    if (num_q_heads <= 0 || num_kv_heads <= 0 || num_q_heads % num_kv_heads != 0) return 1;
    if (head_dim <= 0 || page_size <= 0 || batch <= 0 || sink_tokens < 0) return 1;
    const int G = num_q_heads / num_kv_heads;
    const int D = head_dim;
    const int64_t rows = (int64_t)batch * num_q_heads;
    const double scale = (double)softmax_scale;
#ifdef _OPENMP
    if (num_threads <= 0) num_threads = omp_get_max_threads();
#else
    (void)num_threads;
#endif
#pragma omp parallel for schedule(dynamic, 1) num_threads(num_threads)
    for (int64_t r = 0; r < rows; ++r) {
        const int b = (int)(r / num_q_heads), h = (int)(r % num_q_heads);
        const int kvh = h / G;
        const int64_t L = seq_lens[b];
        const int64_t first_in_window = (window <= 0 || window >= L) ? 0 : L - window;
        const int32_t *bt = block_table + (int64_t)b * max_pages_per_seq;
        double *o = out + r * D;
        for (int d = 0; d < D; ++d) o[d] = 0.0;
        if (L <= 0) {
            if (lse) lse[r] = -INFINITY;
            continue;
        }
        double *qd = (double *)malloc(sizeof(double) * D);
        double *s = (double *)malloc(sizeof(double) * (size_t)L);
        const uint16_t *qrow = q + ((int64_t)b * num_q_heads + h) * D;
        for (int d = 0; d < D; ++d) qd[d] = bf16_to_double(qrow[d]);
        double m = -INFINITY;
        for (int64_t t = 0; t < L; ++t) {
            if (!(t < sink_tokens || t >= first_in_window)) continue; /* not in the kept set */
            const uint16_t *krow = paged_row(k_pages, bt, t, kvh, num_kv_heads, D, page_size);
            double dot = 0.0;
            for (int d = 0; d < D; ++d) dot += qd[d] * bf16_to_double(krow[d]);
            s[t] = scale * dot;
            if (s[t] > m) m = s[t];
        }
        double Z = 0.0;
        for (int64_t t = 0; t < L; ++t) {
            if (!(t < sink_tokens || t >= first_in_window)) continue;
            const double w = exp(s[t] - m);
            const uint16_t *vrow = paged_row(v_pages, bt, t, kvh, num_kv_heads, D, page_size);
            Z += w;
            for (int d = 0; d < D; ++d) o[d] += w * bf16_to_double(vrow[d]);
        }
        for (int d = 0; d < D; ++d) o[d] /= Z;
        if (lse) lse[r] = m + log(Z);
        free(s);
        free(qd);
    }
    return 0;
}

/*
 * FP8 (E4M3) KV-cache variant (the paper names "KV Cache Quantization (Hooper et
 * al., 2024)" as an orthogonal byte-reducing technique, and gives no format, so the reading is
 * DESIGN.md R18): K and V are stored one byte per element in the OCP FP8 E4M3 ("fn") encoding
 *     byte = s eeee mmm :  e = 0      -> (-1)^s * (m / 8) * 2^-6          (subnormal, incl. +-0)
 *                          e = 1..15  -> (-1)^s * (1 + m / 8) * 2^(e - 7)  (max 0x7e = 448)
 *                          0x7f, 0xff -> NaN (there is no infinity)
 * with one fp32 scale per (physical page, kv head) and per pool:
 *     k_t[d] = k_scale[pid][kvh] * e4m3(K8[pid][slot][kvh][d]),   v_t likewise with v_scale.
 * Attention over the dequantised cache is then exactly oracle_decode_attn_window (and, with
 * window <= 0, oracle_decode_attn): same two-pass fp64 statement.  q stays bf16.
 * kv_hnd != 0: the pools are laid out [P][Hkv][ps][D] ("HND") instead of [P][ps][Hkv][D]; only the
 * address of a token row changes.
 */
static double e4m3_to_double(uint8_t byte)
{
    const int sign = byte >> 7, e = (byte >> 3) & 15, m = byte & 7;
    double mag;
    if (e == 15 && m == 7) return NAN;
    if (e == 0) mag = ldexp((double)m / 8.0, -6);
    else mag = ldexp(1.0 + (double)m / 8.0, e - 7);
    return sign ? -mag : mag;
}

/* exported so that the decode table itself can be pinned against the format's published values */
double oracle_e4m3_decode(int byte) { return e4m3_to_double((uint8_t)byte); }

int oracle_decode_attn_fp8(const uint16_t *q,          /* bf16 [batch][Hq][D] */
                           const uint8_t *k_pages,     /* e4m3 [P][ps][Hkv][D] */
                           const uint8_t *v_pages,     /* e4m3 [P][ps][Hkv][D] */
                           const float *k_scale,       /* fp32 [P][Hkv] */
                           const float *v_scale,       /* fp32 [P][Hkv] */
                           const int32_t *block_table, const int32_t *seq_lens, int num_q_heads,
                           int num_kv_heads, int head_dim, int page_size, float softmax_scale,
                           int window, int sink_tokens, int kv_hnd, double *out, double *lse, int batch,
                           int max_pages_per_seq, int num_threads)
{
    if (!q || !k_pages || !v_pages || !k_scale || !v_scale || !block_table || !seq_lens || !out) return 1;
    if (num_q_heads <= 0 || num_kv_heads <= 0 || num_q_heads % num_kv_heads != 0) return 1;
    if (head_dim <= 0 || page_size <= 0 || batch <= 0 || sink_tokens < 0) return 1;
    const int G = num_q_heads / num_kv_heads;
    const int D = head_dim;
    const int64_t rows = (int64_t)batch * num_q_heads;
    const double scale = (double)softmax_scale;
#ifdef _OPENMP
    if (num_threads <= 0) num_threads = omp_get_max_threads();
#else
    (void)num_threads;
#endif
#pragma omp parallel for schedule(dynamic, 1) num_threads(num_threads)
    for (int64_t r = 0; r < rows; ++r) {
        const int b = (int)(r / num_q_heads), h = (int)(r % num_q_heads);
        const int kvh = h / G;
        const int64_t L = seq_lens[b];
        const int64_t first_in_window = (window <= 0 || window >= L) ? 0 : L - window;
        const int32_t *bt = block_table + (int64_t)b * max_pages_per_seq;
        double *o = out + r * D;
        for (int d = 0; d < D; ++d) o[d] = 0.0;
        if (L <= 0) {
            if (lse) lse[r] = -INFINITY;
            continue;
        }
        double *qd = (double *)malloc(sizeof(double) * D);
        double *s = (double *)malloc(sizeof(double) * (size_t)L);
        const uint16_t *qrow = q + ((int64_t)b * num_q_heads + h) * D;
        for (int d = 0; d < D; ++d) qd[d] = bf16_to_double(qrow[d]);
        double m = -INFINITY;
        for (int64_t t = 0; t < L; ++t) {
            if (!(t < sink_tokens || t >= first_in_window)) continue;
            const int64_t pid = bt[t / page_size], slot = t % page_size;
            const uint8_t *krow = k_pages + (kv_hnd ? (pid * num_kv_heads + kvh) * page_size + slot
                                                    : (pid * page_size + slot) * num_kv_heads + kvh) * (int64_t)D;
            const double ks = (double)k_scale[pid * num_kv_heads + kvh];
            double dot = 0.0;
            for (int d = 0; d < D; ++d) dot += qd[d] * (ks * e4m3_to_double(krow[d]));
            s[t] = scale * dot;
            if (s[t] > m) m = s[t];
        }
        double Z = 0.0;
        for (int64_t t = 0; t < L; ++t) {
            if (!(t < sink_tokens || t >= first_in_window)) continue;
            const int64_t pid = bt[t / page_size], slot = t % page_size;
            const uint8_t *vrow = v_pages + (kv_hnd ? (pid * num_kv_heads + kvh) * page_size + slot
                                                    : (pid * page_size + slot) * num_kv_heads + kvh) * (int64_t)D;
            const double vs = (double)v_scale[pid * num_kv_heads + kvh];
            const double w = exp(s[t] - m);
            Z += w;
            for (int d = 0; d < D; ++d) o[d] += w * (vs * e4m3_to_double(vrow[d]));
        }
        for (int d = 0; d < D; ++d) o[d] /= Z;
        if (lse) lse[r] = m + log(Z);
        free(s);
        free(qd);
    }
    return 0;
}

/*
 * Un-normalised partial over the token range [t0, t1) of ONE (b, h) row:
 *   m = max_t s_t, l = sum_t exp(s_t - m), acc[d] = sum_t exp(s_t - m) v_t[d].
 * Empty range -> m = -inf, l = 0, acc = 0 (reading R11).  This is the quantity
 * a split-KV worker hands to the combine step.
 */
int oracle_decode_attn_partial(const uint16_t *q, const uint16_t *k_pages,
                               const uint16_t *v_pages, const int32_t *block_table,
                               const int32_t *seq_lens, int num_q_heads, int num_kv_heads,
                               int head_dim, int page_size, float softmax_scale, int b, int h,
                               int64_t t0, int64_t t1, int max_pages_per_seq, double *acc,
                               double *m_out, double *l_out)
{
    if (!q || !k_pages || !v_pages || !block_table || !seq_lens || !acc) return 1;
    const int G = num_q_heads / num_kv_heads;
    const int D = head_dim;
    const int kvh = h / G;
    const int64_t L = seq_lens[b];
    const int32_t *bt = block_table + (int64_t)b * max_pages_per_seq;
    const double scale = (double)softmax_scale;
    if (t0 < 0) t0 = 0;
    if (t1 > L) t1 = L;
    for (int d = 0; d < D; ++d) acc[d] = 0.0;
    double m = -INFINITY, l = 0.0;
    if (t1 > t0) {
        const uint16_t *qrow = q + ((int64_t)b * num_q_heads + h) * D;
        double *s = (double *)malloc(sizeof(double) * (size_t)(t1 - t0));
        for (int64_t t = t0; t < t1; ++t) {
            const uint16_t *krow = paged_row(k_pages, bt, t, kvh, num_kv_heads, D, page_size);
            double dot = 0.0;
            for (int d = 0; d < D; ++d) dot += bf16_to_double(qrow[d]) * bf16_to_double(krow[d]);
            s[t - t0] = scale * dot;
            if (s[t - t0] > m) m = s[t - t0];
        }
        for (int64_t t = t0; t < t1; ++t) {
            const double w = exp(s[t - t0] - m);
            const uint16_t *vrow = paged_row(v_pages, bt, t, kvh, num_kv_heads, D, page_size);
            l += w;
            for (int d = 0; d < D; ++d) acc[d] += w * bf16_to_double(vrow[d]);
        }
        free(s);
    }
    *m_out = m;
    *l_out = l;
    return 0;
}

/*
 * Log-sum-exp combine of S partials of one row, merged in
 * split-index order:
 *   M = max_s m_s;  w_s = exp(m_s - M);
 *   out = (sum_s w_s acc_s) / (sum_s w_s l_s);   lse = M + log(sum_s w_s l_s).
 * Splits with l_s == 0 (m_s = -inf) contribute nothing; if every split is
 * empty the row is +0.0 and lse = -inf.
 */
int oracle_lse_merge(const double *acc /* [S][D] */, const double *m /* [S] */,
                     const double *l /* [S] */, int num_splits, int head_dim, double *out,
                     double *lse)
{
    const int D = head_dim;
    double M = -INFINITY;
    for (int s = 0; s < num_splits; ++s)
        if (l[s] > 0.0 && m[s] > M) M = m[s];
    for (int d = 0; d < D; ++d) out[d] = 0.0;
    if (M == -INFINITY) {
        if (lse) *lse = -INFINITY;
        return 0;
    }
    double Lsum = 0.0;
    for (int s = 0; s < num_splits; ++s) {
        if (!(l[s] > 0.0)) continue;
        const double w = exp(m[s] - M);
        Lsum += w * l[s];
        for (int d = 0; d < D; ++d) out[d] += w * acc[(int64_t)s * D + d];
    }
    for (int d = 0; d < D; ++d) out[d] /= Lsum;
    if (lse) *lse = M + log(Lsum);
    return 0;
}

/*
 * KV append (K_cache^(t) = [K_cache^(t-1); K^(t)]): write one new K row
 * and one new V row per sequence at logical position seq_lens[b], then
 * seq_lens[b] += 1.  new_k/new_v are bf16 [batch][Hkv][D].
 */
int oracle_kv_append(uint16_t *k_pages, uint16_t *v_pages, const int32_t *block_table,
                     int32_t *seq_lens, const uint16_t *new_k, const uint16_t *new_v,
                     int num_kv_heads, int head_dim, int page_size, int batch,
                     int max_pages_per_seq)
{
    const int64_t row = (int64_t)num_kv_heads * head_dim;
    for (int b = 0; b < batch; ++b) {
        const int64_t t = seq_lens[b];
        if (t / page_size >= max_pages_per_seq) return 1;
        const int64_t pid = block_table[(int64_t)b * max_pages_per_seq + t / page_size];
        const int64_t dst = (pid * page_size + t % page_size) * row;
        memcpy(k_pages + dst, new_k + b * row, sizeof(uint16_t) * row);
        memcpy(v_pages + dst, new_v + b * row, sizeof(uint16_t) * row);
        seq_lens[b] = (int32_t)(t + 1);
    }
    return 0;
}

/*
 * E4M3 encoder (round-to-nearest-even, saturating to +-448, "satfinite"): the grid is the decode table above.
 * NaN -> 0x7f.  Written from the format's definition (bias 7, 3 mantissa bits, subnormal step 2^-9).
 */
static uint8_t e4m3_from_float(float xf)
{
    if (xf != xf) return 0x7f;
    const uint8_t sign = signbit(xf) ? 0x80 : 0x00;
    const double a = fabs((double)xf);
    if (a > 448.0) return sign | 0x7e;          /* includes +-inf; (448, 464) would round to 448 anyway */
    if (a < ldexp(1.0, -6)) {                   /* subnormal range: multiples of 2^-9; 8 steps = 2^-6 = code 0x08 */
        const double q = nearbyint(a * 512.0);  /* default rounding mode: to nearest, ties to even */
        return sign | (uint8_t)q;
    }
    int e;
    const double f = frexp(a, &e);              /* a = f * 2^e, f in [0.5, 1) */
    e -= 1;                                     /* a = m * 2^e, m = 2f in [1, 2) */
    int q = (int)nearbyint((2.0 * f - 1.0) * 8.0);
    if (q == 8) { q = 0; e += 1; }
    if (e > 8 || (e == 8 && q == 7)) return sign | 0x7e;
    return sign | (uint8_t)(((e + 7) << 3) | q);
}

int oracle_e4m3_encode(float x) { return (int)e4m3_from_float(x); }

/*
 * KV append into the FP8 cache (the step right before the path, for reading R18's cache): the new
 * token's bf16 K row of kv head h is stored as   byte = e4m3_rne_sat( (float)k[h][d] / k_scale[pid][h] )
 * -- the IEEE fp32 quotient, then the encoder above -- with pid the page that holds position seq_lens[b]; the
 * page's scale is whatever the caller has put there (how it was chosen is the serving engine's policy);
 * V likewise; then seq_lens[b] += 1.  kv_hnd as in oracle_decode_attn_fp8.
 */
int oracle_kv_append_fp8(uint8_t *k_pages, uint8_t *v_pages, const float *k_scale, const float *v_scale,
                         const int32_t *block_table, int32_t *seq_lens, const uint16_t *new_k,
                         const uint16_t *new_v, int num_kv_heads, int head_dim, int page_size, int batch,
                         int max_pages_per_seq, int kv_hnd)
{
    for (int b = 0; b < batch; ++b) {
        const int64_t t = seq_lens[b];
        if (t / page_size >= max_pages_per_seq) return 1;
        const int64_t pid = block_table[(int64_t)b * max_pages_per_seq + t / page_size];
        const int64_t slot = t % page_size;
        for (int h = 0; h < num_kv_heads; ++h) {
            const int64_t dst = (kv_hnd ? (pid * num_kv_heads + h) * page_size + slot
                                        : (pid * page_size + slot) * num_kv_heads + h) * (int64_t)head_dim;
            const float ks = k_scale[pid * num_kv_heads + h], vs = v_scale[pid * num_kv_heads + h];
            for (int d = 0; d < head_dim; ++d) {
                const int64_t src = ((int64_t)b * num_kv_heads + h) * head_dim + d;
                const float kq = (float)bf16_to_double(new_k[src]) / ks;
                const float vq = (float)bf16_to_double(new_v[src]) / vs;
                k_pages[dst + d] = e4m3_from_float(kq);
                v_pages[dst + d] = e4m3_from_float(vq);
            }
        }
        seq_lens[b] = (int32_t)(t + 1);
    }
    return 0;
}

/*
 * Prefill attention over the paged cache (Alg. 1 lines 9-13: "Prefill new tokens
 * only" (cached) / "Prefill full context" (uncached); reading R20).  Sequence b has seq_lens[b] = L cached tokens,
 * the LAST n_b = q_start[b+1] - q_start[b] of which are the new ones; their queries are rows
 * q[q_start[b] .. q_start[b+1]) of the ragged q [total_q][Hq][D].  Query i of the chunk sits at position
 * pos = L - n_b + i and attends causally: keys t <= pos.
 *     out[row][h] = softmax_{t <= pos}(softmax_scale * q[row][h] . k_t) . V
 * n_b = 1 is the decode step (oracle_decode_attn); n_b = L is the uncached full prefill.  Same two-pass fp64
 * statement per (row, h).  Rows with n_b > L are invalid (return 1).
 */
int oracle_prefill_attn(const uint16_t *q,           /* bf16 [total_q][Hq][D] */
                        const uint16_t *k_pages, const uint16_t *v_pages, const int32_t *block_table,
                        const int32_t *seq_lens, const int32_t *q_start /* [batch + 1] */, int num_q_heads,
                        int num_kv_heads, int head_dim, int page_size, float softmax_scale, double *out,
                        double *lse, int batch, int max_pages_per_seq, int num_threads)
{
    if (!q || !k_pages || !v_pages || !block_table || !seq_lens || !q_start || !out) return 1;
    if (num_q_heads <= 0 || num_kv_heads <= 0 || num_q_heads % num_kv_heads != 0) return 1;
    if (head_dim <= 0 || page_size <= 0 || batch <= 0 || q_start[0] != 0) return 1;
    for (int b = 0; b < batch; ++b) {
        const int n = q_start[b + 1] - q_start[b];
        if (n < 0 || n > seq_lens[b]) return 1;
    }
    const int G = num_q_heads / num_kv_heads;
    const int D = head_dim;
    const int64_t rows = (int64_t)q_start[batch] * num_q_heads;
    const double scale = (double)softmax_scale;
#ifdef _OPENMP
    if (num_threads <= 0) num_threads = omp_get_max_threads();
#else
    (void)num_threads;
#endif
#pragma omp parallel for schedule(dynamic, 1) num_threads(num_threads)
    for (int64_t r = 0; r < rows; ++r) {
        const int row = (int)(r / num_q_heads), h = (int)(r % num_q_heads);
        int b = 0;
        while (q_start[b + 1] <= row) ++b;            /* the sequence this query row belongs to */
        const int kvh = h / G;
        const int64_t L = seq_lens[b];
        const int64_t n = q_start[b + 1] - q_start[b];
        const int64_t pos = L - n + (row - q_start[b]);  /* position of this query; attends t <= pos */
        const int32_t *bt = block_table + (int64_t)b * max_pages_per_seq;
        double *o = out + r * D;
        for (int d = 0; d < D; ++d) o[d] = 0.0;
        double *qd = (double *)malloc(sizeof(double) * D);
        double *s = (double *)malloc(sizeof(double) * (size_t)(pos + 1));
        const uint16_t *qrow = q + r * D;
        for (int d = 0; d < D; ++d) qd[d] = bf16_to_double(qrow[d]);
        double m = -INFINITY;
        for (int64_t t = 0; t <= pos; ++t) {
            const uint16_t *krow = paged_row(k_pages, bt, t, kvh, num_kv_heads, D, page_size);
            double dot = 0.0;
            for (int d = 0; d < D; ++d) dot += qd[d] * bf16_to_double(krow[d]);
            s[t] = scale * dot;
            if (s[t] > m) m = s[t];
        }
        double Z = 0.0;
        for (int64_t t = 0; t <= pos; ++t) {
            const double w = exp(s[t] - m);
            const uint16_t *vrow = paged_row(v_pages, bt, t, kvh, num_kv_heads, D, page_size);
            Z += w;
            for (int d = 0; d < D; ++d) o[d] += w * bf16_to_double(vrow[d]);
        }
        for (int d = 0; d < D; ++d) o[d] /= Z;
        if (lse) lse[r] = m + log(Z);
        free(s);
        free(qd);
    }
    return 0;
}
