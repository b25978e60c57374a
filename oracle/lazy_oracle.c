/*
 * lazy_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU statement of what the LazyAttention hot path computes
 * (arxiv/paper_2606_04302).  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load this file.  It shares no code,
 * header, table or constant with the CUDA path under paper_2606_04302_b200/.
 *
 * Result definition (PAPER.md: LazyAttention "is mathematically identical to
 * existing methods that duplicate KV caches for position re-encoding"):
 *   1. materialise, per request, a RoPE-rotated copy of every visible key at its
 *      logical position ("deferred encoding", L164-166 rotation
 *      formula, Fig. 3b "K1/K2 denote the RoPE half-dimensions");
 *   2. run textbook causal softmax attention softmax(f(Q,m) f(K,n)^T / sqrt(d_k)) V
 *      (Eq. 4 and its RoPE form) with the GQA head mapping
 *      hk = hq / (Hq/Hkv).
 * No tiling, no online softmax, no fusion: every step is the definition written out.
 * OpenMP only distributes independent output rows over host cores.
 *
 * Readings of the paper taken here: half-split pairing
 * (j, j+D/2); theta_j = theta^(-2j/D); q arrives un-rotated and is rotated by the
 * position of its own token; causal mask by sequence index (s <= sq), positions feed
 * only RoPE; scale 1/sqrt(D).
 *
 * Pins: tests/test_oracle_pins.py (brute force, closed forms, shift invariance,
 * SDPA reduction, sharing equivalence, golden worked examples) and tests/test_oracle_fp8.py
 * (FP8 pages: the E4M3 code table, nearest-value and tie rules, round trips, scale closed form,
 * equality with the pinned fp64 path on dequantised pools).  No function here is
 * "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define DT_F64 0
#define DT_BF16 1
#define DT_E4M3 2

/* exact bf16 -> double (bf16 is the top 16 bits of an IEEE fp32) */
static double bf16_to_double(uint16_t b) {
    uint32_t u = ((uint32_t)b) << 16;
    float f;
    memcpy(&f, &u, sizeof f);
    return (double)f;
}

/* OCP 8-bit floating point, E4M3 ("FN" flavour: no infinities): bit 7 sign, bits 6-3 exponent E (bias 7), bits 2-0
 * mantissa M.  E = 0: subnormal, value M/8 * 2^-6.  Otherwise (1 + M/8) * 2^(E-7), except E = 15, M = 7, which is
 * NaN; the largest finite value is therefore 1.75 * 2^8 = 448 (code 0x7e). */
double lazy_oracle_e4m3_to_double(uint8_t c) {
    int E = (c >> 3) & 15, M = c & 7;
    double v;
    if (E == 15 && M == 7) return NAN;
    if (E == 0) v = ldexp((double)M / 8.0, -6);
    else v = ldexp(1.0 + (double)M / 8.0, E - 7);
    return (c & 0x80) ? -v : v;
}

/* Nearest E4M3 code of x: round to nearest, ties to the code with an even mantissa bit, magnitudes beyond 448
 * saturate to +-448 (never NaN, never infinity); NaN gives the NaN code.  Written as a search (bisection) over the
 * 127 non-negative finite values (codes 0x00..0x7e are increasing in value), not as bit manipulation. */
uint8_t lazy_oracle_e4m3_from_float(float x) {
    static double val[0x7f];                     /* values of codes 0x00..0x7e (every thread writes the same numbers) */
    static volatile int ready = 0;
    if (!ready) {
        for (int c = 0; c < 0x7f; ++c) val[c] = lazy_oracle_e4m3_to_double((uint8_t)c);
        ready = 1;
    }
    if (x != x) return 0x7f;
    uint8_t sign = (x < 0.0f || (x == 0.0f && 1.0f / x < 0.0f)) ? 0x80 : 0x00;
    double a = fabs((double)x);
    if (a >= 448.0) return sign | 0x7e;
    int lo_c = 0, hi_c = 0x7e;                   /* bisection: largest code c with val[c] <= a (val[0] = 0 <= a < val[0x7e]) */
    while (hi_c - lo_c > 1) {
        int mid = (lo_c + hi_c) / 2;
        if (val[mid] <= a) lo_c = mid; else hi_c = mid;
    }
    int c = lo_c;
    double dl = a - val[c], dh = val[c + 1] - a; /* exact: fp32 and E4M3 values are dyadic, differences fit in fp64 */
    if (dh < dl || (dh == dl && (c & 1))) ++c;
    return sign | (uint8_t)c;
}

static inline double load_elem(const void* base, int dtype, int64_t idx) {
    if (dtype == DT_BF16) return bf16_to_double(((const uint16_t*)base)[idx]);
    if (dtype == DT_E4M3) return lazy_oracle_e4m3_to_double(((const uint8_t*)base)[idx]);
    return ((const double*)base)[idx];
}

/* RoPE, half-split pairing.  PAPER.md L164-166:
 *   k1' = k1 cos(D) - k2 sin(D),  k2' = k1 sin(D) + k2 cos(D)
 * with k1 = x[0:D/2], k2 = x[D/2:D]; angle for pair j is pos * theta^(-2j/D) (RoPE, Su et al.,
 * cited at PAPER.md L102; stateless, from the absolute index: PAPER.md L455). */
void lazy_oracle_rope(const double* x, double pos, int D, double theta, double* y) {
    int half = D / 2;
    for (int j = 0; j < half; ++j) {
        double a = pos * pow(theta, -2.0 * (double)j / (double)D);
        double c = cos(a), s = sin(a);
        y[j] = x[j] * c - x[j + half] * s;
        y[j + half] = x[j] * s + x[j + half] * c;
    }
}

/* Positional variants (section 3.5).  NULL means the default above.
 *   rope_style 0  half-split pairing (j, j + D/2)
 *              1  interleaved pairing (2j, 2j + 1)                       (L215 "interleaved")
 *   inv_freq      optional [D/2] rotation frequency of pair j, replacing theta^(-2j/D): frequency-scaled RoPE
 *                 families (Llama-3.1 / NTK / YaRN, L213 "variant-specific scaling metadata"); a pair with
 *                 frequency 0 is not rotated (partial rotary)
 *   scale         softmax scale replacing 1/sqrt(D) when > 0 (YaRN's attention temperature folds in here)
 *   alibi_slopes  optional [Hq]: ALiBi (L221): NO rotation at all; the score of query position m and key position
 *                 n gets the bias  slope_h * (n - m)  added after scaling                                        */
typedef struct lazy_oracle_variant {
    int rope_style;
    const double* inv_freq;
    double scale;
    const double* alibi_slopes;
} lazy_oracle_variant;

void lazy_oracle_rope_variant(const double* x, double pos, int D, double theta, const lazy_oracle_variant* var,
                              double* y) {
    int half = D / 2;
    if (var && var->alibi_slopes) { for (int d = 0; d < D; ++d) y[d] = x[d]; return; }
    for (int j = 0; j < half; ++j) {
        double f = (var && var->inv_freq) ? var->inv_freq[j] : pow(theta, -2.0 * (double)j / (double)D);
        double a = pos * f;
        double c = cos(a), s = sin(a);
        int i1 = (var && var->rope_style == 1) ? 2 * j : j;
        int i2 = (var && var->rope_style == 1) ? 2 * j + 1 : j + half;
        y[i1] = x[i1] * c - x[i2] * s;
        y[i2] = x[i1] * s + x[i2] * c;
    }
}

/* Core: attention of n_q query rows over L keys with explicit positions.
 *   q      [n_q][Hq][D]   un-rotated queries
 *   k, v   [L][Hkv][D]    un-rotated keys, values (already gathered)
 *   pos_q  [n_q], pos_k [L]  logical positions (doubles so tests may pass any value)
 *   vis    [n_q]          query i sees key indices s <= vis[i]  (index-based causal mask)
 *   out    [n_q][Hq][D]
 *   probs  optional [n_q][Hq][L] softmax weights (0 beyond vis); may be NULL
 *   khat_out optional [L][Hkv][D] the materialised rotated keys; may be NULL
 *   qhat_out optional [n_q][Hq][D]; may be NULL
 * Step 1 materialises Khat = R_{pos_k} K (the "duplicate + re-encode" copy),
 * step 2 is Eq. 4 on (R_{pos_q} q, Khat, V).
 */
int lazy_oracle_attend_core_ex(const double* q, const double* k, const double* v,
                               const double* pos_q, const double* pos_k, const int64_t* vis,
                               int n_q, int64_t L, int Hq, int Hkv, int D, double theta,
                               const lazy_oracle_variant* var, const double* bias_pos_k,
                               const uint8_t* row_select,
                               double* out, double* probs, double* khat_out, double* qhat_out);

int lazy_oracle_attend_core(const double* q, const double* k, const double* v,
                            const double* pos_q, const double* pos_k, const int64_t* vis,
                            int n_q, int64_t L, int Hq, int Hkv, int D, double theta,
                            const uint8_t* row_select,
                            double* out, double* probs, double* khat_out, double* qhat_out) {
    return lazy_oracle_attend_core_ex(q, k, v, pos_q, pos_k, vis, n_q, L, Hq, Hkv, D, theta, NULL, NULL,
                                      row_select, out, probs, khat_out, qhat_out);
}

/* Same with a positional variant.  bias_pos_k (optional, [L]) are the key positions the ALiBi bias uses when they
 * differ from pos_k (pos_k is the rotation still owed to a key, which a stored-position cache makes different from
 * its logical position); NULL = pos_k. */
int lazy_oracle_attend_core_ex(const double* q, const double* k, const double* v,
                               const double* pos_q, const double* pos_k, const int64_t* vis,
                               int n_q, int64_t L, int Hq, int Hkv, int D, double theta,
                               const lazy_oracle_variant* var, const double* bias_pos_k,
                               const uint8_t* row_select,
                               double* out, double* probs, double* khat_out, double* qhat_out) {
    if (Hq % Hkv != 0 || D % 2 != 0) return -1;
    const double sm_scale = (var && var->scale > 0.0) ? var->scale : 1.0 / sqrt((double)D);
    if (!bias_pos_k) bias_pos_k = pos_k;
    int group = Hq / Hkv;
    double* khat = (double*)malloc(sizeof(double) * (size_t)(L > 0 ? L : 1) * Hkv * D);
    if (!khat) return -2;
    /* 1. materialise the rotated copy */
#pragma omp parallel for schedule(static)
    for (int64_t s = 0; s < L; ++s)
        for (int hk = 0; hk < Hkv; ++hk)
            lazy_oracle_rope_variant(k + ((size_t)s * Hkv + hk) * D, pos_k[s], D, theta, var,
                                     khat + ((size_t)s * Hkv + hk) * D);
    if (khat_out) memcpy(khat_out, khat, sizeof(double) * (size_t)L * Hkv * D);
    /* 2. standard attention, one (query row, head) at a time */
    int64_t n_rows = (int64_t)n_q * Hq;
    int err = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t row = 0; row < n_rows; ++row) {
        int i = (int)(row / Hq), hq = (int)(row % Hq);
        if (row_select && !row_select[i]) continue;
        int hk = hq / group;
        int64_t last = vis[i];               /* keys 0..last visible */
        if (last >= L) last = L - 1;
        double* o = out + ((size_t)i * Hq + hq) * D;
        for (int d = 0; d < D; ++d) o[d] = 0.0;
        double* qhat = (double*)malloc(sizeof(double) * D);
        double* sc = (double*)malloc(sizeof(double) * (size_t)(last >= 0 ? last + 1 : 1));
        if (!qhat || !sc) { err = 1; free(qhat); free(sc); continue; }
        lazy_oracle_rope_variant(q + ((size_t)i * Hq + hq) * D, pos_q[i], D, theta, var, qhat);
        if (qhat_out) memcpy(qhat_out + ((size_t)i * Hq + hq) * D, qhat, sizeof(double) * D);
        if (probs) for (int64_t s = 0; s < L; ++s) probs[((size_t)i * Hq + hq) * L + s] = 0.0;
        if (last >= 0) {
            double m = -INFINITY;
            for (int64_t s = 0; s <= last; ++s) {
                const double* kr = khat + ((size_t)s * Hkv + hk) * D;
                double acc = 0.0;
                for (int d = 0; d < D; ++d) acc += qhat[d] * kr[d];
                sc[s] = acc * sm_scale;
                if (var && var->alibi_slopes) sc[s] += var->alibi_slopes[hq] * (bias_pos_k[s] - pos_q[i]);
                if (sc[s] > m) m = sc[s];
            }
            double l = 0.0;
            for (int64_t s = 0; s <= last; ++s) { sc[s] = exp(sc[s] - m); l += sc[s]; }
            for (int64_t s = 0; s <= last; ++s) {
                double p = sc[s] / l;
                if (probs) probs[((size_t)i * Hq + hq) * L + s] = p;
                const double* vr = v + ((size_t)s * Hkv + hk) * D;
                for (int d = 0; d < D; ++d) o[d] += p * vr[d];
            }
        }
        free(qhat); free(sc);
    }
    free(khat);
    return err ? -2 : 0;
}

/* Paged wrapper (the three-call boundary's read side; PAPER.md L83-88 problem statement, L173/L182
 * per-document offsets carried as metadata -- here one logical start per page, north_star).
 * For request r: sequence index s lives in table slot s/P at in-page offset s%P, physical page
 * block_table[r][s/P], logical position page_logical_pos[r][s/P] + s%P.  The n_q query tokens are the
 * last n_q tokens of the sequence (already written to the cache): sq = L - n_q + i.
 *   q [total_q][Hq][D] (dtype_q), k_pool/v_pool [num_pages][Hkv][P][D] (dtype_kv)
 *   out [total_q][Hq][D] double.  row_select optional [total_q] (0 = skip row, left untouched).
 * Rows of requests with seq_len == 0 are written as zeros.
 */
int lazy_oracle_attend_paged_stored(const void* q, int dtype_q, const void* k_pool, const void* v_pool,
                                    int dtype_kv, const int32_t* block_table, const int32_t* page_logical_pos,
                                    int64_t table_stride, const int32_t* seq_lens, const int32_t* cu_q_lens,
                                    int num_reqs, int Hq, int Hkv, int D, int P, double theta,
                                    int k_storage, const int32_t* page_stored_pos,
                                    const uint8_t* row_select, double* out);

int lazy_oracle_attend_paged(const void* q, int dtype_q, const void* k_pool, const void* v_pool, int dtype_kv,
                             const int32_t* block_table, const int32_t* page_logical_pos, int64_t table_stride,
                             const int32_t* seq_lens, const int32_t* cu_q_lens, int num_reqs,
                             int Hq, int Hkv, int D, int P, double theta,
                             const uint8_t* row_select, double* out) {
    return lazy_oracle_attend_paged_stored(q, dtype_q, k_pool, v_pool, dtype_kv, block_table, page_logical_pos,
                                           table_stride, seq_lens, cu_q_lens, num_reqs, Hq, Hkv, D, P, theta,
                                           0, NULL, row_select, out);
}

/* Same call for the three ways a page's K can be STORED:
 *   k_storage 0  un-rotated (north_star): key s is rotated by its logical position;
 *   k_storage 1  the paper's own layout ("local position ... indexing from 0", L409): token t of
 *                physical page g was stored rotated by page_stored_pos[g] + t, so reaching logical position
 *                page_logical_pos + t needs ONE relative rotation by D = page_logical_pos - page_stored_pos[g]
 *                for the whole page (R_{p+D} = R_D R_p);
 *   k_storage 2  position-dependent cache (the standard-attention baseline of PAPER.md Fig. 5 / Table 12):
 *                K is stored already rotated at its final position, no rotation is left to do.
 * In every mode q is rotated by the logical position of its own token and the rest is Eq. 4. */
int lazy_oracle_attend_paged_variant(const void* q, int dtype_q, const void* k_pool, const void* v_pool,
                                     int dtype_kv, const int32_t* block_table, const int32_t* page_logical_pos,
                                     int64_t table_stride, const int32_t* seq_lens, const int32_t* cu_q_lens,
                                     int num_reqs, int Hq, int Hkv, int D, int P, double theta,
                                     int k_storage, const int32_t* page_stored_pos,
                                     int rope_style, const double* inv_freq, double scale, const double* alibi_slopes,
                                     const uint8_t* row_select, double* out);

int lazy_oracle_attend_paged_stored(const void* q, int dtype_q, const void* k_pool, const void* v_pool,
                                    int dtype_kv, const int32_t* block_table, const int32_t* page_logical_pos,
                                    int64_t table_stride, const int32_t* seq_lens, const int32_t* cu_q_lens,
                                    int num_reqs, int Hq, int Hkv, int D, int P, double theta,
                                    int k_storage, const int32_t* page_stored_pos,
                                    const uint8_t* row_select, double* out) {
    return lazy_oracle_attend_paged_variant(q, dtype_q, k_pool, v_pool, dtype_kv, block_table, page_logical_pos,
                                            table_stride, seq_lens, cu_q_lens, num_reqs, Hq, Hkv, D, P, theta,
                                            k_storage, page_stored_pos, 0, NULL, 0.0, NULL, row_select, out);
}

/* ... and with a positional variant (lazy_oracle_variant above). */
static int attend_paged_impl(const void* q, int dtype_q, const void* k_pool, const void* v_pool,
                             int dtype_kv, const float* k_scale, const float* v_scale,
                             const int32_t* block_table, const int32_t* page_logical_pos,
                             int64_t table_stride, const int32_t* seq_lens, const int32_t* cu_q_lens,
                             int num_reqs, int Hq, int Hkv, int D, int P, double theta,
                             int k_storage, const int32_t* page_stored_pos,
                             int rope_style, const double* inv_freq, double scale, const double* alibi_slopes,
                             const uint8_t* row_select, double* out);

int lazy_oracle_attend_paged_variant(const void* q, int dtype_q, const void* k_pool, const void* v_pool,
                                     int dtype_kv, const int32_t* block_table, const int32_t* page_logical_pos,
                                     int64_t table_stride, const int32_t* seq_lens, const int32_t* cu_q_lens,
                                     int num_reqs, int Hq, int Hkv, int D, int P, double theta,
                                     int k_storage, const int32_t* page_stored_pos,
                                     int rope_style, const double* inv_freq, double scale, const double* alibi_slopes,
                                     const uint8_t* row_select, double* out) {
    if (dtype_kv == DT_E4M3) return -1;     /* FP8 pages need their scales: lazy_oracle_attend_paged_fp8 */
    return attend_paged_impl(q, dtype_q, k_pool, v_pool, dtype_kv, NULL, NULL, block_table, page_logical_pos,
                             table_stride, seq_lens, cu_q_lens, num_reqs, Hq, Hkv, D, P, theta, k_storage,
                             page_stored_pos, rope_style, inv_freq, scale, alibi_slopes, row_select, out);
}

/* FP8 KV pages (the paper's cache holds "purely content-based keys and values", PAPER.md
 * L108, which is what makes a quantised page shareable at any position; decode traffic is the 2LD of L204-209).
 * The paper defines no quantised format; the format is this repository's: pages hold OCP FP8 E4M3
 * codes of the un-rotated K and of V, with one fp32 scale per (page, kv head, token) in k_scale / v_scale
 * [num_pages][Hkv][P].  The result is DEFINED as: dequantise every element exactly (code value x scale, exact in
 * fp64), then the unchanged definition above.  Nothing else differs. */
int lazy_oracle_attend_paged_fp8(const void* q, int dtype_q, const uint8_t* k_codes, const uint8_t* v_codes,
                                 const float* k_scale, const float* v_scale,
                                 const int32_t* block_table, const int32_t* page_logical_pos,
                                 int64_t table_stride, const int32_t* seq_lens, const int32_t* cu_q_lens,
                                 int num_reqs, int Hq, int Hkv, int D, int P, double theta,
                                 int rope_style, const double* inv_freq, double scale, const double* alibi_slopes,
                                 const uint8_t* row_select, double* out) {
    if (!k_scale || !v_scale) return -1;
    return attend_paged_impl(q, dtype_q, k_codes, v_codes, DT_E4M3, k_scale, v_scale, block_table, page_logical_pos,
                             table_stride, seq_lens, cu_q_lens, num_reqs, Hq, Hkv, D, P, theta, 0, NULL,
                             rope_style, inv_freq, scale, alibi_slopes, row_select, out);
}

static int attend_paged_impl(const void* q, int dtype_q, const void* k_pool, const void* v_pool,
                             int dtype_kv, const float* k_scale, const float* v_scale,
                             const int32_t* block_table, const int32_t* page_logical_pos,
                             int64_t table_stride, const int32_t* seq_lens, const int32_t* cu_q_lens,
                             int num_reqs, int Hq, int Hkv, int D, int P, double theta,
                             int k_storage, const int32_t* page_stored_pos,
                             int rope_style, const double* inv_freq, double scale, const double* alibi_slopes,
                             const uint8_t* row_select, double* out) {
    lazy_oracle_variant var;
    var.rope_style = rope_style; var.inv_freq = inv_freq; var.scale = scale; var.alibi_slopes = alibi_slopes;
    if (k_storage < 0 || k_storage > 2 || (k_storage == 1 && !page_stored_pos)) return -1;
    for (int r = 0; r < num_reqs; ++r) {
        int64_t L = seq_lens[r];
        int q0 = cu_q_lens[r], n_q = cu_q_lens[r + 1] - cu_q_lens[r];
        if (n_q <= 0) continue;
        if (row_select) {
            int any = 0;
            for (int i = 0; i < n_q; ++i) any |= row_select[q0 + i];
            if (!any) continue;
        }
        if (L <= 0) {
            for (int64_t e = 0; e < (int64_t)n_q * Hq * D; ++e) out[(size_t)q0 * Hq * D + e] = 0.0;
            continue;
        }
        if (n_q > L) return -1;
        double* kg = (double*)malloc(sizeof(double) * (size_t)L * Hkv * D);
        double* vg = (double*)malloc(sizeof(double) * (size_t)L * Hkv * D);
        double* pos = (double*)malloc(sizeof(double) * (size_t)L);
        double* rot = (double*)malloc(sizeof(double) * (size_t)L);   /* rotation still owed to key s */
        double* qd = (double*)malloc(sizeof(double) * (size_t)n_q * Hq * D);
        double* pos_q = (double*)malloc(sizeof(double) * (size_t)n_q);
        int64_t* vis = (int64_t*)malloc(sizeof(int64_t) * (size_t)n_q);
        if (!kg || !vg || !pos || !rot || !qd || !pos_q || !vis) return -2;
        /* gather the request's rows through the block table */
#pragma omp parallel for schedule(static)
        for (int64_t s = 0; s < L; ++s) {
            int64_t slot = s / P, t = s % P;
            int64_t page = block_table[(size_t)r * table_stride + slot];
            pos[s] = (double)page_logical_pos[(size_t)r * table_stride + slot] + (double)t;
            if (k_storage == 0) rot[s] = pos[s];
            else if (k_storage == 1)
                rot[s] = (double)page_logical_pos[(size_t)r * table_stride + slot] - (double)page_stored_pos[page];
            else rot[s] = 0.0;
            for (int hk = 0; hk < Hkv; ++hk) {
                int64_t base = (((int64_t)page * Hkv + hk) * P + t) * D;
                /* FP8 pages: exact dequantisation, code value x the (page, head, token) scale */
                double sk = k_scale ? (double)k_scale[((int64_t)page * Hkv + hk) * P + t] : 1.0;
                double sv = v_scale ? (double)v_scale[((int64_t)page * Hkv + hk) * P + t] : 1.0;
                for (int d = 0; d < D; ++d) {
                    kg[((size_t)s * Hkv + hk) * D + d] = load_elem(k_pool, dtype_kv, base + d) * sk;
                    vg[((size_t)s * Hkv + hk) * D + d] = load_elem(v_pool, dtype_kv, base + d) * sv;
                }
            }
        }
        for (int64_t e = 0; e < (int64_t)n_q * Hq * D; ++e) qd[e] = load_elem(q, dtype_q, (int64_t)q0 * Hq * D + e);
        for (int i = 0; i < n_q; ++i) {
            int64_t sq = L - n_q + i;        /* sequence index of this query token */
            vis[i] = sq;
            pos_q[i] = pos[sq];
        }
        int rc = lazy_oracle_attend_core_ex(qd, kg, vg, pos_q, rot, vis, n_q, L, Hq, Hkv, D, theta, &var, pos,
                                            row_select ? row_select + q0 : NULL,
                                            out + (size_t)q0 * Hq * D, NULL, NULL, NULL);
        free(kg); free(vg); free(pos); free(rot); free(qd); free(pos_q); free(vis);
        if (rc) return rc;
    }
    return 0;
}

/* lazy_cache_write oracle: bit copy of un-rotated rows into pages (the cache is
 * "purely content-based keys and values").  slot = page*P + off; slot < 0 skips the token.
 *   k_new/v_new [T][Hkv][D] 16-bit words, pools [num_pages][Hkv][P][D] 16-bit words. */
int lazy_oracle_cache_write(const uint16_t* k_new, const uint16_t* v_new, const int64_t* slot_mapping,
                            int64_t num_tokens, int Hkv, int D, int P, int64_t num_pages,
                            uint16_t* k_pool, uint16_t* v_pool) {
    for (int64_t t = 0; t < num_tokens; ++t) {
        int64_t slot = slot_mapping[t];
        if (slot < 0) continue;
        int64_t page = slot / P, off = slot % P;
        if (page >= num_pages) return -1;
        for (int hk = 0; hk < Hkv; ++hk) {
            int64_t dst = ((page * Hkv + hk) * P + off) * D;
            int64_t src = (t * Hkv + hk) * D;
            memcpy(k_pool + dst, k_new + src, sizeof(uint16_t) * D);
            memcpy(v_pool + dst, v_new + src, sizeof(uint16_t) * D);
        }
    }
    return 0;
}

/* lazy_cache_write for FP8 pages: quantise each new (token, kv head) row of K and of V on its own.
 *   amax  = max_d |x[d]|                        (bf16 inputs, exact)
 *   scale = amax / 448 in fp32 (round to nearest), or 1 if that is not a positive number (an all-zero row)
 *   code[d] = nearest E4M3 code of  x[d] / scale  (the quotient formed in fp32, round to nearest)
 * so the row's largest element lands on +-448, the top of the E4M3 range.  Both decisions that produce integers
 * (the scale's fp32 bits and the codes) are taken in fp32, the precision the CUDA kernel uses; IEEE division is
 * correctly rounded on both sides, so codes and scales must agree bit for bit.  Inputs are finite.
 *   k_new/v_new [T][Hkv][D] bf16 words; code pools [num_pages][Hkv][P][D] bytes; scale pools [num_pages][Hkv][P]. */
int lazy_oracle_cache_write_fp8(const uint16_t* k_new, const uint16_t* v_new, const int64_t* slot_mapping,
                                int64_t num_tokens, int Hkv, int D, int P, int64_t num_pages,
                                uint8_t* k_codes, uint8_t* v_codes, float* k_scale, float* v_scale) {
    for (int64_t t = 0; t < num_tokens; ++t)
        if (slot_mapping[t] >= 0 && slot_mapping[t] / P >= num_pages) return -1;
    /* tokens are independent (distinct slots): OpenMP only distributes them over host cores */
#pragma omp parallel for schedule(static)
    for (int64_t t = 0; t < num_tokens; ++t) {
        int64_t slot = slot_mapping[t];
        if (slot < 0) continue;
        int64_t page = slot / P, off = slot % P;
        for (int hk = 0; hk < Hkv; ++hk) {
            int64_t dst = ((page * Hkv + hk) * P + off) * D;
            int64_t src = (t * Hkv + hk) * D;
            for (int which = 0; which < 2; ++which) {
                const uint16_t* x = (which ? v_new : k_new) + src;
                uint8_t* codes = (which ? v_codes : k_codes) + dst;
                float* sc = (which ? v_scale : k_scale) + (page * Hkv + hk) * P + off;
                float amax = 0.0f;
                for (int d = 0; d < D; ++d) {
                    float a = fabsf((float)bf16_to_double(x[d]));
                    if (a > amax) amax = a;
                }
                volatile float scale = amax / 448.0f;       /* volatile: keep the quotient in fp32 (no excess precision) */
                if (!(scale > 0.0f)) scale = 1.0f;
                *sc = scale;
                for (int d = 0; d < D; ++d) {
                    volatile float y = (float)bf16_to_double(x[d]) / scale;
                    codes[d] = lazy_oracle_e4m3_from_float(y);
                }
            }
        }
    }
    return 0;
}

/* Materialising re-encoding of whole pages -- what position-dependent caches do on a position mismatch
 * ("allocate + copy + rotate", App. B) and what LazyAttention avoids.  For i < num:
 *   out[i][hk][t][:] = rope(K[src_pages[i]][hk][t][:], rot_pos[i] + (per_token ? t : 0))
 * per_token = 1 encodes an un-rotated page at logical start rot_pos[i]; per_token = 0 applies one relative
 * rotation D = rot_pos[i] (may be negative) to a page that already carries positions.
 * out is fp64 [num][Hkv][P][D]; the CUDA call rounds the same quantity to bf16. */
int lazy_oracle_materialize_pages(const void* k_pool, int dtype_kv, const int32_t* src_pages,
                                  const int32_t* rot_pos, int per_token, int64_t num,
                                  int Hkv, int D, int P, double theta, double* out) {
    double* x = (double*)malloc(sizeof(double) * D);
    if (!x) return -2;
    for (int64_t i = 0; i < num; ++i)
        for (int hk = 0; hk < Hkv; ++hk)
            for (int t = 0; t < P; ++t) {
                int64_t base = (((int64_t)src_pages[i] * Hkv + hk) * P + t) * D;
                for (int d = 0; d < D; ++d) x[d] = load_elem(k_pool, dtype_kv, base + d);
                lazy_oracle_rope(x, (double)rot_pos[i] + (per_token ? (double)t : 0.0), D, theta,
                                 out + ((((size_t)i * Hkv + hk) * P) + t) * D);
            }
    free(x);
    return 0;
}

int lazy_oracle_num_threads(void) {
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}
