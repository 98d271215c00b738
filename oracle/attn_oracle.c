/*
 * attn_oracle.c — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU statement of what one SlidingServe batch execution computes on the
 * attention path: for a batch B = {(c_i, u_i)} (§3.2 "c_i ... tokens allocated to
 * request i, u_i ... tokens cached by request i") every one of request i's c_i new query rows
 * attends causally over its u_i cached keys plus its own new keys, all requests independent of one
 * another inside the batch (§2.3; §3.1 step 9 "GPU Execution").
 * Chunked prefill only changes WHEN rows are computed, never their value.
 *
 * The method reaches the textbook result exactly (up to rounding order), so this file is the
 * textbook definition written out: materialised scores, max, exp, sum, weighted
 * sum.  No tiling, no online softmax, no split-KV, no SIMD intrinsics, no code shared with the
 * CUDA path.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may build or call this file.
 *
 * Pins (tests/test_oracle_pins.py, all -m "not gpu"): long-double brute force without
 * max-subtraction on dense un-paged inputs, scale=0 prefix mean, needle keys at mask/page
 * boundaries, single cached key returns V exactly, convexity, torch fp64 softmax on de-paged
 * tensors, chunking invariance (bitwise), decode == last prefill row, page-permutation and
 * batch-composition invariance (bitwise), GQA == replicated MHA, visit count == Table 1 identity
 * (PAPER.md:140-146), kv_append sentinel test.  Nothing here is "parity unpinned".
 *
 * Data layout (the paper is silent, SURVEY.md §8(c) reading 6):
 *   k_cache, v_cache : [num_pages][Hkv][page_size][D] bf16 (as uint16 bit patterns)
 *   block_table      : [R][max_pages_per_req] int32, entries past ceil((u+c)/page_size) undefined
 *   query_start_loc  : [R+1] int32 prefix sums of c_i ; ctx_lens : [R] int32 = u_i
 *   q / k_new / v_new: [T][H][D] bf16
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* bf16 -> double, exact: bf16 is the top 16 bits of an IEEE binary32. */
static double bf16_to_f64(uint16_t b) {
    uint32_t w = ((uint32_t)b) << 16;
    float f;
    memcpy(&f, &w, sizeof f);
    return (double)f;
}

static const uint16_t *kv_row(const uint16_t *cache, const int32_t *bt_row, int64_t t, int g,
                              int Hkv, int D, int page_size) {
    /* K(r,t,g,.) = cache[ block_table[r][t / page] ][ g ][ t % page ][ . ] */
    int64_t page = bt_row[t / page_size];
    int64_t slot = t % page_size;
    return cache + ((page * Hkv + g) * page_size + slot) * (int64_t)D;
}

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/*
 * kv_append (PAPER.md:99 step 10: after execution u_i grows by c_i; the write is implicit in the
 * paper).  Token j of request r goes to logical position u_r + j.  Pure uint16 copies.
 */
int oracle_kv_append(uint16_t *k_cache, uint16_t *v_cache, const uint16_t *k_new,
                     const uint16_t *v_new, const int32_t *block_table,
                     const int32_t *query_start_loc, const int32_t *ctx_lens, int R,
                     int max_pages_per_req, int Hkv, int D, int page_size) {
    for (int r = 0; r < R; ++r) {
        int c = query_start_loc[r + 1] - query_start_loc[r];
        int u = ctx_lens[r];
        const int32_t *bt = block_table + (int64_t)r * max_pages_per_req;
        for (int j = 0; j < c; ++j) {
            int64_t pos = (int64_t)u + j;
            int64_t page = bt[pos / page_size];
            int64_t slot = pos % page_size;
            int64_t tok = (int64_t)query_start_loc[r] + j;
            for (int g = 0; g < Hkv; ++g) {
                int64_t dst = ((page * Hkv + g) * page_size + slot) * (int64_t)D;
                int64_t src = (tok * Hkv + g) * (int64_t)D;
                for (int d = 0; d < D; ++d) {
                    k_cache[dst + d] = k_new[src + d];
                    v_cache[dst + d] = v_new[src + d];
                }
            }
        }
    }
    return 0;
}

/*
 * mixed_attention.  For request r, row j (0 <= j < c_r), query head h (kv head g = h / (Hq/Hkv)):
 *     n   = u_r + j + 1                       keys 0 .. u_r + j inclusive are visible
 *     s_t = scale * sum_d q[d] * K(r,t,g,d)   t = 0 .. n-1      (scale: the fp32 value, widened)
 *     m   = max_t s_t ; p_t = exp(s_t - m) ; l = sum_t p_t
 *     out[e] = (sum_t p_t * V(r,t,g,e)) / l ; lse = m + log(l)
 * Requests with c_r <= 1 are the paper's decode set D, c_r > 1 the prefill set P (PAPER.md:111
 * Eq. 2); the arithmetic is the same for both, c_r == 0 contributes no rows.
 *
 * rows: optional list of n_rows flat row indices (0 <= row < T) to compute; NULL = all T rows.
 * out  : [n_out][Hq][D] double, lse: [n_out][Hq] double (may be NULL), where n_out = n_rows or T
 *        and output slot i corresponds to rows[i] (or row i).
 * pairs_out: if non-NULL receives the number of (row, visible key) visits per query head.
 */
int oracle_mixed_attention(const uint16_t *q, const uint16_t *k_cache, const uint16_t *v_cache,
                           const int32_t *block_table, const int32_t *query_start_loc,
                           const int32_t *ctx_lens, int R, int max_pages_per_req, int Hq, int Hkv,
                           int D, int page_size, float scale, const int32_t *rows, int n_rows,
                           double *out, double *lse, int64_t *pairs_out) {
    if (Hkv <= 0 || Hq % Hkv != 0) return -1;
    const int G = Hq / Hkv;
    const int T = R > 0 ? query_start_loc[R] : 0;
    const int n_out = rows ? n_rows : T;
    const double scale_d = (double)scale;
    int64_t pairs = 0;
    int bad = 0;

    /* row -> request map */
    int32_t *row_req = (int32_t *)malloc(sizeof(int32_t) * (size_t)(T > 0 ? T : 1));
    if (!row_req) return -2;
    for (int r = 0; r < R; ++r)
        for (int t = query_start_loc[r]; t < query_start_loc[r + 1]; ++t) row_req[t] = r;

#pragma omp parallel for schedule(dynamic, 1) reduction(+ : pairs) reduction(| : bad)
    for (int i = 0; i < n_out; ++i) {
        const int row = rows ? rows[i] : i;
        if (row < 0 || row >= T) { bad |= 1; continue; }
        const int r = row_req[row];
        const int j = row - query_start_loc[r];
        const int64_t n = (int64_t)ctx_lens[r] + j + 1;
        const int32_t *bt = block_table + (int64_t)r * max_pages_per_req;
        double *s = (double *)malloc(sizeof(double) * (size_t)n);
        double *acc = (double *)malloc(sizeof(double) * (size_t)D);
        if (!s || !acc) { bad |= 2; free(s); free(acc); continue; }
        pairs += n;
        for (int h = 0; h < Hq; ++h) {
            const int g = h / G;
            const uint16_t *qv = q + ((int64_t)row * Hq + h) * D;
            double m = -INFINITY;
            for (int64_t t = 0; t < n; ++t) {
                const uint16_t *kr = kv_row(k_cache, bt, t, g, Hkv, D, page_size);
                double dot = 0.0;
                for (int d = 0; d < D; ++d) dot += bf16_to_f64(qv[d]) * bf16_to_f64(kr[d]);
                s[t] = scale_d * dot;
                if (s[t] > m) m = s[t];
            }
            double l = 0.0;
            for (int64_t t = 0; t < n; ++t) {
                s[t] = exp(s[t] - m);
                l += s[t];
            }
            for (int d = 0; d < D; ++d) acc[d] = 0.0;
            for (int64_t t = 0; t < n; ++t) {
                const uint16_t *vr = kv_row(v_cache, bt, t, g, Hkv, D, page_size);
                const double p = s[t];
                for (int d = 0; d < D; ++d) acc[d] += p * bf16_to_f64(vr[d]);
            }
            double *o = out + ((int64_t)i * Hq + h) * D;
            for (int d = 0; d < D; ++d) o[d] = acc[d] / l;
            if (lse) lse[(int64_t)i * Hq + h] = m + log(l);
        }
        free(s);
        free(acc);
    }
    free(row_req);
    if (pairs_out) *pairs_out = pairs;
    return bad ? -3 : 0;
}
