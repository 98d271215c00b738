/*
 * next_oracle.c — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * fp64 CPU statements of the two "next" steps around the hot path:
 *
 *  (A) rope_qkv_append — the step BEFORE the path: the fused QKV projection output of the models the paper
 *      serves (Llama3-8B, Qwen2.5-7B) is split into q, k, v; rotary position embedding is applied
 *      to q and k at the token's absolute position u_r + j; k and v go to the paged cache (the a1 write), q to
 *      the buffer mixed_attention reads.  The paper is silent on all of it (it runs unmodified vLLM models);
 *      the definition is the public one of those model families ("rotate-half" RoPE), reading 22:
 *          inv_freq_i = theta^(-2 i / D),  i = 0 .. D/2-1        angle = pos * inv_freq_i
 *          y_i       = x_i cos(angle) - x_{i+D/2} sin(angle)
 *          y_{i+D/2} = x_{i+D/2} cos(angle) + x_i sin(angle)
 *      computed in double from the bf16 inputs and rounded ONCE to bf16 (round to nearest even).  v is a bit copy.
 *
 *  (B) FP8 KV cache — K and V stored as OCP FP8 E4M3 ("e4m3fn": bias 7, no infinities, max 448, S.1111.111 = NaN)
 *      with one fp32 scale per (tensor, kv head), reading 23:
 *          append  : code = e4m3_rne_satfinite( x / scale[g] )        (x widened exactly from bf16; the quotient is
 *                    taken in fp32 - the precision in which the decision is made on both sides - then rounded to
 *                    nearest even, magnitudes above 448 clamp to 448, NaN stays NaN)
 *          attention: K(r,t,g,d) = e4m3_to_double(code) * (double)k_scale[g], V likewise; everything else is the
 *                    plain definition of attn_oracle.c (materialised scores, max, exp, sum, weighted sum).
 *
 * Pins (tests/test_next_oracle_pins.py, all -m "not gpu"): RoPE - position 0 is the identity, norm of every
 * (i, i+D/2) pair preserved, <rope(q,m), rope(k,n)> depends on m - n only, complex-multiplication form with
 * numpy, torch fp64 cos/sin/rotate_half formula; bf16 rounding - exhaustive over every bf16 pattern and every
 * midpoint between neighbours (ties to even, just above / below a tie); e4m3 - every one of the 256 codes decodes
 * to the value the OCP table gives, encode(decode(code)) == code, midpoints tie to even, saturation at 448, and
 * torch.float8_e4m3fn agrees on every bf16 input; FP8 attention - scale = 1 on inputs that are exactly
 * representable equals the bf16 oracle bit for bit.  Nothing here is "parity unpinned".
 *
 * Shares no code with the CUDA path; only tests/ (and bench legs that time the oracle) may call it.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

static double bf16_to_f64_(uint16_t b) {
    uint32_t w = ((uint32_t)b) << 16;
    float f;
    memcpy(&f, &w, sizeof f);
    return (double)f;
}

/* double -> bf16, ONE rounding to nearest even (not double -> float -> bf16, which rounds twice). */
uint16_t oracle_f64_to_bf16(double x) {
    if (x != x) return 0x7FC0;
    float f = (float)x; /* first rounding: 24 significant bits */
    uint32_t w;
    memcpy(&w, &f, sizeof w);
    if ((w & 0x7F800000u) == 0x7F800000u) return (uint16_t)(w >> 16); /* +-inf */
    uint32_t low = w & 0xFFFFu, hi = w >> 16;
    if (low > 0x8000u) return (uint16_t)(hi + 1);
    if (low < 0x8000u) return (uint16_t)hi;
    /* f sits exactly on a bf16 tie: the discarded part of x decides, else ties to even */
    double fd = (double)f;
    if (fabs(x) > fabs(fd)) return (uint16_t)(hi + 1);
    if (fabs(x) < fabs(fd)) return (uint16_t)hi;
    return (uint16_t)(hi + (hi & 1u));
}

/* (A) one head vector: out[0..D) = RoPE(x[0..D), pos) in double */
void oracle_rope_rotate(const double *x, int D, int64_t pos, double theta, double *out) {
    int half = D / 2;
    for (int i = 0; i < half; ++i) {
        double inv_freq = pow(theta, -2.0 * (double)i / (double)D);
        double ang = (double)pos * inv_freq;
        double c = cos(ang), s = sin(ang);
        out[i] = x[i] * c - x[i + half] * s;
        out[i + half] = x[i + half] * c + x[i] * s;
    }
}

/*
 * qkv: [T][(Hq + 2 Hkv) * D] bf16 - per token the Hq query heads, then the Hkv key heads, then the Hkv value heads.
 * Writes q_out [T][Hq][D] bf16 (RoPE'd), K (RoPE'd) and V (copied) into the paged caches [P][Hkv][page][D].
 */
int oracle_rope_qkv_append(const uint16_t *qkv, uint16_t *q_out, uint16_t *k_cache, uint16_t *v_cache,
                           const int32_t *block_table, const int32_t *query_start_loc, const int32_t *ctx_lens,
                           int R, int max_pages_per_req, int Hq, int Hkv, int D, int page_size, double theta) {
    double *x = (double *)malloc(sizeof(double) * 2 * (size_t)D);
    if (!x) return -1;
    double *y = x + D;
    int64_t row_elems = (int64_t)(Hq + 2 * Hkv) * D;
    for (int r = 0; r < R; ++r) {
        int c = query_start_loc[r + 1] - query_start_loc[r];
        int u = ctx_lens[r];
        const int32_t *bt = block_table + (int64_t)r * max_pages_per_req;
        for (int j = 0; j < c; ++j) {
            int64_t pos = (int64_t)u + j;
            int64_t tok = (int64_t)query_start_loc[r] + j;
            int64_t page = bt[pos / page_size], slot = pos % page_size;
            const uint16_t *src = qkv + tok * row_elems;
            for (int h = 0; h < Hq; ++h) {
                for (int d = 0; d < D; ++d) x[d] = bf16_to_f64_(src[(int64_t)h * D + d]);
                oracle_rope_rotate(x, D, pos, theta, y);
                for (int d = 0; d < D; ++d) q_out[(tok * Hq + h) * (int64_t)D + d] = oracle_f64_to_bf16(y[d]);
            }
            for (int g = 0; g < Hkv; ++g) {
                int64_t dst = ((page * Hkv + g) * page_size + slot) * (int64_t)D;
                const uint16_t *ks = src + (int64_t)(Hq + g) * D;
                const uint16_t *vs = src + (int64_t)(Hq + Hkv + g) * D;
                for (int d = 0; d < D; ++d) x[d] = bf16_to_f64_(ks[d]);
                oracle_rope_rotate(x, D, pos, theta, y);
                for (int d = 0; d < D; ++d) {
                    k_cache[dst + d] = oracle_f64_to_bf16(y[d]);
                    v_cache[dst + d] = vs[d];
                }
            }
        }
    }
    free(x);
    return 0;
}

/* ------------------------------------------------------------------------------------------------------------ */
/* (B) FP8 E4M3 (e4m3fn) */

double oracle_e4m3_to_f64(uint8_t code) {
    int sign = code >> 7, e = (code >> 3) & 0xF, m = code & 7;
    double v;
    if (e == 0xF && m == 7) return NAN;
    if (e == 0) v = ldexp((double)m, -9);                 /* subnormal: m/8 * 2^-6 */
    else v = ldexp(1.0 + (double)m / 8.0, e - 7);
    return sign ? -v : v;
}

/* fp32 value -> e4m3, round to nearest even, saturate to +-448, NaN -> 0x7F | sign.  Written on the value grid:
 * find the two neighbouring representable magnitudes, pick the nearer, ties to the even code. */
uint8_t oracle_f32_to_e4m3(float xf) {
    if (xf != xf) return 0x7F;
    uint8_t sign = signbit(xf) ? 0x80 : 0;
    double a = fabs((double)xf);
    if (a >= 448.0) return (uint8_t)(sign | 0x7E);        /* satfinite (also +-inf) */
    /* codes 0x00..0x7E are ordered by magnitude: binary search for the largest code with value <= a */
    int lo = 0, hi = 0x7E;
    while (lo < hi) {
        int mid = (lo + hi + 1) / 2;
        if (oracle_e4m3_to_f64((uint8_t)mid) <= a) lo = mid; else hi = mid - 1;
    }
    if (lo == 0x7E) return (uint8_t)(sign | lo);
    double dlo = a - oracle_e4m3_to_f64((uint8_t)lo), dhi = oracle_e4m3_to_f64((uint8_t)(lo + 1)) - a;
    int code = dlo < dhi ? lo : (dhi < dlo ? lo + 1 : ((lo & 1) ? lo + 1 : lo));
    return (uint8_t)(sign | code);
}

/* FP8 kv_append: k_new / v_new [T][Hkv][D] bf16 -> caches [P][Hkv][page][D] uint8 codes; scale [Hkv] fp32 each. */
int oracle_kv_append_fp8(uint8_t *k_cache, uint8_t *v_cache, const uint16_t *k_new, const uint16_t *v_new,
                         const float *k_scale, const float *v_scale, const int32_t *block_table,
                         const int32_t *query_start_loc, const int32_t *ctx_lens, int R, int max_pages_per_req,
                         int Hkv, int D, int page_size) {
    for (int r = 0; r < R; ++r) {
        int c = query_start_loc[r + 1] - query_start_loc[r];
        int u = ctx_lens[r];
        const int32_t *bt = block_table + (int64_t)r * max_pages_per_req;
        for (int j = 0; j < c; ++j) {
            int64_t pos = (int64_t)u + j, page = bt[pos / page_size], slot = pos % page_size;
            int64_t tok = (int64_t)query_start_loc[r] + j;
            for (int g = 0; g < Hkv; ++g) {
                int64_t dst = ((page * Hkv + g) * page_size + slot) * (int64_t)D;
                int64_t src = (tok * Hkv + g) * (int64_t)D;
                for (int d = 0; d < D; ++d) {
                    /* the quotient is an fp32 division on both sides (IEEE, correctly rounded) */
                    float kq = (float)bf16_to_f64_(k_new[src + d]) / k_scale[g];
                    float vq = (float)bf16_to_f64_(v_new[src + d]) / v_scale[g];
                    k_cache[dst + d] = oracle_f32_to_e4m3(kq);
                    v_cache[dst + d] = oracle_f32_to_e4m3(vq);
                }
            }
        }
    }
    return 0;
}

/* FP8 attention: the plain definition of attn_oracle.c with K, V = e4m3 code * scale[g].  rows / out / lse as there. */
int oracle_mixed_attention_fp8(const uint16_t *q, const uint8_t *k_cache, const uint8_t *v_cache,
                               const float *k_scale, const float *v_scale, const int32_t *block_table,
                               const int32_t *query_start_loc, const int32_t *ctx_lens, int R,
                               int max_pages_per_req, int Hq, int Hkv, int D, int page_size, float scale_f32,
                               const int32_t *rows, int n_rows, double *out, double *lse) {
    const int G = Hq / Hkv;
    const double scale = (double)scale_f32;
    int T = R > 0 ? query_start_loc[R] : 0;
    int n_out = rows ? n_rows : T;
    int rc = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int i = 0; i < n_out; ++i) {
        int row = rows ? rows[i] : i;
        int r = 0;
        while (r < R && !(query_start_loc[r] <= row && row < query_start_loc[r + 1])) ++r;
        if (r >= R) { rc = -2; continue; }
        int j = row - query_start_loc[r];
        int64_t n = (int64_t)ctx_lens[r] + j + 1;
        const int32_t *bt = block_table + (int64_t)r * max_pages_per_req;
        double *s = (double *)malloc(sizeof(double) * (size_t)n);
        if (!s) { rc = -1; continue; }
        for (int h = 0; h < Hq; ++h) {
            int g = h / G;
            const uint16_t *qv = q + ((int64_t)row * Hq + h) * D;
            double m = -INFINITY;
            for (int64_t t = 0; t < n; ++t) {
                const uint8_t *kr = k_cache + (((int64_t)bt[t / page_size] * Hkv + g) * page_size + t % page_size) * (int64_t)D;
                double acc = 0.0;
                for (int d = 0; d < D; ++d) acc += bf16_to_f64_(qv[d]) * (oracle_e4m3_to_f64(kr[d]) * (double)k_scale[g]);
                s[t] = scale * acc;
                if (s[t] > m) m = s[t];
            }
            double l = 0.0;
            for (int64_t t = 0; t < n; ++t) { s[t] = exp(s[t] - m); l += s[t]; }
            double *o = out + ((int64_t)i * Hq + h) * D;
            for (int d = 0; d < D; ++d) o[d] = 0.0;
            for (int64_t t = 0; t < n; ++t) {
                const uint8_t *vr = v_cache + (((int64_t)bt[t / page_size] * Hkv + g) * page_size + t % page_size) * (int64_t)D;
                for (int d = 0; d < D; ++d) o[d] += s[t] * (oracle_e4m3_to_f64(vr[d]) * (double)v_scale[g]);
            }
            for (int d = 0; d < D; ++d) o[d] /= l;
            if (lse) lse[(int64_t)i * Hq + h] = m + log(l);
        }
        free(s);
    }
    return rc;
}

/* array forms for the pin tests */
void oracle_f64_to_bf16_array(const double *x, int64_t n, uint16_t *out) {
    for (int64_t i = 0; i < n; ++i) out[i] = oracle_f64_to_bf16(x[i]);
}
void oracle_f32_to_e4m3_array(const float *x, int64_t n, uint8_t *out) {
    for (int64_t i = 0; i < n; ++i) out[i] = oracle_f32_to_e4m3(x[i]);
}
void oracle_e4m3_to_f64_array(const uint8_t *c, int64_t n, double *out) {
    for (int64_t i = 0; i < n; ++i) out[i] = oracle_e4m3_to_f64(c[i]);
}
