// The step before the path (GPU side): RoPE + QKV split fused into kv_append.  The fused QKV
// projection output of one iteration's T tokens - per token Hq query heads, Hkv key heads, Hkv value heads, D bf16
// each - is split; q and k are rotated by the token's absolute position u_r + j ("rotate-half" RoPE of the Llama / Qwen
// families the paper serves; reading 22):
//     angle_i = pos * theta^(-2i/D),   y_i = x_i cos - x_{i+D/2} sin,   y_{i+D/2} = x_{i+D/2} cos + x_i sin
// q goes to the [T][Hq][D] buffer ss_mixed_attention reads, k (rotated) and v (bit copy) straight into their page slots
// (the a1 write).  One CTA per token: cos / sin of the D/2 angles are evaluated ONCE per token in double (range reduction
// at positions up to 2^30 needs it; 64 values, negligible) and shared through smem by all Hq + Hkv heads.  The rotation
// is done in double too, products and sums rounded separately (no fma), and the result is rounded to bf16 ONCE - the
// arithmetic of the oracle's definition, so q and k match it bit for bit (reading 25; the inverse
// frequencies theta^(-2i/D) come from the host's pow(), handed over as a kernel parameter).  The kernel is HBM-bound -
// (Hq + 2 Hkv) D 2 bytes in and out per token against ~6 fp64 operations per element pair - so double costs nothing.
// A thread owns 8 consecutive elements of BOTH halves of a head: two 16-byte loads, two 16-byte stores (8-byte stores
// of E4M3 codes over an FP8 cache).
#include <math.h>

#include "append.cuh"
#include "common.cuh"
#include "ptx.cuh"

namespace ss {

constexpr int kRopeThreads = kAppendThreads;

__device__ __forceinline__ float2 bf2_to_f2(uint32_t w) {
    return make_float2(__uint_as_float(w << 16), __uint_as_float(w & 0xffff0000u));
}

// two bf16 (one word) -> two E4M3 codes: exact widening, IEEE fp32 division by the head's scale, RNE with saturation -
// the quantisation of kv_append_fp8_kernel applied to the bf16 value the bf16 path would have stored
__device__ __forceinline__ uint32_t bf16x2_to_e4m3x2(uint32_t w, float sc) {
    return ptx::f32x2_to_e4m3x2(ptx::div_rn_ieee(__uint_as_float(w << 16), sc), ptx::div_rn_ieee(__uint_as_float(w & 0xffff0000u), sc));
}

struct RopeFreqs { double inv_freq[64]; };       // theta^(-2i/D), i < D/2 <= 64 (host pow(), launch_qkv_rope_append)

// double -> bf16 with a single rounding: to fp32 with round-to-odd (truncate, then set the last bit if anything was
// lost), then fp32 -> bf16 round-to-nearest-even.  fp32 keeps 16 bits more than bf16, so the sticky last bit makes the
// second rounding decide exactly as a direct one would.
__device__ __forceinline__ uint32_t f64_to_bf16_bits(double x) {
    float f = __double2float_rz(x);
    if ((double)f != x) f = __uint_as_float(__float_as_uint(f) | 1u);
    return (uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(f));
}

// FP8 (SS_FLAG_KV_FP8): q as before; the rotated k is rounded to bf16 exactly as on the bf16 path and THEN quantised like
// ss_kv_append does (so is v): the caches are byte arrays, k_cache / v_cache are passed as their byte addresses.
template <bool FP8>
__global__ void __launch_bounds__(kRopeThreads)
qkv_rope_append_kernel(const uint32_t* __restrict__ qkv, uint32_t* __restrict__ q_out, uint32_t* __restrict__ k_cache,
                       uint4* __restrict__ v_cache, const float* __restrict__ k_scale, const float* __restrict__ v_scale,
                       const int32_t* __restrict__ block_table,
                       const int32_t* __restrict__ qsl, const int32_t* __restrict__ ctx_lens, int R, int max_pages,
                       int Hq, int Hkv, int D, const __grid_constant__ RopeFreqs freqs, const int32_t* __restrict__ err_flag) {
    __shared__ double s_cos[64], s_sin[64];
    ptx::pdl_launch_dependents();
    ptx::pdl_wait();
    if (err_flag && *reinterpret_cast<const volatile int32_t*>(err_flag)) return;    // debug checks tripped: write nothing
    const int tok = blockIdx.x, tid = threadIdx.x;
    const int r = request_of_token(qsl, R, tok);
    const int pos = __ldg(ctx_lens + r) + (tok - __ldg(qsl + r));
    const int64_t page = __ldg(block_table + (int64_t)r * max_pages + (pos >> 4));
    const int slot = pos & (kPage - 1);
    const int half = D >> 1;
    if (tid < half) {
        double sn, cs;
        sincos((double)pos * freqs.inv_freq[tid], &sn, &cs);
        s_cos[tid] = cs;
        s_sin[tid] = sn;
    }
    __syncthreads();

    const int wpr = D >> 1;                                          // 32-bit words (bf16 pairs) per head
    const uint32_t* src = qkv + (int64_t)tok * (Hq + 2 * Hkv) * wpr;
    // ---- q and k heads: elements 8u .. 8u+7 of the first half pair with the same elements of the second half ----
    const int uph = half >> 3;                                       // 8-element units per half head
    for (int e = tid; e < (Hq + Hkv) * uph; e += kRopeThreads) {
        const int h = e / uph, u = e - h * uph;
        const uint4 av = __ldg(reinterpret_cast<const uint4*>(src + h * wpr) + u);
        const uint4 bv = __ldg(reinterpret_cast<const uint4*>(src + h * wpr + (half >> 1)) + u);
        const uint32_t aw[4] = {av.x, av.y, av.z, av.w}, bw[4] = {bv.x, bv.y, bv.z, bv.w};
        uint32_t ylo[4], yhi[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float2 a = bf2_to_f2(aw[i]), b = bf2_to_f2(bw[i]);
            const double c0 = s_cos[8 * u + 2 * i], c1 = s_cos[8 * u + 2 * i + 1];
            const double s0 = s_sin[8 * u + 2 * i], s1 = s_sin[8 * u + 2 * i + 1];
            const double ax = a.x, ay = a.y, bx = b.x, by = b.y;
            ylo[i] = f64_to_bf16_bits(__dsub_rn(__dmul_rn(ax, c0), __dmul_rn(bx, s0))) |
                     (f64_to_bf16_bits(__dsub_rn(__dmul_rn(ay, c1), __dmul_rn(by, s1))) << 16);
            yhi[i] = f64_to_bf16_bits(__dadd_rn(__dmul_rn(bx, c0), __dmul_rn(ax, s0))) |
                     (f64_to_bf16_bits(__dadd_rn(__dmul_rn(by, c1), __dmul_rn(ay, s1))) << 16);
        }
        if (FP8 && h >= Hq) {
            const int g = h - Hq;
            const float sc = __ldg(k_scale + g);
            uint2* kd = reinterpret_cast<uint2*>(reinterpret_cast<uint8_t*>(k_cache) + ((page * Hkv + g) * kPage + slot) * (int64_t)D);
            kd[u] = make_uint2(bf16x2_to_e4m3x2(ylo[0], sc) | (bf16x2_to_e4m3x2(ylo[1], sc) << 16),
                               bf16x2_to_e4m3x2(ylo[2], sc) | (bf16x2_to_e4m3x2(ylo[3], sc) << 16));       // elements 8u .. 8u+7
            kd[uph + u] = make_uint2(bf16x2_to_e4m3x2(yhi[0], sc) | (bf16x2_to_e4m3x2(yhi[1], sc) << 16),
                                     bf16x2_to_e4m3x2(yhi[2], sc) | (bf16x2_to_e4m3x2(yhi[3], sc) << 16)); // D/2 + 8u ..
            continue;
        }
        uint32_t* dst = h < Hq ? q_out + ((int64_t)tok * Hq + h) * wpr
                               : k_cache + ((page * Hkv + (h - Hq)) * kPage + slot) * (int64_t)wpr;
        reinterpret_cast<uint4*>(dst)[u] = make_uint4(ylo[0], ylo[1], ylo[2], ylo[3]);
        reinterpret_cast<uint4*>(dst)[uph + u] = make_uint4(yhi[0], yhi[1], yhi[2], yhi[3]);
    }
    // ---- v heads: 16-byte bit copies ----
    const int vph = D >> 3;                                          // uint4 per head
    const uint4* vsrc = reinterpret_cast<const uint4*>(src + (Hq + Hkv) * wpr);
    for (int e = tid; e < Hkv * vph; e += kRopeThreads) {
        const int g = e / vph, dv = e - g * vph;
        const uint4 v = __ldg(vsrc + e);
        if (FP8) {
            const float sc = __ldg(v_scale + g);
            uint2* vd = reinterpret_cast<uint2*>(reinterpret_cast<uint8_t*>(v_cache) + ((page * Hkv + g) * kPage + slot) * (int64_t)D);
            vd[dv] = make_uint2(bf16x2_to_e4m3x2(v.x, sc) | (bf16x2_to_e4m3x2(v.y, sc) << 16),
                                bf16x2_to_e4m3x2(v.z, sc) | (bf16x2_to_e4m3x2(v.w, sc) << 16));
        } else {
            v_cache[((page * Hkv + g) * kPage + slot) * (int64_t)vph + dv] = v;
        }
    }
}

cudaError_t launch_qkv_rope_append(const Handle* h, const void* qkv, const int32_t* bt, const int32_t* qsl,
                                   const int32_t* ctx, int R, int T, float rope_theta, void* q_out, cudaStream_t stream) {
    const ss_config& c = h->cfg;
    // theta^(-2i/D) with the host's pow(): 64 values that depend on (theta, D) only, kept from the previous call
    static thread_local RopeFreqs freqs;
    static thread_local float cached_theta = 0.f;
    static thread_local int cached_d = 0;
    if (cached_theta != rope_theta || cached_d != c.head_dim) {
        for (int i = 0; i < c.head_dim / 2; ++i) freqs.inv_freq[i] = pow((double)rope_theta, -2.0 * (double)i / (double)c.head_dim);
        for (int i = c.head_dim / 2; i < 64; ++i) freqs.inv_freq[i] = 0.0;
        cached_theta = rope_theta;
        cached_d = c.head_dim;
    }
    const int32_t* flag = h->debug_checks ? h->state + kStateErr : nullptr;
    if (h->kv_fp8)
        return launch_pdl(qkv_rope_append_kernel<true>, dim3((unsigned)T), dim3(kRopeThreads), 0, stream, (const uint32_t*)qkv,
                          (uint32_t*)q_out, (uint32_t*)h->k_cache, (uint4*)h->v_cache, h->k_scale, h->v_scale, bt, qsl, ctx, R,
                          c.max_pages_per_req, c.num_q_heads, c.num_kv_heads, c.head_dim, freqs, flag);
    return launch_pdl(qkv_rope_append_kernel<false>, dim3((unsigned)T), dim3(kRopeThreads), 0, stream, (const uint32_t*)qkv,
                      (uint32_t*)q_out, (uint32_t*)h->k_cache, (uint4*)h->v_cache, (const float*)nullptr, (const float*)nullptr, bt,
                      qsl, ctx, R, c.max_pages_per_req, c.num_q_heads, c.num_kv_heads, c.head_dim, freqs, flag);
}

}  // namespace ss
