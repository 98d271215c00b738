// The step before the path (GPU side): RoPE + QKV split fused into kv_append.  The fused QKV
// projection output of one iteration's T tokens - per token Hq query heads, Hkv key heads, Hkv value heads, D bf16
// each - is split; q and k are rotated by the token's absolute position u_r + j ("rotate-half" RoPE of the Llama / Qwen
// families the paper serves; reading 22):
//     angle_i = pos * theta^(-2i/D),   y_i = x_i cos - x_{i+D/2} sin,   y_{i+D/2} = x_{i+D/2} cos + x_i sin
// q goes to the [T][Hq][D] buffer ss_mixed_attention reads, k (rotated) and v (bit copy) straight into their page slots
// (the a1 write).  One CTA per token: cos / sin of the D/2 angles are evaluated ONCE per token in double (range reduction
// at positions up to 2^30 needs it; 64 values, negligible) and shared through smem by all Hq + Hkv heads; the rotation
// itself is fp32 on bf16 pairs, one rounding to bf16.  HBM-bound: reads (Hq + 2 Hkv) D 2 bytes per token, writes the same.
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

// FP8 (SS_FLAG_KV_FP8): q as before; the rotated k is rounded to bf16 exactly as on the bf16 path and THEN quantised like
// ss_kv_append does (so is v): the caches are byte arrays, k_cache / v_cache are passed as their byte addresses.
template <bool FP8>
__global__ void __launch_bounds__(kRopeThreads)
qkv_rope_append_kernel(const uint32_t* __restrict__ qkv, uint32_t* __restrict__ q_out, uint32_t* __restrict__ k_cache,
                       uint4* __restrict__ v_cache, const float* __restrict__ k_scale, const float* __restrict__ v_scale,
                       const int32_t* __restrict__ block_table,
                       const int32_t* __restrict__ qsl, const int32_t* __restrict__ ctx_lens, int R, int max_pages,
                       int Hq, int Hkv, int D, double neg2_log2_theta_over_d, const int32_t* __restrict__ err_flag) {
    __shared__ float s_cos[64], s_sin[64];
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
        const double inv_freq = exp2((double)tid * neg2_log2_theta_over_d);      // theta^(-2 i / D)
        double sn, cs;
        sincos((double)pos * inv_freq, &sn, &cs);
        s_cos[tid] = (float)cs;
        s_sin[tid] = (float)sn;
    }
    __syncthreads();

    const int wpr = D >> 1;                                          // 32-bit words (bf16 pairs) per head
    const uint32_t* src = qkv + (int64_t)tok * (Hq + 2 * Hkv) * wpr;
    // ---- q and k heads: word w of the first half pairs with word w of the second half ----
    const int hw = half >> 1;                                        // words per half head
    for (int e = tid; e < (Hq + Hkv) * hw; e += kRopeThreads) {
        const int h = e / hw, w = e - h * hw;
        const float2 a = bf2_to_f2(__ldg(src + h * wpr + w)), b = bf2_to_f2(__ldg(src + h * wpr + hw + w));
        const float c0 = s_cos[2 * w], c1 = s_cos[2 * w + 1], s0 = s_sin[2 * w], s1 = s_sin[2 * w + 1];
        const uint32_t ylo = ptx::pack_bf16(__fmaf_rn(a.x, c0, -(b.x * s0)), __fmaf_rn(a.y, c1, -(b.y * s1)));
        const uint32_t yhi = ptx::pack_bf16(__fmaf_rn(b.x, c0, a.x * s0), __fmaf_rn(b.y, c1, a.y * s1));
        if (FP8 && h >= Hq) {
            const int g = h - Hq;
            const float sc = __ldg(k_scale + g);
            uint16_t* kd = reinterpret_cast<uint16_t*>(reinterpret_cast<uint8_t*>(k_cache) + ((page * Hkv + g) * kPage + slot) * (int64_t)D);
            kd[w] = (uint16_t)bf16x2_to_e4m3x2(ylo, sc);                 // elements 2w, 2w + 1
            kd[hw + w] = (uint16_t)bf16x2_to_e4m3x2(yhi, sc);            // elements D/2 + 2w, + 1
            continue;
        }
        uint32_t* dst = h < Hq ? q_out + ((int64_t)tok * Hq + h) * wpr
                               : k_cache + ((page * Hkv + (h - Hq)) * kPage + slot) * (int64_t)wpr;
        dst[w] = ylo;
        dst[hw + w] = yhi;
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
    const double k = -2.0 * log2((double)rope_theta) / (double)c.head_dim;
    const int32_t* flag = h->debug_checks ? h->state + kStateErr : nullptr;
    if (h->kv_fp8)
        return launch_pdl(qkv_rope_append_kernel<true>, dim3((unsigned)T), dim3(kRopeThreads), 0, stream, (const uint32_t*)qkv,
                          (uint32_t*)q_out, (uint32_t*)h->k_cache, (uint4*)h->v_cache, h->k_scale, h->v_scale, bt, qsl, ctx, R,
                          c.max_pages_per_req, c.num_q_heads, c.num_kv_heads, c.head_dim, k, flag);
    return launch_pdl(qkv_rope_append_kernel<false>, dim3((unsigned)T), dim3(kRopeThreads), 0, stream, (const uint32_t*)qkv,
                      (uint32_t*)q_out, (uint32_t*)h->k_cache, (uint4*)h->v_cache, (const float*)nullptr, (const float*)nullptr, bt,
                      qsl, ctx, R, c.max_pages_per_req, c.num_q_heads, c.num_kv_heads, c.head_dim, k, flag);
}

}  // namespace ss
