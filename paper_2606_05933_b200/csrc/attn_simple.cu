// Plain CUDA-core attention (one warp per (query row, query head), online softmax over 32-key blocks).
//
// The warp kernel is the library's in-CUDA fallback for shapes the tensor-core kernels do not cover and
// a debugging second opinion (ss_debug_force_simple_path); it is NOT the fast path and never a CPU
// fallback.  Same definition as everywhere: row j of request r sees keys 0..u_r+j.
#include <cuda_fp16.h>

#include "common.cuh"
#include "ptx.cuh"

namespace ss {

constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;

__device__ __forceinline__ float bf16_bits_to_float(uint32_t hi16) { return __uint_as_float(hi16 << 16); }

// two E4M3 codes (low 16 bits) -> two floats, exact
__device__ __forceinline__ float2 e4m3x2_to_float2(uint32_t pair) {
    const uint32_t h2 = ptx::e4m3x2_to_f16x2(pair);
    return __half22float2(*reinterpret_cast<const __half2*>(&h2));
}

// FP8: the caches hold E4M3 codes (one byte per element) with one fp32 scale per (tensor, kv head): K = code * k_scale[g]
// (folded into the score scale), V = code * v_scale[g] (folded into the final normalisation).  DESIGN.md reading 23.
template <int D, bool FP8>
__global__ void __launch_bounds__(128)
simple_attention_kernel(const __nv_bfloat16* __restrict__ q, const void* __restrict__ k_cache_v,
                        const void* __restrict__ v_cache_v, const float* __restrict__ k_scale,
                        const float* __restrict__ v_scale, const int32_t* __restrict__ block_table,
                        const int32_t* __restrict__ qsl, const int32_t* __restrict__ ctx_lens, int R, int T,
                        int Hq, int Hkv, int max_pages, float scale, __nv_bfloat16* __restrict__ out,
                        float* __restrict__ lse, int prefill_only, const int32_t* __restrict__ err_flag) {
    constexpr int EPL = D / 32;                       // output elements per lane
    if (err_flag && *reinterpret_cast<const volatile int32_t*>(err_flag) != 0) return;   // tripped debug check: touch nothing
    __shared__ float s_q[4][D];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t unit = (int64_t)blockIdx.x * 4 + warp;   // (row, head)
    if (unit >= (int64_t)T * Hq) return;
    const int row = (int)(unit / Hq), h = (int)(unit % Hq);
    const int g = h / (Hq / Hkv);

    int lo = 0, hi = R;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (__ldg(qsl + mid) <= row) lo = mid; else hi = mid;
    }
    const int r = lo;
    if (prefill_only && __ldg(qsl + r + 1) - __ldg(qsl + r) <= 1) return;   // decode rows are served by K4
    const int n = __ldg(ctx_lens + r) + (row - __ldg(qsl + r)) + 1;      // visible keys
    const int32_t* bt = block_table + (int64_t)r * max_pages;

    const __nv_bfloat16* qrow = q + ((int64_t)row * Hq + h) * D;
    for (int d = lane; d < D; d += 32) s_q[warp][d] = __bfloat162float(qrow[d]);
    __syncwarp();

    const __nv_bfloat16* k_cache = static_cast<const __nv_bfloat16*>(k_cache_v);
    const __nv_bfloat16* v_cache = static_cast<const __nv_bfloat16*>(v_cache_v);
    const uint8_t* k_codes = static_cast<const uint8_t*>(k_cache_v);
    const uint8_t* v_codes = static_cast<const uint8_t*>(v_cache_v);
    const float sl2 = scale * kLog2e * (FP8 ? __ldg(k_scale + g) : 1.f);
    float m = -INFINITY, l = 0.f, acc[EPL];
#pragma unroll
    for (int e = 0; e < EPL; ++e) acc[e] = 0.f;

    for (int base = 0; base < n; base += 32) {
        const int t = base + lane;
        const bool valid = t < n;
        int64_t row_off = 0;
        float s = -INFINITY;
        if (valid) {
            const int64_t page = __ldg(bt + (t >> 4));
            row_off = ((page * Hkv + g) * kPage + (t & 15)) * (int64_t)D;
            float dot = 0.f;
            if (FP8) {
                const uint2* kr = reinterpret_cast<const uint2*>(k_codes + row_off);
#pragma unroll 4
                for (int v = 0; v < D / 8; ++v) {
                    const uint2 w = __ldg(kr + v);
                    const float* qq = &s_q[warp][v * 8];
                    const float2 a = e4m3x2_to_float2(w.x), b = e4m3x2_to_float2(w.x >> 16);
                    const float2 c = e4m3x2_to_float2(w.y), d = e4m3x2_to_float2(w.y >> 16);
                    dot += qq[0] * a.x + qq[1] * a.y + qq[2] * b.x + qq[3] * b.y;
                    dot += qq[4] * c.x + qq[5] * c.y + qq[6] * d.x + qq[7] * d.y;
                }
            } else {
            const uint4* kr = reinterpret_cast<const uint4*>(k_cache + row_off);
#pragma unroll 4
            for (int v = 0; v < D / 8; ++v) {
                const uint4 w = __ldg(kr + v);
                const float* qq = &s_q[warp][v * 8];
                dot += qq[0] * bf16_bits_to_float(w.x & 0xffffu) + qq[1] * bf16_bits_to_float(w.x >> 16);
                dot += qq[2] * bf16_bits_to_float(w.y & 0xffffu) + qq[3] * bf16_bits_to_float(w.y >> 16);
                dot += qq[4] * bf16_bits_to_float(w.z & 0xffffu) + qq[5] * bf16_bits_to_float(w.z >> 16);
                dot += qq[6] * bf16_bits_to_float(w.w & 0xffffu) + qq[7] * bf16_bits_to_float(w.w >> 16);
            }
            }
            s = dot * sl2;
        }
        float bm = s;
#pragma unroll
        for (int o = 16; o; o >>= 1) bm = fmaxf(bm, __shfl_xor_sync(0xffffffffu, bm, o));
        const float m_new = fmaxf(m, bm);                 // finite: lane 0 of every block is valid
        const float alpha = exp2f(m - m_new);             // exp2(-inf) = 0 on the first block
        const float p = valid ? exp2f(s - m_new) : 0.f;
        float ps = p;
#pragma unroll
        for (int o = 16; o; o >>= 1) ps += __shfl_xor_sync(0xffffffffu, ps, o);
        l = l * alpha + ps;
#pragma unroll
        for (int e = 0; e < EPL; ++e) acc[e] *= alpha;
        m = m_new;
        const int cnt = min(32, n - base);
        for (int i = 0; i < cnt; ++i) {
            const float pi = __shfl_sync(0xffffffffu, p, i);
            const int64_t off = __shfl_sync(0xffffffffu, row_off, i);
            if (FP8) {
                static_assert(!FP8 || EPL == 4, "FP8 path: 4 codes per lane");
                const float2 a = e4m3x2_to_float2(*reinterpret_cast<const uint32_t*>(v_codes + off + lane * EPL));
                const float2 b = e4m3x2_to_float2(*reinterpret_cast<const uint32_t*>(v_codes + off + lane * EPL) >> 16);
                acc[0] += pi * a.x; acc[1] += pi * a.y; acc[2 % EPL] += pi * b.x; acc[3 % EPL] += pi * b.y;
            } else {
                const __nv_bfloat16* vr = v_cache + off + lane * EPL;
#pragma unroll
                for (int e = 0; e < EPL; ++e) acc[e] += pi * __bfloat162float(vr[e]);
            }
        }
    }
    const float inv = (FP8 ? __ldg(v_scale + g) : 1.f) / l;
    __nv_bfloat16* orow = out + ((int64_t)row * Hq + h) * D + lane * EPL;
#pragma unroll
    for (int e = 0; e < EPL; ++e) orow[e] = __float2bfloat16_rn(acc[e] * inv);
    if (lse && lane == 0) lse[(int64_t)row * Hq + h] = (m + log2f(l)) * kLn2;
}

cudaError_t launch_simple_attention(const Handle* h, const void* q, const int32_t* bt, const int32_t* qsl,
                                    const int32_t* ctx, int R, int T, float scale, void* out, float* lse,
                                    cudaStream_t stream, int prefill_only) {
    const ss_config& c = h->cfg;
    const int64_t units = (int64_t)T * c.num_q_heads;
    const unsigned blocks = (unsigned)((units + 3) / 4);
    const int32_t* err = h->debug_checks ? h->state + kStateErr : nullptr;
    if (h->kv_fp8)
        simple_attention_kernel<128, true><<<blocks, 128, 0, stream>>>(
            (const __nv_bfloat16*)q, h->k_cache, h->v_cache, h->k_scale, h->v_scale, bt, qsl, ctx, R, T, c.num_q_heads,
            c.num_kv_heads, c.max_pages_per_req, scale, (__nv_bfloat16*)out, lse, prefill_only, err);
    else if (c.head_dim == 128)
        simple_attention_kernel<128, false><<<blocks, 128, 0, stream>>>(
            (const __nv_bfloat16*)q, h->k_cache, h->v_cache, nullptr, nullptr, bt, qsl, ctx, R, T, c.num_q_heads,
            c.num_kv_heads, c.max_pages_per_req, scale, (__nv_bfloat16*)out, lse, prefill_only, err);
    else
        simple_attention_kernel<64, false><<<blocks, 128, 0, stream>>>(
            (const __nv_bfloat16*)q, h->k_cache, h->v_cache, nullptr, nullptr, bt, qsl, ctx, R, T, c.num_q_heads,
            c.num_kv_heads, c.max_pages_per_req, scale, (__nv_bfloat16*)out, lse, prefill_only, err);
    return cudaGetLastError();
}

}  // namespace ss
