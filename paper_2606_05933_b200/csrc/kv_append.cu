// K1 kv_append (a1; PAPER.md:99 step 10 — request r's cached length grows by c_r).
// One CTA per (token, K|V): the token's Hkv*D bf16 row is moved as 16-byte vectors straight into its
// page slot.  Integer index math + bit copies only (never through a float type) => bit-exact.
// Roofline: HBM; algorithmic bytes = 4*T*Hkv*D*2 (read + write, K and V).
#include "append.cuh"
#include "common.cuh"
#include "ptx.cuh"

namespace ss {

__global__ void __launch_bounds__(kAppendThreads)
kv_append_kernel(const uint4* __restrict__ k_new, const uint4* __restrict__ v_new,
                 uint4* __restrict__ k_cache, uint4* __restrict__ v_cache,
                 const int32_t* __restrict__ block_table, const int32_t* __restrict__ qsl,
                 const int32_t* __restrict__ ctx_lens, int R, int max_pages, int Hkv, int vec_per_head,
                 const int32_t* __restrict__ err_flag) {
    ptx::pdl_launch_dependents();
    ptx::pdl_wait();
    if (err_flag && *reinterpret_cast<const volatile int32_t*>(err_flag)) return;    // debug checks tripped: write nothing
    const int tok = blockIdx.x;
    const uint4* __restrict__ src = blockIdx.y ? v_new : k_new;
    uint4* __restrict__ dst = blockIdx.y ? v_cache : k_cache;

    // the token's first vectors are requested before the (dependent) metadata chain, so the two overlap
    const int vec_per_tok = Hkv * vec_per_head;
    const uint4* s = src + (int64_t)tok * vec_per_tok;
    uint4 first = make_uint4(0u, 0u, 0u, 0u);
    if ((int)threadIdx.x < vec_per_tok) first = __ldg(s + threadIdx.x);

    const int r = request_of_token(qsl, R, tok);
    const int pos = __ldg(ctx_lens + r) + (tok - __ldg(qsl + r));
    const int64_t page = __ldg(block_table + (int64_t)r * max_pages + (pos >> 4));
    const int slot = pos & (kPage - 1);

    for (int v = threadIdx.x; v < vec_per_tok; v += kAppendThreads) {
        const int g = v / vec_per_head;
        const int dv = v - g * vec_per_head;
        const int64_t d = ((page * Hkv + g) * kPage + slot) * (int64_t)vec_per_head + dv;
        dst[d] = v == (int)threadIdx.x ? first : __ldg(s + v);
    }
}

// FP8 variant (SS_FLAG_KV_FP8, reading 23): the same placement, each bf16 element quantised to an E4M3 code,
// code = e4m3_rne_satfinite(x / scale[g]) with the quotient an IEEE fp32 division (the precision in which the oracle
// takes the decision too).  One thread = 8 elements: 16 bytes in, 8 bytes out.  Bit-exact against the oracle.
__global__ void __launch_bounds__(kAppendThreads)
kv_append_fp8_kernel(const uint4* __restrict__ k_new, const uint4* __restrict__ v_new, uint2* __restrict__ k_cache,
                     uint2* __restrict__ v_cache, const float* __restrict__ k_scale, const float* __restrict__ v_scale,
                     const int32_t* __restrict__ block_table, const int32_t* __restrict__ qsl,
                     const int32_t* __restrict__ ctx_lens, int R, int max_pages, int Hkv, int vec_per_head,
                     const int32_t* __restrict__ err_flag) {
    ptx::pdl_launch_dependents();
    ptx::pdl_wait();
    if (err_flag && *reinterpret_cast<const volatile int32_t*>(err_flag)) return;
    const int tok = blockIdx.x;
    const uint4* __restrict__ src = blockIdx.y ? v_new : k_new;
    uint2* __restrict__ dst = blockIdx.y ? v_cache : k_cache;
    const float* __restrict__ scale = blockIdx.y ? v_scale : k_scale;
    const int r = request_of_token(qsl, R, tok);
    const int pos = __ldg(ctx_lens + r) + (tok - __ldg(qsl + r));
    const int64_t page = __ldg(block_table + (int64_t)r * max_pages + (pos >> 4));
    const int slot = pos & (kPage - 1);
    const int vec_per_tok = Hkv * vec_per_head;
    const uint4* s = src + (int64_t)tok * vec_per_tok;
    for (int v = threadIdx.x; v < vec_per_tok; v += kAppendThreads) {
        const int g = v / vec_per_head;
        const int dv = v - g * vec_per_head;
        const float sc = __ldg(scale + g);
        const uint4 w = __ldg(s + v);
        const uint32_t in[4] = {w.x, w.y, w.z, w.w};
        uint32_t out[2] = {0u, 0u};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float lo = __uint_as_float(in[i] << 16), hi = __uint_as_float(in[i] & 0xffff0000u);   // exact widening
            const uint32_t c2 = ptx::f32x2_to_e4m3x2(ptx::div_rn_ieee(lo, sc), ptx::div_rn_ieee(hi, sc));
            out[i >> 1] |= c2 << (16 * (i & 1));
        }
        dst[((page * Hkv + g) * kPage + slot) * (int64_t)vec_per_head + dv] = make_uint2(out[0], out[1]);
    }
}

cudaError_t launch_kv_append(const Handle* h, const void* k_new, const void* v_new, const int32_t* bt,
                             const int32_t* qsl, const int32_t* ctx, int R, int T, cudaStream_t stream) {
    const ss_config& c = h->cfg;
    dim3 grid((unsigned)T, 2, 1);
    if (h->kv_fp8)
        return launch_pdl(kv_append_fp8_kernel, grid, dim3(kAppendThreads), 0, stream, (const uint4*)k_new, (const uint4*)v_new,
                          (uint2*)h->k_cache, (uint2*)h->v_cache, h->k_scale, h->v_scale, bt, qsl, ctx, R, c.max_pages_per_req,
                          c.num_kv_heads, c.head_dim / 8, (const int32_t*)(h->debug_checks ? h->state + kStateErr : nullptr));
    return launch_pdl(kv_append_kernel, grid, dim3(kAppendThreads), 0, stream, (const uint4*)k_new, (const uint4*)v_new,
                      (uint4*)h->k_cache, (uint4*)h->v_cache, bt, qsl, ctx, R, c.max_pages_per_req, c.num_kv_heads,
                      c.head_dim / 8, (const int32_t*)(h->debug_checks ? h->state + kStateErr : nullptr));
}

}  // namespace ss
