// Debug-check kernel of the boundary ("a debug build bounds-checks in-kernel and sets a device flag").
// Runs before ss_kv_append / ss_mixed_attention when the handle was created with SS_FLAG_DEBUG_CHECKS and verifies the
// device-resident metadata the host cannot see without a sync:
//   kChkQsl           query_start_loc[0] == 0, non-decreasing, query_start_loc[R] == T
//   kChkCtxNegative   ctx_lens[r] >= 0
//   kChkTooManyPages  ceil((u_r + c_r) / 16) <= max_pages_per_req            (requests with c_r > 0)
//   kChkPageId        0 <= block_table[r][p] < num_pages for every page p < ceil((u_r + c_r) / 16)
//   kChkKvScale       FP8 handles: k_scale[g], v_scale[g] finite and > 0 (value = the scale's bit pattern; request = g for
//                     k_scale, Hkv + g for v_scale) - the kernels' running max of raw scores needs k_scale > 0
// The first violation wins (atomicCAS on the code word) and records (code, request, offending value, limit).  The hot
// kernels read the code word after their grid-dependency wait and, if it is set, touch neither caches nor outputs;
// the flag stays set until ss_poll_device_error clears it.  Integer work only.
#include "common.cuh"
#include "ptx.cuh"

namespace ss {

constexpr int kValThreads = 256;

__device__ __forceinline__ void report(int32_t* err, int code, int req, long long value, long long limit) {
    if (atomicCAS(err, 0, code) == 0) {
        err[1] = req;
        err[2] = (int32_t)(value > 0x7fffffffll ? 0x7fffffff : (value < -0x7fffffffll ? -0x7fffffff : value));
        err[3] = (int32_t)(limit > 0x7fffffffll ? 0x7fffffff : limit);
    }
}

__global__ void __launch_bounds__(kValThreads)
validate_kernel(const int32_t* __restrict__ block_table, const int32_t* __restrict__ qsl,
                const int32_t* __restrict__ ctx_lens, int R, int T, int max_pages, long long num_pages, int32_t* err,
                const float* __restrict__ k_scale, const float* __restrict__ v_scale, int Hkv) {
    ptx::pdl_wait();
    const int warp = (blockIdx.x * kValThreads + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    const int nwarps = gridDim.x * (kValThreads / 32);
    if (k_scale && blockIdx.x == 0)
        for (int i = threadIdx.x; i < 2 * Hkv; i += kValThreads) {
            const float s = i < Hkv ? __ldg(k_scale + i) : __ldg(v_scale + i - Hkv);
            if (!(s > 0.f) || !(s <= 3.4028234e38f)) report(err, kChkKvScale, i, (long long)__float_as_int(s), 0);   // NaN fails both
        }
    if (warp == 0 && lane == 0) {
        if (__ldg(qsl) != 0) report(err, kChkQsl, 0, __ldg(qsl), 0);
        if (__ldg(qsl + R) != T) report(err, kChkQsl, R, __ldg(qsl + R), T);
    }
    for (int r = warp; r < R; r += nwarps) {
        const long long q0 = __ldg(qsl + r), q1 = __ldg(qsl + r + 1), u = __ldg(ctx_lens + r);
        const long long c = q1 - q0;
        bool ok = true;
        if (c < 0 || q0 < 0 || q1 > T) { if (lane == 0) report(err, kChkQsl, r, q1, q0); ok = false; }
        if (u < 0) { if (lane == 0) report(err, kChkCtxNegative, r, u, 0); ok = false; }
        if (!ok || c == 0) continue;
        const long long need = (u + c + kPage - 1) / kPage;
        if (need > max_pages) { if (lane == 0) report(err, kChkTooManyPages, r, need, max_pages); continue; }
        const int32_t* row = block_table + (int64_t)r * max_pages;
        for (int p = lane; p < (int)need; p += 32) {
            const long long pg = __ldg(row + p);
            if (pg < 0 || pg >= num_pages) report(err, kChkPageId, r, pg, num_pages);
        }
    }
}

cudaError_t launch_validate(const Handle* h, const int32_t* bt, const int32_t* qsl, const int32_t* ctx, int R, int T,
                            cudaStream_t stream) {
    const int warps_per_cta = kValThreads / 32;
    int grid = (R + warps_per_cta - 1) / warps_per_cta;
    if (grid > 4 * h->num_sms) grid = 4 * h->num_sms;
    if (grid < 1) grid = 1;
    validate_kernel<<<grid, kValThreads, 0, stream>>>(bt, qsl, ctx, R, T, h->cfg.max_pages_per_req,
                                                      (long long)h->cfg.num_pages, h->state + kStateErr,
                                                      h->kv_fp8 ? h->k_scale : nullptr, h->v_scale, h->cfg.num_kv_heads);
    return cudaGetLastError();
}

}  // namespace ss
