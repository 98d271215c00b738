// Measurement aid (include/slidingattn_debug.h, ss_debug_stream_read): a read-only streaming pass over a device buffer.
// The HBM roofline of the decode path is a READ roofline - the path reads every visible K / V row once and writes almost
// nothing - while MEASURED_PEAKS.json's hbm_gbs is a copy (read + write) figure, which the decode kernel beats (C4:
// 1.09 of it).  bench.py times this kernel next to the workload and reports fractions against max(copy peak, this)
// as well, so that no HBM fraction can exceed 1.  No arithmetic of the method here.
#include "common.cuh"
#include "ptx.cuh"

namespace ss {

constexpr int kProbeChunk = 16 * 1024;   // bytes per bulk copy
constexpr int kProbeStages = 12;         // 192 KB in flight per SM, one CTA per SM

// One thread per CTA keeps kProbeStages bulk copies (global -> shared, cp.async.bulk) in flight and re-arms a stage as
// soon as its bytes have landed; nobody consumes the data.  Chunks are interleaved across the CTAs.  This is the access
// pattern of the decode path (TMA slabs into a shared-memory ring) without any of its work.
__global__ void __launch_bounds__(32)
stream_read_kernel(const char* __restrict__ src, size_t nchunks) {
    extern __shared__ __align__(128) char stage[];
    __shared__ __align__(8) uint64_t bars[kProbeStages];
    if (threadIdx.x != 0) return;
    for (int s = 0; s < kProbeStages; ++s) ptx::mbar_init(ptx::smem_u32(&bars[s]), 1);
    ptx::fence_barrier_init();
    size_t next = blockIdx.x;
    for (int s = 0; s < kProbeStages && next < nchunks; ++s, next += gridDim.x) {
        ptx::mbar_arrive_expect_tx(ptx::smem_u32(&bars[s]), kProbeChunk);
        ptx::bulk_load_1d(ptx::smem_u32(stage + s * kProbeChunk), src + next * kProbeChunk, kProbeChunk, ptx::smem_u32(&bars[s]));
    }
    int s = 0;
    uint32_t phase = 0;
    for (size_t done = blockIdx.x; done < nchunks; done += gridDim.x) {
        ptx::mbar_wait(ptx::smem_u32(&bars[s]), phase);
        if (next < nchunks) {
            ptx::mbar_arrive_expect_tx(ptx::smem_u32(&bars[s]), kProbeChunk);
            ptx::bulk_load_1d(ptx::smem_u32(stage + s * kProbeChunk), src + next * kProbeChunk, kProbeChunk, ptx::smem_u32(&bars[s]));
            next += gridDim.x;
        }
        if (++s == kProbeStages) { s = 0; phase ^= 1u; }
    }
}

}  // namespace ss

extern "C" int ss_debug_stream_read(ss_handle* hh, const void* buf, size_t bytes, void* cuda_stream) {
    ss::Handle* h = (ss::Handle*)hh;
    if (!h || !buf || (((uintptr_t)buf) & 15u) || bytes < (size_t)ss::kProbeChunk) return SS_ERR_INVALID_ARG;
    const int smem = ss::kProbeChunk * ss::kProbeStages;
    if (cudaFuncSetAttribute(ss::stream_read_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) return SS_ERR_CUDA;
    ss::stream_read_kernel<<<h->num_sms, 32, smem, (cudaStream_t)cuda_stream>>>((const char*)buf, bytes / ss::kProbeChunk);
    return cudaGetLastError() == cudaSuccess ? SS_OK : SS_ERR_CUDA;
}
