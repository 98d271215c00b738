// Shared by the append kernels (a1 and its RoPE / FP8 variants): token -> request lookup.
#pragma once
#include "common.cuh"

namespace ss {

constexpr int kAppendThreads = 128;

// Request of token `tok`: the last r with qsl[r] <= tok (requests with c_r = 0 are skipped by construction).  Every
// thread of the CTA calls it.  The CTA counts the entries <= tok with independent loads - one memory round trip
// instead of the log2(R) dependent ones of a binary search, which after an L2 flush was most of the kernel's latency.
__device__ __forceinline__ int request_of_token(const int32_t* __restrict__ qsl, int R, int tok) {
    __shared__ int s_cnt;
    if (threadIdx.x == 0) s_cnt = 0;
    __syncthreads();
    int n = 0;
    for (int r = threadIdx.x; r < R; r += kAppendThreads) n += (__ldg(qsl + r) <= tok) ? 1 : 0;
    n = __reduce_add_sync(0xffffffffu, n);
    if ((threadIdx.x & 31) == 0 && n) atomicAdd(&s_cnt, n);
    __syncthreads();
    return s_cnt - 1;
}

}  // namespace ss
