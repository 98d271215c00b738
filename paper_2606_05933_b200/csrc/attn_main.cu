// Main attention path dispatcher (a3 prefill tiles, a4 decode splits, a5 merge).
#include "common.cuh"

namespace ss {

cudaError_t launch_main_attention(const Handle* h, const void* q, const int32_t* bt, const int32_t* qsl,
                                  const int32_t* ctx, int R, int T, float scale, void* out, float* lse,
                                  void* workspace, cudaStream_t stream, int* n_launches) {
    cudaError_t e = launch_decode(h, q, bt, scale, workspace, out, lse, stream);
    if (e != cudaSuccess) return e;
    e = launch_merge(h, qsl, R, workspace, out, lse, stream);
    if (e != cudaSuccess) return e;
    e = launch_prefill(h, q, bt, ctx, T, scale, workspace, out, lse, stream);
    *n_launches = 3;
    return e;
}

}  // namespace ss
