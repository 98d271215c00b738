// ss_mixed_attention_static (include/slidingattn.h): the attention step for callers that cannot allocate device memory.
//
// The regular route needs two pieces of scratch: the handle's queue tickets / split-arrival counters (ss_create
// cudaMallocs them) and the caller's workspace (work list + split-KV partials).  A serving engine that hands every free
// byte of HBM to its paged KV cache at start-up has nothing left to cudaMalloc from when an iteration runs, and a
// cudaMalloc on the iteration path would stall every stream of the device anyway.  For such callers both pieces live
// in ONE array that is part of the library image, g_static_scratch below: SS_STATIC_SCRATCH_BYTES on every GPU that
// loads the library, from load to process exit.  This file calls no cudaMalloc / cudaFree and builds its handle on the
// host stack; the kernels are the ones ss_mixed_attention launches (attn_mixed.cu, worklist.cu), given other pointers.
#include <math.h>
#include <mutex>
#include <stdarg.h>
#include <string.h>

#include "common.cuh"

using namespace ss;

namespace {

// The scratch itself.  In host code this NAME is only a stand-in the runtime uses to look the array up - it is not a
// device address, and a kernel handed `g_static_scratch` from the host would read or write the wrong memory.  Host code
// below therefore only ever uses the pointer cudaGetSymbolAddress returned for the current device (device_setup).
static __device__ __align__(256) unsigned char g_static_scratch[SS_STATIC_SCRATCH_BYTES];

constexpr int kMaxDevices = 64;
struct DeviceSetup {
    bool ready;
    unsigned char* scratch;      // device address of g_static_scratch ON THIS DEVICE (every device has its own copy)
    int num_sms;
};
DeviceSetup g_setup[kMaxDevices];
std::mutex g_setup_mutex;

int fail(char* msg, size_t len, int code, const char* fmt, ...) {
    if (msg && len) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(msg, len, fmt, ap);
        va_end(ap);
    }
    return code;
}

// Once per device, with that device current: resolve the array's device address, read the SM count, opt the main
// kernel in to its shared-memory window.  Nothing here allocates on our side (the runtime loads the module image - the
// array included - the first time any symbol of it is touched on a device).
int device_setup(const DeviceSetup** out, char* msg, size_t len) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(msg, len, SS_ERR_CUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices) return fail(msg, len, SS_ERR_UNSUPPORTED_DEVICE, "device ordinal %d outside [0, %d)", dev, kMaxDevices);
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    DeviceSetup& s = g_setup[dev];
    if (!s.ready) {
        int major = 0, sms = 0;
        if ((e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev)) != cudaSuccess ||
            (e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess)
            return fail(msg, len, SS_ERR_CUDA, "cudaDeviceGetAttribute: %s", cudaGetErrorString(e));
        if (major != 10) return fail(msg, len, SS_ERR_UNSUPPORTED_DEVICE, "device %d is compute capability %d.x, need 10.x", dev, major);
        unsigned char* ptr = nullptr;
        e = cudaGetSymbolAddress((void**)&ptr, g_static_scratch);
        if (e != cudaSuccess || !ptr)
            return fail(msg, len, SS_ERR_CUDA, "cudaGetSymbolAddress(static scratch) on device %d: %s", dev, cudaGetErrorString(e));
        if ((e = init_main_attention(64, 0)) != cudaSuccess || (e = init_main_attention(128, 0)) != cudaSuccess)
            return fail(msg, len, SS_ERR_CUDA, "cudaFuncSetAttribute: %s", cudaGetErrorString(e));
        s.scratch = ptr;
        s.num_sms = sms;
        s.ready = true;
    }
    *out = &s;
    return SS_OK;
}

bool aligned16(const void* p) { return (((uintptr_t)p) & 15u) == 0; }
bool aligned4(const void* p) { return (((uintptr_t)p) & 3u) == 0; }

}  // namespace

extern "C" int ss_mixed_attention_static(const ss_config* cfg, void* k_cache, void* v_cache, const void* q,
                                         const int32_t* block_table, const int32_t* query_start_loc,
                                         const int32_t* ctx_lens, int32_t R, int32_t T, float scale, void* out,
                                         float* lse_or_null, void* cuda_stream, char* err_msg, size_t err_msg_len) {
    if (err_msg && err_msg_len) err_msg[0] = 0;
    // the config rules of ss_create, minus the two flags this entry point does not serve
    if (!cfg || !k_cache || !v_cache || !aligned16(k_cache) || !aligned16(v_cache))
        return fail(err_msg, err_msg_len, SS_ERR_INVALID_ARG, "null or misaligned config / cache pointer");
    if (cfg->page_size != kPage || (cfg->head_dim != 64 && cfg->head_dim != 128) || cfg->num_q_heads <= 0 ||
        cfg->num_kv_heads <= 0 || cfg->num_q_heads % cfg->num_kv_heads || cfg->num_q_heads / cfg->num_kv_heads > kMaxGroup ||
        cfg->num_pages <= 0 || cfg->max_requests <= 0 || cfg->max_requests > 2048 || cfg->max_tokens <= 0 ||
        cfg->max_pages_per_req <= 0 || (int64_t)cfg->max_pages_per_req * kPage > (int64_t)1 << 30)
        return fail(err_msg, err_msg_len, SS_ERR_INVALID_ARG, "config outside what ss_create accepts");
    if (cfg->flags != 0)
        return fail(err_msg, err_msg_len, SS_ERR_INVALID_ARG, "flags must be 0: the static-scratch entry point serves bf16 caches without device checks");
    if (R < 0 || T < 0 || R > cfg->max_requests || T > cfg->max_tokens)
        return fail(err_msg, err_msg_len, SS_ERR_INVALID_ARG, "R = %d / T = %d outside the config's bounds", R, T);
    if (R == 0 || T == 0) return SS_OK;
    if (!q || !out || !block_table || !query_start_loc || !ctx_lens || !aligned16(q) || !aligned16(out) ||
        !aligned4(block_table) || !aligned4(query_start_loc) || !aligned4(ctx_lens) || (lse_or_null && !aligned4(lse_or_null)))
        return fail(err_msg, err_msg_len, SS_ERR_INVALID_ARG, "null or misaligned batch pointer");
    if (!(scale > 0.f) || !isfinite(scale)) return fail(err_msg, err_msg_len, SS_ERR_INVALID_ARG, "scale must be finite and > 0");

    const DeviceSetup* dev = nullptr;
    int rc = device_setup(&dev, err_msg, err_msg_len);
    if (rc != SS_OK) return rc;

    // A handle on the host stack: the launchers only read it, and the kernels get their parameters by value.
    Handle h;
    memset(&h, 0, sizeof h);
    h.cfg = *cfg;
    h.num_sms = dev->num_sms;
    h.group = cfg->num_q_heads / cfg->num_kv_heads;
    h.k_cache = k_cache;
    h.v_cache = v_cache;
    h.ws = workspace_layout(h.cfg, h.num_sms);
    if (!h.ws.ok) return fail(err_msg, err_msg_len, SS_ERR_INVALID_ARG, "worst-case item count of this config overflows int32");

    // [0, state_bytes): what ss_create would have cudaMalloc'ed (queue tickets, error record, arrival counters);
    // [state_bytes, state_bytes + ws.total): what the caller of ss_mixed_attention would have passed as workspace.
    const size_t state_bytes =
        (sizeof(int32_t) * ((size_t)kStateCounters + (size_t)cfg->max_requests * cfg->num_kv_heads) + 255) & ~(size_t)255;
    const size_t need = state_bytes + h.ws.total;
    if (need > (size_t)SS_STATIC_SCRATCH_BYTES)
        return fail(err_msg, err_msg_len, SS_ERR_WORKSPACE_TOO_SMALL,
                    "this config needs %zu bytes of scratch, the library's static array holds %zu (SS_STATIC_SCRATCH_BYTES): "
                    "lower max_requests / max_tokens / max_pages_per_req, or use ss_create + ss_mixed_attention with your own workspace",
                    need, (size_t)SS_STATIC_SCRATCH_BYTES);
    h.state = (int32_t*)dev->scratch;
    h.state_bytes = state_bytes;
    void* workspace = dev->scratch + state_bytes;

    if ((rc = encode_cache_map(&h, &h.tmap_k, k_cache)) != SS_OK || (rc = encode_cache_map(&h, &h.tmap_v, v_cache)) != SS_OK)
        return fail(err_msg, err_msg_len, rc, "%s", h.err);
    h.have_tmaps = true;

    cudaStream_t st = (cudaStream_t)cuda_stream;
    // The array keeps whatever the previous call (any config) left in it.  The tickets and arrival counters must start
    // at zero and a different config puts them elsewhere, so they are cleared here, in stream order before the kernels;
    // the work list and the partials are written before they are read and need no clearing.
    cudaError_t e = cudaMemsetAsync(h.state, 0, state_bytes, st);
    if (e != cudaSuccess) return fail(err_msg, err_msg_len, SS_ERR_CUDA, "state clear: %s", cudaGetErrorString(e));
    if (!main_self_plans(&h, R, T)) {
        e = launch_worklist(&h, query_start_loc, ctx_lens, R, T, workspace, st);
        if (e != cudaSuccess) return fail(err_msg, err_msg_len, SS_ERR_CUDA, "worklist launch: %s", cudaGetErrorString(e));
    }
    int n = 0;
    e = launch_main_attention(&h, q, block_table, query_start_loc, ctx_lens, R, T, scale, out, lse_or_null, workspace, st, &n);
    if (e != cudaSuccess) return fail(err_msg, err_msg_len, SS_ERR_CUDA, "main attention launch: %s", cudaGetErrorString(e));
    return SS_OK;
}
