// C ABI of libslidingattn (include/slidingattn.h): argument checks, handle, launch sequencing.
// No arithmetic of the method lives here; every step of the path runs in the kernels.
#include <math.h>
#include <new>
#include <string.h>

#include "common.cuh"

using namespace ss;

namespace {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

bool aligned16(const void* p) { return (((uintptr_t)p) & 15u) == 0; }

int fail_cuda(Handle* h, cudaError_t e, const char* where) {
    if (h) snprintf(h->err, sizeof h->err, "%s: %s", where, cudaGetErrorString(e));
    return SS_ERR_CUDA;
}

#define SS_CUDA(h, call, where)                                  \
    do {                                                         \
        cudaError_t e__ = (call);                                \
        if (e__ != cudaSuccess) return fail_cuda(h, e__, where); \
    } while (0)

int check_batch_args(const Handle* h, const void* a, const void* b, const void* c, const void* d, int R, int T) {
    if (!h) return SS_ERR_INVALID_ARG;
    if (R < 0 || T < 0 || R > h->cfg.max_requests || T > h->cfg.max_tokens) return SS_ERR_INVALID_ARG;
    if (R == 0 || T == 0) return SS_OK;
    if (!a || !b || !c || !d) return SS_ERR_INVALID_ARG;
    if (!aligned16(a) || !aligned16(b)) return SS_ERR_INVALID_ARG;
    if ((((uintptr_t)c) & 3u) || (((uintptr_t)d) & 3u)) return SS_ERR_INVALID_ARG;
    return SS_OK;
}

}  // namespace

// KV cache [num_pages][Hkv][16][D] bf16 viewed as a 4-D tensor (innermost first): 64 columns of a 128-byte half row,
// 8 rows of an 8-key group (stride D*2 bytes), D/64 halves (stride 128 bytes), 8-key groups (stride 8*D*2 bytes; a
// (page, kv head) slab is two consecutive groups).  One TMA box = one whole slab: 2 groups x halves x 8 rows x 64
// columns, written to shared memory as [group][half][8 rows][128 B] with SWIZZLE_128B - every [8 rows][128 B] block is a
// canonical UMMA / ldmatrix core group, groups uniformly D/64 KB apart.  One operation per slab instead of one per
// (slab, half): the per-SM copy engine costs ~31 ns per operation whatever its size (profiles/r2b.md).
int ss::encode_cache_map(Handle* h, CUtensorMap* map, void* base) {
    EncodeTiledFn enc = get_encode_fn();
    if (!enc) {
        snprintf(h->err, sizeof h->err, "cuTensorMapEncodeTiled entry point not found");
        return SS_ERR_CUDA;
    }
    const ss_config& c = h->cfg;
    // FP8 cache: a row is head_dim bytes; the same map in units of 2-byte words (64 words = 128 bytes per half row)
    const cuuint64_t row_bytes = (cuuint64_t)c.head_dim * (h->kv_fp8 ? 1 : 2);
    const cuuint32_t halves = (cuuint32_t)(row_bytes / 128);
    cuuint64_t gdim[4] = {64, 8, halves, (cuuint64_t)c.num_pages * c.num_kv_heads * 2};
    cuuint64_t gstride[3] = {row_bytes, 128, row_bytes * 8};
    cuuint32_t box[4] = {64u, 8u, halves, 2u};
    cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
    CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, base, gdim, gstride, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(h->err, sizeof h->err, "cuTensorMapEncodeTiled failed: %d", (int)r);
        return SS_ERR_CUDA;
    }
    return SS_OK;
}

extern "C" {

int ss_version(void) { return SS_VERSION; }

const char* ss_status_string(int s) {
    switch (s) {
        case SS_OK: return "SS_OK";
        case SS_ERR_INVALID_ARG: return "SS_ERR_INVALID_ARG";
        case SS_ERR_WORKSPACE_TOO_SMALL: return "SS_ERR_WORKSPACE_TOO_SMALL";
        case SS_ERR_UNSUPPORTED_DEVICE: return "SS_ERR_UNSUPPORTED_DEVICE";
        case SS_ERR_CUDA: return "SS_ERR_CUDA";
        case SS_ERR_NOT_IMPLEMENTED: return "SS_ERR_NOT_IMPLEMENTED";
        case SS_ERR_DEVICE_CHECK: return "SS_ERR_DEVICE_CHECK";
        default: return "SS_ERR_UNKNOWN";
    }
}

const char* ss_last_error_string(const ss_handle* hh) {
    const Handle* h = (const Handle*)hh;
    return h ? h->err : "null handle";
}

int ss_create(ss_handle** out_handle, const ss_config* cfg, void* k_cache, void* v_cache) {
    if (!out_handle) return SS_ERR_INVALID_ARG;
    *out_handle = nullptr;
    if (!cfg || !k_cache || !v_cache || !aligned16(k_cache) || !aligned16(v_cache)) return SS_ERR_INVALID_ARG;
    if (cfg->page_size != kPage) return SS_ERR_INVALID_ARG;
    if (cfg->head_dim != 64 && cfg->head_dim != 128) return SS_ERR_INVALID_ARG;
    if (cfg->num_q_heads <= 0 || cfg->num_kv_heads <= 0 || cfg->num_q_heads % cfg->num_kv_heads) return SS_ERR_INVALID_ARG;
    if (cfg->num_q_heads / cfg->num_kv_heads > kMaxGroup) return SS_ERR_INVALID_ARG;
    if (cfg->num_pages <= 0 || cfg->max_requests <= 0 || cfg->max_requests > 2048 || cfg->max_tokens <= 0 ||
        cfg->max_pages_per_req <= 0)
        return SS_ERR_INVALID_ARG;
    if ((int64_t)cfg->max_pages_per_req * kPage > (int64_t)1 << 30) return SS_ERR_INVALID_ARG;
    if (cfg->flags & ~(uint32_t)(SS_FLAG_DEBUG_CHECKS | SS_FLAG_KV_FP8)) return SS_ERR_INVALID_ARG;
    if ((cfg->flags & SS_FLAG_KV_FP8) && cfg->head_dim != 128) return SS_ERR_INVALID_ARG;
    if (!workspace_layout(*cfg, 256).ok) return SS_ERR_INVALID_ARG;   // worst-case item count must fit the int32 index space

    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return SS_ERR_CUDA;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return SS_ERR_CUDA;
    if (prop.major != 10) return SS_ERR_UNSUPPORTED_DEVICE;

    Handle* h = new (std::nothrow) Handle();
    if (!h) return SS_ERR_CUDA;
    memset(h, 0, sizeof *h);
    h->cfg = *cfg;
    h->device = dev;
    h->num_sms = prop.multiProcessorCount;
    h->group = cfg->num_q_heads / cfg->num_kv_heads;
    h->k_cache = k_cache;
    h->v_cache = v_cache;
    h->debug_checks = (cfg->flags & SS_FLAG_DEBUG_CHECKS) ? 1 : 0;
    h->kv_fp8 = (cfg->flags & SS_FLAG_KV_FP8) ? 1 : 0;
    h->ws = workspace_layout(h->cfg, h->num_sms);
    if (!h->ws.ok) {                 // worst-case item count of this config overflows the int32 index space
        delete h;
        return SS_ERR_INVALID_ARG;
    }
    if (init_main_attention(cfg->head_dim, h->kv_fp8) != cudaSuccess) {
        delete h;
        return SS_ERR_CUDA;
    }
    int rc = encode_cache_map(h, &h->tmap_k, k_cache);
    if (rc == SS_OK) rc = encode_cache_map(h, &h->tmap_v, v_cache);
    if (rc != SS_OK) {
        delete h;
        return rc;
    }
    h->have_tmaps = true;
    const size_t state_bytes = sizeof(int32_t) * ((size_t)kStateCounters + (size_t)cfg->max_requests * cfg->num_kv_heads);
    h->state_bytes = state_bytes;
    if (cudaMalloc((void**)&h->state, state_bytes) != cudaSuccess || cudaMemset(h->state, 0, state_bytes) != cudaSuccess) {
        if (h->state) cudaFree(h->state);
        delete h;
        return SS_ERR_CUDA;
    }
    *out_handle = (ss_handle*)h;
    return SS_OK;
}

int ss_destroy(ss_handle* hh) {
    Handle* h = (Handle*)hh;
    if (!h) return SS_ERR_INVALID_ARG;
    if (h->ev0) cudaEventDestroy(h->ev0);
    if (h->ev1) cudaEventDestroy(h->ev1);
    if (h->state) cudaFree(h->state);
    void* bufs[] = {h->st_q, h->st_knew, h->st_vnew, h->st_out, h->st_ws, h->st_bt, h->st_qsl, h->st_ctx};
    for (void* b : bufs)
        if (b) cudaFree(b);
    delete h;
    return SS_OK;
}

int ss_set_kv_scales(ss_handle* hh, const float* k_scale, const float* v_scale) {
    Handle* h = (Handle*)hh;
    if (!h || !h->kv_fp8 || !k_scale || !v_scale || (((uintptr_t)k_scale) & 3u) || (((uintptr_t)v_scale) & 3u)) return SS_ERR_INVALID_ARG;
    h->k_scale = k_scale;
    h->v_scale = v_scale;
    return SS_OK;
}

size_t ss_workspace_bytes(const ss_handle* hh) {
    const Handle* h = (const Handle*)hh;
    return h ? h->ws.total : 0;
}

int ss_last_launch_count(const ss_handle* hh) {
    const Handle* h = (const Handle*)hh;
    return h ? h->last_launches : 0;
}

int ss_set_kernel_timing(ss_handle* hh, int on) {
    Handle* h = (Handle*)hh;
    if (!h) return SS_ERR_INVALID_ARG;
    if (on && !h->ev0) {
        SS_CUDA(h, cudaEventCreate(&h->ev0), "event create");
        SS_CUDA(h, cudaEventCreate(&h->ev1), "event create");
    }
    h->timing_on = on ? 1 : 0;
    h->timing_valid = 0;
    return SS_OK;
}

int ss_last_kernel_time_us(ss_handle* hh, float* main_us) {
    Handle* h = (Handle*)hh;
    if (!h || !main_us || !h->timing_on || !h->timing_valid) return SS_ERR_INVALID_ARG;
    SS_CUDA(h, cudaEventSynchronize(h->ev1), "timing sync");
    float ms = 0.f;
    SS_CUDA(h, cudaEventElapsedTime(&ms, h->ev0, h->ev1), "timing elapsed");
    *main_us = ms * 1000.f;
    return SS_OK;
}

int ss_debug_force_simple_path(ss_handle* hh, int on) {
    Handle* h = (Handle*)hh;
    if (!h) return SS_ERR_INVALID_ARG;
    h->force_simple = on ? 1 : 0;
    return SS_OK;
}

int ss_debug_set_param(ss_handle* hh, int which, int value) {
    Handle* h = (Handle*)hh;
    if (!h || which < 1 || which >= 8) return SS_ERR_INVALID_ARG;
    if (which == kDbgSplitKeys && value > 0) {
        // the workspace's item / partial slots are sized for the automatic split length; the plan raises a forced
        // length until the batch's splits fit them (plan.cuh), so the knob can never write past the workspace
        value = (value + kTileKeys - 1) / kTileKeys * kTileKeys;
        if (value < kMinSplitKeys) value = kMinSplitKeys;
        if (value > kMaxSplitKeys) value = kMaxSplitKeys;
    }
    h->dbg[which] = value;
    return SS_OK;
}

int ss_debug_set_trace(ss_handle* hh, void* trace_dev, int32_t words_per_cta) {
    Handle* h = (Handle*)hh;
    if (!h || (trace_dev && words_per_cta < 6) || (((uintptr_t)trace_dev) & 7u)) return SS_ERR_INVALID_ARG;
    h->trace = (unsigned long long*)trace_dev;
    h->trace_words = trace_dev ? words_per_cta : 0;
    return SS_OK;
}

int ss_kv_append(ss_handle* hh, const void* k_new, const void* v_new, const int32_t* block_table,
                 const int32_t* query_start_loc, const int32_t* ctx_lens, int32_t R, int32_t T, void* cuda_stream) {
    Handle* h = (Handle*)hh;
    int rc = check_batch_args(h, k_new, v_new, query_start_loc, ctx_lens, R, T);
    if (rc != SS_OK) return rc;
    h->last_launches = 0;
    if (R == 0 || T == 0) return SS_OK;
    if (!block_table || (((uintptr_t)block_table) & 3u)) return SS_ERR_INVALID_ARG;
    if (h->kv_fp8 && !h->k_scale) return SS_ERR_INVALID_ARG;          // ss_set_kv_scales first
    if (h->debug_checks)
        SS_CUDA(h, launch_validate(h, block_table, query_start_loc, ctx_lens, R, T, (cudaStream_t)cuda_stream), "validate launch");
    SS_CUDA(h, launch_kv_append(h, k_new, v_new, block_table, query_start_loc, ctx_lens, R, T, (cudaStream_t)cuda_stream),
            "kv_append launch");
    h->last_launches = 1 + h->debug_checks;
    return SS_OK;
}

int ss_qkv_rope_append(ss_handle* hh, const void* qkv, const int32_t* block_table, const int32_t* query_start_loc,
                       const int32_t* ctx_lens, int32_t R, int32_t T, float rope_theta, void* q_out, void* cuda_stream) {
    Handle* h = (Handle*)hh;
    int rc = check_batch_args(h, qkv, q_out, query_start_loc, ctx_lens, R, T);
    if (rc != SS_OK) return rc;
    h->last_launches = 0;
    if (R == 0 || T == 0) return SS_OK;
    if (!block_table || (((uintptr_t)block_table) & 3u)) return SS_ERR_INVALID_ARG;
    if (!(rope_theta > 1.f) || !isfinite(rope_theta)) return SS_ERR_INVALID_ARG;
    if (h->kv_fp8 && !h->k_scale) return SS_ERR_INVALID_ARG;          // ss_set_kv_scales first
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (h->debug_checks) SS_CUDA(h, launch_validate(h, block_table, query_start_loc, ctx_lens, R, T, st), "validate launch");
    SS_CUDA(h, launch_qkv_rope_append(h, qkv, block_table, query_start_loc, ctx_lens, R, T, rope_theta, q_out, st),
            "qkv_rope_append launch");
    h->last_launches = 1 + h->debug_checks;
    return SS_OK;
}

int ss_mixed_attention(ss_handle* hh, const void* q, const int32_t* block_table, const int32_t* query_start_loc,
                       const int32_t* ctx_lens, int32_t R, int32_t T, float scale, void* out, float* lse_or_null,
                       void* workspace, size_t workspace_bytes, void* cuda_stream) {
    Handle* h = (Handle*)hh;
    int rc = check_batch_args(h, q, out, query_start_loc, ctx_lens, R, T);
    if (rc != SS_OK) return rc;
    h->last_launches = 0;
    if (R == 0 || T == 0) return SS_OK;
    if (!block_table || (((uintptr_t)block_table) & 3u)) return SS_ERR_INVALID_ARG;
    if (lse_or_null && (((uintptr_t)lse_or_null) & 3u)) return SS_ERR_INVALID_ARG;
    if (!workspace || !aligned16(workspace)) return SS_ERR_INVALID_ARG;
    if (workspace_bytes < h->ws.total) return SS_ERR_WORKSPACE_TOO_SMALL;
    if (!(scale > 0.f) || !isfinite(scale)) return SS_ERR_INVALID_ARG;      // see slidingattn.h: running max of raw scores
    if (h->kv_fp8 && !h->k_scale) return SS_ERR_INVALID_ARG;                // ss_set_kv_scales first
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (h->debug_checks) SS_CUDA(h, launch_validate(h, block_table, query_start_loc, ctx_lens, R, T, st), "validate launch");

    if (h->force_simple) {
        SS_CUDA(h, launch_simple_attention(h, q, block_table, query_start_loc, ctx_lens, R, T, scale, out, lse_or_null, st),
                "simple attention launch");
        h->last_launches = 1 + h->debug_checks;
        return SS_OK;
    }
    const bool two_kernels = !main_self_plans(h, R, T);
    if (two_kernels) SS_CUDA(h, launch_worklist(h, query_start_loc, ctx_lens, R, T, workspace, st), "worklist launch");
    int n = 1;
    if (h->timing_on) SS_CUDA(h, cudaEventRecord(h->ev0, st), "timing event");
    SS_CUDA(h, launch_main_attention(h, q, block_table, query_start_loc, ctx_lens, R, T, scale, out, lse_or_null,
                                     workspace, st, &n),
            "main attention launch");
    if (h->timing_on) {
        SS_CUDA(h, cudaEventRecord(h->ev1, st), "timing event");
        h->timing_valid = 1;
    }
    h->last_launches = (two_kernels ? 1 : 0) + n + h->debug_checks;
    return SS_OK;
}

int ss_reset(ss_handle* hh, void* cuda_stream) {
    Handle* h = (Handle*)hh;
    if (!h) return SS_ERR_INVALID_ARG;
    SS_CUDA(h, cudaMemsetAsync(h->state, 0, h->state_bytes, (cudaStream_t)cuda_stream), "state reset");
    return SS_OK;
}

int ss_poll_device_error(ss_handle* hh, void* cuda_stream) {
    Handle* h = (Handle*)hh;
    if (!h) return SS_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int32_t rec[4] = {0, 0, 0, 0};
    SS_CUDA(h, cudaMemcpyAsync(rec, h->state + kStateErr, sizeof rec, cudaMemcpyDeviceToHost, st), "error flag copy");
    SS_CUDA(h, cudaStreamSynchronize(st), "error flag sync");
    if (rec[0] == 0) return SS_OK;
    SS_CUDA(h, cudaMemsetAsync(h->state + kStateErr, 0, sizeof rec, st), "error flag clear");
    SS_CUDA(h, cudaStreamSynchronize(st), "error flag sync");
    const char* what = rec[0] == kChkQsl            ? "query_start_loc is not 0 = qsl[0] <= ... <= qsl[R] = T"
                       : rec[0] == kChkCtxNegative  ? "negative ctx_len"
                       : rec[0] == kChkTooManyPages ? "ceil((u+c)/16) exceeds max_pages_per_req"
                       : rec[0] == kChkPageId       ? "block_table page id outside [0, num_pages)"
                       : rec[0] == kChkKvScale      ? "FP8 k_scale / v_scale entry not finite and > 0 (request = kv head, + Hkv for v_scale; value = its bits)"
                                                    : "unknown check";
    snprintf(h->err, sizeof h->err, "device check %d: %s (request %d, value %d, limit %d)", rec[0], what, rec[1], rec[2], rec[3]);
    return SS_ERR_DEVICE_CHECK;
}

int ss_build_worklist(ss_handle* hh, const int32_t* query_start_loc, const int32_t* ctx_lens, int32_t R, int32_t T,
                      void* workspace, size_t workspace_bytes, ss_work_item* items_host, int32_t max_items,
                      int32_t counts_host[3], void* cuda_stream) {
    Handle* h = (Handle*)hh;
    if (!h || !counts_host || R < 0 || T < 0 || R > h->cfg.max_requests || T > h->cfg.max_tokens) return SS_ERR_INVALID_ARG;
    counts_host[0] = counts_host[1] = counts_host[2] = 0;
    if (R == 0) return SS_OK;
    if (!query_start_loc || !ctx_lens || !workspace) return SS_ERR_INVALID_ARG;
    if (workspace_bytes < h->ws.total) return SS_ERR_WORKSPACE_TOO_SMALL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    SS_CUDA(h, launch_worklist(h, query_start_loc, ctx_lens, R, T, workspace, st), "worklist launch");
    WorkHeader hdr;
    SS_CUDA(h, cudaMemcpyAsync(&hdr, (char*)workspace + h->ws.header_off, sizeof hdr, cudaMemcpyDeviceToHost, st),
            "worklist header copy");
    SS_CUDA(h, cudaStreamSynchronize(st), "worklist sync");
    counts_host[0] = hdr.n_prefill;
    counts_host[1] = hdr.n_decode;
    counts_host[2] = hdr.n_partial;
    if (items_host) {
        int n = hdr.n_prefill + hdr.n_decode;
        if (n > max_items) n = max_items;
        if (n > 0) {
            SS_CUDA(h, cudaMemcpyAsync(items_host, (char*)workspace + h->ws.items_off, sizeof(ss_work_item) * (size_t)n,
                                       cudaMemcpyDeviceToHost, st),
                    "worklist items copy");
            SS_CUDA(h, cudaStreamSynchronize(st), "worklist sync");
        }
    }
    return SS_OK;
}

int ss_iteration_host(ss_handle* hh, const void* q_host, const void* k_new_host, const void* v_new_host,
                      const int32_t* block_table_host, const int32_t* qsl_host, const int32_t* ctx_host, int32_t R,
                      int32_t T, float scale, void* out_host, void* cuda_stream) {
    Handle* h = (Handle*)hh;
    if (!h || R < 0 || T < 0 || R > h->cfg.max_requests || T > h->cfg.max_tokens) return SS_ERR_INVALID_ARG;
    if (R == 0 || T == 0) return SS_OK;
    if (!q_host || !block_table_host || !qsl_host || !ctx_host || !out_host) return SS_ERR_INVALID_ARG;
    if ((k_new_host == nullptr) != (v_new_host == nullptr)) return SS_ERR_INVALID_ARG;
    const ss_config& c = h->cfg;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t q_max = (size_t)c.max_tokens * c.num_q_heads * c.head_dim * 2;
    const size_t kv_max = (size_t)c.max_tokens * c.num_kv_heads * c.head_dim * 2;
    if (!h->st_ctx) {
        // all or nothing: st_ctx (allocated last) doubles as the "staging ready" mark
        void** slots[] = {&h->st_q, &h->st_out, &h->st_knew, &h->st_vnew, &h->st_ws, (void**)&h->st_bt, (void**)&h->st_qsl,
                          (void**)&h->st_ctx};
        const size_t sizes[] = {q_max, q_max, kv_max, kv_max, h->ws.total,
                                sizeof(int32_t) * (size_t)c.max_requests * c.max_pages_per_req,
                                sizeof(int32_t) * (size_t)(c.max_requests + 1), sizeof(int32_t) * (size_t)c.max_requests};
        cudaError_t e = cudaSuccess;
        for (int i = 0; i < 8 && e == cudaSuccess; ++i) e = cudaMalloc(slots[i], sizes[i]);
        if (e != cudaSuccess) {
            for (int i = 0; i < 8; ++i) {
                if (*slots[i]) cudaFree(*slots[i]);
                *slots[i] = nullptr;
            }
            return fail_cuda(h, e, "staging alloc");
        }
    }
    const size_t q_bytes = (size_t)T * c.num_q_heads * c.head_dim * 2;
    const size_t kv_bytes = (size_t)T * c.num_kv_heads * c.head_dim * 2;
    SS_CUDA(h, cudaMemcpyAsync(h->st_q, q_host, q_bytes, cudaMemcpyHostToDevice, st), "h2d q");
    SS_CUDA(h, cudaMemcpyAsync(h->st_bt, block_table_host, sizeof(int32_t) * (size_t)R * c.max_pages_per_req,
                               cudaMemcpyHostToDevice, st), "h2d block_table");
    SS_CUDA(h, cudaMemcpyAsync(h->st_qsl, qsl_host, sizeof(int32_t) * (size_t)(R + 1), cudaMemcpyHostToDevice, st), "h2d qsl");
    SS_CUDA(h, cudaMemcpyAsync(h->st_ctx, ctx_host, sizeof(int32_t) * (size_t)R, cudaMemcpyHostToDevice, st), "h2d ctx");
    int launches = 0;
    if (k_new_host) {
        SS_CUDA(h, cudaMemcpyAsync(h->st_knew, k_new_host, kv_bytes, cudaMemcpyHostToDevice, st), "h2d k_new");
        SS_CUDA(h, cudaMemcpyAsync(h->st_vnew, v_new_host, kv_bytes, cudaMemcpyHostToDevice, st), "h2d v_new");
        int rc = ss_kv_append(hh, h->st_knew, h->st_vnew, h->st_bt, h->st_qsl, h->st_ctx, R, T, cuda_stream);
        if (rc != SS_OK) return rc;
        launches += h->last_launches;
    }
    int rc = ss_mixed_attention(hh, h->st_q, h->st_bt, h->st_qsl, h->st_ctx, R, T, scale, h->st_out, nullptr, h->st_ws,
                                h->ws.total, cuda_stream);
    if (rc != SS_OK) return rc;
    launches += h->last_launches;
    SS_CUDA(h, cudaMemcpyAsync(out_host, h->st_out, q_bytes, cudaMemcpyDeviceToHost, st), "d2h out");
    SS_CUDA(h, cudaStreamSynchronize(st), "iteration sync");
    h->last_launches = launches;
    return SS_OK;
}

}  // extern "C"
