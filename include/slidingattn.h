/*
 * slidingattn.h — C ABI of the B200 (sm_100a) mixed chunked-prefill + decode paged-attention library.
 *
 * What it executes: one continuous-batching iteration of SlidingServe's "GPU Execution" step
 * (§3.1 step 9) restricted to attention + KV-cache access, the part of batch latency that
 * depends on the batch composition B = {(c_i, u_i)} (§3.2; §2.2 "attention
 * computation, and key-value cache access times"; Table 1).  c_i -> q_len
 * (query_start_loc differences), u_i -> ctx_lens.
 *
 * Conventions for every entry point
 *   - "device" pointers are CUDA device memory of the current device, 16-byte aligned, caller-owned.
 *     "host" pointers are ordinary (ideally pinned) host memory.
 *   - bf16 tensors are raw 16-bit patterns; row-major with the last dimension contiguous.
 *   - cuda_stream is a cudaStream_t passed as void* (NULL = legacy default stream).  All work is
 *     enqueued on it; no entry point below synchronises or reads device data on the host unless it
 *     says so.
 *   - Return value: 0 = SS_OK, negative = error (see ss_status).  No exceptions, no abort().
 *   - Layouts (the paper is silent on them):
 *       k_cache, v_cache : [num_pages][num_kv_heads][page_size][head_dim] bf16   (4 KB slab per page,head)
 *       block_table      : [R][max_pages_per_req] int32; entry p of row r is the physical page holding
 *                          logical tokens 16p..16p+15 of request r; entries past ceil((u_r+c_r)/16)
 *                          are never read
 *       query_start_loc  : [R+1] int32, qsl[0]=0, non-decreasing, qsl[R]=T   (prefix sums of c_r)
 *       ctx_lens         : [R] int32 = u_r, tokens cached BEFORE this iteration (excludes the c_r new)
 *       q, out           : [T][num_q_heads][head_dim] bf16 ;  k_new, v_new : [T][num_kv_heads][head_dim]
 *     Query head h uses KV head h / (num_q_heads/num_kv_heads).
 *   - Slots past u_r+c_r in a last page, pages in no block table and block-table tail entries may
 *     hold ANY bit pattern; they never influence results and are never written.
 *   - Device-resident metadata cannot be validated without a sync: page ids >= num_pages, a
 *     non-monotone query_start_loc or ceil((u_r+c_r)/16) > max_pages_per_req are undefined behaviour.
 */
#ifndef SLIDINGATTN_H
#define SLIDINGATTN_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SS_VERSION 100

typedef enum ss_status {
    SS_OK = 0,
    SS_ERR_INVALID_ARG = -1,         /* null / misaligned pointer, negative size, R or T above the handle's bounds, bad config */
    SS_ERR_WORKSPACE_TOO_SMALL = -2,
    SS_ERR_UNSUPPORTED_DEVICE = -3,  /* current device is not compute capability 10.x */
    SS_ERR_CUDA = -4,                /* a CUDA runtime/driver call failed; see ss_last_error_string */
    SS_ERR_NOT_IMPLEMENTED = -5
} ss_status;

typedef struct ss_handle ss_handle;  /* opaque; owns tensor maps, SM count, small staging buffers */

typedef struct ss_config {
    int32_t num_q_heads;        /* Hq; Hq % Hkv == 0, Hq/Hkv <= 16 */
    int32_t num_kv_heads;       /* Hkv */
    int32_t head_dim;           /* 64 or 128 */
    int32_t page_size;          /* must be 16 */
    int64_t num_pages;          /* pages per cache tensor */
    int32_t max_requests;       /* upper bound on R */
    int32_t max_tokens;         /* upper bound on T */
    int32_t max_pages_per_req;  /* second dimension of block_table */
} ss_config;

/* One entry of the device work list (a2); exposed so tests can check the builder.
 * kind 1 = prefill tile: query rows [row0, row0+nrows) of request req (c_r > 1, Eq. 2),
 *          query head `head`, keys [0, kv_end);
 * kind 2 = decode split: the single row of request req (c_r == 1), KV head `head`, keys
 *          [kv_begin, kv_end); partial results go to slot `partial` unless nsplit == 1. */
typedef struct ss_work_item {
    int32_t kind;
    int32_t req;
    int32_t head;
    int32_t row0;       /* flat row index into q/out */
    int32_t nrows;
    int32_t kv_begin;
    int32_t kv_end;
    int32_t split;      /* index of this split, 0 <= split < nsplit */
    int32_t nsplit;
    int32_t partial;    /* decode: first partial slot of this (req, kv head), slot = partial + split */
    int32_t q_pos0;     /* prefill: chunk-relative index j of the first row (row j sees keys 0..u+j) */
    int32_t reserved;
} ss_work_item;

/* Lifetime.  ss_create binds the handle to the two cache tensors (TMA descriptors are encoded once)
 * and to the current CUDA device.  The caches stay caller-owned and must outlive the handle. */
int ss_create(ss_handle** out_handle, const ss_config* cfg, void* k_cache_device, void* v_cache_device);
int ss_destroy(ss_handle* h);

/* Upper bound (from the config) of the device workspace ss_mixed_attention needs: work list,
 * counters and split-KV partials. */
size_t ss_workspace_bytes(const ss_handle* h);

/*
 * a1  kv_append (PAPER.md:99 step 10: after a batch runs, request r's cached length grows by c_r;
 * north_star "kv_append(k_new, v_new, block_table, slot offsets)").  Token j of request r is written
 * to logical position ctx_lens[r] + j, i.e. page block_table[r][(u_r+j)/16], slot (u_r+j)%16.
 * Pure 16-byte bit copies: bit-exact incl. NaN payloads and -0.  Writes exactly T*Hkv*D elements per
 * cache tensor and nothing else.  All pointers device.  R == 0 or T == 0: returns SS_OK, no launch.
 */
int ss_kv_append(ss_handle* h, const void* k_new, const void* v_new, const int32_t* block_table,
                 const int32_t* query_start_loc, const int32_t* ctx_lens, int32_t R, int32_t T,
                 void* cuda_stream);

/*
 * a2..a5  mixed_attention (north_star "mixed_attention(q, k_cache, v_cache,
 * block_table, query_start_loc, ctx_lens, scale, out)"; the caches were bound at ss_create).
 * For request r, row j < c_r, head h:  out = softmax(scale * q . K[0..u_r+j]^T) V[0..u_r+j]  with
 * bf16 operands, fp32 accumulation and softmax state, bf16 round-to-nearest-even output.  The cache
 * must already hold the u_r + c_r tokens (run ss_kv_append for the same batch earlier on the same
 * stream).  Requests with c_r == 1 take the split-KV decode path, c_r > 1 the tensor-core chunk path,
 * c_r == 0 contributes nothing; any mix and any request order is served by one call.
 * lse_or_null: optional [T][Hq] fp32 log-sum-exp (natural log) of the scaled scores, a test aid.
 * workspace: device memory of at least ss_workspace_bytes(h), contents undefined in/out.
 * Bitwise reproducible run to run for identical inputs.  All pointers device.
 */
int ss_mixed_attention(ss_handle* h, const void* q, const int32_t* block_table,
                       const int32_t* query_start_loc, const int32_t* ctx_lens, int32_t R, int32_t T,
                       float scale, void* out, float* lse_or_null, void* workspace,
                       size_t workspace_bytes, void* cuda_stream);

/*
 * a2 alone (test aid): build the work list for a batch into `workspace` exactly as ss_mixed_attention
 * does, then copy it to the host (this call DOES synchronise the stream).  items_host may be NULL to
 * query counts only.  counts_host[0] = number of prefill items, [1] = decode items, [2] = partial slots.
 */
int ss_build_worklist(ss_handle* h, const int32_t* query_start_loc, const int32_t* ctx_lens, int32_t R,
                      int32_t T, void* workspace, size_t workspace_bytes, ss_work_item* items_host,
                      int32_t max_items, int32_t counts_host[3], void* cuda_stream);

/*
 * End-to-end iteration from HOST buffers (what a serving loop without device-resident activations
 * calls; bench.py's "e2e" leg): copies q / k_new / v_new / metadata host->device into handle-owned
 * staging buffers, runs ss_kv_append (if k_new_host != NULL) and ss_mixed_attention, copies `out`
 * device->host and synchronises the stream before returning.  block_table_host is [R][max_pages_per_req].
 */
int ss_iteration_host(ss_handle* h, const void* q_host, const void* k_new_host, const void* v_new_host,
                      const int32_t* block_table_host, const int32_t* query_start_loc_host,
                      const int32_t* ctx_lens_host, int32_t R, int32_t T, float scale, void* out_host,
                      void* cuda_stream);

/* Which kernels the last ss_mixed_attention / ss_kv_append on this handle launched (count), so a
 * caller can report launches per iteration without a profiler. */
int ss_last_launch_count(const ss_handle* h);

/* Measurement aid: when on, ss_mixed_attention brackets its dominant kernel(s) (a3+a4 main launch) with
 * CUDA events on the caller's stream; ss_last_kernel_time_us then synchronises on them and returns the
 * device time of the last call's main launch in microseconds (SS_ERR_INVALID_ARG if timing was off). */
int ss_set_kernel_timing(ss_handle* h, int on);
int ss_last_kernel_time_us(ss_handle* h, float* main_us);

/* Debug: force the plain one-warp-per-row CUDA kernel (no tensor cores) for every row. 0 = off. */
int ss_debug_force_simple_path(ss_handle* h, int on);

/* Debug / tuning knobs; value 0 restores the automatic choice.  which: 1 = CTAs of the main launch (default one
 * per SM), 2 = number of CTAs that drain the decode queue first (default: balanced from the batch's decode bytes and
 * prefill flops by the planner; -1 = none), 3 = decode split length in keys (multiple of 128), 4 = nonzero forces the
 * two-launch route (stand-alone work-list kernel + main kernel reading its items) that batches of more than 256
 * requests take; by default smaller batches are planned inside the main kernel (one launch).
 * Results never depend on these; only timing does.  SS_ERR_INVALID_ARG for an unknown key. */
int ss_debug_set_param(ss_handle* h, int which, int value);

/* Measurement aid: per-CTA timeline of the main launch.  `trace_dev` is a DEVICE buffer of
 * num_ctas * words_per_cta uint64 words (caller-owned; NULL switches tracing off; words_per_cta >= 6).  Per CTA the
 * kernel writes word 0 = %globaltimer at entry (ns), 1 = after setup + grid dependency wait, 2 = worker warps' exit,
 * 3 = item count, 4 = exit of the MMA / split-merge warp, 5 = unused, then 9 words per item while they fit: start ns,
 * end ns, kind << 32 | KV tiles, first tile ready ns, tile loop end ns, and 4 epilogue stamps (decode items only).
 * Results never depend on it. */
int ss_debug_set_trace(ss_handle* h, void* trace_dev, int32_t words_per_cta);

const char* ss_status_string(int status);
const char* ss_last_error_string(const ss_handle* h);   /* detail of the last SS_ERR_CUDA on this handle */
int ss_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SLIDINGATTN_H */
