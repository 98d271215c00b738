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
 *       k_cache, v_cache : [num_pages][num_kv_heads][page_size][head_dim] bf16   (4 KB slab per page,head;
 *                          one byte per element with SS_FLAG_KV_FP8)
 *       block_table      : [R][max_pages_per_req] int32; entry p of row r is the physical page holding
 *                          logical tokens 16p..16p+15 of request r; entries past ceil((u_r+c_r)/16)
 *                          are never read
 *       query_start_loc  : [R+1] int32, qsl[0]=0, non-decreasing, qsl[R]=T   (prefix sums of c_r)
 *       ctx_lens         : [R] int32 = u_r, tokens cached BEFORE this iteration (excludes the c_r new)
 *       q, out           : [T][num_q_heads][head_dim] bf16 ;  k_new, v_new : [T][num_kv_heads][head_dim]
 *     Query head h uses KV head h / (num_q_heads/num_kv_heads).
 *   - Slots past u_r+c_r in a last page, pages in no block table and block-table tail entries may
 *     hold ANY bit pattern; they never influence results and are never written.
 *   - Device-resident metadata cannot be validated on the host without a sync.  Without
 *     SS_FLAG_DEBUG_CHECKS, page ids outside [0, num_pages), a query_start_loc that is not
 *     0 = qsl[0] <= ... <= qsl[R] = T, a negative ctx_len or ceil((u_r+c_r)/16) > max_pages_per_req are
 *     undefined behaviour.  With the flag, every ss_kv_append / ss_mixed_attention first runs a device-side
 *     check of exactly these conditions (on FP8 handles also: every k_scale / v_scale entry finite and > 0); on a violation it records (code, request, value) in a device flag
 *     and the call - and every later call on the handle - touches neither the caches nor `out` until
 *     ss_poll_device_error has reported and cleared it.
 *   - ONE CALL IN FLIGHT PER HANDLE: the work-queue tickets and split-arrival counters are handle-owned
 *     device memory that the kernels re-arm themselves, so all calls on one handle must be ordered on one
 *     stream (or by events).  Use one handle per stream for concurrency.  If a launch was aborted
 *     (sticky CUDA error, device reset), call ss_reset before reusing the handle.
 *   - scale must be finite and > 0 (SS_ERR_INVALID_ARG otherwise): the kernels fold log2(e) into it and
 *     take the running maximum of the raw scores, which is the maximum of the scaled scores only for scale > 0.
 */
#ifndef SLIDINGATTN_H
#define SLIDINGATTN_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SS_VERSION 200

typedef enum ss_status {
    SS_OK = 0,
    SS_ERR_INVALID_ARG = -1,         /* null / misaligned pointer, negative size, R or T above the handle's bounds, bad config */
    SS_ERR_WORKSPACE_TOO_SMALL = -2,
    SS_ERR_UNSUPPORTED_DEVICE = -3,  /* current device is not compute capability 10.x */
    SS_ERR_CUDA = -4,                /* a CUDA runtime/driver call failed; see ss_last_error_string */
    SS_ERR_NOT_IMPLEMENTED = -5,
    SS_ERR_DEVICE_CHECK = -6         /* ss_poll_device_error: the in-kernel metadata check (SS_FLAG_DEBUG_CHECKS) tripped */
} ss_status;

/* ss_config.flags */
#define SS_FLAG_DEBUG_CHECKS 1u      /* "debug build" of SURVEY.md section 8(b): bounds-check device metadata in-kernel */
#define SS_FLAG_KV_FP8 2u            /* FP8 E4M3 KV cache (reading 23): see ss_set_kv_scales */

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
    uint32_t flags;             /* bitwise or of SS_FLAG_* (0 = bf16 cache, no device checks) */
} ss_config;

/* Lifetime.  ss_create binds the handle to the two cache tensors (TMA descriptors are encoded once)
 * and to the current CUDA device.  The caches stay caller-owned and must outlive the handle. */
int ss_create(ss_handle** out_handle, const ss_config* cfg, void* k_cache_device, void* v_cache_device);
int ss_destroy(ss_handle* h);

/*
 * FP8 KV cache (SS_FLAG_KV_FP8; head_dim must be 128).  k_cache / v_cache are [num_pages][num_kv_heads][16][head_dim]
 * bytes holding OCP FP8 E4M3 codes ("e4m3fn": bias 7, no infinities, max 448, S.1111.111 = NaN) with one fp32 scale per
 * (tensor, kv head): value = decode(code) * scale[g].  k_scale_device / v_scale_device are DEVICE arrays of
 * num_kv_heads floats, caller-owned, read by every later hot call (they must stay valid and may be rewritten between
 * calls in stream order); every scale must be finite and > 0.  Required before the first ss_kv_append /
 * ss_mixed_attention on an FP8 handle (SS_ERR_INVALID_ARG otherwise).
 *   ss_kv_append       quantises: code = e4m3(x / scale[g]), the quotient an IEEE fp32 division, rounded to nearest
 *                      even, magnitudes above 448 saturate to 448, NaN -> 0x7F.  Bit-exact against that definition.
 *   ss_mixed_attention same definition as the bf16 path with K = decode(code) * k_scale[g], V likewise; bf16 q / out.
 *                      The staged codes are widened exactly to fp16 and every product runs on fp16 tensor-core operands
 *                      (decode: half the HBM bytes; prefill chunks: tcgen05 on fp16 copies of the tiles); q is rounded
 *                      to fp16 for them - exact for |q| in [2^-14, 65504], clamped above - and P is rounded to fp16.
 *   ss_qkv_rope_append rotates as on a bf16 handle (k rounded to bf16 once), then quantises k and v exactly as ss_kv_append does.
 */
int ss_set_kv_scales(ss_handle* h, const float* k_scale_device, const float* v_scale_device);

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
 * The step before the path: RoPE + QKV split fused into the append.  qkv is the fused
 * projection output [T][(Hq + 2 Hkv) * D] bf16 - per token the Hq query heads, then the Hkv key heads, then the Hkv value
 * heads.  q and k are rotated by the token's absolute position ctx_lens[r] + j with the "rotate-half" rotary embedding
 * of the model families the paper serves (reading 22):
 *     angle_i = pos * rope_theta^(-2i/D);  y_i = x_i cos - x_{i+D/2} sin;  y_{i+D/2} = x_{i+D/2} cos + x_i sin
 * (cos / sin and the rotation evaluated in double, products and sums rounded separately, ONE rounding to bf16: bit-exact
 * against that definition up to the last place of cos / sin).  Rotated q -> q_out [T][Hq][D] (the q
 * argument of ss_mixed_attention), rotated k and the untouched v bits -> their page slots exactly as ss_kv_append places
 * them.  Replaces ss_kv_append for the batch.  rope_theta must be finite and > 1.  All pointers device.
 */
int ss_qkv_rope_append(ss_handle* h, const void* qkv, const int32_t* block_table, const int32_t* query_start_loc,
                       const int32_t* ctx_lens, int32_t R, int32_t T, float rope_theta, void* q_out,
                       void* cuda_stream);

/*
 * a2..a5  mixed_attention (north_star "mixed_attention(q, k_cache, v_cache,
 * block_table, query_start_loc, ctx_lens, scale, out)"; the caches were bound at ss_create).
 * For request r, row j < c_r, head h:  out = softmax(scale * q . K[0..u_r+j]^T) V[0..u_r+j]  with
 * bf16 operands, fp32 accumulation and softmax state, bf16 round-to-nearest-even output.  The cache
 * must already hold the u_r + c_r tokens (run ss_kv_append for the same batch earlier on the same
 * stream).  Requests with c_r == 1 take the split-KV decode path, c_r > 1 the tensor-core chunk path,
 * c_r == 0 contributes nothing; any mix and any request order is served by one call.
 * scale: finite and > 0, else SS_ERR_INVALID_ARG (benchmarks pass 1/sqrt(head_dim)).
 * lse_or_null: optional [T][Hq] fp32 log-sum-exp (natural log) of the scaled scores, a test aid.
 * workspace: device memory of at least ss_workspace_bytes(h), contents undefined in/out.
 * Bitwise reproducible run to run for identical inputs.  All pointers device.
 */
int ss_mixed_attention(ss_handle* h, const void* q, const int32_t* block_table,
                       const int32_t* query_start_loc, const int32_t* ctx_lens, int32_t R, int32_t T,
                       float scale, void* out, float* lse_or_null, void* workspace,
                       size_t workspace_bytes, void* cuda_stream);

/*
 * ss_mixed_attention for callers that CANNOT ALLOCATE device memory.  Who that is: a serving engine that gives every
 * free byte of HBM to its paged KV cache when it starts has nothing left for a cudaMalloc by the time an iteration
 * runs; a plugin living inside someone else's memory pool may not be allowed one; and a cudaMalloc on the iteration
 * path stalls the whole device.  The regular route allocates twice on such a caller's behalf (ss_create mallocs the
 * handle's counters, and somebody has to malloc the workspace).  This entry point needs neither: no handle, no
 * workspace, and it calls no cudaMalloc / cudaFree or any other allocating routine.  Its scratch is an array compiled
 * into the library: SS_STATIC_SCRATCH_BYTES of device memory on every GPU that loads the library, held until the
 * process exits whether or not this function is ever called.
 *
 * Same operation, same kernels, same results as ss_mixed_attention (a2..a5 above) on a handle created with this `cfg`,
 * flags == 0 and these caches; the caches must already hold the batch's u_r + c_r tokens.  Inputs and outputs are still
 * the caller's device memory.
 *   cfg                flags must be 0 (bf16 cache, no device checks).  The scratch a config needs grows with
 *                      max_requests, max_tokens, max_pages_per_req and the head counts exactly as ss_workspace_bytes
 *                      does (plus 4 * (8 + max_requests * num_kv_heads) bytes of counters).  A config that needs more than
 *                      SS_STATIC_SCRATCH_BYTES is refused with SS_ERR_WORKSPACE_TOO_SMALL and both byte counts in
 *                      err_msg; nothing is launched.  Guide: Llama-3-8B shapes (32 / 8 heads, D = 128) with 129 requests,
 *                      2176 tokens and 8K context need 5.1 MB; the 70B batch C5 (64 / 8 heads, 30K context) needs 21 MB
 *                      and does not fit - so size cfg to the iteration's real bounds, not the engine's global ones.
 *   err_msg            optional host buffer (err_msg_len bytes) that receives a one-line reason on any non-zero return.
 * FIRST CALL ON EACH DEVICE does a one-time set-up with that device current (looks up the array's device address,
 * reads the SM count, sets the kernels' shared-memory attribute).  Make that first call during start-up, outside any
 * stream capture; it needs real arguments, so a small warm-up batch is the way to do it.
 * SHARED STATE: every call on a device uses the same array, and the array keeps the previous call's contents.  The
 * call itself clears (cudaMemsetAsync on `cuda_stream`) the counters that must start at zero; everything else is
 * written before it is read.  Two calls whose GPU work overlaps - different streams, or different host threads on one
 * device - race on the array and produce garbage: order them on one stream or by events.  Calls on ss_create handles
 * do not touch the array and may overlap with it freely.
 */
#define SS_STATIC_SCRATCH_BYTES (8u << 20)
int ss_mixed_attention_static(const ss_config* cfg, void* k_cache_device, void* v_cache_device, const void* q,
                              const int32_t* block_table, const int32_t* query_start_loc, const int32_t* ctx_lens,
                              int32_t R, int32_t T, float scale, void* out, float* lse_or_null, void* cuda_stream,
                              char* err_msg, size_t err_msg_len);

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

/*
 * Debug-check report.  Synchronises `cuda_stream`, reads the device error flag and
 * clears it.  SS_OK if no check tripped (always, when the handle was created without SS_FLAG_DEBUG_CHECKS);
 * SS_ERR_DEVICE_CHECK otherwise, with ss_last_error_string naming the violated condition, the request index
 * and the offending value.  Calls issued between the violation and this poll did nothing.
 */
int ss_poll_device_error(ss_handle* h, void* cuda_stream);

/* Re-zero the handle-owned device state (queue tickets, split-arrival counters, error flag) on `cuda_stream`.
 * Only needed after a launch on this handle was aborted mid-flight. */
int ss_reset(ss_handle* h, void* cuda_stream);

const char* ss_status_string(int status);
const char* ss_last_error_string(const ss_handle* h);   /* detail of the last SS_ERR_CUDA / SS_ERR_DEVICE_CHECK on this handle */
int ss_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SLIDINGATTN_H */
