/*
 * slidingattn_debug.h - test, tuning and measurement aids of libslidingattn.  NOT part of the product boundary
 * (include/slidingattn.h lists the calls of SURVEY.md section 8(b)); nothing here changes results.
 */
#ifndef SLIDINGATTN_DEBUG_H
#define SLIDINGATTN_DEBUG_H

#include "slidingattn.h"

#ifdef __cplusplus
extern "C" {
#endif

/* One entry of the device work list (a2); exposed so tests can check the builder.
 * kind 1 = prefill tile: query rows [row0, row0+nrows) of request req (c_r > 1, Eq. 2),
 *          query heads head .. head+nheads-1 (1 or 2 heads of one KV head), keys [0, kv_end);
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
    int32_t nheads;     /* prefill: 1 or 2 query heads served by the item; decode: the G heads of the KV head */
} ss_work_item;

/*
 * a2 alone (test aid): build the work list for a batch into `workspace` exactly as ss_mixed_attention
 * does, then copy it to the host (this call DOES synchronise the stream).  items_host may be NULL to
 * query counts only.  counts_host[0] = number of prefill items, [1] = decode items, [2] = partial slots.
 */
int ss_build_worklist(ss_handle* h, const int32_t* query_start_loc, const int32_t* ctx_lens, int32_t R,
                      int32_t T, void* workspace, size_t workspace_bytes, ss_work_item* items_host,
                      int32_t max_items, int32_t counts_host[3], void* cuda_stream);

/* Which kernels the last ss_mixed_attention / ss_kv_append on this handle launched (count), so a
 * caller can report launches per iteration without a profiler. */
int ss_last_launch_count(const ss_handle* h);

/* Measurement aid: when on, ss_mixed_attention brackets its dominant kernel(s) (a3+a4 main launch) with
 * CUDA events on the caller's stream; ss_last_kernel_time_us then synchronises on them and returns the
 * device time of the last call's main launch in microseconds (SS_ERR_INVALID_ARG if timing was off). */
int ss_set_kernel_timing(ss_handle* h, int on);
int ss_last_kernel_time_us(ss_handle* h, float* main_us);

/* Measurement aid: one read-only streaming pass (16 KB bulk copies into shared memory, whole chunks only) over `bytes` of device memory at `buf` (16-byte aligned), enqueued on
 * the stream.  bench.py times it to get the HBM READ peak of this GPU: the decode path only reads, and the copy
 * (read + write) peak in MEASURED_PEAKS.json understates what a read-only stream can reach.  Touches no library state. */
int ss_debug_stream_read(ss_handle* h, const void* buf, size_t bytes, void* cuda_stream);

/* Debug: force the plain one-warp-per-row CUDA kernel (no tensor cores) for every row. 0 = off. */
int ss_debug_force_simple_path(ss_handle* h, int on);

/* Debug / tuning knobs; value 0 restores the automatic choice.  which: 1 = CTAs of the main launch (default one
 * per SM), 2 = number of CTAs that drain the decode queue first (default: balanced from the batch's decode bytes and
 * prefill flops by the planner; -1 = none), 3 = decode split length in keys (multiple of 128, within [512, 16384]; raised per batch until
 * the splits fit the workspace's partial slots, which are sized for the automatic length), 4 = nonzero forces the
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

#ifdef __cplusplus
}
#endif
#endif /* SLIDINGATTN_DEBUG_H */
