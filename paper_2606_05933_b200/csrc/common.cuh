// Internal declarations shared by the translation units of libslidingattn (CUDA product path only;
// the CPU oracle under oracle/ shares nothing with this directory).
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "slidingattn.h"
#include "slidingattn_debug.h"

namespace ss {

constexpr int kPage = 16;             // tokens per KV page (BASELINE.json configs: "page 16")
constexpr int kTileKeys = 128;        // keys per prefill KV step (MMA N; two 64-key ring slots) and the alignment of decode splits
constexpr int kTileRows = 128;        // query rows per prefill tile / MMA M
constexpr int kMaxGroup = 16;         // max q heads per kv head on the decode path (MMA M = 16)
constexpr int kDecodeWaves = 1;       // target decode items per SM when choosing the split length (a split costs ~2 us of
                                      // first-tile wait + merge: 3 or 6 per SM over-split every batch with >= 2 units per SM)
constexpr int kMinSplitKeys = 512;    // never split a decode KV range finer than this
constexpr int kMaxSplitKeys = 16384;  // never leave a decode item longer than this (4096: 50 % more items on C5, +3 % time)
// SM partition model of the two-queue scheduler (measured on B200): bytes/us one SM streams on the
// decode path, flop/us one SM sustains on the prefill path, and the CTA count past which decode is HBM-limited.
constexpr float kDecodeBytesPerUsPerSm = 80e3f;
constexpr float kPrefillFlopsPerUsPerSm = 8.0e6f;
constexpr int kMaxDecodeCtas = 88;
// ss_debug_set_param keys (tuning / measurement aids; 0 restores the automatic choice)
enum { kDbgGrid = 1, kDbgDecodeCtas = 2, kDbgSplitKeys = 3, kDbgTwoKernel = 4 };
constexpr int kPlanMaxR = 256;        // requests the main kernel's in-kernel plan tables hold (larger batches: work-list kernel)

// Workspace header written by the work-list kernel (device side, int32 words).
struct WorkHeader {
    int32_t n_prefill;      // prefill tile items
    int32_t n_decode;       // decode split items
    int32_t n_partial;      // partial slots (one per split of a split (req, kv head))
    int32_t split_keys;     // chosen split length L (multiple of kTileKeys)
    int32_t next_prefill;   // dynamic queue heads of the main kernel (zeroed by the work-list kernel)
    int32_t next_decode;
    int32_t n_decode_ctas;  // CTAs [0, n_decode_ctas) drain the decode queue first, the others the prefill queue first
    int32_t pad[9];
};

struct WorkspaceLayout {
    size_t header_off, items_off, counters_off, partial_off, total;
    int32_t max_items, max_partials;
    bool ok;                         // false: the config's worst case does not fit the int32 item / slot index space
};

constexpr int kStateErr = 4;         // Handle::state word offsets
constexpr int kStateCounters = 8;
// debug-check codes (ss_poll_device_error)
enum { kChkQsl = 1, kChkCtxNegative = 2, kChkTooManyPages = 3, kChkPageId = 4, kChkKvScale = 5 };

struct Handle {
    ss_config cfg;
    int device;
    int num_sms;
    int group;                       // Hq / Hkv
    void* k_cache;
    void* v_cache;
    CUtensorMap tmap_k, tmap_v;      // 4-D slab maps, one box = one (page, kv head) slab, 128B swizzle (encode_cache_map, api.cu)
    bool have_tmaps;
    WorkspaceLayout ws;
    // host-iteration staging (lazy)
    void *st_q, *st_knew, *st_vnew, *st_out, *st_ws;
    int32_t *st_bt, *st_qsl, *st_ctx;
    int last_launches;
    int force_simple;
    int dbg[8];                      // ss_debug_set_param knobs (0 = automatic)
    int32_t* state;                  // device: [0..3] self-cleaning queue tickets, [4..7] debug-check record (code, request,
                                     // value, limit), [8..) split arrival counters (max_requests*Hkv)
    size_t state_bytes;
    int kv_fp8;                      // SS_FLAG_KV_FP8: caches hold E4M3 codes, one byte per element
    const float* k_scale;            // device, [Hkv] (ss_set_kv_scales); null until set
    const float* v_scale;
    int debug_checks;                // SS_FLAG_DEBUG_CHECKS: validate device metadata before every hot call
    unsigned long long* trace;       // ss_debug_set_trace buffer (device) or null
    int trace_words;
    int timing_on, timing_valid;
    cudaEvent_t ev0, ev1;
    char err[256];
};

inline WorkspaceLayout workspace_layout(const ss_config& c, int num_sms) {
    WorkspaceLayout w{};
    const int64_t group = c.num_q_heads / c.num_kv_heads;
    const int64_t tiles = ((int64_t)c.max_tokens + kTileRows - 1) / kTileRows + c.max_requests;   // widen BEFORE the add
    const int64_t max_prefill = (int64_t)c.num_q_heads * tiles;
    // decode items: Hkv * sum_r nsplit_r.  Unclamped split length: <= Hkv*R + num_sms*kDecodeWaves;
    // split length clamped at kMaxSplitKeys: <= Hkv * R * (ceil(max ctx / kMaxSplitKeys) + 1).
    const int64_t max_ctx = (int64_t)c.max_pages_per_req * kPage;
    const int64_t max_decode = (int64_t)c.num_kv_heads * c.max_requests * ((max_ctx + kMaxSplitKeys - 1) / kMaxSplitKeys + 1) +
                               (int64_t)num_sms * kDecodeWaves + 64;
    w.ok = max_prefill + max_decode <= (int64_t)0x7fffffff / 4;     // item / partial-slot indices stay far inside int32
    w.max_items = (int32_t)(w.ok ? max_prefill + max_decode : 0);
    w.max_partials = (int32_t)(w.ok ? max_decode : 0);
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = (off + bytes + 255) & ~(size_t)255; return o; };
    w.header_off = take(sizeof(WorkHeader));
    w.items_off = take(sizeof(ss_work_item) * (size_t)w.max_items);
    w.counters_off = take(sizeof(int32_t) * (size_t)c.max_requests * (size_t)c.num_kv_heads);   // split arrival counters
    // partial slot = group rows of (m, l, o[D]) fp32
    w.partial_off = take(sizeof(float) * (size_t)w.max_partials * (size_t)group * (size_t)(c.head_dim + 2));
    w.total = off;
    return w;
}

// Launch with programmatic stream serialization: the grid may start while its predecessor in the stream drains;
// every kernel launched this way executes griddepcontrol.wait before it touches global memory.
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

// ---- launchers implemented in the .cu files (all enqueue on `stream`, return cudaError_t) ----
cudaError_t launch_kv_append(const Handle* h, const void* k_new, const void* v_new, const int32_t* bt,
                             const int32_t* qsl, const int32_t* ctx, int R, int T, cudaStream_t stream);
cudaError_t launch_qkv_rope_append(const Handle* h, const void* qkv, const int32_t* bt, const int32_t* qsl,
                                   const int32_t* ctx, int R, int T, float rope_theta, void* q_out, cudaStream_t stream);
cudaError_t launch_worklist(const Handle* h, const int32_t* qsl, const int32_t* ctx, int R, int T,
                            void* workspace, cudaStream_t stream);
cudaError_t launch_simple_attention(const Handle* h, const void* q, const int32_t* bt, const int32_t* qsl,
                                    const int32_t* ctx, int R, int T, float scale, void* out, float* lse,
                                    cudaStream_t stream, int prefill_only = 0);
bool main_self_plans(const Handle* h, int R, int T);
// TMA descriptor of one cache tensor (api.cu; host-only encode, needs h->cfg / h->kv_fp8, writes h->err on failure)
int encode_cache_map(Handle* h, CUtensorMap* map, void* base);
cudaError_t init_main_attention(int head_dim, int kv_fp8);   // one-time function attributes (ss_create)
// SS_FLAG_DEBUG_CHECKS: device-side validation of (qsl, ctx_lens, block_table); records the first violation in
// h->state[kStateErr..] - the hot kernels of this and later calls then skip every cache / output access
cudaError_t launch_validate(const Handle* h, const int32_t* bt, const int32_t* qsl, const int32_t* ctx, int R, int T,
                            cudaStream_t stream);
// Main path (a3 + a4 + a5): consumes the work list in `workspace`; *n_launches receives the kernel count.
cudaError_t launch_main_attention(const Handle* h, const void* q, const int32_t* bt, const int32_t* qsl,
                                  const int32_t* ctx, int R, int T, float scale, void* out, float* lse,
                                  void* workspace, cudaStream_t stream, int* n_launches);

}  // namespace ss
