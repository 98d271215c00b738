// K2 stand-alone work-list kernel (a2): builds the plan of plan.cuh and materialises every item as a
// 48-byte record in the workspace.  Used by ss_build_worklist (test / inspection aid) and by ss_mixed_attention for
// batches whose request count exceeds the main kernel's in-kernel plan tables; smaller batches are planned inside
// the main kernel's prologue from the same device functions, so both routes yield identical items.
#include "common.cuh"
#include "plan.cuh"
#include "ptx.cuh"

namespace ss {

constexpr int kWlThreads = 512;
constexpr int kWlCtas = 8;            // every CTA rebuilds the (small) plan and writes its slice of the items

__global__ void __launch_bounds__(kWlThreads)
worklist_kernel(const int32_t* __restrict__ qsl, const int32_t* __restrict__ ctx_lens, int R, int Hq, int Hkv,
                int num_sms, int D, int force_split_keys, int force_decode_ctas, WorkHeader* __restrict__ hdr,
                ss_work_item* __restrict__ items, int32_t* __restrict__ merge_counters, int max_items,
                int max_decode_items, const int32_t* __restrict__ err_flag) {
    extern __shared__ __align__(16) int32_t sm[];
    const int Rp = (R + 3) & ~3;
    int32_t* scratch = sm;                                        // 3 Rp
    PlanTables<int32_t> tb;
    tb.off = sm + 3 * Rp;                                         // R
    tb.ord = reinterpret_cast<uint16_t*>(sm + 4 * Rp);            // R x u16
    __shared__ PlanHeader ph;
    const int tid = threadIdx.x, nt = blockDim.x;

    ptx::pdl_launch_dependents();
    ptx::pdl_wait();            // qsl / ctx_lens may come from the preceding kernel in the stream
    // SS_FLAG_DEBUG_CHECKS: a tripped check means the metadata is not to be trusted (a negative ctx_len would divide by
    // zero in the plan); like the append and main kernels, do nothing until ss_poll_device_error has cleared the flag
    if (err_flag && *reinterpret_cast<const volatile int32_t*>(err_flag) != 0) return;
    build_plan<kWlThreads, int32_t>(qsl, ctx_lens, R, Hq, Hkv, D, num_sms, force_split_keys, force_decode_ctas, max_decode_items,
                                    scratch, tb, &ph);
    if (blockIdx.x == 0)
        for (int i = tid; i < R * Hkv; i += nt) merge_counters[i] = 0;     // "last split merges" arrival counters
    const int total = ph.tot_p + ph.tot_d;
    for (int idx = blockIdx.x * nt + tid; idx < total && idx < max_items; idx += nt * gridDim.x) {
        union { ss_work_item it; uint4 v[3]; } wu;
        plan_decode_item(idx, &ph, tb, qsl, ctx_lens, Hq, Hkv, wu.it);
        uint4* dst = reinterpret_cast<uint4*>(items + idx);
        dst[0] = wu.v[0]; dst[1] = wu.v[1]; dst[2] = wu.v[2];
    }
    if (tid == 0 && blockIdx.x == 0) {
        hdr->n_prefill = ph.tot_p;
        hdr->n_decode = ph.tot_d;
        hdr->n_partial = ph.tot_d;          // partial slots are numbered like the decode items
        hdr->split_keys = ph.L;
        hdr->next_prefill = 0;
        hdr->next_decode = 0;
        hdr->n_decode_ctas = ph.n_decode_ctas;
    }
}

cudaError_t launch_worklist(const Handle* h, const int32_t* qsl, const int32_t* ctx, int R, int T,
                            void* workspace, cudaStream_t stream) {
    (void)T;
    char* ws = (char*)workspace;
    const WorkspaceLayout& w = h->ws;
    const size_t smem = sizeof(int32_t) * 5 * (size_t)((R + 3) & ~3);
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(worklist_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    return launch_pdl(worklist_kernel, dim3(kWlCtas), dim3(kWlThreads), smem, stream, qsl, ctx, R, h->cfg.num_q_heads,
                      h->cfg.num_kv_heads, h->num_sms, h->cfg.head_dim, h->dbg[kDbgSplitKeys], h->dbg[kDbgDecodeCtas],
                      (WorkHeader*)(ws + w.header_off), (ss_work_item*)(ws + w.items_off),
                      (int32_t*)(ws + w.counters_off), w.max_items, w.max_partials,
                      (const int32_t*)(h->debug_checks ? h->state + kStateErr : nullptr));
}

}  // namespace ss
