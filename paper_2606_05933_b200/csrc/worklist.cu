// K2 work-list builder (a2).  Partitions the ragged batch {(c_r, u_r)} into CTA-sized
// work items on the device, from query_start_loc and ctx_lens only:
//   c_r == 0 -> nothing;  c_r == 1 -> decode set D;  c_r > 1 -> prefill set P   (Eq. 2)
//   prefill: one item per (request, 128-row tile, query head), keys [0, u + last row + 1)
//   decode : one item per (request, KV split, kv head); the split length L is chosen so that the batch
//            yields ~kDecodeWaves items per SM (tile aligned, clamped to [kMinSplitKeys, kMaxSplitKeys])
// Items of each kind are ordered heavy-first by request (longest KV range first) so the tail of the
// persistent main kernel is short.  Integer work only; a few CTAs that each recompute the (tiny) per-request phases and write a slice of
// the items; no host read-back.
// Phases: (A) per-request counts, (B) heavy-first ranks, (C) block scans in rank order, (D) one thread
// per item writes its 48-byte record with three 16-byte stores.
#include "common.cuh"
#include "ptx.cuh"

namespace ss {

__device__ __forceinline__ int ceil_div(int a, int b) { return (a + b - 1) / b; }

constexpr int kWlThreads = 512;
constexpr int kWlCtas = 8;            // every CTA recomputes phases A-C (R is small) and writes its slice of the items

// Exclusive scan of three int arrays at once (x[0..n0), y[0..n1), z[0..n2)) in place; totals returned through tot[3].
// Each thread owns a contiguous chunk; chunk sums are scanned with warp shuffles (two levels).
__device__ void block_exclusive_scan3(int32_t* x, int n0, int32_t* y, int n1, int32_t* z, int n2, int32_t* warp_tmp,
                                      int32_t* tot) {
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    constexpr int kWarps = kWlThreads / 32;
    int32_t* arr[3] = {x, y, z};
    const int nn[3] = {n0, n1, n2};
    int sum[3], chunk[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        chunk[a] = (nn[a] + kWlThreads - 1) / kWlThreads;
        int sacc = 0;
        for (int i = tid * chunk[a]; i < min(nn[a], (tid + 1) * chunk[a]); ++i) sacc += arr[a][i];
        sum[a] = sacc;
    }
    int incl[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        int v = sum[a];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, v, o); if (lane >= o) v += t; }
        incl[a] = v;
        if (lane == 31) warp_tmp[a * kWarps + wid] = v;
    }
    __syncthreads();
    if (wid == 0) {
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            int v = lane < kWarps ? warp_tmp[a * kWarps + lane] : 0;
#pragma unroll
            for (int o = 1; o < kWarps; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, v, o); if (lane >= o) v += t; }
            if (lane < kWarps) warp_tmp[a * kWarps + lane] = v;           // inclusive over warps
            if (lane == kWarps - 1) tot[a] = v;
        }
    }
    __syncthreads();
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        int run = incl[a] - sum[a] + (wid > 0 ? warp_tmp[a * kWarps + wid - 1] : 0);
        for (int i = tid * chunk[a]; i < min(nn[a], (tid + 1) * chunk[a]); ++i) { const int v = arr[a][i]; arr[a][i] = run; run += v; }
    }
    __syncthreads();
}

__global__ void __launch_bounds__(kWlThreads)
worklist_kernel(const int32_t* __restrict__ qsl, const int32_t* __restrict__ ctx_lens, int R, int Hq, int Hkv,
                int num_sms, int D, int force_split_keys, int force_decode_ctas, WorkHeader* __restrict__ hdr,
                ss_work_item* __restrict__ items, int32_t* __restrict__ merge_counters, int max_items) {
    extern __shared__ int32_t sm[];
    int32_t* s_c = sm;               // c_r
    int32_t* s_u = s_c + R;          // u_r
    int32_t* s_ns = s_u + R;         // decode splits of r
    int32_t* s_cost = s_ns + R;      // ordering key (KV length of the heaviest item)
    int32_t* s_ordP = s_cost + R;    // rank k -> request (prefill)
    int32_t* s_ordD = s_ordP + R;    // rank k -> request (decode)
    int32_t* s_offP = s_ordD + R;    // rank k -> first prefill item
    int32_t* s_offD = s_offP + R;    // rank k -> first decode item (relative to the decode base)
    int32_t* s_part = s_offD + R;    // request -> partial slot base
    __shared__ unsigned long long s_total_keys, s_total_pairs;
    __shared__ int s_L, s_nP, s_nD;
    __shared__ int32_t s_warp_tmp[3 * (kWlThreads / 32)];
    __shared__ int32_t s_tot[3];
    const int tid = threadIdx.x, nt = blockDim.x, lane = tid & 31;

    ptx::pdl_launch_dependents();
    if (tid == 0) { s_total_keys = 0ull; s_total_pairs = 0ull; s_nP = 0; s_nD = 0; }
    __syncthreads();
    ptx::pdl_wait();            // qsl / ctx_lens may come from the preceding kernel in the stream
    // ---- (A) ----
    unsigned long long my_keys = 0, my_pairs = 0;
    int my_p = 0, my_d = 0;
    for (int r = tid; r < R; r += nt) {
        const int c = qsl[r + 1] - qsl[r];
        const int u = ctx_lens[r];
        s_c[r] = c;
        s_u[r] = u;
        if (c == 1) { my_keys += (unsigned long long)(u + 1); ++my_d; }
        if (c > 1) { ++my_p; my_pairs += (unsigned long long)c * (unsigned long long)u + (unsigned long long)c * (c + 1) / 2; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        my_keys += __shfl_xor_sync(0xffffffffu, my_keys, o);
        my_pairs += __shfl_xor_sync(0xffffffffu, my_pairs, o);
        my_p += __shfl_xor_sync(0xffffffffu, my_p, o);
        my_d += __shfl_xor_sync(0xffffffffu, my_d, o);
    }
    if (lane == 0) {
        if (my_keys) atomicAdd(&s_total_keys, my_keys);
        if (my_pairs) atomicAdd(&s_total_pairs, my_pairs);
        if (my_p) atomicAdd(&s_nP, my_p);
        if (my_d) atomicAdd(&s_nD, my_d);
    }
    __syncthreads();
    if (tid == 0) {
        const unsigned long long units = s_total_keys * (unsigned long long)Hkv;
        const unsigned long long target = (unsigned long long)num_sms * kDecodeWaves;
        unsigned long long L = (units + target - 1) / target;
        L = (L + kTileKeys - 1) / kTileKeys * kTileKeys;
        if (L < (unsigned long long)kMinSplitKeys) L = kMinSplitKeys;
        if (L > (unsigned long long)kMaxSplitKeys) L = kMaxSplitKeys;
        if (force_split_keys > 0) L = (unsigned long long)(force_split_keys + kTileKeys - 1) / kTileKeys * kTileKeys;
        s_L = (int)L;
    }
    __syncthreads();
    const int L = s_L, nP = s_nP, nD = s_nD;
    for (int r = tid; r < R; r += nt) {
        const int c = s_c[r], u = s_u[r];
        int ns = 0, cost = 0;
        if (c > 1) {
            cost = u + c;
        } else if (c == 1) {
            const int n = u + 1;
            const int chunk = ceil_div(ceil_div(n, ceil_div(n, L)), kTileKeys) * kTileKeys;
            ns = ceil_div(n, chunk);
            cost = chunk < n ? chunk : n;
        }
        s_ns[r] = ns;
        s_cost[r] = cost;
    }
    __syncthreads();
    // ---- (B) heavy-first rank inside each kind; partial-slot sizes in request order ----
    for (int r = tid; r < R; r += nt) {
        const int c = s_c[r], my_cost = s_cost[r];
        if (c >= 1) {
            const bool is_p = c > 1;
            int rank = 0;
            for (int o = 0; o < R; ++o) {
                const int co = s_c[o];
                const bool same = is_p ? (co > 1) : (co == 1);
                rank += (same && (s_cost[o] > my_cost || (s_cost[o] == my_cost && o < r))) ? 1 : 0;
            }
            (is_p ? s_ordP : s_ordD)[rank] = r;
        }
        s_part[r] = (c == 1 && s_ns[r] > 1) ? s_ns[r] * Hkv : 0;
    }
    __syncthreads();
    // ---- (C) scans ----
    for (int k = tid; k < nP; k += nt) s_offP[k] = ceil_div(s_c[s_ordP[k]], kTileRows) * Hq;
    for (int k = tid; k < nD; k += nt) s_offD[k] = s_ns[s_ordD[k]] * Hkv;
    __syncthreads();
    block_exclusive_scan3(s_offP, nP, s_offD, nD, s_part, R, s_warp_tmp, s_tot);
    const int tot_p = s_tot[0], tot_d = s_tot[1], tot_part = s_tot[2];
    if (blockIdx.x == 0)
        for (int i = tid; i < R * Hkv; i += nt) merge_counters[i] = 0;     // "last split merges" arrival counters
    // ---- (D) one thread per item ----
    const int total = tot_p + tot_d;
    for (int idx = blockIdx.x * nt + tid; idx < total && idx < max_items; idx += nt * gridDim.x) {
        union { ss_work_item it; uint4 v[3]; } wu;
        ss_work_item& it = wu.it;
        if (idx < tot_p) {
            int lo = 0, hi = nP;                         // last k with offP[k] <= idx
            while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (s_offP[mid] <= idx) lo = mid; else hi = mid; }
            const int r = s_ordP[lo], local = idx - s_offP[lo];
            const int c = s_c[r], u = s_u[r];
            const int ntile = ceil_div(c, kTileRows);
            const int mt = ntile - 1 - local / Hq;       // heaviest (last) tile first
            const int nrows = min(kTileRows, c - mt * kTileRows);
            it.kind = 1; it.req = r; it.head = local % Hq; it.row0 = qsl[r] + mt * kTileRows; it.nrows = nrows;
            it.kv_begin = 0; it.kv_end = u + mt * kTileRows + nrows; it.split = 0; it.nsplit = 1;
            it.partial = -1; it.q_pos0 = mt * kTileRows; it.reserved = 0;
        } else {
            const int didx = idx - tot_p;
            int lo = 0, hi = nD;
            while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (s_offD[mid] <= didx) lo = mid; else hi = mid; }
            const int r = s_ordD[lo], local = didx - s_offD[lo];
            const int n = s_u[r] + 1, ns = s_ns[r];
            const int chunk = ceil_div(ceil_div(n, ceil_div(n, L)), kTileKeys) * kTileKeys;
            const int s = local / Hkv, g = local % Hkv;
            it.kind = 2; it.req = r; it.head = g; it.row0 = qsl[r]; it.nrows = 1;
            it.kv_begin = s * chunk; it.kv_end = min(n, (s + 1) * chunk); it.split = s; it.nsplit = ns;
            it.partial = ns > 1 ? s_part[r] + g * ns : -1; it.q_pos0 = 0; it.reserved = 0;
        }
        uint4* dst = reinterpret_cast<uint4*>(items + idx);
        dst[0] = wu.v[0]; dst[1] = wu.v[1]; dst[2] = wu.v[2];
    }
    if (tid == 0 && blockIdx.x == 0) {
        hdr->n_prefill = tot_p;
        hdr->n_decode = tot_d;
        hdr->n_partial = tot_part;
        hdr->split_keys = L;
        hdr->next_prefill = 0;
        hdr->next_decode = 0;
        // SM partition between the two queues: SM-time of the decode items at the per-SM streaming rate vs
        // SM-time of the prefill tiles at the per-SM tensor rate; never more decode-first CTAs than saturate HBM.
        int nd = 0;
        if (tot_d > 0 && tot_p == 0) nd = num_sms;
        else if (tot_d > 0) {
            const float t_d = (float)s_total_keys * (float)(Hkv * D * 4) / kDecodeBytesPerUsPerSm;
            const float t_p = (float)s_total_pairs * (float)Hq * (float)(4 * D) / kPrefillFlopsPerUsPerSm;
            nd = (int)((float)num_sms * t_d / (t_d + t_p) + 0.5f);
            if (nd < 1) nd = 1;
            if (nd > kMaxDecodeCtas) nd = kMaxDecodeCtas;
            if (nd > num_sms - 1) nd = num_sms - 1;
        }
        if (force_decode_ctas > 0) nd = force_decode_ctas;
        if (force_decode_ctas < 0) nd = 0;
        hdr->n_decode_ctas = nd;
    }
}

cudaError_t launch_worklist(const Handle* h, const int32_t* qsl, const int32_t* ctx, int R, int T,
                            void* workspace, cudaStream_t stream) {
    (void)T;
    char* ws = (char*)workspace;
    const WorkspaceLayout& w = h->ws;
    const size_t smem = sizeof(int32_t) * 9 * (size_t)R;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(worklist_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    return launch_pdl(worklist_kernel, dim3(kWlCtas), dim3(kWlThreads), smem, stream, qsl, ctx, R, h->cfg.num_q_heads,
                      h->cfg.num_kv_heads, h->num_sms, h->cfg.head_dim, h->dbg[kDbgSplitKeys], h->dbg[kDbgDecodeCtas],
                      (WorkHeader*)(ws + w.header_off), (ss_work_item*)(ws + w.items_off),
                      (int32_t*)(ws + w.counters_off), w.max_items);
}

}  // namespace ss
