// K2 work-list builder (a2).  Partitions the ragged batch {(c_r, u_r)} into CTA-sized
// work items on the device, from query_start_loc and ctx_lens only:
//   c_r == 0 -> nothing;  c_r == 1 -> decode set D;  c_r > 1 -> prefill set P   (Eq. 2)
//   prefill: one item per (request, 128-row tile, query head), keys [0, u + last row + 1)
//   decode : one item per (request, KV split, kv head); the split length L is chosen so that the batch
//            yields ~kDecodeWaves items per SM (tile aligned, clamped to [kMinSplitKeys, kMaxSplitKeys])
// Items of each kind are ordered heavy-first by request (longest KV range first) so the tail of the
// persistent main kernel is short.  Integer work only; one CTA; no host read-back.
#include "common.cuh"

namespace ss {

__device__ __forceinline__ int ceil_div(int a, int b) { return (a + b - 1) / b; }

__global__ void __launch_bounds__(1024)
worklist_kernel(const int32_t* __restrict__ qsl, const int32_t* __restrict__ ctx_lens, int R, int Hq, int Hkv,
                int num_sms, WorkHeader* __restrict__ hdr, ss_work_item* __restrict__ items,
                int32_t* __restrict__ req_nsplit, int32_t* __restrict__ req_partial, int max_items) {
    extern __shared__ int32_t sm[];
    int32_t* s_c = sm;              // c_r
    int32_t* s_u = s_c + R;         // u_r
    int32_t* s_np = s_u + R;        // prefill items of r
    int32_t* s_nd = s_np + R;       // decode items of r
    int32_t* s_ns = s_nd + R;       // splits of r (decode)
    int32_t* s_cost = s_ns + R;     // ordering key (KV length of the heaviest item)
    __shared__ unsigned long long s_total_keys;
    __shared__ int s_L;
    const int tid = threadIdx.x, nt = blockDim.x;

    if (tid == 0) s_total_keys = 0ull;
    __syncthreads();
    unsigned long long my_keys = 0;
    for (int r = tid; r < R; r += nt) {
        const int c = qsl[r + 1] - qsl[r];
        const int u = ctx_lens[r];
        s_c[r] = c;
        s_u[r] = u;
        if (c == 1) my_keys += (unsigned long long)(u + 1);
    }
    if (my_keys) atomicAdd(&s_total_keys, my_keys);
    __syncthreads();
    if (tid == 0) {
        const unsigned long long units = s_total_keys * (unsigned long long)Hkv;
        const unsigned long long target = (unsigned long long)num_sms * kDecodeWaves;
        unsigned long long L = (units + target - 1) / target;
        L = (L + kTileKeys - 1) / kTileKeys * kTileKeys;
        if (L < (unsigned long long)kMinSplitKeys) L = kMinSplitKeys;
        if (L > (unsigned long long)kMaxSplitKeys) L = kMaxSplitKeys;
        s_L = (int)L;
    }
    __syncthreads();
    const int L = s_L;
    for (int r = tid; r < R; r += nt) {
        const int c = s_c[r], u = s_u[r];
        int np = 0, nd = 0, ns = 0, cost = 0;
        if (c > 1) {
            np = ceil_div(c, kTileRows) * Hq;
            cost = u + c;
        } else if (c == 1) {
            const int n = u + 1;
            const int ns0 = ceil_div(n, L);
            const int chunk = ceil_div(ceil_div(n, ns0), kTileKeys) * kTileKeys;
            ns = ceil_div(n, chunk);
            nd = ns * Hkv;
            cost = chunk < n ? chunk : n;
        }
        s_np[r] = np; s_nd[r] = nd; s_ns[r] = ns; s_cost[r] = cost;
    }
    __syncthreads();

    // Per request: item offsets in heavy-first order (rank by cost desc, ties by index) and the
    // partial-slot base (request order).  O(R^2 / threads) integer compares; R is a few hundred.
    int tot_p = 0, tot_d = 0, tot_part = 0;
    for (int r = tid; r < R; r += nt) {
        const int my_cost = s_cost[r];
        const bool is_p = s_c[r] > 1, is_d = s_c[r] == 1;
        int off = 0, part = 0;
        for (int o = 0; o < R; ++o) {
            const bool before = (s_cost[o] > my_cost) || (s_cost[o] == my_cost && o < r);
            if (is_p && before) off += s_np[o];
            if (is_d && before) off += s_nd[o];
            if (o < r && s_ns[o] > 1) part += s_ns[o] * Hkv;
        }
        const int c = s_c[r], u = s_u[r];
        if (is_p) {
            const int ntile = ceil_div(c, kTileRows);
            for (int k = 0; k < ntile; ++k) {           // heaviest (last) tile first
                const int mt = ntile - 1 - k;
                const int nrows = min(kTileRows, c - mt * kTileRows);
                for (int hq = 0; hq < Hq; ++hq) {
                    const int idx = off + k * Hq + hq;
                    if (idx >= max_items) continue;
                    ss_work_item it;
                    it.kind = 1; it.req = r; it.head = hq; it.row0 = qsl[r] + mt * kTileRows; it.nrows = nrows;
                    it.kv_begin = 0; it.kv_end = u + mt * kTileRows + nrows; it.split = 0; it.nsplit = 1;
                    it.partial = -1; it.q_pos0 = mt * kTileRows; it.reserved = 0;
                    items[idx] = it;                    // prefill items occupy [0, n_prefill)
                }
            }
        }
        req_nsplit[r] = is_d ? s_ns[r] : 0;
        req_partial[r] = (is_d && s_ns[r] > 1) ? part : -1;
    }
    // totals
    __shared__ int s_tot[3];
    if (tid == 0) { s_tot[0] = s_tot[1] = s_tot[2] = 0; }
    __syncthreads();
    for (int r = tid; r < R; r += nt) {
        tot_p += s_np[r]; tot_d += s_nd[r];
        if (s_ns[r] > 1) tot_part += s_ns[r] * Hkv;
    }
    if (tot_p) atomicAdd(&s_tot[0], tot_p);
    if (tot_d) atomicAdd(&s_tot[1], tot_d);
    if (tot_part) atomicAdd(&s_tot[2], tot_part);
    __syncthreads();
    const int n_prefill = s_tot[0];

    // decode items: second pass now that the prefill count (their base index) is known
    for (int r = tid; r < R; r += nt) {
        if (s_c[r] != 1) continue;
        const int my_cost = s_cost[r];
        int off = 0, part = 0;
        for (int o = 0; o < R; ++o) {
            const bool before = (s_cost[o] > my_cost) || (s_cost[o] == my_cost && o < r);
            if (before) off += s_nd[o];
            if (o < r && s_ns[o] > 1) part += s_ns[o] * Hkv;
        }
        const int n = s_u[r] + 1;
        const int ns = s_ns[r];
        const int chunk = ceil_div(ceil_div(n, ceil_div(n, L)), kTileKeys) * kTileKeys;
        for (int s = 0; s < ns; ++s)
            for (int g = 0; g < Hkv; ++g) {
                const int idx = n_prefill + off + s * Hkv + g;
                if (idx >= max_items) continue;
                ss_work_item it;
                it.kind = 2; it.req = r; it.head = g; it.row0 = qsl[r]; it.nrows = 1;
                it.kv_begin = s * chunk; it.kv_end = min(n, (s + 1) * chunk); it.split = s; it.nsplit = ns;
                it.partial = ns > 1 ? part + g * ns : -1; it.q_pos0 = 0; it.reserved = 0;
                items[idx] = it;
            }
    }
    if (tid == 0) {
        hdr->n_prefill = s_tot[0];
        hdr->n_decode = s_tot[1];
        hdr->n_partial = s_tot[2];
        hdr->split_keys = L;
        hdr->n_merge = 0;
    }
}

cudaError_t launch_worklist(const Handle* h, const int32_t* qsl, const int32_t* ctx, int R, int T,
                            void* workspace, cudaStream_t stream) {
    (void)T;
    char* ws = (char*)workspace;
    const WorkspaceLayout& w = h->ws;
    const size_t smem = sizeof(int32_t) * 6 * (size_t)R;
    int threads = R >= 512 ? 1024 : (R >= 128 ? 512 : 256);
    worklist_kernel<<<1, threads, smem, stream>>>(
        qsl, ctx, R, h->cfg.num_q_heads, h->cfg.num_kv_heads, h->num_sms, (WorkHeader*)(ws + w.header_off),
        (ss_work_item*)(ws + w.items_off), (int32_t*)(ws + w.req_nsplit_off), (int32_t*)(ws + w.req_partial_off),
        w.max_items);
    return cudaGetLastError();
}

}  // namespace ss
