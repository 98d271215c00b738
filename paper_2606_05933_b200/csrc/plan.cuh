// a2 work-list plan (SURVEY.md §8(a) "work-list build"; north_star (d)): partitions the ragged batch {(c_r, u_r)}
// into CTA-sized work items from query_start_loc and ctx_lens only.
//   c_r == 0 -> nothing;  c_r == 1 -> decode set D;  c_r > 1 -> prefill set P   (Eq. 2)
//   prefill: one item per (request, 128-row tile, PAIR of query heads of one kv head), keys [0, u + last row + 1),
//            heaviest tile first.  The two heads share every staged K/V tile and run as two independent softmax
//            chains (attn_mixed.cu); a group with an odd number of heads (G = 1, 7) ends in a single-head item
//   decode : one item per (request, KV split, kv head); the split length L is chosen so that the batch yields
//            ~kDecodeWaves items per SM (tile aligned, clamped to [kMinSplitKeys, kMaxSplitKeys])
// Requests of each kind are ranked heavy-first (longest KV range first) so the tail of the persistent main kernel
// is short.  The plan is a pair of small rank tables; an item is decoded from its queue index on demand, so the main
// kernel can build the plan in its own prologue (one launch, no global round trip) and the stand-alone work-list
// kernel (ss_build_worklist; batches too large for the in-kernel tables) materialises exactly the same items.
// Integer work only.
#pragma once
#include "common.cuh"

namespace ss {

struct PlanHeader {                  // lives in shared memory
    int32_t L;                       // decode split length in keys (multiple of kTileKeys)
    int32_t nP, nD;                  // prefill / decode requests
    int32_t tot_p, tot_d;            // prefill / decode items
    int32_t n_decode_ctas;           // CTAs [0, n) drain the decode queue first
    int32_t pair_heads;              // 1: a prefill item serves two query heads of a kv head (two softmax chains per CTA)
    unsigned long long total_keys;   // sum over D of (u + 1)
    unsigned long long total_pairs;  // sum over P of c*u + c(c+1)/2
};

// ord[k] = request of rank k; ranks [0, nP) are the prefill requests, ranks [nP, nP + nD) the decode requests, each
// kind heavy-first.  off[k] = exclusive prefix, inside the kind, of row tiles (prefill) or KV splits (decode).
template <typename OffT>
struct PlanTables {
    uint16_t* ord;
    OffT* off;
};

__device__ __forceinline__ int plan_ceil_div(int a, int b) { return (a + b - 1) / b; }

// prefill items per (request, row tile): Hkv groups x ceil(G / 2) head pairs, or one per query head
__host__ __device__ __forceinline__ int plan_head_pairs(int Hq, int Hkv) { return Hkv * ((Hq / Hkv + 1) / 2); }
// Pair two heads per item unless the single-head items would all fit in one wave of CTAs anyway: a pair item keeps a
// CTA ~1.6x as long as a single-head item (two chains share the SM), so pairing pays only from the second wave on.
__host__ __device__ __forceinline__ int plan_pair_heads(int row_tiles, int Hq, int Hkv, int prefill_ctas) {
    return Hq / Hkv > 1 && row_tiles * Hq > prefill_ctas;
}

// balanced split of n keys into ceil(n / L) tile-aligned chunks
__device__ __forceinline__ int plan_decode_chunk(int n, int L) {
    return plan_ceil_div(plan_ceil_div(n, plan_ceil_div(n, L)), kTileKeys) * kTileKeys;
}

// All NT threads of the CTA call this; `scratch` = 3*R + 4 int32 of 16-byte aligned shared memory, dead afterwards
// (u + c < 2^29).
template <int NT, typename OffT>
__device__ void build_plan(const int32_t* __restrict__ qsl, const int32_t* __restrict__ ctx_lens, int R, int Hq, int Hkv,
                           int D, int num_sms, int force_split_keys, int force_decode_ctas, int max_decode_items,
                           int32_t* scratch, PlanTables<OffT> tb, PlanHeader* ph) {
    int32_t* s_c = scratch;
    int32_t* s_u = scratch + R;
    int32_t* s_cost = scratch + 2 * ((R + 3) & ~3);          // 16-byte aligned: read as int4
    const int tid = threadIdx.x, lane = tid & 31;
    if (tid == 0) { ph->total_keys = 0ull; ph->total_pairs = 0ull; ph->nP = 0; ph->nD = 0; }
    __syncthreads();
    // ---- (A) classify ----
    unsigned long long my_keys = 0, my_pairs = 0;
    int my_p = 0, my_d = 0;
    for (int r = tid; r < R; r += NT) {
        const int c = __ldg(qsl + r + 1) - __ldg(qsl + r);
        const int u = __ldg(ctx_lens + r);
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
        if (my_keys) atomicAdd(&ph->total_keys, my_keys);
        if (my_pairs) atomicAdd(&ph->total_pairs, my_pairs);
        if (my_p) atomicAdd(&ph->nP, my_p);
        if (my_d) atomicAdd(&ph->nD, my_d);
    }
    __syncthreads();
    if (tid == 0) {
        const unsigned long long units = ph->total_keys * (unsigned long long)Hkv;
        const unsigned long long target = (unsigned long long)num_sms * kDecodeWaves;
        unsigned long long L = (units + target - 1) / target;
        L = (L + kTileKeys - 1) / kTileKeys * kTileKeys;
        if (L < (unsigned long long)kMinSplitKeys) L = kMinSplitKeys;
        if (L > (unsigned long long)kMaxSplitKeys) L = kMaxSplitKeys;
        if (force_split_keys > 0) {
            L = (unsigned long long)(force_split_keys + kTileKeys - 1) / kTileKeys * kTileKeys;
            // The workspace's item / partial slots are sized for the automatic L (workspace_layout).  A forced, shorter L
            // can ask for more: sum_r ceil(n_r / L) <= total_keys / L + nD splits per kv head.  Raise it until the batch
            // fits; at kMaxSplitKeys it always does.
            while (L < (unsigned long long)kMaxSplitKeys &&
                   (ph->total_keys / L + (unsigned long long)ph->nD) * (unsigned long long)Hkv > (unsigned long long)max_decode_items)
                L += kTileKeys;
        }
        ph->L = (int)L;
    }
    __syncthreads();
    const int L = ph->L, nP = ph->nP, nD = ph->nD;
    // sort key: kind in the high bits (2 = prefill, 1 = decode, none = -1), cost (KV length of the heaviest item) below
    const int Rpad = (R + 3) & ~3;
    for (int r = tid; r < Rpad; r += NT) {
        int key = -1;
        if (r < R) {
            const int c = s_c[r], u = s_u[r];
            if (c > 1) {
                key = (2 << 29) | (u + c);
            } else if (c == 1) {
                const int n = u + 1, chunk = plan_decode_chunk(n, L);
                key = (1 << 29) | (chunk < n ? chunk : n);
            }
        }
        s_cost[r] = key;
    }
    __syncthreads();
    // ---- (B) heavy-first rank inside each kind (ties: lower request index first) ----
    for (int r = tid; r < R; r += NT) {
        const int my = s_cost[r];
        if (my >= 0) {
            const int hi = (my | ((1 << 29) - 1)) + 1;           // first key of the next kind
            int rank = 0;
            const int4* keys = reinterpret_cast<const int4*>(s_cost);
#pragma unroll 4
            for (int o4 = 0; o4 < Rpad / 4; ++o4) {
                const int4 k = keys[o4];
                const int o = o4 * 4;
                rank += ((k.x > my && k.x < hi) || (k.x == my && o + 0 < r)) ? 1 : 0;
                rank += ((k.y > my && k.y < hi) || (k.y == my && o + 1 < r)) ? 1 : 0;
                rank += ((k.z > my && k.z < hi) || (k.z == my && o + 2 < r)) ? 1 : 0;
                rank += ((k.w > my && k.w < hi) || (k.w == my && o + 3 < r)) ? 1 : 0;
            }
            tb.ord[((my >> 29) == 2 ? 0 : nP) + rank] = (uint16_t)r;
        }
    }
    __syncthreads();
    // ---- (C) exclusive prefix per kind, by warp 0 in rank order ----
    if (tid < 32) {
        int carry = 0;
        for (int base = 0; base < nP; base += 32) {
            const int k = base + lane;
            const int v = k < nP ? plan_ceil_div(s_c[tb.ord[k]], kTileRows) : 0;
            int incl = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += t; }
            if (k < nP) tb.off[k] = (OffT)(carry + incl - v);
            carry += __shfl_sync(0xffffffffu, incl, 31);
        }
        const int tiles_p = carry;
        carry = 0;
        for (int base = 0; base < nD; base += 32) {
            const int k = base + lane;
            const int v = k < nD ? plan_ceil_div(s_u[tb.ord[nP + k]] + 1, plan_decode_chunk(s_u[tb.ord[nP + k]] + 1, L)) : 0;
            int incl = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += t; }
            if (k < nD) tb.off[nP + k] = (OffT)(carry + incl - v);
            carry += __shfl_sync(0xffffffffu, incl, 31);
        }
        if (lane == 0) {
            const int tot_d = carry * Hkv;
            // SM partition between the two queues: SM-time of the decode items at the per-SM streaming rate vs SM-time
            // of the prefill tiles at the per-SM tensor rate; never more decode-first CTAs than saturate HBM.
            int nd = 0;
            if (tot_d > 0 && tiles_p == 0) nd = num_sms;
            else if (tot_d > 0) {
                const float t_d = (float)ph->total_keys * (float)(Hkv * D * 4) / kDecodeBytesPerUsPerSm;
                const float t_p = (float)ph->total_pairs * (float)Hq * (float)(4 * D) / kPrefillFlopsPerUsPerSm;
                nd = (int)((float)num_sms * t_d / (t_d + t_p) + 0.5f);
                if (nd < 1) nd = 1;
                if (nd > kMaxDecodeCtas) nd = kMaxDecodeCtas;
                if (nd > num_sms - 1) nd = num_sms - 1;
            }
            if (force_decode_ctas > 0) nd = force_decode_ctas;
            if (force_decode_ctas < 0) nd = 0;
            const int pair = plan_pair_heads(tiles_p, Hq, Hkv, num_sms - (nd < num_sms ? nd : 0));
            ph->pair_heads = pair;
            const int tot_p = tiles_p * (pair ? plan_head_pairs(Hq, Hkv) : Hq);
            ph->tot_p = tot_p;
            ph->tot_d = tot_d;
            ph->n_decode_ctas = nd;
        }
    }
    __syncthreads();
}

// Item `idx` of the queue order: [0, tot_p) prefill items, [tot_p, tot_p + tot_d) decode items.
template <typename OffT>
__device__ __forceinline__ void plan_decode_item(int idx, const PlanHeader* ph, PlanTables<OffT> tb,
                                                 const int32_t* __restrict__ qsl, const int32_t* __restrict__ ctx_lens,
                                                 int Hq, int Hkv, ss_work_item& it) {
    const int nP = ph->nP;
    if (idx < ph->tot_p) {
        const int G = Hq / Hkv, GP = ph->pair_heads ? (G + 1) / 2 : G, HP = Hkv * GP, hpi = ph->pair_heads ? 2 : 1;
        const int unit = idx / HP;
        int lo = 0, hi = nP;                             // last k with off[k] <= unit
        while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if ((int)tb.off[mid] <= unit) lo = mid; else hi = mid; }
        const int r = tb.ord[lo], local = idx - (int)tb.off[lo] * HP;
        const int q0 = __ldg(qsl + r), c = __ldg(qsl + r + 1) - q0, u = __ldg(ctx_lens + r);
        const int ntile = plan_ceil_div(c, kTileRows);
        const int mt = ntile - 1 - local / HP;           // heaviest (last) tile first
        const int nrows = min(kTileRows, c - mt * kTileRows);
        const int hp = local % HP, g = hp / GP, j = hp % GP;
        it.kind = 1; it.req = r; it.head = g * G + hpi * j; it.row0 = q0 + mt * kTileRows; it.nrows = nrows;
        it.kv_begin = 0; it.kv_end = u + mt * kTileRows + nrows; it.split = 0; it.nsplit = 1;
        it.partial = -1; it.q_pos0 = mt * kTileRows; it.nheads = (hpi == 2 && 2 * j + 1 < G) ? 2 : 1;
    } else {
        const int didx = idx - ph->tot_p, unit = didx / Hkv;
        int lo = 0, hi = ph->nD;
        while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if ((int)tb.off[nP + mid] <= unit) lo = mid; else hi = mid; }
        const int r = tb.ord[nP + lo], base = (int)tb.off[nP + lo] * Hkv, local = didx - base;
        const int n = __ldg(ctx_lens + r) + 1;
        const int chunk = plan_decode_chunk(n, ph->L), ns = plan_ceil_div(n, chunk);
        const int s = local / Hkv, g = local % Hkv;
        it.kind = 2; it.req = r; it.head = g; it.row0 = __ldg(qsl + r); it.nrows = 1;
        it.kv_begin = s * chunk; it.kv_end = min(n, (s + 1) * chunk); it.split = s; it.nsplit = ns;
        it.partial = ns > 1 ? base + g * ns : -1;        // partial slots share the decode items' index space
        it.q_pos0 = 0; it.nheads = Hq / Hkv;
    }
}

}  // namespace ss
