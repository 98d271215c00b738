// K4 decode splits (a4): the single query row of a request with c_r == 1 (the paper's
// decode set D, Eq. 2) attends keys [kv_begin, kv_end) of one KV head for all G query heads
// of the group at once.  HBM-bound (arithmetic intensity G flop/B); the roofline that bounds it is the
// measured HBM copy bandwidth, algorithmic bytes per cached token per kv head = 2 * D * 2.
//
// Design (B200): persistent CTAs, one per SM, static striding over the device work list.
//   warp 0          : TMA producer.  Per 128-key tile, 8 pages x {K,V} x D/64 boxes of 16 rows x 128 B
//                     (SWIZZLE_128B) land in a 3-stage ring; one lane per box, one mbarrier per stage.
//   warps 1..4      : consumers.  Warp w owns keys [32w, 32w+32) of every tile: S = Q K^T with
//                     mma.sync.m16n8k16 (the G heads padded to the 16 MMA rows — wasted rows are free, the
//                     path is bandwidth-bound), online softmax in registers (quad shuffles), O += P V.
//   item end        : the four warps' (m, l, O) are merged through shared memory with the log-sum-exp
//                     rule, then written as the final bf16 row (unsplit item) or as an fp32 partial
//                     (o, m, l) for the merge kernel K5.
// Unused slots / stale smem rows never reach the result: masked scores are replaced (not multiplied) and
// V rows past kv_end are zeroed in shared memory before the PV MMA (0 * NaN would poison the row).
#include "common.cuh"
#include "ptx.cuh"

namespace ss {

using namespace ptx;

constexpr int kDecStages = 3;
constexpr int kDecConsumerWarps = 4;
constexpr int kDecThreads = 32 * (1 + kDecConsumerWarps);
constexpr float kLog2eF = 1.4426950408889634f;
constexpr float kLn2F = 0.6931471805599453f;

template <int D>
struct DecodeSmem {
    static constexpr int kHalves = D / 64;
    static constexpr int kTileBytes = kHalves * kTileKeys * 128;         // K (or V) tile: [half][128 rows][128 B]
    static constexpr int kStageBytes = 2 * kTileBytes;
    static constexpr int kMergeFloats = kDecConsumerWarps * kMaxGroup * (D + 2);
    static constexpr int kBarOff = kDecStages * kStageBytes;
    static constexpr int kMergeOff = kBarOff + 128;
    static constexpr int kTotal = kMergeOff + kMergeFloats * 4 + 1024;   // + slack for 1024 B alignment
};

template <int D>
__global__ void __launch_bounds__(kDecThreads, 1)
decode_kernel(const __grid_constant__ CUtensorMap tmap_k, const __grid_constant__ CUtensorMap tmap_v,
              const __nv_bfloat16* __restrict__ q, const int32_t* __restrict__ block_table,
              const WorkHeader* __restrict__ hdr, const ss_work_item* __restrict__ items, int max_pages, int Hq,
              int Hkv, float scale, float* __restrict__ partials, __nv_bfloat16* __restrict__ out,
              float* __restrict__ lse) {
    using SM = DecodeSmem<D>;
    constexpr int kHalves = SM::kHalves;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* smem = smem_raw + (smem_base - smem_u32(smem_raw));
    const uint32_t bar_full = smem_base + SM::kBarOff;             // kDecStages x 8 B
    const uint32_t bar_empty = bar_full + 8 * kDecStages;
    float* merge = reinterpret_cast<float*>(smem + SM::kMergeOff);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int G = Hq / Hkv;
    const int n_prefill = hdr->n_prefill;
    const int n_decode = hdr->n_decode;
    items += n_prefill;

    if (threadIdx.x == 0) {
        for (int s = 0; s < kDecStages; ++s) {
            mbar_init(bar_full + 8 * s, 1);
            mbar_init(bar_empty + 8 * s, kDecConsumerWarps);
        }
        fence_barrier_init();
        prefetch_tmap(&tmap_k);
        prefetch_tmap(&tmap_v);
    }
    __syncthreads();

    if (warp == 0) {
        // ===================== TMA producer =====================
        int stage = 0;
        uint32_t phase = 0;
        constexpr int kBoxes = 8 * 2 * kHalves;                    // boxes per tile
        for (int it = blockIdx.x; it < n_decode; it += gridDim.x) {
            const ss_work_item w = items[it];
            const int32_t* bt = block_table + (int64_t)w.req * max_pages;
            for (int key0 = w.kv_begin; key0 < w.kv_end; key0 += kTileKeys) {
                const int npages = min(8, (w.kv_end - key0 + kPage - 1) / kPage);
                mbar_wait(bar_empty + 8 * stage, phase ^ 1);
                if (lane == 0) mbar_arrive_expect_tx(bar_full + 8 * stage, (uint32_t)npages * 2 * kHalves * 2048);
                __syncwarp();
                if (lane < kBoxes) {
                    const int p = lane / (2 * kHalves);
                    const int which = lane % (2 * kHalves);          // [K halves..., V halves...]
                    const int is_v = which / kHalves, half = which % kHalves;
                    if (p < npages) {
                        const int page = __ldg(bt + (key0 >> 4) + p);
                        const uint32_t dst = smem_base + stage * SM::kStageBytes + is_v * SM::kTileBytes +
                                             half * (kTileKeys * 128) + p * (kPage * 128);
                        tma_load_2d(dst, is_v ? &tmap_v : &tmap_k, half * 64, (page * Hkv + w.head) * kPage,
                                    bar_full + 8 * stage);
                    }
                }
                if (++stage == kDecStages) { stage = 0; phase ^= 1; }
            }
        }
    } else {
        // ===================== consumers =====================
        const int cw = warp - 1;                                   // 0..3 -> keys [32cw, 32cw+32) of a tile
        const int qrow = lane >> 2, qcol = (lane & 3) * 2;
        const float sl2 = scale * kLog2eF;
        int stage = 0;
        uint32_t phase = 0;
        for (int it = blockIdx.x; it < n_decode; it += gridDim.x) {
            const ss_work_item w = items[it];
            // ---- Q fragments: rows = the G heads of kv head w.head (rows >= G are zero) ----
            uint32_t qa[D / 16][4];
            {
                const __nv_bfloat16* qb = q + ((int64_t)w.row0 * Hq + (int64_t)w.head * G) * D;
#pragma unroll
                for (int ks = 0; ks < D / 16; ++ks) {
                    const int d0 = ks * 16 + qcol;
                    qa[ks][0] = qrow < G ? *reinterpret_cast<const uint32_t*>(qb + (int64_t)qrow * D + d0) : 0u;
                    qa[ks][1] = qrow + 8 < G ? *reinterpret_cast<const uint32_t*>(qb + (int64_t)(qrow + 8) * D + d0) : 0u;
                    qa[ks][2] = qrow < G ? *reinterpret_cast<const uint32_t*>(qb + (int64_t)qrow * D + d0 + 8) : 0u;
                    qa[ks][3] = qrow + 8 < G ? *reinterpret_cast<const uint32_t*>(qb + (int64_t)(qrow + 8) * D + d0 + 8) : 0u;
                }
            }
            float o[D / 8][4];
#pragma unroll
            for (int i = 0; i < D / 8; ++i) o[i][0] = o[i][1] = o[i][2] = o[i][3] = 0.f;
            float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;     // rows qrow, qrow+8 (log2 units)

            for (int key0 = w.kv_begin; key0 < w.kv_end; key0 += kTileKeys) {
                mbar_wait(bar_full + 8 * stage, phase);
                const int nvalid = w.kv_end - (key0 + 32 * cw);          // valid keys in my 32-key slice
                if (nvalid > 0) {
                    const uint32_t kbase = smem_base + stage * SM::kStageBytes;
                    const uint32_t vbase = kbase + SM::kTileBytes;
                    if (nvalid < 32) {
                        // zero V rows [nvalid, 32) of my slice (stale or never-written data may be NaN)
                        for (int i = lane; i < (32 - nvalid) * kHalves * 8; i += 32) {
                            const int r = 32 * cw + nvalid + i / (kHalves * 8);
                            const int c = i % (kHalves * 8);
                            const uint32_t a = vbase + (c >> 3) * (kTileKeys * 128) + r * 128 + (c & 7) * 16;
                            asm volatile("st.shared.v4.b32 [%0], {%1,%1,%1,%1};" ::"r"(a), "r"(0u) : "memory");
                        }
                        __syncwarp();
                    }
                    // ---- S = Q K^T : 16 x 32 ----
                    float s[4][4];
#pragma unroll
                    for (int nt = 0; nt < 4; ++nt) s[nt][0] = s[nt][1] = s[nt][2] = s[nt][3] = 0.f;
#pragma unroll
                    for (int j = 0; j < D / 32; ++j) {                  // pairs of k-steps (4 chunks of 16 B)
#pragma unroll
                        for (int nt = 0; nt < 4; ++nt) {
                            const int row = 32 * cw + nt * 8 + (lane & 7);
                            const int cd = 4 * j + (lane >> 3);         // 16-byte chunk of d
                            const uint32_t a = kbase + (cd >> 3) * (kTileKeys * 128) + row * 128 + (((cd & 7) ^ (row & 7)) << 4);
                            uint32_t b0, b1, b2, b3;
                            ldmatrix_x4(b0, b1, b2, b3, a);
                            mma_bf16_16816(s[nt], qa[2 * j], b0, b1);
                            mma_bf16_16816(s[nt], qa[2 * j + 1], b2, b3);
                        }
                    }
                    // ---- mask + online softmax (rows qrow and qrow+8) ----
                    float bm0 = -INFINITY, bm1 = -INFINITY;
#pragma unroll
                    for (int nt = 0; nt < 4; ++nt) {
                        const int c = nt * 8 + qcol;
                        if (c >= nvalid) { s[nt][0] = -INFINITY; s[nt][2] = -INFINITY; }
                        if (c + 1 >= nvalid) { s[nt][1] = -INFINITY; s[nt][3] = -INFINITY; }
                        bm0 = fmaxf(bm0, fmaxf(s[nt][0], s[nt][1]));
                        bm1 = fmaxf(bm1, fmaxf(s[nt][2], s[nt][3]));
                    }
                    bm0 = fmaxf(bm0, __shfl_xor_sync(0xffffffffu, bm0, 1));
                    bm0 = fmaxf(bm0, __shfl_xor_sync(0xffffffffu, bm0, 2));
                    bm1 = fmaxf(bm1, __shfl_xor_sync(0xffffffffu, bm1, 1));
                    bm1 = fmaxf(bm1, __shfl_xor_sync(0xffffffffu, bm1, 2));
                    const float mn0 = fmaxf(m0, bm0 * sl2), mn1 = fmaxf(m1, bm1 * sl2);   // finite: key 0 of the slice is valid
                    const float al0 = exp2f(m0 - mn0), al1 = exp2f(m1 - mn1);
                    float ps0 = 0.f, ps1 = 0.f;
                    uint32_t pa[2][4];
#pragma unroll
                    for (int nt = 0; nt < 4; ++nt) {
                        const float p0 = exp2f(s[nt][0] * sl2 - mn0), p1 = exp2f(s[nt][1] * sl2 - mn0);
                        const float p2 = exp2f(s[nt][2] * sl2 - mn1), p3 = exp2f(s[nt][3] * sl2 - mn1);
                        ps0 += p0 + p1;
                        ps1 += p2 + p3;
                        pa[nt >> 1][(nt & 1) * 2 + 0] = pack_bf16(p0, p1);
                        pa[nt >> 1][(nt & 1) * 2 + 1] = pack_bf16(p2, p3);
                    }
                    l0 = l0 * al0 + ps0;
                    l1 = l1 * al1 + ps1;
                    m0 = mn0;
                    m1 = mn1;
#pragma unroll
                    for (int i = 0; i < D / 8; ++i) { o[i][0] *= al0; o[i][1] *= al0; o[i][2] *= al1; o[i][3] *= al1; }
                    // ---- O += P V : k-steps of 16 keys, n-tiles of 8 d ----
#pragma unroll
                    for (int kk = 0; kk < 2; ++kk) {
#pragma unroll
                        for (int np = 0; np < D / 16; ++np) {
                            const int row = 32 * cw + kk * 16 + ((lane >> 3) & 1) * 8 + (lane & 7);
                            const int cd = 2 * np + (lane >> 4);
                            const uint32_t a = vbase + (cd >> 3) * (kTileKeys * 128) + row * 128 + (((cd & 7) ^ (row & 7)) << 4);
                            uint32_t b0, b1, b2, b3;
                            ldmatrix_x4_trans(b0, b1, b2, b3, a);
                            mma_bf16_16816(o[2 * np], pa[kk], b0, b1);
                            mma_bf16_16816(o[2 * np + 1], pa[kk], b2, b3);
                        }
                    }
                    if (nvalid < 32) fence_proxy_async();    // order my generic zero-fill before the next TMA into this stage
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_empty + 8 * stage);
                if (++stage == kDecStages) { stage = 0; phase ^= 1; }
            }

            // ---- item end: quad-reduce l, then merge the four warps through shared memory ----
            l0 += __shfl_xor_sync(0xffffffffu, l0, 1);
            l0 += __shfl_xor_sync(0xffffffffu, l0, 2);
            l1 += __shfl_xor_sync(0xffffffffu, l1, 1);
            l1 += __shfl_xor_sync(0xffffffffu, l1, 2);
            float* mine = merge + cw * kMaxGroup * (D + 2);
#pragma unroll
            for (int i = 0; i < D / 8; ++i) {
                *reinterpret_cast<float2*>(mine + qrow * (D + 2) + i * 8 + qcol) = make_float2(o[i][0], o[i][1]);
                *reinterpret_cast<float2*>(mine + (qrow + 8) * (D + 2) + i * 8 + qcol) = make_float2(o[i][2], o[i][3]);
            }
            if ((lane & 3) == 0) {
                mine[qrow * (D + 2) + D] = m0;
                mine[qrow * (D + 2) + D + 1] = l0;
                mine[(qrow + 8) * (D + 2) + D] = m1;
                mine[(qrow + 8) * (D + 2) + D + 1] = l1;
            }
            named_bar_sync(1, 32 * kDecConsumerWarps);
            {
                const int ct = threadIdx.x - 32;                         // 0..127
                for (int e = ct; e < G * D; e += 32 * kDecConsumerWarps) {
                    const int row = e / D, d = e % D;
                    float M = -INFINITY;
#pragma unroll
                    for (int x = 0; x < kDecConsumerWarps; ++x) M = fmaxf(M, merge[(x * kMaxGroup + row) * (D + 2) + D]);
                    float L = 0.f, acc = 0.f;
#pragma unroll
                    for (int x = 0; x < kDecConsumerWarps; ++x) {
                        const float* src = merge + (x * kMaxGroup + row) * (D + 2);
                        const float wgt = exp2f(src[D] - M);            // exp2(-inf) = 0 for warps that saw no key
                        L += src[D + 1] * wgt;
                        acc += src[d] * wgt;
                    }
                    if (w.nsplit == 1) {
                        const int64_t orow = (int64_t)w.row0 * Hq + (int64_t)w.head * G + row;
                        out[orow * D + d] = __float2bfloat16_rn(acc / L);
                        if (lse && d == 0) lse[orow] = (M + log2f(L)) * kLn2F;
                    } else {
                        float* dst = partials + ((int64_t)(w.partial + w.split) * G + row) * (D + 2);
                        dst[d] = acc;
                        if (d == 0) { dst[D] = M; dst[D + 1] = L; }
                    }
                }
            }
            named_bar_sync(1, 32 * kDecConsumerWarps);
        }
    }
}

cudaError_t launch_decode(const Handle* h, const void* q, const int32_t* bt, float scale, void* workspace,
                          void* out, float* lse, cudaStream_t stream) {
    const ss_config& c = h->cfg;
    char* ws = (char*)workspace;
    const WorkHeader* hdr = (const WorkHeader*)(ws + h->ws.header_off);
    const ss_work_item* items = (const ss_work_item*)(ws + h->ws.items_off);
    float* partials = (float*)(ws + h->ws.partial_off);
    cudaError_t e;
    if (c.head_dim == 128) {
        auto kern = decode_kernel<128>;
        constexpr int smem = DecodeSmem<128>::kTotal;
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        kern<<<h->num_sms, kDecThreads, smem, stream>>>(h->tmap_k, h->tmap_v, (const __nv_bfloat16*)q, bt, hdr, items,
                                                        c.max_pages_per_req, c.num_q_heads, c.num_kv_heads, scale,
                                                        partials, (__nv_bfloat16*)out, lse);
    } else {
        auto kern = decode_kernel<64>;
        constexpr int smem = DecodeSmem<64>::kTotal;
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        kern<<<h->num_sms, kDecThreads, smem, stream>>>(h->tmap_k, h->tmap_v, (const __nv_bfloat16*)q, bt, hdr, items,
                                                        c.max_pages_per_req, c.num_q_heads, c.num_kv_heads, scale,
                                                        partials, (__nv_bfloat16*)out, lse);
    }
    return cudaGetLastError();
}

}  // namespace ss
