// K3 prefill-chunk tiles (a3): for a request with c_r > 1 (the paper's prefill set P,
// PAPER.md:111 Eq. 2), query head h and a tile of up to 128 query rows, row j attends keys 0..u_r+j.
// This is the dense contraction of the path (x1 - x2/2 of PAPER.md:140-141 drives its FLOPs) and runs on
// the 5th-gen tensor cores: the roofline that bounds it is bf16 tensor throughput, 4*D flop per
// (row, visible key) pair per head.
//
// Design (B200): persistent CTAs, static striding over the device work list, 6 warps:
//   warp 0      TMA producer: Q tile (2 boxes of 128 rows x 64 cols) once per item; per 128-key step the
//               K and V tiles as 8 pages x 16-row boxes, SWIZZLE_128B, into a 2-stage ring.
//   warp 1      tcgen05.mma issuer (one elected thread) and TMEM owner:
//                 S[128x128 fp32, TMEM cols 0..127]   = Q K^T      (A, B K-major from smem)
//                 O[128xD  fp32, TMEM cols 128..]    += P V        (A = P K-major from smem, B = V MN-major)
//   warps 2..5  softmax: thread = query row (TMEM lane).  tcgen05.ld S, causal/length mask by select,
//               online softmax in fp32 (exp2 with log2e folded into the scale), P -> bf16 into a swizzled
//               smem tile, O rescaled in TMEM only when some row's max moved; epilogue normalises and
//               stores rows < nrows only (rows past the chunk belong to the next request).
// V rows at or past kv_end are zeroed in smem before the PV MMA (unused slots may hold NaN; 0*NaN = NaN).
#include "common.cuh"
#include "ptx.cuh"

namespace ss {

using namespace ptx;

constexpr int kPreStages = 2;
constexpr int kPreThreads = 192;
constexpr float kPLog2e = 1.4426950408889634f;
constexpr float kPLn2 = 0.6931471805599453f;

template <int D>
struct PrefillSmem {
    static constexpr int kHalves = D / 64;
    static constexpr int kQBytes = kHalves * kTileRows * 128;
    static constexpr int kKBytes = kHalves * kTileKeys * 128;
    static constexpr int kVBytes = kKBytes;
    static constexpr int kPBytes = 2 * kTileRows * 128;                 // 128 keys = 2 halves of 64
    static constexpr int kQOff = 0;
    static constexpr int kKVOff = kQOff + kQBytes;                       // stage s: K at kKVOff + s*(K+V), V after K
    static constexpr int kStageBytes = kKBytes + kVBytes;
    static constexpr int kPOff = kKVOff + kPreStages * kStageBytes;
    static constexpr int kBarOff = kPOff + kPBytes;
    static constexpr int kTotal = kBarOff + 256 + 1024;
    static constexpr int kTmemCols = (128 + D) <= 256 ? 256 : 512;
};

// 64-bit UMMA shared-memory descriptor, SWIZZLE_128B, sm_100 version bits.
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
    uint64_t d = 0;
    d |= (uint64_t)((saddr & 0x3FFFFu) >> 4);
    d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFFu) << 16;
    d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFFu) << 32;
    d |= (uint64_t)1 << 46;                 // descriptor version (Blackwell)
    d |= (uint64_t)2 << 61;                 // layout type: SWIZZLE_128B
    return d;
}
// kind::f16 instruction descriptor: bf16 x bf16 -> fp32, M x N, A K-major, B K- or MN-major.
__host__ __device__ constexpr uint32_t umma_idesc(int M, int N, int b_mn_major) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)b_mn_major << 16) | ((uint32_t)(N >> 3) << 17) |
           ((uint32_t)(M >> 4) << 24);
}

template <int D>
__global__ void __launch_bounds__(kPreThreads, 1)
prefill_kernel(const __grid_constant__ CUtensorMap tmap_q, const __grid_constant__ CUtensorMap tmap_k,
               const __grid_constant__ CUtensorMap tmap_v, const int32_t* __restrict__ block_table,
               const int32_t* __restrict__ ctx_lens, const WorkHeader* __restrict__ hdr,
               const ss_work_item* __restrict__ items, int max_pages, int Hq, int Hkv, float scale,
               __nv_bfloat16* __restrict__ out, float* __restrict__ lse) {
    using SM = PrefillSmem<D>;
    constexpr int kHalves = SM::kHalves;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* smem = smem_raw + (sbase - smem_u32(smem_raw));

    // barriers
    const uint32_t bar0 = sbase + SM::kBarOff;
    const uint32_t bar_q_full = bar0 + 0, bar_q_empty = bar0 + 8;
    const uint32_t bar_kv_full = bar0 + 16;                 // [kPreStages]
    const uint32_t bar_kv_empty = bar0 + 16 + 8 * kPreStages;
    const uint32_t bar_s_full = bar0 + 16 + 16 * kPreStages;
    const uint32_t bar_p_full = bar_s_full + 8;
    const uint32_t bar_o_full = bar_s_full + 16;
    const uint32_t bar_o_free = bar_s_full + 24;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + SM::kBarOff + 128);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int G = Hq / Hkv;
    const int n_items = hdr->n_prefill;

    if (threadIdx.x == 0) {
        mbar_init(bar_q_full, 1);
        mbar_init(bar_q_empty, 1);
        for (int s = 0; s < kPreStages; ++s) {
            mbar_init(bar_kv_full + 8 * s, 1);
            mbar_init(bar_kv_empty + 8 * s, 1);
        }
        mbar_init(bar_s_full, 1);
        mbar_init(bar_p_full, 128);
        mbar_init(bar_o_full, 1);
        mbar_init(bar_o_free, 128);
        fence_barrier_init();
        prefetch_tmap(&tmap_q);
        prefetch_tmap(&tmap_k);
        prefetch_tmap(&tmap_v);
    }
    if (warp == 1) {
        tmem_alloc(smem_u32(tmem_slot), SM::kTmemCols);
        tmem_relinquish();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;
    const uint32_t tmem_s = tmem_base;               // columns [0,128)
    const uint32_t tmem_o = tmem_base + 128;         // columns [128,128+D)

    if (warp == 0) {
        // ===================== TMA producer =====================
        int stage = 0;
        uint32_t kv_phase = 0, q_phase = 0;
        constexpr int kBoxes = 8 * 2 * kHalves;
        for (int it = blockIdx.x; it < n_items; it += gridDim.x) {
            const ss_work_item w = items[it];
            const int32_t* bt = block_table + (int64_t)w.req * max_pages;
            const int g = w.head / G;
            mbar_wait(bar_q_empty, q_phase ^ 1);
            if (lane == 0) {
                mbar_arrive_expect_tx(bar_q_full, (uint32_t)SM::kQBytes);
#pragma unroll
                for (int hh = 0; hh < kHalves; ++hh)
                    tma_load_2d(sbase + SM::kQOff + hh * (kTileRows * 128), &tmap_q, w.head * D + hh * 64, w.row0, bar_q_full);
            }
            q_phase ^= 1;
            for (int key0 = 0; key0 < w.kv_end; key0 += kTileKeys) {
                const int npages = min(8, (w.kv_end - key0 + kPage - 1) / kPage);
                mbar_wait(bar_kv_empty + 8 * stage, kv_phase ^ 1);
                if (lane == 0) mbar_arrive_expect_tx(bar_kv_full + 8 * stage, (uint32_t)npages * 2 * kHalves * 2048);
                __syncwarp();
                if (lane < kBoxes) {
                    const int p = lane / (2 * kHalves);
                    const int which = lane % (2 * kHalves);
                    const int is_v = which / kHalves, half = which % kHalves;
                    if (p < npages) {
                        const int page = __ldg(bt + (key0 >> 4) + p);
                        const uint32_t dst = sbase + SM::kKVOff + stage * SM::kStageBytes + is_v * SM::kKBytes +
                                             half * (kTileKeys * 128) + p * (kPage * 128);
                        tma_load_2d(dst, is_v ? &tmap_v : &tmap_k, half * 64, (page * Hkv + g) * kPage, bar_kv_full + 8 * stage);
                    }
                }
                if (++stage == kPreStages) { stage = 0; kv_phase ^= 1; }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer =====================
        constexpr uint32_t idesc_qk = umma_idesc(kTileRows, kTileKeys, 0);
        constexpr uint32_t idesc_pv = umma_idesc(kTileRows, D, 1);
        int stage = 0;
        uint32_t kv_phase = 0, q_phase = 0, p_phase = 0, ofree_phase = 0;
        for (int it = blockIdx.x; it < n_items; it += gridDim.x) {
            const ss_work_item w = items[it];
            const int ntiles = (w.kv_end + kTileKeys - 1) / kTileKeys;
            mbar_wait(bar_q_full, q_phase);
            q_phase ^= 1;
            mbar_wait(bar_o_free, ofree_phase ^ 1);          // previous item's epilogue has drained O
            ofree_phase ^= 1;
            for (int t = 0; t < ntiles; ++t) {
                mbar_wait(bar_kv_full + 8 * stage, kv_phase);
                tc_fence_after();
                const uint32_t kaddr = sbase + SM::kKVOff + stage * SM::kStageBytes;
                const uint32_t vaddr = kaddr + SM::kKBytes;
                if (lane == 0) {
#pragma unroll
                    for (int ks = 0; ks < D / 16; ++ks) {
                        const uint32_t off = (ks >> 2) * (kTileRows * 128) + (ks & 3) * 32;
                        umma_ss(tmem_s, umma_desc(sbase + SM::kQOff + off, 16, 1024), umma_desc(kaddr + off, 16, 1024),
                                idesc_qk, ks > 0);
                    }
                    umma_commit(bar_s_full);
                    if (t == ntiles - 1) umma_commit(bar_q_empty);
                }
                __syncwarp();
                mbar_wait(bar_p_full, p_phase);
                p_phase ^= 1;
                tc_fence_after();
                if (lane == 0) {
#pragma unroll
                    for (int kk = 0; kk < kTileKeys / 16; ++kk) {
                        const uint32_t poff = (kk >> 2) * (kTileRows * 128) + (kk & 3) * 32;
                        umma_ss(tmem_o, umma_desc(sbase + SM::kPOff + poff, 16, 1024),
                                umma_desc(vaddr + kk * 2048, kTileKeys * 128, 1024), idesc_pv, (t > 0 || kk > 0));
                    }
                    umma_commit(bar_kv_empty + 8 * stage);
                    if (t == ntiles - 1) umma_commit(bar_o_full);
                }
                __syncwarp();
                if (++stage == kPreStages) { stage = 0; kv_phase ^= 1; }
            }
        }
    } else {
        // ===================== softmax / correction / epilogue: thread = query row =====================
        const int quarter = warp & 3;                         // TMEM lane quarter this warp may access
        const int row = quarter * 32 + lane;                  // row inside the tile
        const uint32_t lane_addr = (uint32_t)(quarter * 32) << 16;
        const float sl2 = scale * kPLog2e;
        int stage = 0;
        uint32_t kv_phase = 0, s_phase = 0, o_phase = 0;
        for (int it = blockIdx.x; it < n_items; it += gridDim.x) {
            const ss_work_item w = items[it];
            const int ntiles = (w.kv_end + kTileKeys - 1) / kTileKeys;
            const int u = __ldg(ctx_lens + w.req);
            const int limit = u + w.q_pos0 + row + 1;           // keys [0, limit) visible to this row
            float m = -INFINITY, l = 0.f;
            for (int t = 0; t < ntiles; ++t) {
                const int key0 = t * kTileKeys;
                const bool last_partial = key0 + kTileKeys > w.kv_end;
                if (last_partial) {
                    // zero V rows [kv_end - key0, 128): stale / unused-slot bits must not meet P = 0 in the MMA
                    mbar_wait(bar_kv_full + 8 * stage, kv_phase);
                    const uint32_t vaddr = sbase + SM::kKVOff + stage * SM::kStageBytes + SM::kKBytes;
                    const int first = w.kv_end - key0;
                    const int tix = threadIdx.x - 64;
                    for (int i = tix; i < (kTileKeys - first) * kHalves * 8; i += 128) {
                        const int r = first + i / (kHalves * 8);
                        const int c = i % (kHalves * 8);
                        const uint32_t a = vaddr + (c >> 3) * (kTileKeys * 128) + r * 128 + (c & 7) * 16;
                        asm volatile("st.shared.v4.b32 [%0], {%1,%1,%1,%1};" ::"r"(a), "r"(0u) : "memory");
                    }
                }
                mbar_wait(bar_s_full, s_phase);
                s_phase ^= 1;
                tc_fence_after();
                // ---- load S row (128 fp32) ----
                uint32_t sr[4][32];
#pragma unroll
                for (int c = 0; c < 4; ++c) tmem_ld_32x32b_x32(tmem_s + lane_addr + c * 32, sr[c]);
                tmem_ld_wait();
                const int nvis = limit - key0;                  // columns [0, nvis) visible (may be <= 0 or >= 128)
                float bm = -INFINITY;
                if (nvis >= kTileKeys) {
#pragma unroll
                    for (int c = 0; c < 4; ++c)
#pragma unroll
                        for (int i = 0; i < 32; ++i) bm = fmaxf(bm, __uint_as_float(sr[c][i]));
                } else {
#pragma unroll
                    for (int c = 0; c < 4; ++c)
#pragma unroll
                        for (int i = 0; i < 32; ++i) {
                            if (c * 32 + i >= nvis) sr[c][i] = 0xff800000u;      // -inf by select, never by arithmetic
                            bm = fmaxf(bm, __uint_as_float(sr[c][i]));
                        }
                }
                const float m_new = fmaxf(m, bm * sl2);          // tile 0 has key 0 visible for every row => finite
                const float alpha = exp2f(m - m_new);
                float psum = 0.f;
                // ---- P = exp2(s*sl2 - m_new) -> bf16 -> swizzled smem (K-major, 2 halves of 64 keys) ----
                const uint32_t prow = sbase + SM::kPOff + row * 128;
#pragma unroll
                for (int c = 0; c < 4; ++c) {
#pragma unroll
                    for (int v = 0; v < 4; ++v) {                 // 8 keys = one 16-byte chunk
                        float p[8];
#pragma unroll
                        for (int e = 0; e < 8; ++e) {
                            p[e] = exp2f(__uint_as_float(sr[c][v * 8 + e]) * sl2 - m_new);
                            psum += p[e];
                        }
                        const int chunk = (c & 1) * 4 + v;        // chunk within the 64-key half
                        const uint32_t a = prow + (c >> 1) * (kTileRows * 128) + ((chunk ^ (row & 7)) << 4);
                        asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(a), "r"(pack_bf16(p[0], p[1])),
                                     "r"(pack_bf16(p[2], p[3])), "r"(pack_bf16(p[4], p[5])), "r"(pack_bf16(p[6], p[7]))
                                     : "memory");
                    }
                }
                l = l * alpha + psum;
                m = m_new;
                // ---- rescale O in TMEM when some row of this warp moved its max (never needed on tile 0) ----
                if (t > 0 && !__all_sync(0xffffffffu, alpha == 1.f)) {
#pragma unroll
                    for (int c = 0; c < D / 32; ++c) {
                        uint32_t orr[32];
                        tmem_ld_32x32b_x32(tmem_o + lane_addr + c * 32, orr);
                        tmem_ld_wait();
#pragma unroll
                        for (int i = 0; i < 32; ++i) orr[i] = __float_as_uint(__uint_as_float(orr[i]) * alpha);
                        tmem_st_32x32b_x32(tmem_o + lane_addr + c * 32, orr);
                    }
                    tmem_st_wait();
                }
                tc_fence_before();
                fence_proxy_async();                              // P (and zeroed V rows) visible to the MMA's async proxy
                mbar_arrive(bar_p_full);
                if (++stage == kPreStages) { stage = 0; kv_phase ^= 1; }
            }
            // ---- epilogue ----
            mbar_wait(bar_o_full, o_phase);
            o_phase ^= 1;
            tc_fence_after();
            const float inv = 1.f / l;
            const bool store = row < w.nrows;
            __nv_bfloat16* orow = out + ((int64_t)(w.row0 + row) * Hq + w.head) * D;
#pragma unroll
            for (int c = 0; c < D / 32; ++c) {
                uint32_t orr[32];
                tmem_ld_32x32b_x32(tmem_o + lane_addr + c * 32, orr);
                tmem_ld_wait();
                if (store) {
#pragma unroll
                    for (int v = 0; v < 4; ++v) {
                        uint4 pk;
                        pk.x = pack_bf16(__uint_as_float(orr[v * 8 + 0]) * inv, __uint_as_float(orr[v * 8 + 1]) * inv);
                        pk.y = pack_bf16(__uint_as_float(orr[v * 8 + 2]) * inv, __uint_as_float(orr[v * 8 + 3]) * inv);
                        pk.z = pack_bf16(__uint_as_float(orr[v * 8 + 4]) * inv, __uint_as_float(orr[v * 8 + 5]) * inv);
                        pk.w = pack_bf16(__uint_as_float(orr[v * 8 + 6]) * inv, __uint_as_float(orr[v * 8 + 7]) * inv);
                        *reinterpret_cast<uint4*>(orow + c * 32 + v * 8) = pk;
                    }
                }
            }
            if (store && lse) lse[(int64_t)(w.row0 + row) * Hq + w.head] = (m + log2f(l)) * kPLn2;
            tc_fence_before();
            mbar_arrive(bar_o_free);
        }
    }

    // ---- teardown ----
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc(tmem_base, SM::kTmemCols);
}

// Encode the per-call Q tensor map: q viewed as [T rows][Hq*D] bf16, box = 128 rows x 64 columns.
static bool encode_q_map(CUtensorMap* map, const void* q, int T, int Hq, int D) {
    typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                      const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                      CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) != cudaSuccess ||
            qres != cudaDriverEntryPointSuccess)
            return false;
        fn = (EncodeTiledFn)p;
    }
    cuuint64_t gdim[2] = {(cuuint64_t)Hq * D, (cuuint64_t)T};
    cuuint64_t gstride[1] = {(cuuint64_t)Hq * D * 2};
    cuuint32_t box[2] = {64u, (cuuint32_t)kTileRows};
    cuuint32_t estr[2] = {1u, 1u};
    return fn(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(q), gdim, gstride, box, estr,
              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

cudaError_t launch_prefill(const Handle* h, const void* q, const int32_t* bt, const int32_t* ctx, int T, float scale,
                           void* workspace, void* out, float* lse, cudaStream_t stream) {
    const ss_config& c = h->cfg;
    char* ws = (char*)workspace;
    const WorkHeader* hdr = (const WorkHeader*)(ws + h->ws.header_off);
    const ss_work_item* items = (const ss_work_item*)(ws + h->ws.items_off);
    CUtensorMap tmap_q;
    if (!encode_q_map(&tmap_q, q, T, c.num_q_heads, c.head_dim)) return cudaErrorInvalidValue;
    cudaError_t e;
    if (c.head_dim == 128) {
        auto kern = prefill_kernel<128>;
        constexpr int smem = PrefillSmem<128>::kTotal;
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        kern<<<h->num_sms, kPreThreads, smem, stream>>>(tmap_q, h->tmap_k, h->tmap_v, bt, ctx, hdr, items,
                                                        c.max_pages_per_req, c.num_q_heads, c.num_kv_heads, scale,
                                                        (__nv_bfloat16*)out, lse);
    } else {
        auto kern = prefill_kernel<64>;
        constexpr int smem = PrefillSmem<64>::kTotal;
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        kern<<<h->num_sms, kPreThreads, smem, stream>>>(tmap_q, h->tmap_k, h->tmap_v, bt, ctx, hdr, items,
                                                        c.max_pages_per_req, c.num_q_heads, c.num_kv_heads, scale,
                                                        (__nv_bfloat16*)out, lse);
    }
    return cudaGetLastError();
}

}  // namespace ss
