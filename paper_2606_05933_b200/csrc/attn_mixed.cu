// Main kernel of the path: ONE launch serves any mix of prefill-chunk tiles (a3) and decode splits (a4) and
// merges split partials (a5) — SURVEY.md §8(a), north_star (b)(c)(d).
//
// Persistent CTAs (one per SM) pull items from the device work list through a dynamic queue (atomic
// counter), so tensor-bound prefill tiles and HBM-bound decode splits overlap across SMs and the batch
// costs ~max(bytes/HBM, flops/tensor) instead of the sum.  12 warps per CTA in 3 warpgroups (bf16 cache); the register
// file is re-partitioned with setmaxnreg (WG0 88 registers per thread, WG1 / WG2 208):
//   WG0 warp 0  scheduler + Q / K producer (one elected thread).  Publishes each item to the other warps through a
//               4-slot smem ring, loads the Q tiles (prefill: the item's 1 or 2 query heads, 128 rows each) and
//               streams 64-key K tiles into a 5-slot K ring: ONE 4-D TMA box per (page, kv head) slab (16 keys x D,
//               SWIZZLE_128B, written as [8-key group][64-column half][8 rows][128 B]).
//   WG0 warp 3  V producer (one elected thread): follows the item ring and streams the V tiles the same way into the
//               V ring (a K slot is free as soon as its S MMAs are done, a V slot as soon as its PV MMAs are done).
//               Two producer threads because one could not issue a 32 KB tile in less than ~600 ns.
//   WG0 warps 1,2  tcgen05.mma issuers (warp 1 also owns the TMEM allocation), one elected thread each: warp 1 issues
//               chain A's MMAs, warp 2 chain B's (prefill items only).  Per query head X (a
//               "chain") TMEM holds S_X[0], S_X[1] (128 rows x 64 keys fp32, 64 columns each) and O_X (128 x D
//               fp32): 2 x 256 = all 512 columns.  P (bf16 pairs) is written IN PLACE over its S buffer, so per
//               chain the order is  S(k) -> softmax -> P(k) -> PV(k) -> S(k+2)  with S(k+1) already done: each
//               chain's softmax never waits for the tensor pipe, and the two chains interleave on it
//               (PV_A(k) S_A(k+2) PV_B(k) S_B(k+2) ...) while sharing every staged K/V tile.
//               Decode items: warp 2 runs a5 - publishes each split (acq_rel ticket) and, when it draws the last
//               ticket of a (request, kv head), merges all splits in fixed order (bitwise reproducible).
//   WG1, WG2    workers (4 warps each; warp % 4 = TMEM lane quarter).
//               prefill item: WG1 = chain A (head), WG2 = chain B (head + 1); thread = query row (TMEM lane):
//                 tcgen05.ld S, causal/length mask by select (only in the warp-uniform diagonal variant), online
//                 softmax (exp2, log2e folded into the scale, packed f32x2 arithmetic, lazy rescale: O is only touched
//                 when a row max grows by more than 2^8), P -> bf16 -> TMEM, epilogue stores rows < nrows only.
//               decode item: all 8 worker warps; a warp owns 16 keys of every other 64-key slot (WG1 the even slots
//                 of the item, WG2 the odd ones): mma.sync.m16n8k16 with the G query heads of the KV head padded to 16
//                 rows (bandwidth-bound, wasted rows are free), online softmax in registers with quad shuffles,
//                 cross-warp log-sum-exp merge through smem (G <= 8: one 8 -> 1 pass by all 256 threads; G > 8: WG2 ->
//                 WG1 in registers, then 4 -> 1), then either the final bf16 row or an fp32 partial.
//   FP8 cache (template FP8, SS_FLAG_KV_FP8): E4M3 codes through the same TMA boxes on 128-byte rows (6-slot rings).
//               Decode: codes widened exactly to fp16 after ldmatrix, f16 mma.sync; a warpgroup visits its own slots only.
//               Prefill: a FOURTH warpgroup (16 warps; registers 88 / 192 / 192 / 40) widens each staged tile into fp16
//               tiles in the bf16 slot layout for the tcgen05 MMAs (kind::f16 on fp16 operands) of both chains; each
//               chain's workers rewrite their Q tile as fp16 in place.
// Rooflines: decode items HBM (2*D*2 bytes per cached token per kv head), prefill items bf16 tensor
// (4*D flop per visible (row,key) pair per head).  V rows at/after kv_end are zeroed in smem before any
// PV product (unused slots may hold NaN; 0*NaN = NaN); masked scores are replaced, never multiplied.
#include "common.cuh"
#include "plan.cuh"
#include "ptx.cuh"

// -DSS_PROFILE (measurement builds only, see profiles/): clock64 phase counters, written into the ss_debug_set_trace
// buffer - prefill items: words 5..8 = chain A's cycles in {S wait, tcgen05.ld, softmax, st + fence + arrive}, and the
// last 4 words of the CTA block = the MMA thread's cycles in {P wait, K/V wait, issue} and its half tiles; decode items:
// words 7, 8 = decode warp 0's cycles in {K wait << 32 | S^T, V wait << 32 | softmax + O^T} summed over the item's tiles.
#ifdef SS_PROFILE
#define SS_PF(i) { const long long c_ = clock64(); pf_acc[i] += c_ - pf_t; pf_t = c_; }
#define SS_MM(i) { const long long c_ = clock64(); mm_acc[i] += c_ - mm_t; mm_t = c_; }
#else
#define SS_PF(i)
#define SS_MM(i)
#endif

namespace ss {

using namespace ptx;

constexpr int kSlotKeys = 64;        // keys per K / V ring slot = keys per S buffer
constexpr int kMaxSt = 8;            // most K / V ring slots of any instantiation (barrier index layout)
constexpr int kBarBytes = 704;       // mbarrier block (8 bytes each)
constexpr int kSchedSlots = 4;
constexpr int kDecKeys = 16;         // keys of a 64-key slot one decode warp owns (4 warps per slot)
// setmaxnreg moves registers inside the CTA's own launch allocation.  bf16 cache: 384 threads x 168 (the __launch_bounds__
// cap ptxas reports) = 64512, so 128*88 + 256*208 = 64512 fits exactly; one register more per worker and the .inc spins
// forever.  (88: the K producer thread keeps the next item, three tiles of page ids and its slot history without spilling.)
// FP8 cache: a fourth warpgroup (the fp8 -> fp16 tile converters of the prefill path) - 512 threads x 128 = 65536 =
// 128*88 + 256*192 + 128*40.
template <bool FP8>
struct MixCta {
    static constexpr int kThreads = FP8 ? 512 : 384;
    static constexpr int kRegsLaunch = FP8 ? 128 : 168, kRegsWg0 = 88, kRegsWorker = FP8 ? 192 : 208, kRegsConv = 40;
    static_assert(128 * kRegsWg0 + 256 * kRegsWorker + (FP8 ? 128 * kRegsConv : 0) <= kThreads * kRegsLaunch,
                  "setmaxnreg.inc could never be granted");
};
constexpr float kMLog2e = 1.4426950408889634f;
constexpr float kMLn2 = 0.6931471805599453f;
constexpr float kRescaleThreshold = 8.f;   // log2 units: P <= 2^8, safe in bf16 / fp32

// FP8: the KV cache holds one byte per element (E4M3 codes): a key row is D bytes = D/128 128-byte chunks.
template <int D, bool FP8 = false>
struct MixSmem {
    static constexpr int kHalves = D / 64;                       // 128-byte chunks of a bf16 row (Q tiles, bf16 K / V rows)
    static constexpr int kKvHalves = FP8 ? D / 128 : D / 64;     // 128-byte chunks of a K / V row in the ring
    static constexpr int kSlot = kKvHalves * kSlotKeys * 128;    // one K (or V) ring slot: 64 keys
    // Ring depth.  bf16: 5 slots of 16 KB per tensor (4: -1.5 % on pure decode, 6 would not leave room for 2 Q tiles);
    // a slot then alternates between the two decode warpgroups, so every decode warp takes part in every slot phase.
    // FP8: 6 slots of 8 KB; with an EVEN ring a slot always belongs to the same decode warpgroup (tile parity = slot
    // parity), so a warp only touches its own slots - no pass-through waits (kOwnSlots).  The space saved holds the
    // fp16 copies of the K / V tiles the tensor-core prefill path works on (kConv*, see the converter warps).
    static constexpr int kNumSt = FP8 ? 6 : 5;
    static constexpr bool kOwnSlots = kNumSt % 2 == 0;
    static_assert(kNumSt <= kMaxSt, "barrier index layout");
    // Slot layout = what ONE 4-D TMA box per (page, kv head) slab writes: [8-key group][64-column half][8 rows][128 B],
    // every [8 rows][128 B] block a SWIZZLE_128B core group.  8-key groups are kGroup bytes apart (uniform over the 4
    // pages of a slot: the UMMA stride-byte-offset), the halves of a group 1024 bytes apart.
    static constexpr int kGroup = kKvHalves * 1024;
    static constexpr int kPageBytes = 2 * kGroup;                // one (page, kv head) slab: 16 keys
    // byte offset of the 16-byte chunk cd (0 .. 8 kKvHalves - 1) of key row r (0 .. 63) inside a slot, swizzle applied
    __device__ static __forceinline__ uint32_t kv_off(int r, int cd) {
        return (uint32_t)((r >> 3) * kGroup + (cd >> 3) * 1024 + (r & 7) * 128 + (((cd & 7) ^ (r & 7)) << 4));
    }
    static constexpr int kQTile = kHalves * kTileRows * 128;     // one Q tile (one query head, 128 rows)
    static constexpr int kKOff = 0;
    static constexpr int kVOff = kKOff + kNumSt * kSlot;
    static constexpr int kQOff = kVOff + kNumSt * kSlot;         // 2 Q tiles (prefill) / decode: cross-warp merge buffer + staged Q rows
    static constexpr int kQBytes = 2 * kQTile;
    static constexpr int kMergeBytes = 4 * kMaxGroup * (D + 2) * 4;
    // decode with G <= 8: merge buffer of 8 rows per warp (8 warps), then kSchedSlots staged Q blocks (G rows x D bf16, one per
    // scheduler slot, bulk-copied by the producer so the workers never wait on a cold global Q load)
    static constexpr int kMerge8Bytes = 8 * 8 * (D + 2) * 4;     // G <= 8: one partial per decode warp, merged 8 -> 1 in one pass
    static constexpr int kQStageOff = kQOff + (kMerge8Bytes + 127) / 128 * 128;
    static constexpr int kQStageBytes = 8 * D * 2;
    static_assert(kMergeBytes <= kQBytes, "decode merge buffer must fit the Q region");
    static_assert(kQStageOff + kSchedSlots * kQStageBytes <= kQOff + kQBytes, "staged Q blocks must fit beside the merge buffer");
    // FP8 prefill: two fp16 K tiles and two fp16 V tiles (64 keys x D) in the bf16 slot layout (8-key groups kConvGroup apart)
    static constexpr int kConvTile = FP8 ? kHalves * kSlotKeys * 128 : 0;
    static constexpr int kConvGroup = kHalves * 1024;
    static constexpr int kKConvOff = kQOff + kQBytes;
    static constexpr int kVConvOff = kKConvOff + 2 * kConvTile;
    __device__ static __forceinline__ uint32_t conv_off(int r, int cd) {      // 16-byte chunk cd (0 .. D/8-1) of key row r
        return (uint32_t)((r >> 3) * kConvGroup + (cd >> 3) * 1024 + (r & 7) * 128 + (((cd & 7) ^ (r & 7)) << 4));
    }
    static constexpr int kBarOff = kVConvOff + 2 * kConvTile;
    static constexpr int kSchedOff = kBarOff + kBarBytes;        // kSchedSlots x 48 B
    static constexpr int kTmemSlotOff = kSchedOff + kSchedSlots * 48;
    // in-kernel plan (plan.cuh): header + rank tables for up to kPlanMaxR requests, alive for the whole kernel
    static constexpr int kPlanOff = kTmemSlotOff + 32;
    static constexpr int kPlanBytes = 64 + 4 * kPlanMaxR;
    static constexpr int kTotal = kPlanOff + kPlanBytes;       // no alignment slack: the dynamic window is declared 1024-aligned
    // TMEM columns per chain X (base 256 X): S[0] [0,64) S[1] [64,128) O [128,128+D); P[b] = first 32 columns of S[b]
    static constexpr int kTmemCols = 512;
    static constexpr int kTmemChain = 256, kTmemO = 128;
    static_assert(kTotal <= 232448, "shared memory budget");
};

// barrier indices (8 bytes each, from kBarOff)
enum : int {
    B_KFULL = 0, B_VFULL = kMaxSt, B_KEMPTY_P = 2 * kMaxSt, B_KEMPTY_D = 3 * kMaxSt, B_VEMPTY_P = 4 * kMaxSt,
    B_VEMPTY_D = 5 * kMaxSt,
    B_SFULL = 6 * kMaxSt, B_PFULL = B_SFULL + 4,      // [chain * 2 + buffer]
    B_QFULL = B_PFULL + 4, B_QEMPTY = B_QFULL + 1, B_OFULL = B_QEMPTY + 1, B_OFREE = B_OFULL + 2, B_PVDONE = B_OFREE + 2,     // [chain]
    B_SCHED_FULL = B_PVDONE + 2, B_SCHED_EMPTY = B_SCHED_FULL + 4, B_PARTIAL = B_SCHED_EMPTY + 4,
    // FP8 prefill: fp16 copies of the staged tiles [buffer], and the Q tile converted in place
    B_KCONV_FULL = B_PARTIAL + 4, B_KCONV_EMPTY = B_KCONV_FULL + 2, B_VCONV_FULL = B_KCONV_EMPTY + 2,
    B_VCONV_EMPTY = B_VCONV_FULL + 2, B_QCONV = B_VCONV_EMPTY + 2 /* [chain] */, B_COUNT = B_QCONV + 2
};
static_assert(B_COUNT * 8 <= kBarBytes, "barrier region");
static_assert(kSchedSlots == 4, "barrier indices assume 4 scheduler slots");

__device__ __forceinline__ uint64_t umma_desc_sw128(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
    uint64_t d = 0;
    d |= (uint64_t)((saddr & 0x3FFFFu) >> 4);
    d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFFu) << 16;
    d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFFu) << 32;
    d |= (uint64_t)1 << 46;                 // descriptor version (Blackwell)
    d |= (uint64_t)2 << 61;                 // layout type: SWIZZLE_128B
    return d;
}
// kind::f16 with fp16 A and B operands (FP8 cache: the staged tiles are widened to fp16), fp32 accumulate
__host__ __device__ constexpr uint32_t umma_idesc_f16(int M, int N, int b_mn_major) {
    return (1u << 4) | ((uint32_t)b_mn_major << 16) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}
__host__ __device__ constexpr uint32_t umma_idesc_bf16(int M, int N, int b_mn_major) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)b_mn_major << 16) | ((uint32_t)(N >> 3) << 17) |
           ((uint32_t)(M >> 4) << 24);
}

struct MixParams {
    const int32_t* block_table;
    const int32_t* ctx_lens;
    WorkHeader* hdr;
    const ss_work_item* items;
    int32_t* merge_counters;
    float* partials;
    const __nv_bfloat16* q;
    __nv_bfloat16* out;
    float* lse;
    int max_pages, Hq, Hkv;
    float scale;
    // a2 inside this kernel (self_plan) or items read from the work-list kernel's output
    const int32_t* qsl;
    int32_t* queue;                // [0] next prefill ticket, [1] next decode ticket, [2] CTAs done (self_plan only)
    int self_plan, R, num_sms, force_split_keys, force_decode_ctas, max_partials;
    unsigned long long* trace;     // ss_debug_set_trace: per-CTA timeline, or null
    int trace_words;
    const float* k_scale;          // SS_FLAG_KV_FP8: per kv head scales (device), else null
    const float* v_scale;
    const int32_t* err_flag;       // SS_FLAG_DEBUG_CHECKS: nonzero = the metadata check tripped, serve no item; else null
};

// exp2 on the FMA / ALU pipes for two values at once (the MUFU pipe does 16 ex2 per clock and SM: at 128 x 64 scores per
// chain and half tile it alone would take as long as the two MMAs): round-to-nearest split x = n + f, |f| <= 0.5, by
// the 1.5 * 2^23 magic add; cubic minimax polynomial for 2^f (max relative error 7.6e-5, P is rounded to bf16 = 3.9e-3
// anyway); 2^n by adding n to the exponent field.  x is clamped at -126 so the result never leaves the normal range.
__device__ __forceinline__ float2 exp2_poly2(float2 x) {
    const float kMagic = 12582912.f;                   // 1.5 * 2^23: the integer part lands in the low mantissa bits
    x.x = fmaxf(x.x, -126.f);
    x.y = fmaxf(x.y, -126.f);
    const float2 t = __fadd2_rn(x, make_float2(kMagic, kMagic));
    const float2 f = __fadd2_rn(x, __ffma2_rn(t, make_float2(-1.f, -1.f), make_float2(kMagic, kMagic)));   // x - round(x)
    float2 q = __ffma2_rn(f, make_float2(0.055170879f, 0.055170879f), make_float2(0.24260919f, 0.24260919f));
    q = __ffma2_rn(q, f, make_float2(0.69326097f, 0.69326097f));
    q = __ffma2_rn(q, f, make_float2(0.99992818f, 0.99992818f));
    return make_float2(__uint_as_float(__float_as_uint(q.x) + (__float_as_uint(t.x) << 23)),
                       __uint_as_float(__float_as_uint(q.y) + (__float_as_uint(t.y) << 23)));
}
#ifndef SS_POLY_EVERY
#define SS_POLY_EVERY 3
#endif
constexpr int kPolyEvery = SS_POLY_EVERY;      // every kPolyEvery-th pair of scores takes exp2_poly2 instead of MUFU.EX2 (0 = none)

// One 64-key half tile of one query row: S (64 fp32 scores in sr) -> P (bf16 pairs in pk), online-softmax state (m, l).
// MASKED: keys at and after nvis are invisible (causal diagonal / end of the KV range); replaced by select.
// Returns alpha (the factor the accumulated O row must be scaled by; 1 unless the reference max moved).
template <bool MASKED, bool F16 = false>
__device__ __forceinline__ float softmax_half(uint32_t (&sr)[2][32], int nvis, float sl2, float& m, float& l, uint32_t (&pk)[32]) {
    float bm[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
#pragma unroll
    for (int c = 0; c < 2; ++c)
#pragma unroll
        for (int i = 0; i < 32; i += 2) {
            if (MASKED && c * 32 + i >= nvis) sr[c][i] = 0xff800000u;   // -inf by select, never by arithmetic
            if (MASKED && c * 32 + i + 1 >= nvis) sr[c][i + 1] = 0xff800000u;
            bm[(i >> 1) & 3] = fmax3(bm[(i >> 1) & 3], __uint_as_float(sr[c][i]), __uint_as_float(sr[c][i + 1]));   // FMNMX3
        }
    const float cand = fmaxf(fmaxf(bm[0], bm[1]), fmaxf(bm[2], bm[3])) * sl2;
    // lazy rescale: only move the reference max when it grows by more than 2^8
    float m_new = m, alpha = 1.f;
    if (cand > m + kRescaleThreshold) { m_new = cand; alpha = exp2f(m - m_new); }   // first tile: m = -inf -> alpha = 0
    const float2 sl2v = make_float2(sl2, sl2), nm = make_float2(-m_new, -m_new);
    float2 ps[4] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
    // P = exp2(s*sl2 - m_new) -> bf16 pairs (A operand of the PV MMA), 32 packed columns per row
#pragma unroll
    for (int i = 0; i < 32; ++i) {
        const float2 x = __ffma2_rn(make_float2(__uint_as_float(sr[i >> 4][(2 * i) & 31]), __uint_as_float(sr[i >> 4][((2 * i) & 31) + 1])), sl2v, nm);
        const float2 p = (kPolyEvery > 0 && i % (kPolyEvery > 0 ? kPolyEvery : 1) == 0) ? exp2_poly2(x) : make_float2(exp2f(x.x), exp2f(x.y));
        ps[i & 3] = __fadd2_rn(ps[i & 3], p);
        pk[i] = F16 ? pack_f16(p.x, p.y) : pack_bf16(p.x, p.y);      // FP8 cache: V is widened to fp16, so is P
    }
    const float2 s01 = __fadd2_rn(__fadd2_rn(ps[0], ps[1]), __fadd2_rn(ps[2], ps[3]));
    l = l * alpha + (s01.x + s01.y);
    m = m_new;
    return alpha;
}

// bf16 pair -> fp16 pair (FP8 cache: the products run as f16 MMAs, every E4M3 value being an fp16 value).  Exact for
// magnitudes in [2^-14, 65504]; clamped above (documented in slidingattn.h), rounded to the fp16 subnormal grid below.
__device__ __forceinline__ uint32_t bf16x2_to_f16x2(uint32_t w) {
    const float lo = fminf(fmaxf(__uint_as_float(w << 16), -65504.f), 65504.f);
    const float hi = fminf(fmaxf(__uint_as_float(w & 0xffff0000u), -65504.f), 65504.f);
    return pack_f16(lo, hi);
}

// One decode split on the 8 worker warps (see the call site).  NT = 8-head column tiles (1: G <= 8, 2: G <= 16).
// FP8 (E4M3 cache, reading 23): the same structure on 128-byte key rows.  ldmatrix moves the codes as 16-bit
// units, so a thread ends up with 4 consecutive d of one key (K) or a 2 x 2 block of (key, d) (V, transposed load):
//   S^T: the contraction index is permuted inside each 16-d step - MMA k = {2c, 2c+1, 2c+8, 2c+9} <-> d = 16 ks + {4c,
//        4c+1, 4c+2, 4c+3} - identically for the K fragment and the Q^T fragment (a sum does not care);
//   O^T: one byte permute per register separates the two d of a block; MMA row i < 8 <-> d = 16 mt + 2i, row i + 8 <->
//        d = 16 mt + 2i + 1, undone when the accumulators are written out.
// Codes widen exactly to fp16 (cvt.rn.f16x2.e4m3x2), P is rounded to fp16, k_scale folds into the score scale and
// v_scale into the output.
template <int D, int NT, bool FP8>
__device__ __forceinline__ void decode_item(const ss_work_item& w, const int n, const int slot, const uint32_t tile_ctr,
                                            const int wg, const int cw, const int lane, const int wtid, const uint32_t sbase,
                                            const uint32_t bar0, const MixParams& prm, float* merge, unsigned long long* tr) {
    using SM = MixSmem<D, FP8>;
    constexpr int kHalves = SM::kKvHalves;
    auto BAR = [&](int i) -> uint32_t { return bar0 + 8u * (uint32_t)i; };
    const int Hq = prm.Hq, Hkv = prm.Hkv, G = Hq / Hkv;
    const float sl2 = prm.scale * kMLog2e * (FP8 ? __ldg(prm.k_scale + w.head) : 1.f);
    const float vs = FP8 ? __ldg(prm.v_scale + w.head) : 1.f;
    const int qr = lane >> 2, qc = (lane & 3) * 2;           // fragment coordinates: row / column pair
    constexpr int mrows = NT * 8;                           // merge-buffer rows (heads) per warp
    // B fragments of Q^T (16 d x 8 heads per k-step): head = 8 nt + qr; bf16: d = 16 ks + qc (+1) and + 8;
    // FP8: d = 16 ks + 2 qc (+1) and + 2 (+3), as fp16 pairs
    uint32_t qb[D / 16][2 * NT];
    if (NT == 1) {
        const uint32_t qs = sbase + SM::kQStageOff + slot * SM::kQStageBytes + (qr * D + (FP8 ? 2 : 1) * qc) * 2;
#pragma unroll
        for (int ks = 0; ks < D / 16; ++ks) {
            const uint32_t w0 = qr < G ? lds32(qs + ks * 32) : 0u, w1 = qr < G ? lds32(qs + ks * 32 + (FP8 ? 4 : 16)) : 0u;
            qb[ks][0] = FP8 ? bf16x2_to_f16x2(w0) : w0;
            qb[ks][1] = FP8 ? bf16x2_to_f16x2(w1) : w1;
        }
    } else {
        const __nv_bfloat16* qg = prm.q + ((int64_t)w.row0 * Hq + (int64_t)w.head * G) * D;
#pragma unroll
        for (int nt = 0; nt < NT; ++nt)
#pragma unroll
            for (int ks = 0; ks < D / 16; ++ks) {
                const int hd = 8 * nt + qr;
                const __nv_bfloat16* src = qg + (int64_t)hd * D + ks * 16 + (FP8 ? 2 : 1) * qc;
                const uint32_t w0 = hd < G ? *reinterpret_cast<const uint32_t*>(src) : 0u;
                const uint32_t w1 = hd < G ? *reinterpret_cast<const uint32_t*>(src + (FP8 ? 2 : 8)) : 0u;
                qb[ks][2 * nt] = FP8 ? bf16x2_to_f16x2(w0) : w0;
                qb[ks][2 * nt + 1] = FP8 ? bf16x2_to_f16x2(w1) : w1;
            }
    }
    // O^T accumulators: [nt][mt] c0 = (d = 16 mt + qr, head 8 nt + qc), c1 = head + 1, c2 = (d + 8, head), c3 = (d + 8, head + 1)
    // (FP8: c0 / c1 at d = 16 mt + 2 qr, c2 / c3 at d + 1)
    float oT[NT][D / 16][4];
    float m[NT][2], l[NT][2];                               // per head qc, qc + 1 (l: this lane's share of the row sum)
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) {
        m[nt][0] = m[nt][1] = -INFINITY;
        l[nt][0] = l[nt][1] = 0.f;
#pragma unroll
        for (int mt = 0; mt < D / 16; ++mt) oT[nt][mt][0] = oT[nt][mt][1] = oT[nt][mt][2] = oT[nt][mt][3] = 0.f;
    }
    // Odd ring (bf16, 5 slots): EVERY warp waits FULL and arrives EMPTY on EVERY slot - an mbarrier parity wait is only
    // sound while the waiter is less than one phase away from the barrier, and a slot alternates between the warpgroups.
    // Even ring (FP8): every item covers an even number of ring tiles, so item-local tile parity = slot parity and a slot
    // always belongs to the same warpgroup: a warp waits and arrives on its own slots only, and sees every use of them.
    const int r16 = cw * kDecKeys;                          // first key row of this warp inside its slots
    const int mi = lane >> 3, l7 = lane & 7;                // ldmatrix: this lane addresses row l7 of matrix mi
    // The swizzled ldmatrix offsets of this lane are loop invariants, pinned in registers (the empty asm makes them opaque:
    // the compiler otherwise recomputes them per tile - FP8 under the 128-register launch bound of the 16-warp CTA: +9 %
    // instructions in a loop that is issue-bound; bf16: ~90 of the loop's 376 instructions)
    constexpr int kFragLoads = FP8 ? D / 32 : D / 16;           // ldmatrix.x4 per tensor per 16-key slice
    uint32_t koffs[kFragLoads], voffs[kFragLoads];
#pragma unroll
    for (int jj = 0; jj < kFragLoads; ++jj) {
        koffs[jj] = SM::kv_off(r16 + (mi & 1) * 8 + l7, 2 * jj + (mi >> 1));
        voffs[jj] = FP8 ? SM::kv_off(r16 + (mi & 1) * 8 + l7, 2 * jj + (mi >> 1)) : SM::kv_off(r16 + (mi >> 1) * 8 + l7, 2 * jj + (mi & 1));
        asm volatile("" : "+r"(koffs[jj]));
        asm volatile("" : "+r"(voffs[jj]));
    }
#ifdef SS_PROFILE
    long long pf_t = clock64(), pf_acc[4] = {0, 0, 0, 0};     // K wait | S^T | V wait | softmax + O^T  (cycles, this warp)
#endif
    // even ring: only the item's tiles of this warpgroup's parity are visited, slot and phase parity advance by 2 slots
    int s_run = (int)((tile_ctr + (uint32_t)wg) % SM::kNumSt);
    uint32_t par_run = ((tile_ctr + (uint32_t)wg) / SM::kNumSt) & 1;
    for (int t = SM::kOwnSlots ? wg : 0; t < n; t += SM::kOwnSlots ? 2 : 1) {
        const uint32_t tc = tile_ctr + t;
        const int s = SM::kOwnSlots ? s_run : (int)(tc % SM::kNumSt);
        const uint32_t fpar = SM::kOwnSlots ? par_run : (tc / SM::kNumSt) & 1;
        if (SM::kOwnSlots) {
            s_run += 2;
            if (s_run >= SM::kNumSt) { s_run -= SM::kNumSt; par_run ^= 1; }
        }
        const int key0 = w.kv_begin + t * kSlotKeys;
        // <= 0: nothing for this warp in this slot (odd ring: the other warpgroup's turn; it still waits and arrives)
        const int nvalid = (SM::kOwnSlots || (t & 1) == wg) ? w.kv_end - (key0 + r16) : 0;
        const uint32_t kbase = sbase + SM::kKOff + s * SM::kSlot;
        const uint32_t vbase = sbase + SM::kVOff + s * SM::kSlot;
        float sT[NT][4];
        mbar_wait(BAR(B_KFULL + s), fpar);
        if (tr && t == 0) tr[3] = globaltimer_ns();
        SS_PF(0)
        if (nvalid > 0) {
            // S^T (16 keys x 8 heads) = K (16 x D) Q^T: two interleaved accumulation chains per head tile
            float sU[NT][4];
#pragma unroll
            for (int nt = 0; nt < NT; ++nt)
#pragma unroll
                for (int i = 0; i < 4; ++i) sT[nt][i] = sU[nt][i] = 0.f;
            // lane's K row: r16 + (mi & 1) * 8 + l7 - a0: keys 0-7, a1: keys 8-15, a2 / a3: the next 8 d (offsets in koffs)
            // every fragment load is issued before the first MMA (the wrappers are asm volatile and keep their order: an
            // interleaved loop exposed one ldmatrix latency per k-step)
            if (FP8) {
                uint32_t r[D / 32][4];                           // one ldmatrix = 16 keys x 32 d of codes = two k-steps
#pragma unroll
                for (int jj = 0; jj < D / 32; ++jj)
                    ldmatrix_x4(r[jj][0], r[jj][1], r[jj][2], r[jj][3], kbase + koffs[jj]);
#pragma unroll
                for (int jj = 0; jj < D / 32; ++jj)
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const int ks = 2 * jj + h;
                        const uint32_t a[4] = {e4m3x2_to_f16x2(r[jj][2 * h]), e4m3x2_to_f16x2(r[jj][2 * h + 1]),
                                               e4m3x2_hi_to_f16x2(r[jj][2 * h]), e4m3x2_hi_to_f16x2(r[jj][2 * h + 1])};
#pragma unroll
                        for (int nt = 0; nt < NT; ++nt) mma_f16_16816(h ? sU[nt] : sT[nt], a, qb[ks][2 * nt], qb[ks][2 * nt + 1]);
                    }
            } else {
                uint32_t a[D / 16][4];
#pragma unroll
                for (int ks = 0; ks < D / 16; ++ks)
                    ldmatrix_x4(a[ks][0], a[ks][1], a[ks][2], a[ks][3], kbase + koffs[ks]);
#pragma unroll
                for (int ks = 0; ks < D / 16; ++ks)
#pragma unroll
                    for (int nt = 0; nt < NT; ++nt) mma_bf16_16816((ks & 1) ? sU[nt] : sT[nt], a[ks], qb[ks][2 * nt], qb[ks][2 * nt + 1]);
            }
#pragma unroll
            for (int nt = 0; nt < NT; ++nt)
#pragma unroll
                for (int i = 0; i < 4; ++i) sT[nt][i] += sU[nt][i];
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(BAR(B_KEMPTY_D + s));
        SS_PF(1)
        mbar_wait(BAR(B_VFULL + s), fpar);
        SS_PF(2)
        if (nvalid > 0) {
            if (nvalid < kDecKeys) {
                // zero the V rows past the end of the KV range (unused slots may hold NaN; 0 * NaN = NaN)
                for (int i = lane; i < (kDecKeys - nvalid) * kHalves * 8; i += 32) {
                    const int r = r16 + nvalid + i / (kHalves * 8);
                    const int c = i % (kHalves * 8);
                    const uint32_t a = vbase + SM::kv_off(r, c);
                    asm volatile("st.shared.v4.b32 [%0], {%1,%1,%1,%1};" ::"r"(a), "r"(0u) : "memory");
                }
                __syncwarp();
            }
            // the V fragments are requested now, ahead of the softmax arithmetic that hides their latency.
            // bf16: a0 = (keys 0-7, d 0-7)^T, a1 = (keys 0-7, d 8-15)^T, a2 / a3: keys 8-15, one ldmatrix per 16 d;
            // FP8: matrices (keys 0-7, chunk), (keys 8-15, chunk), the same for chunk + 1, one ldmatrix per 32 d
            constexpr int kVLoads = FP8 ? D / 32 : D / 16;
            uint32_t va[kVLoads][4];
#pragma unroll
            for (int i = 0; i < kVLoads; ++i)
                ldmatrix_x4_trans(va[i][0], va[i][1], va[i][2], va[i][3], vbase + voffs[i]);
            uint32_t pb[NT][2];                              // B fragments of P^T (16 keys x 8 heads)
            bool moved = false;
            float mn[NT][2];
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) {
                // c0 / c1: key qr, heads qc / qc + 1;  c2 / c3: key qr + 8.  Masked by select, never by arithmetic.
                if (qr >= nvalid) { sT[nt][0] = -INFINITY; sT[nt][1] = -INFINITY; }
                if (qr + 8 >= nvalid) { sT[nt][2] = -INFINITY; sT[nt][3] = -INFINITY; }
                float b0 = fmaxf(sT[nt][0], sT[nt][2]), b1 = fmaxf(sT[nt][1], sT[nt][3]);
#pragma unroll
                for (int o = 4; o < 32; o <<= 1) {
                    b0 = fmaxf(b0, __shfl_xor_sync(0xffffffffu, b0, o));
                    b1 = fmaxf(b1, __shfl_xor_sync(0xffffffffu, b1, o));
                }
                mn[nt][0] = fmaxf(m[nt][0], b0 * sl2);
                mn[nt][1] = fmaxf(m[nt][1], b1 * sl2);
                moved |= mn[nt][0] != m[nt][0] || mn[nt][1] != m[nt][1];
                const float p0 = exp2f(sT[nt][0] * sl2 - mn[nt][0]), p1 = exp2f(sT[nt][1] * sl2 - mn[nt][1]);
                const float p2 = exp2f(sT[nt][2] * sl2 - mn[nt][0]), p3 = exp2f(sT[nt][3] * sl2 - mn[nt][1]);
                sT[nt][0] = p0 + p2;                         // this lane's share of the two row sums
                sT[nt][1] = p1 + p3;
                pb[nt][0] = movmatrix_trans(FP8 ? pack_f16(p0, p1) : pack_bf16(p0, p1));   // keys 0-7:  (key qr, heads qc..) -> (head qr, keys qc..)
                pb[nt][1] = movmatrix_trans(FP8 ? pack_f16(p2, p3) : pack_bf16(p2, p3));   // keys 8-15
            }
            // the accumulators are only rescaled when some head's maximum moved (warp-uniform test)
            if (__any_sync(0xffffffffu, moved)) {
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) {
                    const float al0 = exp2f(m[nt][0] - mn[nt][0]), al1 = exp2f(m[nt][1] - mn[nt][1]);   // first tile: exp2(-inf) = 0
                    l[nt][0] *= al0;
                    l[nt][1] *= al1;
#pragma unroll
                    for (int mt = 0; mt < D / 16; ++mt) { oT[nt][mt][0] *= al0; oT[nt][mt][1] *= al1; oT[nt][mt][2] *= al0; oT[nt][mt][3] *= al1; }
                    m[nt][0] = mn[nt][0];
                    m[nt][1] = mn[nt][1];
                }
            }
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) { l[nt][0] += sT[nt][0]; l[nt][1] += sT[nt][1]; }
            // O^T (D x 8 heads) += V^T (D x 16 keys) P^T
            if (FP8) {
#pragma unroll
                for (int mm = 0; mm < D / 32; ++mm)
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        // register = codes [key 2c][d 2qr], [2c][2qr+1], [2c+1][2qr], [2c+1][2qr+1] -> (d 2qr | d 2qr+1) x keys (2c, 2c+1)
                        const uint32_t x0 = __byte_perm(va[mm][2 * h], 0u, 0x3120), x1 = __byte_perm(va[mm][2 * h + 1], 0u, 0x3120);
                        const uint32_t a[4] = {e4m3x2_to_f16x2(x0), e4m3x2_hi_to_f16x2(x0), e4m3x2_to_f16x2(x1), e4m3x2_hi_to_f16x2(x1)};
#pragma unroll
                        for (int nt = 0; nt < NT; ++nt) mma_f16_16816(oT[nt][2 * mm + h], a, pb[nt][0], pb[nt][1]);
                    }
            } else {
#pragma unroll
                for (int mt = 0; mt < D / 16; ++mt)
#pragma unroll
                    for (int nt = 0; nt < NT; ++nt) mma_bf16_16816(oT[nt][mt], va[mt], pb[nt][0], pb[nt][1]);
            }
            if (nvalid < kDecKeys) fence_proxy_async();
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(BAR(B_VEMPTY_D + s));
        SS_PF(3)
    }
#ifdef SS_PROFILE
    if (tr) { tr[7] = ((unsigned long long)pf_acc[0] << 32) | (unsigned)pf_acc[1]; tr[8] = ((unsigned long long)pf_acc[2] << 32) | (unsigned)pf_acc[3]; }
#endif
    // ---- cross-warp log-sum-exp merge through smem, two stages over one 4-warp buffer [warp][head][D + 2] ----
    if (tr) tr[4] = globaltimer_ns();
#pragma unroll
    for (int nt = 0; nt < NT; ++nt)
#pragma unroll
        for (int o = 4; o < 32; o <<= 1) {
            l[nt][0] += __shfl_xor_sync(0xffffffffu, l[nt][0], o);
            l[nt][1] += __shfl_xor_sync(0xffffffffu, l[nt][1], o);
        }
    // G <= 8 (NT = 1): every warp writes its partial, one 8 -> 1 pass by all 256 threads.  G > 8: eight 16-row partials
    // do not fit the buffer - two stages over a 4-warp buffer (WG2 -> WG1 in registers, then 4 -> 1 by WG1).
    float* mine = merge + (NT == 1 ? wg * 4 + cw : cw) * mrows * (D + 2);
    const int dA = FP8 ? 2 * qr : qr, dB = FP8 ? 2 * qr + 1 : qr + 8;     // d (inside a 16-d block) of accumulator rows qr, qr + 8
    auto put = [&]() {
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) {
            float* h0 = mine + (8 * nt + qc) * (D + 2);
            float* h1 = h0 + (D + 2);
#pragma unroll
            for (int mt = 0; mt < D / 16; ++mt) {
                h0[16 * mt + dA] = oT[nt][mt][0];
                h1[16 * mt + dA] = oT[nt][mt][1];
                h0[16 * mt + dB] = oT[nt][mt][2];
                h1[16 * mt + dB] = oT[nt][mt][3];
            }
            if (qr == 0) {
                h0[D] = m[nt][0]; h0[D + 1] = l[nt][0];
                h1[D] = m[nt][1]; h1[D + 1] = l[nt][1];
            }
        }
    };
    if (NT == 1) {
        named_bar_sync(2, 256);                   // every thread is done reading the previous decode item's partials
        put();
        named_bar_sync(2, 256);
        if (tr) tr[5] = globaltimer_ns();
        for (int e = wg * 128 + wtid; e < G * D; e += 256) {
            const int r = e / D, d = e % D;
            float M = -INFINITY;
#pragma unroll
            for (int x = 0; x < 8; ++x) M = fmaxf(M, merge[(x * mrows + r) * (D + 2) + D]);
            float L = 0.f, acc = 0.f;
#pragma unroll
            for (int x = 0; x < 8; ++x) {
                const float* src = merge + (x * mrows + r) * (D + 2);
                const float wgt = exp2f(src[D] - M);           // a warp that saw no key: m = -inf -> weight 0
                L += src[D + 1] * wgt;
                acc += src[d] * wgt;
            }
            acc *= vs;
            if (w.nsplit == 1) {
                const int64_t orow = (int64_t)w.row0 * Hq + (int64_t)w.head * G + r;
                prm.out[orow * D + d] = __float2bfloat16_rn(acc / L);
                if (prm.lse && d == 0) prm.lse[orow] = (M + log2f(L)) * kMLn2;
            } else {
                float* dst = prm.partials + ((int64_t)(w.partial + w.split) * G + r) * (D + 2);
                dst[d] = acc;
                if (d == 0) { dst[D] = M; dst[D + 1] = L; }
            }
        }
        if (tr) tr[6] = globaltimer_ns();
        mbar_arrive(BAR(B_PARTIAL + slot));       // release (CTA) of this thread's partial stores to the a5 warp; count 256
        return;
    }
    if (wg == 1) {
        // stage A: WG2's warp cw hands its partial to WG1's warp cw (same fragment coordinates).  The buffer is free
        // once WG1 has finished the previous decode item's merge (named barrier 3: WG1 arrives, WG2 syncs).
        named_bar_sync(3, 256);
        put();
        named_bar_arrive(2, 256);
        return;
    }
    named_bar_sync(2, 256);
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) {
        const float* h0 = mine + (8 * nt + qc) * (D + 2);
        const float* h1 = h0 + (D + 2);
        const float mb0 = h0[D], lb0 = h0[D + 1], mb1 = h1[D], lb1 = h1[D + 1];
        const float M0 = fmaxf(m[nt][0], mb0), M1 = fmaxf(m[nt][1], mb1);
        // a side that saw no key has m = -inf: weight 0 (and never exp2(-inf - -inf))
        const float wa0 = m[nt][0] == -INFINITY ? 0.f : exp2f(m[nt][0] - M0), wb0 = mb0 == -INFINITY ? 0.f : exp2f(mb0 - M0);
        const float wa1 = m[nt][1] == -INFINITY ? 0.f : exp2f(m[nt][1] - M1), wb1 = mb1 == -INFINITY ? 0.f : exp2f(mb1 - M1);
#pragma unroll
        for (int mt = 0; mt < D / 16; ++mt) {
            oT[nt][mt][0] = oT[nt][mt][0] * wa0 + h0[16 * mt + dA] * wb0;
            oT[nt][mt][1] = oT[nt][mt][1] * wa1 + h1[16 * mt + dA] * wb1;
            oT[nt][mt][2] = oT[nt][mt][2] * wa0 + h0[16 * mt + dB] * wb0;
            oT[nt][mt][3] = oT[nt][mt][3] * wa1 + h1[16 * mt + dB] * wb1;
        }
        l[nt][0] = l[nt][0] * wa0 + lb0 * wb0;
        l[nt][1] = l[nt][1] * wa1 + lb1 * wb1;
        m[nt][0] = M0;
        m[nt][1] = M1;
    }
    __syncwarp();                                 // this warp's reads of `mine` are done before it rewrites it
    put();
    named_bar_sync(1, 128);
    if (tr) tr[5] = globaltimer_ns();
    for (int e = wtid; e < G * D; e += 128) {
        const int r = e / D, d = e % D;
        float M = -INFINITY;
#pragma unroll
        for (int x = 0; x < 4; ++x) M = fmaxf(M, merge[(x * mrows + r) * (D + 2) + D]);
        float L = 0.f, acc = 0.f;
#pragma unroll
        for (int x = 0; x < 4; ++x) {
            const float* src = merge + (x * mrows + r) * (D + 2);
            const float wgt = exp2f(src[D] - M);           // a warp pair that saw no key: m = -inf -> weight 0
            L += src[D + 1] * wgt;
            acc += src[d] * wgt;
        }
        acc *= vs;
        if (w.nsplit == 1) {
            const int64_t orow = (int64_t)w.row0 * Hq + (int64_t)w.head * G + r;
            prm.out[orow * D + d] = __float2bfloat16_rn(acc / L);
            if (prm.lse && d == 0) prm.lse[orow] = (M + log2f(L)) * kMLn2;
        } else {
            float* dst = prm.partials + ((int64_t)(w.partial + w.split) * G + r) * (D + 2);
            dst[d] = acc;
            if (d == 0) { dst[D] = M; dst[D + 1] = L; }
        }
    }
    if (tr) tr[6] = globaltimer_ns();
    // a5 hand-off: warp 3 publishes this split and, if it was the last of its (request, kv head), merges all of them; the
    // decode warps go straight on to the next item.  mbarrier arrive = release at CTA scope for this thread's partial stores.
    mbar_arrive(BAR(B_PARTIAL + slot));           // once per item and slot use (phase = slot use count)
    named_bar_sync(1, 128);                       // every WG1 thread is done reading the merge buffer ...
    named_bar_arrive(3, 256);                     // ... so WG2 may write the next decode item's partials
}

// One tensor's tile stream (K by warp 0, V by warp 3), run by ONE thread: 64-key tiles of an item's KV range into the
// ring, one 4-D TMA box per (page, kv head) slab.  What the loop is shaped around (measured, profiles/r2b.md): the thread
// pays ~115 ns per barrier phase (try_wait round trip + arrive.expect_tx) and ~25 ns per TMA operation whose
// coordinates must first reach uniform registers (LDG -> IMAD -> R2UR).  So: the EMPTY test of the NEXT slot is issued
// before this tile's operations (its round trip overlaps them), full tiles take a branch-free path so the four R2UR /
// UTMALDG pairs can be scheduled together, and page ids are loaded two tiles ahead of their use.
// Slot history as bit fields: parity of the next EMPTY wait per consumer type, and the type (1 prefill / 2 decode) of
// the slot's last consumer, which names the EMPTY barrier that consumer will arrive on.
template <int D, bool FP8, int B_FULL0, int B_EMPTY_P0, int B_EMPTY_D0>
struct TileStreamer {
    using SM = MixSmem<D, FP8>;
    uint32_t parP = 0, parD = 0, lastT = 0;
    int s = 0;                     // ring slot of the next tile
    uint32_t eb = 0, epar = 0;     // EMPTY barrier (0: slot never used) and parity the next tile must see
    bool ok = true;                // ... and whether an early test already found it complete
    uint32_t bar0, ring;           // shared addresses: barrier block, this tensor's ring
    const CUtensorMap* tmap;

    __device__ __forceinline__ uint32_t BAR(int i) const { return bar0 + 8u * (uint32_t)i; }
    __device__ __forceinline__ void look(int slot, uint32_t& b, uint32_t& par) const {
        const uint32_t lt = (lastT >> (2 * slot)) & 3u;
        par = ((lt == 1 ? parP : parD) >> slot) & 1u;
        b = lt ? BAR((lt == 1 ? B_EMPTY_P0 : B_EMPTY_D0) + slot) : 0u;
    }
    // streams keys [w.kv_begin, w.kv_end) of request row `bt`, kv head g; pg = page ids of the first tile;
    // on_last() runs just before the item's last tile is issued
    template <typename F>
    __device__ __forceinline__ void item(const ss_work_item& w, const int32_t* __restrict__ bt, const int g, const int Hkv,
                                         int (&pg)[4], F on_last) {
        auto load_pages = [&](int key0, int (&dst)[4]) {
#pragma unroll
            for (int p = 0; p < 4; ++p) dst[p] = (key0 + p * kPage < w.kv_end) ? __ldg(bt + (key0 >> 4) + p) : 0;
        };
        int pg1[4];
        load_pages(w.kv_begin + kSlotKeys, pg1);
        const int ntiles = (w.kv_end - w.kv_begin + kSlotKeys - 1) / kSlotKeys;
        const int nring = SM::kOwnSlots ? (ntiles + 1) & ~1 : ntiles;      // even ring: pad with an empty tile (see the consumers)
        for (int i = 0, key0 = w.kv_begin; i < nring; ++i, key0 += kSlotKeys) {
            if (i == ntiles - 1) on_last();              // (drawing the next ticket 3 or 5 tiles earlier changes nothing)
            int pg2[4];
            load_pages(key0 + 2 * kSlotKeys, pg2);                 // used two iterations from now
            int cg[4];                                             // first 8-key group of each (page, kv head) slab
#pragma unroll
            for (int p = 0; p < 4; ++p) cg[p] = (pg[p] * Hkv + g) * 2;
            const int s1 = s + 1 == SM::kNumSt ? 0 : s + 1;
            uint32_t eb1, epar1;
            look(s1, eb1, epar1);                                  // slot s1's history cannot change while tile s is issued
            while (!ok) ok = mbar_try_wait(eb, epar);
            const bool ok1 = eb1 ? mbar_try_wait(eb1, epar1) : true;   // early test: its round trip overlaps the issue below
            const uint32_t full = BAR(B_FULL0 + s), dst = ring + s * SM::kSlot;
            const int nkeys = w.kv_end - key0;
            if (nkeys >= kSlotKeys) {
                mbar_arrive_expect_tx(full, 4u * SM::kPageBytes);
#pragma unroll
                for (int p = 0; p < 4; ++p) tma_load_slab(dst + p * SM::kPageBytes, tmap, cg[p], full);
            } else {
                const int npages = nkeys > 0 ? (nkeys + kPage - 1) / kPage : 0;      // 0: the padding tile, a plain arrival
                mbar_arrive_expect_tx(full, (uint32_t)npages * SM::kPageBytes);
#pragma unroll
                for (int p = 0; p < 4; ++p)
                    if (p < npages) tma_load_slab(dst + p * SM::kPageBytes, tmap, cg[p], full);
            }
            const uint32_t lt = (lastT >> (2 * s)) & 3u;
            if (lt == 1) parP ^= 1u << s; else if (lt == 2) parD ^= 1u << s;
            lastT = (lastT & ~(3u << (2 * s))) | ((uint32_t)w.kind << (2 * s));
            s = s1; eb = eb1; epar = epar1; ok = ok1;
#pragma unroll
            for (int p = 0; p < 4; ++p) { pg[p] = pg1[p]; pg1[p] = pg2[p]; }
        }
    }
};

// a5: publish one decode split (acq_rel ticket) and, if it was the last of its (request, kv head), merge all splits in
// fixed split order (bitwise reproducible).  One whole warp; `use` = how many times the scheduler slot has been used.
template <int D>
__device__ __forceinline__ void split_merge(const ss_work_item& w, const int slot, const uint32_t use, const int lane,
                                            const uint32_t bar0, const MixParams& prm) {
    auto BAR = [&](int i) -> uint32_t { return bar0 + 8u * (uint32_t)i; };
    const int Hq = prm.Hq, Hkv = prm.Hkv, G = Hq / Hkv;
    mbar_wait(BAR(B_PARTIAL + slot), use & 1);   // acquire (CTA): all 128 merge threads' partial stores
    int last = 0;
    if (lane == 0) last = atom_add_acq_rel_gpu(prm.merge_counters + w.req * Hkv + w.head, 1) == w.nsplit - 1;
    last = __shfl_sync(0xffffffffu, last, 0);
    __syncwarp();
    if (last) {
        // lane owns columns d = lane + 32 j; 2 rows (q heads) per pass; per split 4 + 2 D/32 independent
        // L2 loads in flight per lane (x2 unrolled), online log-sum-exp merge in split order
        constexpr int DJ = D / 32;
        const int64_t sstride = (int64_t)G * (D + 2);
        const float* pbase = prm.partials + (int64_t)w.partial * sstride;
        for (int r0 = 0; r0 < G; r0 += 2) {
            float M[2], L[2], A[2][DJ];
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                M[i] = -INFINITY; L[i] = 0.f;
#pragma unroll
                for (int j = 0; j < DJ; ++j) A[i][j] = 0.f;
            }
#pragma unroll 2
            for (int x = 0; x < w.nsplit; ++x) {
                const float* px = pbase + x * sstride;
                float mx[2], lx[2], ox[2][DJ];
#pragma unroll
                for (int i = 0; i < 2; ++i) {
                    const float* pr = px + min(r0 + i, G - 1) * (D + 2);
                    mx[i] = __ldcg(pr + D);
                    lx[i] = __ldcg(pr + D + 1);
#pragma unroll
                    for (int j = 0; j < DJ; ++j) ox[i][j] = __ldcg(pr + lane + 32 * j);
                }
#pragma unroll
                for (int i = 0; i < 2; ++i) {
                    const float Mn = fmaxf(M[i], mx[i]);
                    const float al = exp2f(M[i] - Mn), bx = exp2f(mx[i] - Mn);
                    L[i] = L[i] * al + lx[i] * bx;
#pragma unroll
                    for (int j = 0; j < DJ; ++j) A[i][j] = A[i][j] * al + ox[i][j] * bx;
                    M[i] = Mn;
                }
            }
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                if (r0 + i < G) {
                    const int64_t orow = (int64_t)w.row0 * Hq + (int64_t)w.head * G + r0 + i;
                    const float inv = 1.f / L[i];
#pragma unroll
                    for (int j = 0; j < DJ; ++j) prm.out[orow * D + lane + 32 * j] = __float2bfloat16_rn(A[i][j] * inv);
                    if (prm.lse && lane == 0) prm.lse[orow] = (M[i] + log2f(L[i])) * kMLn2;
                }
            }
        }
        if (lane == 0) prm.merge_counters[w.req * Hkv + w.head] = 0;     // re-armed for the next call
    }
}

template <int D, bool FP8>
__global__ void __launch_bounds__(MixCta<FP8>::kThreads, 1)
mixed_kernel(const __grid_constant__ CUtensorMap tmap_q, const __grid_constant__ CUtensorMap tmap_k,
             const __grid_constant__ CUtensorMap tmap_v, const MixParams prm) {
    using SM = MixSmem<D, FP8>;
    constexpr int kHalves = SM::kHalves;
    extern __shared__ __align__(1024) uint8_t smem_raw[];       // SWIZZLE_128B tiles need 1024-byte alignment
    const uint32_t sbase = smem_u32(smem_raw);
    uint8_t* smem = smem_raw;
    if (sbase & 1023u) __trap();                                // never observed; a misaligned window would corrupt every tile
    const uint32_t bar0 = sbase + SM::kBarOff;
    auto BAR = [&](int i) -> uint32_t { return bar0 + 8u * (uint32_t)i; };
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + SM::kTmemSlotOff);
    const ss_work_item* sched = reinterpret_cast<const ss_work_item*>(smem + SM::kSchedOff);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int Hq = prm.Hq, Hkv = prm.Hkv, G = Hq / Hkv;
    unsigned long long* const trace = prm.trace ? prm.trace + (size_t)blockIdx.x * prm.trace_words : nullptr;
    if (trace && threadIdx.x == 0) trace[0] = globaltimer_ns();

    if (threadIdx.x == 0) {
        for (int s = 0; s < SM::kNumSt; ++s) {
            mbar_init(BAR(B_KFULL + s), 1);
            mbar_init(BAR(B_VFULL + s), 1);
            mbar_init(BAR(B_KEMPTY_P + s), FP8 ? 1 : 2);     // one commit per chain; FP8: the K converter warps
            mbar_init(BAR(B_VEMPTY_P + s), FP8 ? 1 : 2);
            mbar_init(BAR(B_KEMPTY_D + s), SM::kOwnSlots ? 4 : 8);   // the owning warpgroup / every decode warp
            mbar_init(BAR(B_VEMPTY_D + s), SM::kOwnSlots ? 4 : 8);
        }
        for (int b = 0; b < 4; ++b) {
            mbar_init(BAR(B_SFULL + b), 1);
            mbar_init(BAR(B_PFULL + b), 128);
        }
        mbar_init(BAR(B_QFULL), 1);
        mbar_init(BAR(B_QEMPTY), 2);
        if (FP8) {
            for (int b = 0; b < 2; ++b) {
                mbar_init(BAR(B_KCONV_FULL + b), 1);
                mbar_init(BAR(B_KCONV_EMPTY + b), 2);             // one commit per chain, like the ring slots
                mbar_init(BAR(B_VCONV_FULL + b), 1);
                mbar_init(BAR(B_VCONV_EMPTY + b), 2);
            }
            mbar_init(BAR(B_QCONV + 0), 128);
            mbar_init(BAR(B_QCONV + 1), 128);
        }
        for (int x = 0; x < 2; ++x) {
            mbar_init(BAR(B_OFULL + x), 1);
            mbar_init(BAR(B_OFREE + x), 128);
            mbar_init(BAR(B_PVDONE + x), 1);
        }
        for (int s = 0; s < kSchedSlots; ++s) {
            mbar_init(BAR(B_PARTIAL + s), G <= 8 ? 256 : 128);   // the threads that store decode partials (see decode_item)
            mbar_init(BAR(B_SCHED_FULL + s), 1);
            mbar_init(BAR(B_SCHED_EMPTY + s), FP8 ? 15 : 11);    // 2 MMA warps (warp 2 = a5) + the V producer + 8 worker warps (+ 4 converter warps)
        }
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
    pdl_wait();                 // everything above overlaps the tail of the preceding kernel (kv_append / work list)
    PlanHeader* const ph = reinterpret_cast<PlanHeader*>(smem + SM::kPlanOff);
    PlanTables<uint16_t> ptb;
    ptb.ord = reinterpret_cast<uint16_t*>(smem + SM::kPlanOff + 64);
    ptb.off = ptb.ord + kPlanMaxR;
    const bool tripped = prm.err_flag && *reinterpret_cast<const volatile int32_t*>(prm.err_flag) != 0;   // CTA-uniform
    if (tripped) {
        // debug checks found bad metadata: an empty plan - every role sees the end-of-list item and leaves
        if (threadIdx.x == 0) { ph->tot_p = 0; ph->tot_d = 0; ph->n_decode_ctas = 0; ph->nP = 0; ph->nD = 0; }
    } else if (prm.self_plan) {
        // a2: every CTA builds the same plan (scratch = the still unused K ring); items are decoded from queue tickets
        build_plan<MixCta<FP8>::kThreads, uint16_t>(prm.qsl, prm.ctx_lens, prm.R, Hq, Hkv, D, prm.num_sms, prm.force_split_keys,
                                          prm.force_decode_ctas, prm.max_partials, reinterpret_cast<int32_t*>(smem + SM::kKOff), ptb, ph);
        fence_proxy_async();    // scratch was written through the generic proxy; TMA writes the same bytes next
    } else if (threadIdx.x == 0) {
        ph->tot_p = prm.hdr->n_prefill;
        ph->tot_d = prm.hdr->n_decode;
        ph->n_decode_ctas = prm.hdr->n_decode_ctas;
    }
    __syncthreads();
    if (trace && threadIdx.x == 0) trace[1] = globaltimer_ns();
    const uint32_t tmem_base = *tmem_slot;

    // Re-partition the register file: the producer / issuer warpgroup gives up what the 8 worker warps need.  The two
    // setmaxnreg sit INSIDE the role branches (which only re-join at the teardown): ptxas allocates each region against
    // the count of the setmaxnreg that dominates it, and code reachable from both would get the smaller one.
    if (warp < 4) {
      setmaxnreg_dec<MixCta<FP8>::kRegsWg0>();
      if (warp == 0) {
        // =============================== scheduler + TMA producer ===============================
        // One elected thread runs the whole loop (waits included) so every TMA operand is uniform.
        if (elect_one()) {
            const int n_pre_items = ph->tot_p, n_dec = ph->tot_d;
            const bool prefer_decode = (int)blockIdx.x < ph->n_decode_ctas;
            int32_t* const q_pre = prm.queue, * const q_dec = prm.queue + 1;
            bool pre_done = n_pre_items == 0, dec_done = n_dec == 0;
            // per-slot history as bit fields: parity of the next EMPTY wait per consumer type, last consumer type
            TileStreamer<D, FP8, B_KFULL, B_KEMPTY_P, B_KEMPTY_D> ks;
            ks.bar0 = bar0; ks.ring = sbase + SM::kKOff; ks.tmap = &tmap_k;
            uint32_t n_sched = 0, n_pre = 0;
            int prev_kind = 0;
            const bool q_staged = G <= 8;
            union WU { ss_work_item it; uint4 v[3]; };
            // two typed queues: this CTA drains its preferred kind first, then helps with the other
            auto fetch = [&](WU& wu) {
                int idx = -1;
                if (prefer_decode) {
                    if (!dec_done) { const int i = atomicAdd(q_dec, 1); if (i < n_dec) idx = n_pre_items + i; else dec_done = true; }
                    if (idx < 0 && !pre_done) { const int i = atomicAdd(q_pre, 1); if (i < n_pre_items) idx = i; else pre_done = true; }
                } else {
                    if (!pre_done) { const int i = atomicAdd(q_pre, 1); if (i < n_pre_items) idx = i; else pre_done = true; }
                    if (idx < 0 && !dec_done) { const int i = atomicAdd(q_dec, 1); if (i < n_dec) idx = n_pre_items + i; else dec_done = true; }
                }
                if (idx >= 0 && prm.self_plan) {
                    plan_decode_item(idx, ph, ptb, prm.qsl, prm.ctx_lens, Hq, Hkv, wu.it);
                } else if (idx >= 0) {
                    const uint4* src = reinterpret_cast<const uint4*>(prm.items + idx);
                    wu.v[0] = __ldg(src); wu.v[1] = __ldg(src + 1); wu.v[2] = __ldg(src + 2);
                } else {
                    wu.v[0] = wu.v[1] = wu.v[2] = make_uint4(0u, 0u, 0u, 0u);
                }
            };
            auto first_pages = [&](const ss_work_item& it, int (&pgs)[4]) {
                const int32_t* b = prm.block_table + (int64_t)it.req * prm.max_pages;
#pragma unroll
                for (int p = 0; p < 4; ++p)
                    pgs[p] = (it.kind != 0 && it.kv_begin + p * kPage < it.kv_end) ? __ldg(b + (it.kv_begin >> 4) + p) : 0;
            };
            // the NEXT item (queue ticket, record, first page ids) is fetched while the current item's tiles are being
            // issued, so the atomic -> record -> block-table latency chain never sits between two items' TMA streams
            WU nxt;
            int nxt_pg[4];
            fetch(nxt);
            first_pages(nxt.it, nxt_pg);
            for (;;) {
                const int slot = n_sched % kSchedSlots;
                mbar_wait(BAR(B_SCHED_EMPTY + slot), ((n_sched / kSchedSlots) & 1) ^ 1);
                uint4* dst = reinterpret_cast<uint4*>(smem + SM::kSchedOff + slot * 48);
                const WU wu = nxt;
                dst[0] = wu.v[0]; dst[1] = wu.v[1]; dst[2] = wu.v[2];
                const ss_work_item& w = wu.it;
                if (w.kind == 2 && q_staged) {
                    // the staged Q block lies inside the prefill Q tiles: the last prefill item's MMAs must be done
                    mbar_wait(BAR(B_QEMPTY), (n_pre & 1) ^ 1);
                    const uint32_t qbytes = (uint32_t)(G * D * 2);
                    mbar_arrive_expect_tx(BAR(B_SCHED_FULL + slot), qbytes);     // release: the record is visible too
                    bulk_load_1d(sbase + SM::kQStageOff + slot * SM::kQStageBytes,
                                 prm.q + ((int64_t)w.row0 * Hq + (int64_t)w.head * G) * D, qbytes, BAR(B_SCHED_FULL + slot));
                } else {
                    mbar_arrive(BAR(B_SCHED_FULL + slot));        // release semantics: the item is visible to the waiters
                }
                ++n_sched;
                if (w.kind == 0) break;
                const int32_t* bt = prm.block_table + (int64_t)w.req * prm.max_pages;
                const int g = w.kind == 1 ? w.head / G : w.head;
                int pg[4];
#pragma unroll
                for (int p = 0; p < 4; ++p) pg[p] = nxt_pg[p];
                if (w.kind == 1) {
                    mbar_wait(BAR(B_QEMPTY), (n_pre & 1) ^ 1);
                    if (prev_kind == 2) {
                        // the Q region doubles as the decode merge buffer: wait until the previous (decode) item is done
                        const uint32_t pn = n_sched - 2;
                        mbar_wait(BAR(B_SCHED_EMPTY + pn % kSchedSlots), (pn / kSchedSlots) & 1);
                    }
                    mbar_arrive_expect_tx(BAR(B_QFULL), (uint32_t)(w.nheads * SM::kQTile));
                    for (int x = 0; x < w.nheads; ++x)
#pragma unroll
                        for (int hh = 0; hh < kHalves; ++hh)
                            tma_load_2d(sbase + SM::kQOff + x * SM::kQTile + hh * (kTileRows * 128), &tmap_q,
                                        (w.head + x) * D + hh * 64, w.row0, BAR(B_QFULL));
                    ++n_pre;
                }
                prev_kind = w.kind;
                // K only: the V tiles of every item are streamed by warp 3 (one thread could not issue both).  At the item's
                // last tile the next ticket is drawn (not earlier, or the tail of the launch grows by an item held while
                // this one is still streaming); the ring hides the atomic -> record -> block-table chain.
                ks.item(w, bt, g, Hkv, pg, [&]() {
                    fetch(nxt);
                    first_pages(nxt.it, nxt_pg);
                });
            }
            if (prm.self_plan) {
                // self-cleaning queue: every CTA checks out after its last ticket; the last one re-arms the counters
                // for the next call on this handle (the state lives in handle-owned memory, zeroed at ss_create)
                if (atomicAdd(prm.queue + 2, 1) == (int)gridDim.x - 1) {
                    atomicExch(prm.queue + 0, 0);
                    atomicExch(prm.queue + 1, 0);
                    atomicExch(prm.queue + 2, 0);
                }
            }
        }
      } else if (warp == 3) {
        // =============================== V producer ===============================
        // Follows the scheduler ring like every consumer and streams the V tiles of each item into the V ring: same slot
        // order and the same typed-EMPTY bookkeeping as warp 0 keeps for K.  One elected thread, waits included.
        if (elect_one()) {
            TileStreamer<D, FP8, B_VFULL, B_VEMPTY_P, B_VEMPTY_D> vs;
            vs.bar0 = bar0; vs.ring = sbase + SM::kVOff; vs.tmap = &tmap_v;
            uint32_t n_sched = 0;
            for (;;) {
                const int slot = n_sched % kSchedSlots;
                mbar_wait(BAR(B_SCHED_FULL + slot), (n_sched / kSchedSlots) & 1);
                const ss_work_item w = sched[slot];
                ++n_sched;
                if (w.kind == 0) break;
                const int32_t* bt = prm.block_table + (int64_t)w.req * prm.max_pages;
                const int g = w.kind == 1 ? w.head / G : w.head;
                int pg[4];
#pragma unroll
                for (int p = 0; p < 4; ++p) pg[p] = (w.kv_begin + p * kPage < w.kv_end) ? __ldg(bt + (w.kv_begin >> 4) + p) : 0;
                vs.item(w, bt, g, Hkv, pg, []() {});
                mbar_arrive(BAR(B_SCHED_EMPTY + slot));
            }
        }
      } else {
        // =============================== tcgen05.mma issuers ===============================
        // Warp 1 issues chain A's MMAs, warp 2 chain B's (one elected thread each, waits included, so descriptors stay
        // in uniform registers).  Two issuers because one thread could not keep the pipe fed: per (chain, half tile)
        // it spent ~250 cycles in three mbarrier round trips and ~740 blocked in issue (profiles/r2_a3.md), serially
        // for both chains.  The chains touch disjoint TMEM and only read the shared K/V slots, so no order is needed
        // between them; the slot / Q-tile release barriers take one commit per chain (chain A commits twice when the
        // item has a single head).  Decode items: warp 1 has nothing to do, warp 2 runs a5 (split_merge).
        // FP8 cache: the operands are the fp16 copies the converter warps (WG3) write into two K and two V buffers (shared
        // by both chains, released by one commit per chain), Q converted in place by each chain's workers; tiles are
        // counted by cv_ctr.
        constexpr uint32_t idesc_qk = FP8 ? umma_idesc_f16(kTileRows, kSlotKeys, 0) : umma_idesc_bf16(kTileRows, kSlotKeys, 0);
        constexpr uint32_t idesc_pv = FP8 ? umma_idesc_f16(kTileRows, D, 1) : umma_idesc_bf16(kTileRows, D, 1);
        const int X = warp - 1;
        const uint32_t tchain = tmem_base + X * SM::kTmemChain;
        uint32_t tile_ctr = 0, n_sched = 0, n_pre = 0, s_ctr = 0, n_chain = 0;   // s_ctr / n_chain: this chain's half tiles / items
        uint32_t cv_ctr = 0;                                                      // FP8: prefill tiles converted so far
        for (;;) {
            const int slot = n_sched % kSchedSlots;
            mbar_wait(BAR(B_SCHED_FULL + slot), (n_sched / kSchedSlots) & 1);
            const ss_work_item w = sched[slot];
            const int kind = w.kind;
            // ring tiles of the item; on an even ring (FP8) padded to an even count with an empty tile, so that every
            // item starts on an even slot and tile parity = slot parity holds with ITEM-LOCAL tile indices (the split of
            // keys between the warpgroups, hence the summation order, must not depend on what the CTA ran before)
            const int n = SM::kOwnSlots ? ((w.kv_end - w.kv_begin + kSlotKeys - 1) / kSlotKeys + 1) & ~1
                                        : (w.kv_end - w.kv_begin + kSlotKeys - 1) / kSlotKeys;
            const int nr = (w.kv_end - w.kv_begin + kSlotKeys - 1) / kSlotKeys;      // real tiles (n may hold a padding tile)
            ++n_sched;
            if (kind == 0) break;
            if (kind == 1) {
                const int nq = w.nheads;
                // Every issuer observes every Q phase, also chain B's on a single-head item it sits out: a parity wait
                // is only exact for a waiter that is at most one phase behind, and the Q phase is what orders an item
                // against the ring (see B_QEMPTY below).
                if (X >= nq && elect_one()) mbar_wait(BAR(B_QFULL), n_pre & 1);
                if (X < nq && elect_one()) {
                    const int ncommit = nq == 1 ? 2 : 1;          // arrivals this chain owes the shared (count 2) barriers
#ifdef SS_PROFILE
                    long long mm_t = 0, mm_acc[4] = {0, 0, 0, 0};      // wait P (+O free) | wait K/V | issue | -
#endif
                    auto issue_s = [&](int kt) {
                        const uint32_t tc = tile_ctr + kt, sc = s_ctr + kt;
                        const int s = tc % SM::kNumSt, b = sc & 1;
                        const uint32_t cv = cv_ctr + kt, cb = cv & 1;
                        SS_MM(2)
                        if (FP8) mbar_wait(BAR(B_KCONV_FULL + cb), (cv >> 1) & 1);
                        else mbar_wait(BAR(B_KFULL + s), (tc / SM::kNumSt) & 1);
                        tc_fence_after();
                        SS_MM(1)
                        const uint64_t qdesc0 = umma_desc_sw128(sbase + SM::kQOff + X * SM::kQTile, 16, 1024);
                        const uint64_t kdesc0 = FP8 ? umma_desc_sw128(sbase + SM::kKConvOff + cb * SM::kConvTile, 16, SM::kConvGroup)
                                                    : umma_desc_sw128(sbase + SM::kKOff + s * SM::kSlot, 16, SM::kGroup);
#pragma unroll
                        for (int ks = 0; ks < D / 16; ++ks) {
                            // bytes; descriptor address unit = 16 B.  64-column halves: Q 128 rows, K 64 rows apart
                            const uint32_t qoff = (ks >> 2) * (kTileRows * 128) + (ks & 3) * 32;
                            const uint32_t koff = (ks >> 2) * 1024 + (ks & 3) * 32;
                            umma_ss(tchain + b * 64, qdesc0 + (qoff >> 4), kdesc0 + (koff >> 4), idesc_qk, ks > 0);
                        }
                        umma_commit(BAR(B_SFULL + X * 2 + b));
                        if (FP8) for (int c = 0; c < ncommit; ++c) umma_commit(BAR(B_KCONV_EMPTY + cb));
                        else for (int c = 0; c < ncommit; ++c) umma_commit(BAR(B_KEMPTY_P + s));
                    };
                    auto issue_pv = [&](int kt) {
                        const uint32_t tc = tile_ctr + kt, sc = s_ctr + kt;
                        const int s = tc % SM::kNumSt, b = sc & 1;
                        SS_MM(2)
                        mbar_wait(BAR(B_PFULL + X * 2 + b), (sc >> 1) & 1);
                        if (kt == 0) mbar_wait(BAR(B_OFREE + X), (n_chain & 1) ^ 1);     // previous epilogue drained O
                        const uint32_t cv = cv_ctr + kt, cb = cv & 1;
                        SS_MM(0)
                        if (FP8) mbar_wait(BAR(B_VCONV_FULL + cb), (cv >> 1) & 1);
                        else mbar_wait(BAR(B_VFULL + s), (tc / SM::kNumSt) & 1);
                        tc_fence_after();
                        SS_MM(1)
                        // halves 1024 apart, 8-key groups kGroup; 16 keys (one k-step) = two groups
                        const uint64_t vdesc0 = FP8 ? umma_desc_sw128(sbase + SM::kVConvOff + cb * SM::kConvTile, 1024, SM::kConvGroup)
                                                    : umma_desc_sw128(sbase + SM::kVOff + s * SM::kSlot, 1024, SM::kGroup);
                        constexpr uint32_t kstep = 2 * (FP8 ? SM::kConvGroup : SM::kGroup);
#pragma unroll
                        for (int kk = 0; kk < kSlotKeys / 16; ++kk)      // A = P[b] from TMEM: 16 keys = 8 packed columns
                            umma_ts(tchain + SM::kTmemO, tchain + b * 64 + kk * 8, vdesc0 + (uint64_t)(kk * kstep >> 4), idesc_pv, (kt > 0 || kk > 0));
                        umma_commit(BAR(B_PVDONE + X));
                        if (FP8) for (int c = 0; c < ncommit; ++c) umma_commit(BAR(B_VCONV_EMPTY + cb));
                        else for (int c = 0; c < ncommit; ++c) umma_commit(BAR(B_VEMPTY_P + s));
                        if (kt == nr - 1) {
                            umma_commit(BAR(B_OFULL + X));
                            // Q tiles free for the next item.  Committed after the LAST MMA of the item (not the last
                            // S): when the next Q tile lands, every K and V tile issued before it has landed too, so a
                            // role that sat out an item (chain B on single-head items, both issuers on decode items)
                            // can never run a parity wait one phase early on a ring slot.
                            for (int c = 0; c < ncommit; ++c) umma_commit(BAR(B_QEMPTY));
                        }
                    };
                    mbar_wait(BAR(B_QFULL), n_pre & 1);
                    if (FP8) { mbar_wait(BAR(B_QCONV + X), n_chain & 1); tc_fence_after(); }   // this chain's Q tile rewritten as fp16
#ifdef SS_PROFILE
                    mm_t = clock64();
#endif
                    for (int kt = 0; kt < 2 && kt < nr; ++kt) issue_s(kt);
                    for (int kt = 0; kt < nr; ++kt) {
                        issue_pv(kt);
                        if (kt + 2 < nr) issue_s(kt + 2);
                    }
#ifdef SS_PROFILE
                    SS_MM(2)
                    if (trace && prm.trace_words >= 16 && X == 0) {
                        unsigned long long* tw = trace + prm.trace_words - 4;
                        tw[0] += mm_acc[0]; tw[1] += mm_acc[1]; tw[2] += mm_acc[2]; tw[3] += (unsigned long long)n;
                    }
#endif
                }
                __syncwarp();
                if (X < nq) { s_ctr += nr; ++n_chain; }
                cv_ctr += nr;
                ++n_pre;
            } else if (X == 1 && w.nsplit > 1) {
                split_merge<D>(w, slot, (n_sched - 1) / kSchedSlots, lane, bar0, prm);
            }
            tile_ctr += n;
            __syncwarp();
            if (lane == 0) mbar_arrive(BAR(B_SCHED_EMPTY + slot));
        }
        if (trace && lane == 0 && X == 1) trace[4] = globaltimer_ns();
      }
    } else if (warp < 12) {
        setmaxnreg_inc<MixCta<FP8>::kRegsWorker>();
        // =============================== workers ===============================
        const int wg = (warp - 4) >> 2;                        // 0: chain A / decode on even slots, 1: chain B / decode on odd slots
        const int cw = (warp - 4) & 3;                         // decode: 16-key slice of the slot
        const int quarter = warp & 3;                          // TMEM lane quarter this warp may access
        const int row = quarter * 32 + lane;                   // prefill: query row inside the tile
        const uint32_t lane_addr = (uint32_t)(quarter * 32) << 16;
        const int wtid = threadIdx.x - 128 - wg * 128;         // 0..127 inside the warpgroup
        const float sl2_base = prm.scale * kMLog2e;
        const uint32_t tchain = tmem_base + wg * SM::kTmemChain;
        const uint32_t tmem_o = tchain + SM::kTmemO;
        uint32_t tile_ctr = 0, s_ctr = 0, n_sched = 0, n_chain = 0, n_pre = 0;
        float* merge = reinterpret_cast<float*>(smem + SM::kQOff);
        if (wg == 0 && G > 8) named_bar_arrive(3, 256);        // G > 8: the decode merge buffer starts out free (stage A of decode_item)
        for (;;) {
            const int slot = n_sched % kSchedSlots;
            mbar_wait(BAR(B_SCHED_FULL + slot), (n_sched / kSchedSlots) & 1);
            const ss_work_item w = sched[slot];
            ++n_sched;
            if (w.kind == 0) break;
            // ring tiles of the item; on an even ring (FP8) padded to an even count with an empty tile, so that every
            // item starts on an even slot and tile parity = slot parity holds with ITEM-LOCAL tile indices (the split of
            // keys between the warpgroups, hence the summation order, must not depend on what the CTA ran before)
            const int n = SM::kOwnSlots ? ((w.kv_end - w.kv_begin + kSlotKeys - 1) / kSlotKeys + 1) & ~1
                                        : (w.kv_end - w.kv_begin + kSlotKeys - 1) / kSlotKeys;
            unsigned long long* const tr = (trace && wg == 0 && wtid == 0 && 6 + 9 * (int)n_sched <= prm.trace_words) ? trace + 6 + 9 * (n_sched - 1) : nullptr;
            if (tr) {
                tr[0] = globaltimer_ns();
                tr[2] = ((unsigned long long)w.kind << 32) | (unsigned)n;
            }
            const int nr = (w.kv_end - w.kv_begin + kSlotKeys - 1) / kSlotKeys;      // real tiles (n may hold a padding tile)
            if (FP8 && w.kind == 1) {
                mbar_wait(BAR(B_QFULL), n_pre & 1);        // every Q phase, also by a chain that sits the item out (exact parity)
                ++n_pre;
            }
            if (w.kind == 1 && wg < w.nheads) {
                // -------------------------- prefill tile, chain wg: thread = query row --------------------------
                if (FP8) {
                    // FP8 cache: the MMAs run on fp16 operands - this chain's Q tile is rewritten in place (same swizzled
                    // positions, bf16 -> fp16: exact for magnitudes in [2^-14, 65504], clamped above) before the first S
                    uint8_t* qt = smem + SM::kQOff + wg * SM::kQTile;
                    for (int i = wtid; i < SM::kQTile / 16; i += 128) {
                        uint4 v = *reinterpret_cast<uint4*>(qt + i * 16);
                        v.x = bf16x2_to_f16x2(v.x); v.y = bf16x2_to_f16x2(v.y); v.z = bf16x2_to_f16x2(v.z); v.w = bf16x2_to_f16x2(v.w);
                        *reinterpret_cast<uint4*>(qt + i * 16) = v;
                    }
                    fence_proxy_async();
                    mbar_arrive(BAR(B_QCONV + wg));
                }
                const float sl2 = sl2_base * (FP8 ? __ldg(prm.k_scale + w.head / G) : 1.f);
                const int u = __ldg(prm.ctx_lens + w.req);
                const int limit = u + w.q_pos0 + row + 1;            // keys [0, limit) visible to this row
                const int limit_w = u + w.q_pos0 + quarter * 32 + 1;  // ... to the first row of this warp (the fewest)
                const int head = w.head + wg;
                float m = -INFINITY, l = 0.f;
#ifdef SS_PROFILE
                long long pf_t = clock64(), pf_acc[4] = {0, 0, 0, 0};     // S wait | tcgen05.ld | softmax | st + fence + arrive
#endif
                for (int kt = 0; kt < nr; ++kt) {
                    const uint32_t sc = s_ctr + kt, tc = tile_ctr + kt;
                    const int b = sc & 1, s = tc % SM::kNumSt;
                    const int key0 = kt * kSlotKeys;
                    const bool tail = key0 + kSlotKeys > w.kv_end;
                    mbar_wait(BAR(B_SFULL + wg * 2 + b), (sc >> 1) & 1);
                    tc_fence_after();
                    if (tail && !FP8) {                          // (FP8: the converter writes zeros for the rows past kv_end)
                        // zero V rows [kv_end - key0, 64): stale / unused-slot bits must not meet P = 0 in the MMA
                        // (both chains write the same zeros; each fences before its own P arrive).  After the S wait:
                        // S(kt) done => this item's Q landed => every earlier tile landed (see B_QEMPTY), so the
                        // V wait below is never a phase early.
                        mbar_wait(BAR(B_VFULL + s), (tc / SM::kNumSt) & 1);
                        const uint32_t vaddr = sbase + SM::kVOff + s * SM::kSlot;
                        const int first = w.kv_end - key0;
                        for (int i = wtid; i < (kSlotKeys - first) * kHalves * 8; i += 128) {
                            const int r = first + i / (kHalves * 8);
                            const int c = i % (kHalves * 8);
                            const uint32_t a = vaddr + SM::kv_off(r, c);
                            asm volatile("st.shared.v4.b32 [%0], {%1,%1,%1,%1};" ::"r"(a), "r"(0u) : "memory");
                        }
                    }
                    if (tr && kt == 0) tr[3] = globaltimer_ns();
                    SS_PF(0)
                    uint32_t sr[2][32];
                    tmem_ld_32x32b_x32(tchain + b * 64 + lane_addr, sr[0]);
                    tmem_ld_32x32b_x32(tchain + b * 64 + lane_addr + 32, sr[1]);
                    tmem_ld_wait();
                    SS_PF(1)
                    uint32_t pk[32];
                    float alpha;
                    if (limit_w - key0 >= kSlotKeys && !tail)       // warp-uniform: every row of this warp sees all 64 keys
                        alpha = softmax_half<false, FP8>(sr, kSlotKeys, sl2, m, l, pk);
                    else
                        alpha = softmax_half<true, FP8>(sr, min(limit, w.kv_end) - key0, sl2, m, l, pk);
                    SS_PF(2)
                    tmem_st_32x32b_x32(tchain + b * 64 + lane_addr, pk);        // P in place over S
                    if (kt > 0 && !__all_sync(0xffffffffu, alpha == 1.f)) {
                        mbar_wait(BAR(B_PVDONE + wg), (sc - 1) & 1);          // PV(kt-1) must have landed in O
                        tc_fence_after();
#pragma unroll
                        for (int c = 0; c < D / 32; ++c) {
                            uint32_t orr[32];
                            tmem_ld_32x32b_x32(tmem_o + lane_addr + c * 32, orr);
                            tmem_ld_wait();
#pragma unroll
                            for (int i = 0; i < 32; ++i) orr[i] = __float_as_uint(__uint_as_float(orr[i]) * alpha);
                            tmem_st_32x32b_x32(tmem_o + lane_addr + c * 32, orr);
                        }
                    }
                    tmem_st_wait();
                    tc_fence_before();
                    if (tail && !FP8) fence_proxy_async();   // zeroed V rows -> visible to the MMA's async proxy
                    mbar_arrive(BAR(B_PFULL + wg * 2 + b));
                    SS_PF(3)
                }
                // ---- epilogue ----
                if (tr) tr[4] = globaltimer_ns();
#ifdef SS_PROFILE
                if (tr) { tr[6] = pf_acc[1]; tr[7] = pf_acc[2]; tr[8] = pf_acc[3]; }
#endif
#ifdef SS_PROFILE
                pf_t = clock64();
#endif
                mbar_wait(BAR(B_OFULL + wg), n_chain & 1);
                tc_fence_after();
#ifdef SS_PROFILE
                if (tr) tr[5] = (unsigned long long)pf_acc[0] | ((unsigned long long)(clock64() - pf_t) << 32);
#endif
                const float inv = (FP8 ? __ldg(prm.v_scale + w.head / G) : 1.f) / l;
                const bool store = row < w.nrows;
                __nv_bfloat16* orow = prm.out + ((int64_t)(w.row0 + row) * Hq + head) * D;
                // thread = row: D fp32 -> D bf16 = 2 D bytes contiguous, written as 32-byte (whole-sector) stores
#pragma unroll
                for (int c = 0; c < D / 64; ++c) {
                    uint32_t orr[2][32];
                    tmem_ld_32x32b_x32(tmem_o + lane_addr + c * 64, orr[0]);
                    tmem_ld_32x32b_x32(tmem_o + lane_addr + c * 64 + 32, orr[1]);
                    tmem_ld_wait();
                    if (store) {
#pragma unroll
                        for (int v = 0; v < 4; ++v) {
                            uint32_t o8[8];
#pragma unroll
                            for (int j = 0; j < 8; ++j) {
                                const int e = v * 16 + 2 * j;
                                o8[j] = pack_bf16(__uint_as_float(orr[e >> 5][e & 31]) * inv, __uint_as_float(orr[e >> 5][(e & 31) + 1]) * inv);
                            }
                            stg_256(orow + c * 64 + v * 16, o8);
                        }
                    }
                }
                if (store && prm.lse) prm.lse[(int64_t)(w.row0 + row) * Hq + head] = (m + log2f(l)) * kMLn2;
                tc_fence_before();
                mbar_arrive(BAR(B_OFREE + wg));
                s_ctr += nr;
                ++n_chain;
            } else if (w.kind == 1) {
                // single-head item: chain B has nothing to do
            } else {
                // -------------------------- decode split: all 8 worker warps --------------------------
                // Warp dw owns 16 keys of every other 64-key slot: warps 0-3 (WG1) the even slots of the item, warps 4-7
                // (WG2) the odd ones.  The products are taken TRANSPOSED, keys on the M = 16 side of mma.sync.m16n8k16
                // and the G query heads of the KV head on the N = 8 side:  S^T = K Q^T  (A = K rows from smem by
                // ldmatrix, B = Q^T from the staged Q rows),  O^T += V^T P^T  (A = V by ldmatrix.trans, B = P^T by
                // movmatrix from the S^T accumulators): half the HMMA count and a quarter of the accumulator registers of
                // padding the heads to M = 16 (64 HMMA per 64-key tile for G <= 8).
                if (G <= 8) decode_item<D, 1, FP8>(w, n, slot, tile_ctr, wg, cw, lane, wtid, sbase, bar0, prm, merge, tr);
                else        decode_item<D, 2, FP8>(w, n, slot, tile_ctr, wg, cw, lane, wtid, sbase, bar0, prm, merge, tr);
            }
            // prefill items: keep B_PARTIAL's per-slot phase count in step (its waiters only look at decode items)
            if (w.kind == 1 && (G <= 8 || wg == 0)) mbar_arrive(BAR(B_PARTIAL + slot));
            tile_ctr += n;
            if (tr) tr[1] = globaltimer_ns();
            __syncwarp();
            if (lane == 0) mbar_arrive(BAR(B_SCHED_EMPTY + slot));
        }
        if (trace && wg == 0 && wtid == 0) { trace[2] = globaltimer_ns(); trace[3] = n_sched - 1; }
    } else if constexpr (FP8) {
        // =============================== fp8 -> fp16 tile converters (FP8 cache only) ===============================
        // The tcgen05 MMAs of a prefill item run on fp16 operands: warps 12, 13 widen every staged K tile, warps 14, 15
        // every V tile, into two K and two V buffers in the bf16 slot layout, each pair at its own pace (K(t) needs
        // S(t-2) of both chains done, V(t) needs PV(t-2)).  A 16-byte chunk of codes becomes two chunks of the fp16
        // tile; rows past kv_end are written as zeros (unused slots may hold NaN codes; 0 * NaN = NaN in the PV
        // product).  Decode items are sat out (their warps widen in registers), so every prefill item starts with its
        // Q phase: once that Q tile has landed, every ring tile issued before it has landed and been released, and the
        // parity waits on the ring are exact again.
        setmaxnreg_dec<MixCta<FP8>::kRegsConv>();
        const int cw = warp - 12;
        const int is_v = cw >> 1;
        const int ct = (cw & 1) * 32 + lane;                                  // 0 .. 63 inside the pair
        const uint32_t ring = sbase + (is_v ? SM::kVOff : SM::kKOff);
        const uint32_t conv = sbase + (is_v ? SM::kVConvOff : SM::kKConvOff);
        const int b_full = is_v ? B_VFULL : B_KFULL, b_empty = is_v ? B_VEMPTY_P : B_KEMPTY_P;
        const int c_full = is_v ? B_VCONV_FULL : B_KCONV_FULL, c_empty = is_v ? B_VCONV_EMPTY : B_KCONV_EMPTY;
        uint32_t tile_ctr = 0, n_sched = 0, cv_ctr = 0, n_pre = 0;
        for (;;) {
            const int slot = n_sched % kSchedSlots;
            mbar_wait(BAR(B_SCHED_FULL + slot), (n_sched / kSchedSlots) & 1);
            const ss_work_item w = sched[slot];
            ++n_sched;
            if (w.kind == 0) break;
            const int nr = (w.kv_end - w.kv_begin + kSlotKeys - 1) / kSlotKeys;      // real tiles
            const int n = (nr + 1) & ~1;                                             // ring tiles (even ring: padded)
            if (w.kind == 1) {
                mbar_wait(BAR(B_QFULL), n_pre & 1);
                ++n_pre;
                for (int t = 0; t < n; ++t) {
                    const uint32_t tc = tile_ctr + t;
                    const int s = tc % SM::kNumSt;
                    mbar_wait(BAR(b_full + s), (tc / SM::kNumSt) & 1);
                    const uint32_t cv = cv_ctr + t, cb = cv & 1;
                    if (t < nr) {
                        mbar_wait(BAR(c_empty + cb), ((cv >> 1) & 1) ^ 1);            // the MMAs that read this buffer are done
                        const int nkeys = w.kv_end - t * kSlotKeys;
                        const uint32_t src = ring + s * SM::kSlot, dst = conv + cb * SM::kConvTile;
#pragma unroll 4
                        for (int q = ct; q < kSlotKeys * 8; q += 64) {
                            const int r = q >> 3, cd = q & 7;
                            uint32_t c0 = 0u, c1 = 0u, c2 = 0u, c3 = 0u;
                            if (r < nkeys)
                                asm volatile("ld.shared.v4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(c0), "=r"(c1), "=r"(c2), "=r"(c3) : "r"(src + SM::kv_off(r, cd)));
                            asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(dst + SM::conv_off(r, 2 * cd)), "r"(e4m3x2_to_f16x2(c0)),
                                         "r"(e4m3x2_hi_to_f16x2(c0)), "r"(e4m3x2_to_f16x2(c1)), "r"(e4m3x2_hi_to_f16x2(c1)) : "memory");
                            asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(dst + SM::conv_off(r, 2 * cd + 1)), "r"(e4m3x2_to_f16x2(c2)),
                                         "r"(e4m3x2_hi_to_f16x2(c2)), "r"(e4m3x2_to_f16x2(c3)), "r"(e4m3x2_hi_to_f16x2(c3)) : "memory");
                        }
                        fence_proxy_async();                                          // generic writes -> the MMA's async proxy
                    }
                    named_bar_sync(4 + is_v, 64);
                    if (ct == 0) {
                        if (t < nr) mbar_arrive(BAR(c_full + cb));
                        mbar_arrive(BAR(b_empty + s));                                // the ring slot is free
                    }
                }
                cv_ctr += nr;
            }
            tile_ctr += n;
            __syncwarp();
            if (lane == 0) mbar_arrive(BAR(B_SCHED_EMPTY + slot));
        }
    }

    // ---- teardown ----
    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        __syncwarp();
        tmem_dealloc(tmem_base, SM::kTmemCols);
    }
}

// Per-call Q tensor map: q viewed as [T rows][Hq*D] bf16, box = 128 rows x 64 columns, 128B swizzle.
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

// The main kernel plans the batch itself when its u16 rank tables can hold it; otherwise the stand-alone work-list
// kernel runs first (ss_mixed_attention asks this before launching).
bool main_self_plans(const Handle* h, int R, int T) {
    if (h->dbg[kDbgTwoKernel] || R > kPlanMaxR) return false;
    const int64_t min_split = h->dbg[kDbgSplitKeys] > 0 ? (h->dbg[kDbgSplitKeys] + kTileKeys - 1) / kTileKeys * kTileKeys : kMinSplitKeys;
    const int64_t max_ctx = (int64_t)h->cfg.max_pages_per_req * kPage;
    if ((max_ctx / min_split + 2) * R > 65535) return false;          // decode split prefix must fit u16
    if ((int64_t)T / kTileRows + R > 65535) return false;              // prefill tile prefix must fit u16
    return true;
}

cudaError_t launch_main_attention(const Handle* h, const void* q, const int32_t* bt, const int32_t* qsl,
                                  const int32_t* ctx, int R, int T, float scale, void* out, float* lse,
                                  void* workspace, cudaStream_t stream, int* n_launches) {
    const ss_config& c = h->cfg;
    char* ws = (char*)workspace;
    CUtensorMap tmap_q;
    if (!encode_q_map(&tmap_q, q, T, c.num_q_heads, c.head_dim)) return cudaErrorInvalidValue;
    MixParams p;
    p.block_table = bt;
    p.ctx_lens = ctx;
    p.hdr = (WorkHeader*)(ws + h->ws.header_off);
    p.items = (const ss_work_item*)(ws + h->ws.items_off);
    p.self_plan = main_self_plans(h, R, T) ? 1 : 0;
    p.merge_counters = p.self_plan ? h->state + kStateCounters : (int32_t*)(ws + h->ws.counters_off);
    p.err_flag = h->debug_checks ? h->state + kStateErr : nullptr;
    p.k_scale = h->k_scale;
    p.v_scale = h->v_scale;
    p.queue = p.self_plan ? h->state : &p.hdr->next_prefill;
    p.qsl = qsl;
    p.R = R;
    p.num_sms = h->num_sms;
    p.force_split_keys = h->dbg[kDbgSplitKeys];
    p.force_decode_ctas = h->dbg[kDbgDecodeCtas];
    p.max_partials = h->ws.max_partials;
    p.partials = (float*)(ws + h->ws.partial_off);
    p.q = (const __nv_bfloat16*)q;
    p.out = (__nv_bfloat16*)out;
    p.lse = lse;
    p.max_pages = c.max_pages_per_req;
    p.Hq = c.num_q_heads;
    p.Hkv = c.num_kv_heads;
    p.scale = scale;
    p.trace = h->trace;
    p.trace_words = h->trace_words;
    *n_launches = 1;
    const int grid = h->dbg[kDbgGrid] > 0 ? h->dbg[kDbgGrid] : h->num_sms;
    cudaError_t e;
    if (h->kv_fp8)
        e = launch_pdl(mixed_kernel<128, true>, dim3(grid), dim3(MixCta<true>::kThreads), MixSmem<128, true>::kTotal, stream, tmap_q, h->tmap_k, h->tmap_v, p);
    else if (c.head_dim == 128)
        e = launch_pdl(mixed_kernel<128, false>, dim3(grid), dim3(MixCta<false>::kThreads), MixSmem<128>::kTotal, stream, tmap_q, h->tmap_k, h->tmap_v, p);
    else
        e = launch_pdl(mixed_kernel<64, false>, dim3(grid), dim3(MixCta<false>::kThreads), MixSmem<64>::kTotal, stream, tmap_q, h->tmap_k, h->tmap_v, p);
    if (e != cudaSuccess) return e;
    return cudaGetLastError();
}

// Opt in to the large dynamic shared-memory window once per process and head_dim (ss_create), not per call.
cudaError_t init_main_attention(int head_dim, int kv_fp8) {
    if (kv_fp8)
        return cudaFuncSetAttribute(mixed_kernel<128, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, MixSmem<128, true>::kTotal);
    if (head_dim == 128)
        return cudaFuncSetAttribute(mixed_kernel<128, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, MixSmem<128>::kTotal);
    return cudaFuncSetAttribute(mixed_kernel<64, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, MixSmem<64>::kTotal);
}

}  // namespace ss
