// attn_core.cuh — the tcgen05 / TMEM / TMA flash-attention core of (a4) prefill cross-attention
// (prefill_kernel.cu; the chunk-major decode has its own swapped-operand kernel in cascade_kernel.cu).
// PAPER.md:112-115 §4.2 Eq. 7-8:
// A = softmax(QK^T/sqrt d) without mask, H = AV; PAPER.md:119 + 149: one joint softmax over the concatenation of the
// linked chunks; Eq. 12 cost.
//
// Flash-style online softmax; both contractions run on tcgen05 tensor cores with TMEM accumulators:
//   S = Q K^T : A = Q tile (smem, K-major, SWIZZLE_128B), B = K tile (smem, K-major)      -> TMEM fp32 [128][128]
//   O += P V  : A = P (TMEM, bf16, written in place over S), B = V tile (smem, MN-major)  -> TMEM fp32 [128][Dv]
// K/V pages are gathered by block table with 2-D TMA boxes of {64 dims, 16 tokens} straight out of the paged
// arena ([page][Hkv][16][D] is a dense [rows][D] matrix), eight pages forming one 128-key tile.
// GQA: the 128 rows of a Q tile are (128/G tokens) x (G heads of one kv-head).
// Softmax statistics (running max in the log2 domain, running sum) are fp32 in registers; one thread owns one row.
//
// MODE selects what an item is and where its rows go:
//   kModeFinal   (request, kv-head, 1-2 Q tiles) over all of the request's KV  -> out / lse
//   kModeRanges  the same over one KV range of the request                       -> fp32 partial rows (merged by LSE)
#pragma once
#include "kernels.h"
#include "ptx.cuh"

#include <cuda.h>
#include <cuda_bf16.h>

namespace comb {
namespace {

enum { kModeFinal = 0, kModeRanges = 1 };

constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;
constexpr int kTileM = 128;  // query rows per tile (= TMEM lanes)
constexpr int kTileN = kTileSlots;  // 128 key slots per tile (8 pages)
constexpr uint64_t kFullTile = 0x1010101010101010ull;  // tile_ntok of eight full pages

struct PrefillArgs {
    const PrefillItem *items;
    const int32_t *page_indptr, *page_ids, *tile_indptr;
    const uint64_t *tile_ntok;
    __nv_bfloat16 *out;  // [sum lq][Hq][Dv]
    float *lse;          // [sum lq][Hq] or null
    int num_q_heads, num_kv_heads, group;
    int layer_row0;      // first arena row of this layer = layer * num_pages * Hkv * 16
    float scale_log2;    // scale * log2(e)
    // KV ranges (items with split >= 0): normalised partial rows and their log2-domain LSE, merged by a second kernel
    float *part_o;       // partial rows in blocks of 128 (range s, tile slot t of an item: PrefillItem::part_base), a block
                         // stored [Dv/4][128 rows][4]: the rows' k-th float4s are contiguous, so a warp (one row per
                         // thread) writes 512 contiguous bytes per store instead of 32 separate lines
    float *part_lse;     // [partial rows]       log2(sum_j 2^(s_j * scale_log2)) over the item's range
    int64_t total_q;
    int nsplit;
};

// Work item `idx` of the launch.
template <int MODE>
__device__ __forceinline__ PrefillItem fetch_item(const PrefillArgs &a, int idx) {
    return a.items[idx];
}

// The slice of a request's tables an item covers: first table entry, number of entries, first tile.
struct ItemKv {
    int pbeg, npages, tile0;
};
// What tile slot t of an item works on: consecutive query rows over the item's KV range.
struct TileView {
    int q_row0, tok_valid;  // first query token row, valid query tokens (<= 0: slot unused)
    int pbeg, npages, tile0;  // KV: first table entry, entries, first tile
    int split;              // -1: final output, else range index of the partial result
};
__device__ __forceinline__ TileView tile_view(const PrefillArgs &a, const PrefillItem &it, int t, int tok_per_tile) {
    const int pb = a.page_indptr[it.request], np = a.page_indptr[it.request + 1] - pb;
    const int skip = min(np, it.kv_tile0 * kTilePages);
    TileView v;
    v.pbeg = pb + skip;
    v.npages = min(np - skip, it.kv_tiles * kTilePages);
    v.tile0 = a.tile_indptr[it.request] + it.kv_tile0;
    v.q_row0 = it.q_row0 + t * tok_per_tile;
    v.tok_valid = it.q_rows - t * tok_per_tile;
    v.split = it.split;
    return v;
}
__device__ __forceinline__ ItemKv item_kv(const PrefillArgs &a, const PrefillItem &it) {
    const int pb = a.page_indptr[it.request], np = a.page_indptr[it.request + 1] - pb;
    ItemKv v;
    const int skip = min(np, it.kv_tile0 * kTilePages);
    v.pbeg = pb + skip;
    v.npages = min(np - skip, it.kv_tiles * kTilePages);
    v.tile0 = a.tile_indptr[it.request] + it.kv_tile0;
    return v;
}

struct Maps {
    CUtensorMap q, k, v;
};

// Timeline of CTA 0 (profiling aid, compiled only into libcomb_trace*.so by `build.py --trace[=1]`, -DCOMB_TRACE=2 or
// 1 = softmax stamps only; the product library has none of it): clock64() stamps of one softmax thread per warpgroup and of the issuing lane, per KV tile.
//   softmax [tile slot][tile #][k]: 0 before / 1 after the s_full wait, 3 row maximum known, 4 / 5 first / second
//                                   hand-over of P;   [1][127][0..3]: kernel entry, set-up done, loop end, exit
//   issuer  [tile slot][tile #][k]: 0 before the wait for the first half of P, 1 / 2 first / second half seen,
//                                   3 P V issued, 5 / 6 before / after the issue of the next S
#ifdef COMB_TRACE
__device__ unsigned long long g_trace_sm[2][128][8];
__device__ unsigned long long g_trace_mma[2][128][8];
__device__ unsigned long long g_trace_cta[1024][4];  // per CTA, %globaltimer (ns): entry, set-up done, loop end, exit
#define COMB_TR_SM(t, seq, k)                                                                                   \
    do {                                                                                                        \
        if (blockIdx.x == 0 && lane == 0 && (warp & 3) == 0 && (seq) < 127u) g_trace_sm[t][seq][k] = clock64(); \
    } while (0)
#if COMB_TRACE >= 2  // the issuer's stamps lengthen the loop by ~10 % (it runs in step with the tensor pipe)
#define COMB_TR_MMA(t, seq, k)                                                                \
    do {                                                                                      \
        if (blockIdx.x == 0 && leader && (seq) < 127u) g_trace_mma[t][seq][k] = clock64();    \
    } while (0)
#else
#define COMB_TR_MMA(t, seq, k)
#endif
#define COMB_TR_CTA(k)                                                                \
    do {                                                                              \
        if (blockIdx.x == 0 && threadIdx.x == 0) g_trace_sm[1][127][k] = clock64();   \
        if (threadIdx.x == 0 && blockIdx.x < 1024) {                                  \
            unsigned long long gt;                                                    \
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(gt));                    \
            g_trace_cta[blockIdx.x][k] = gt;                                          \
        }                                                                             \
    } while (0)
#else
#define COMB_TR_SM(t, seq, k)
#define COMB_TR_MMA(t, seq, k)
#define COMB_TR_CTA(k)
#endif

// ============================================================================================
// Persistent, warp-specialised, two Q tiles in ping-pong per CTA.
//   warps 0-3 : softmax + epilogue of Q tile 0 (one thread per row)      warp 8 : TMA loader (Q tiles, K/V ring)
//   warps 4-7 : softmax + epilogue of Q tile 1                           warp 9 : tcgen05.mma issuer (one lane)
// TMEM (512 columns): S0/P0 @0, S1/P1 @128, O0 @256, O1 @256+DV.  While the softmax warps of one tile work on
// S_j, the tensor pipe runs P V_j and Q K_{j+1}^T of the other tile.  The running max is only advanced when it
// grows by more than 2^8 (lazy rescale), so the accumulator in TMEM is almost never touched by the softmax warps.
// ============================================================================================
// NT = Q tiles per CTA. NT = 2 is the configuration described above (one CTA per SM). NT = 1 is for calls in
// which no request has more than one 128-row tile per kv-head (the paper's regime, < 50 dynamic tokens): a CTA then
// has a single softmax warpgroup, 256 TMEM columns and half the shared memory, so TWO CTAs share an SM and the
// ping-pong happens between CTAs, each with its own K/V stream (inside one CTA a lone tile would leave the tensor
// pipe idle during its softmax).
template <int DQK, int DV, int NT>
struct V1Cfg {
    static constexpr int KH = DQK / 64, VH = DV / 64;
    static constexpr int HALF = kTileM * 128;  // [128 rows][64 bf16]
    static constexpr int Q_BYTES = KH * HALF;
    static constexpr int K_BYTES = KH * HALF, V_BYTES = VH * HALF;
    static constexpr int SLOT = K_BYTES > V_BYTES ? K_BYTES : V_BYTES;  // K and V tiles alternate in one ring
    // 227 KB for a CTA that owns the SM; half of 228 KB less the 1 KB the system reserves per CTA for two per SM.
    // A single-tile CTA whose ring would not get two slots in half an SM (Dqk = 192) takes the whole SM instead
    // and spends the second Q tile's space on a third ring slot.
    static constexpr bool HALF_SM = NT == 1 && (115712 - 1024 - 512 - Q_BYTES) / SLOT >= 2;
    static constexpr int CTAS_PER_SM = HALF_SM ? 2 : 1;
    static constexpr int SMEM_MAX = HALF_SM ? 115712 : 232448;
    static constexpr int NSLOT_RAW = (SMEM_MAX - 1024 - 512 - NT * Q_BYTES) / SLOT;
    static constexpr int NSLOT = NSLOT_RAW > 8 ? 8 : NSLOT_RAW;
    static constexpr bool FITS = NSLOT >= 2;  // at least a K and a V slot
    static constexpr int SMEM = 1024 + NT * Q_BYTES + (FITS ? NSLOT : 2) * SLOT + 512;
    static constexpr int TMEM_COLS = 256 * NT;           // S_t/P_t @ 128 t, O_t @ 128 NT + t DV
    static constexpr int NSW = 4 * NT;                   // softmax warps; then the loader warp, then the issuer warp
    static constexpr int THREADS = 128 * (NT + 1);       // + one warpgroup {loader, MMA issuer, 2 idle warps}
    // register file per CTA = THREADS x the launch-bound count (168 at NT = 2, 128 at NT = 1); setmaxnreg moves it:
    //   NT = 2: 2 x 128 x 208 + 128 x 88 = 384 x 168        NT = 1: 128 x 208 + 128 x 48 = 256 x 128
    static constexpr int REG_SOFTMAX = 208;
    static constexpr int REG_OTHER = NT == 2 ? 88 : 48;
};

__device__ __forceinline__ float fmax3(float a, float b, float c) {
    float d;
    asm("max.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c));
    return d;
}

// CL = 2 (two-tile kernel, whole-KV items only): a thread-block CLUSTER of two CTAs works on two consecutive items that
// share their K/V stream (two Q-tile pairs of one (request, kv-head)).  Each CTA's loader fetches every second page of
// a tile and TMA-multicasts it into BOTH CTAs' ring slots, so a K/V tile crosses L2 -> SM once per cluster instead of
// once per CTA; a ring slot is refilled when both CTAs' MMAs have released it (tcgen05.commit multicast on kv_empty,
// which counts two arrivals).  The two CTAs run the same number of items with the same KV lengths, in lockstep by
// construction of the ring.
template <int DQK, int DV, int MODE, int NT, int CL = 1>
__global__ void __launch_bounds__(V1Cfg<DQK, DV, NT>::THREADS, 3 - NT)  // registers: 168 (NT = 2) or 128 (NT = 1)
attn_core_kernel(const PrefillArgs a, const __grid_constant__ Maps maps, const int num_items) {
    using C = V1Cfg<DQK, DV, NT>;
    extern __shared__ unsigned char smem_raw[];
    unsigned char *smem = ptx::align_smem_1024(smem_raw);
    unsigned char *sQ = smem;                    // [2 tiles][KH][128][64]
    unsigned char *sKV = smem + NT * C::Q_BYTES;  // ring of NSLOT tiles
    uint64_t *bars = reinterpret_cast<uint64_t *>(sKV + C::NSLOT * C::SLOT);
    // p_full is indexed [tile * 2 + half]: P goes to the tensor pipe in two 64-key halves, one barrier each (a parity
    // wait cannot tell phase k from phase k - 2, so a barrier must never have two phases outstanding)
    uint64_t *q_full = bars, *q_empty = bars + 2, *s_full = bars + 4, *p_full = bars + 6, *o_done = bars + 10;
    uint64_t *kv_full = bars + 12, *kv_empty = bars + 12 + C::NSLOT;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(bars + 12 + 2 * C::NSLOT);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    COMB_TR_CTA(0);
    if (tid == 0) {
        for (int t = 0; t < 2; ++t) {
            ptx::mbar_init(&q_full[t], 1);
            ptx::mbar_init(&q_empty[t], 1);
            ptx::mbar_init(&s_full[t], 1);
            ptx::mbar_init(&p_full[t * 2], 128);
            ptx::mbar_init(&p_full[t * 2 + 1], 128);
            ptx::mbar_init(&o_done[t], 1);
        }
        for (int s = 0; s < C::NSLOT; ++s) {
            ptx::mbar_init(&kv_full[s], 1);
            ptx::mbar_init(&kv_empty[s], CL);  // one tcgen05.commit per CTA of the cluster
        }
        ptx::fence_barrier_init();
        ptx::tma_prefetch_desc(&maps.q);
        ptx::tma_prefetch_desc(&maps.k);
        ptx::tma_prefetch_desc(&maps.v);
    }
    if (warp == C::NSW) {
        ptx::tmem_alloc(tmem_slot, C::TMEM_COLS);
        ptx::tmem_relinquish();
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (CL > 1) ptx::cluster_sync();  // the peer's barriers are initialised before anything is multicast into them
    ptx::tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const uint32_t cta_rank = CL > 1 ? ptx::cluster_ctarank() : 0u;
    constexpr uint16_t kClusterMask = (uint16_t)((1u << CL) - 1u);
    COMB_TR_CTA(1);
    const int G = a.group, Hq = a.num_q_heads;
    const int tok_per_tile = kTileM / G;

    // register file: 384 x 168 at launch; the softmax warpgroups take what the third warpgroup gives up
    // (2 x 128 x 208 + 128 x 88 = 384 x 168: asking for more than the CTA owns would block forever)
    if (warp < C::NSW) {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(C::REG_SOFTMAX));
    } else {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(C::REG_OTHER));
    }

    if (warp < C::NSW) {
        // ===================== softmax + epilogue of Q tile t =====================
        const int t = warp >> 2;
        const int row = (warp & 3) * 32 + lane;
        const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
        const uint32_t tS = tmem + lane_base + t * 128;
        const uint32_t tO = tmem + lane_base + 128 * NT + t * DV;
        const int row_tok = row / G, row_head = row % G;
        const float c = a.scale_log2;
        const float2 c2 = make_float2(c, c);
        uint32_t s_cnt = 0, o_cnt = 0;
        for (int idx = blockIdx.x; idx < num_items; idx += gridDim.x) {
            const PrefillItem it = fetch_item<MODE>(a, idx);
            const TileView tv = tile_view(a, it, t, tok_per_tile);
            const int tok_valid = tv.tok_valid;
            if (tok_valid <= 0) continue;  // this item does not use the second tile slot
            const int n_kv = (tv.npages + kTilePages - 1) / kTilePages;
            const int tile0 = tv.tile0;
            const bool row_valid = row_tok < tok_valid;
            const int tok = tv.q_row0 + row_tok, head = it.kv_head * G + row_head;
            __nv_bfloat16 *orow = a.out + ((size_t)tok * Hq + head) * DV;
            if (n_kv == 0) {  // no contexts linked (reading I13): zero contribution, lse = -inf
                if (row_valid && tv.split < 0) {
                    for (int e = 0; e < DV / 8; ++e) reinterpret_cast<uint4 *>(orow)[e] = make_uint4(0, 0, 0, 0);
                    if (a.lse) a.lse[(size_t)tok * Hq + head] = -INFINITY;
                } else if (MODE == kModeRanges && row_valid) {  // an empty KV range: weight zero in the merge
                    const size_t pblk = (size_t)it.part_base + (size_t)tv.split * (2 * kTileM) + t * kTileM;
                    for (int e = 0; e < DV / 4; ++e)
                        reinterpret_cast<float4 *>(a.part_o + pblk * DV)[e * kTileM + row] = make_float4(0.f, 0.f, 0.f, 0.f);
                    a.part_lse[pblk + row] = -INFINITY;
                }
                continue;
            }
            float m_used = -INFINITY, l_run = 0.f;
            for (int j = 0; j < n_kv; ++j) {
                const uint64_t ntok8 = a.tile_ntok[tile0 + j];
                COMB_TR_SM(t, s_cnt, 0);
                ptx::mbar_wait(&s_full[t], s_cnt & 1);
                COMB_TR_SM(t, s_cnt, 1);
                ++s_cnt;
                ptx::tc_fence_after();
                uint32_t r[kTileN];
#pragma unroll
                for (int q = 0; q < kTileN / 32; ++q)
                    ptx::tmem_ld32(tS + q * 32, *reinterpret_cast<uint32_t(*)[32]>(&r[q * 32]));
                ptx::tmem_wait_ld();
                if (ntok8 != kFullTile) {  // interior partial pages / missing pages of the last tile
#pragma unroll
                    for (int e = 0; e < kTileN; ++e) {
                        const int nt = (int)((ntok8 >> (8 * (e / kPage))) & 0xffu);
                        if ((e % kPage) >= nt) r[e] = 0xff800000u;  // -inf
                    }
                }
                float mx4[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
#pragma unroll
                for (int e = 0; e < kTileN; e += 2)
                    mx4[(e >> 1) & 3] = fmax3(mx4[(e >> 1) & 3], __uint_as_float(r[e]), __uint_as_float(r[e + 1]));
                const float m_new = fmaxf(fmax3(mx4[0], mx4[1], mx4[2]), fmaxf(mx4[3], m_used));
                if (j == 0) {
                    m_used = m_new;
                } else if (__any_sync(0xffffffffu, (m_new - m_used) * c > 8.f)) {
                    // rare: move the reference max and rescale this warp's rows of the accumulator
                    // P V_{j-1} has landed: the MMAs of the issuing thread complete in order and s_full was committed
                    // after S_j, which it issued after P V_{j-1}
                    const float alpha = ptx::ex2((m_used - m_new) * c);
                    l_run *= alpha;
                    m_used = m_new;
#pragma unroll
                    for (int q = 0; q < DV / 32; ++q) {
                        uint32_t o[32];
                        ptx::tmem_ld32(tO + q * 32, o);
                        ptx::tmem_wait_ld();
#pragma unroll
                        for (int e = 0; e < 32; ++e) o[e] = __float_as_uint(__uint_as_float(o[e]) * alpha);
                        ptx::tmem_st32(tO + q * 32, o);
                    }
                }
                COMB_TR_SM(t, s_cnt - 1, 3);
                const float neg = -m_used * c;
                const float2 neg2 = make_float2(neg, neg);
                float2 sum4[4] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
#pragma unroll
                for (int half = 0; half < 2; ++half) {
                    // P (bf16, written over S columns this thread has already consumed) is handed over in two 64-key
                    // halves: the tensor pipe runs the first half of P V under the second half's exponentials
#pragma unroll
                    for (int e = half * 64; e < half * 64 + 64; e += 2) {
                        const float2 x = ptx::ffma2(make_float2(__uint_as_float(r[e]), __uint_as_float(r[e + 1])), c2, neg2);
                        const float p0 = ptx::ex2(x.x), p1 = ptx::ex2(x.y);
                        sum4[(e >> 1) & 3] = ptx::fadd2(sum4[(e >> 1) & 3], make_float2(p0, p1));
                        r[e >> 1] = ptx::pack_bf16x2(p0, p1);
                    }
                    ptx::tmem_st32(tS + half * 32, *reinterpret_cast<uint32_t(*)[32]>(&r[half * 32]));
                    ptx::tmem_wait_st();
                    ptx::tc_fence_before();
                    ptx::mbar_arrive(&p_full[t * 2 + half]);
                    COMB_TR_SM(t, s_cnt - 1, 4 + half);
                }
                const float2 sA = ptx::fadd2(sum4[0], sum4[1]), sB = ptx::fadd2(sum4[2], sum4[3]);
                l_run += (sA.x + sA.y) + (sB.x + sB.y);
            }
            // ---- epilogue: O / l -> bf16 (or an fp32 partial row) ----
            ptx::mbar_wait(&o_done[t], o_cnt & 1);  // committed once per item, after its last P V
            ++o_cnt;
            ptx::tc_fence_after();
            const float inv = 1.f / l_run;
            // partial: one KV range of several (compiled in only then)
            const bool partial = MODE == kModeRanges && tv.split >= 0;
            size_t prow = 0;
            if (MODE == kModeRanges && partial) prow = (size_t)it.part_base + (size_t)tv.split * (2 * kTileM) + t * kTileM + row;
#pragma unroll
            for (int q = 0; q < DV / 32; ++q) {
                uint32_t o[32];
                ptx::tmem_ld32(tO + q * 32, o);
                ptx::tmem_wait_ld();
                if (row_valid && !partial) {
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        uint4 w;
                        w.x = ptx::pack_bf16x2(__uint_as_float(o[8 * e + 0]) * inv, __uint_as_float(o[8 * e + 1]) * inv);
                        w.y = ptx::pack_bf16x2(__uint_as_float(o[8 * e + 2]) * inv, __uint_as_float(o[8 * e + 3]) * inv);
                        w.z = ptx::pack_bf16x2(__uint_as_float(o[8 * e + 4]) * inv, __uint_as_float(o[8 * e + 5]) * inv);
                        w.w = ptx::pack_bf16x2(__uint_as_float(o[8 * e + 6]) * inv, __uint_as_float(o[8 * e + 7]) * inv);
                        reinterpret_cast<uint4 *>(orow)[q * 4 + e] = w;
                    }
                } else if (MODE != kModeFinal && row_valid) {  // fp32 partial row for the merge kernel
                    float4 *pblk_o = reinterpret_cast<float4 *>(a.part_o + (prow - row) * DV) + row;
#pragma unroll
                    for (int e = 0; e < 8; ++e)
                        pblk_o[(q * 8 + e) * kTileM] = make_float4(__uint_as_float(o[4 * e + 0]) * inv, __uint_as_float(o[4 * e + 1]) * inv,
                                                __uint_as_float(o[4 * e + 2]) * inv, __uint_as_float(o[4 * e + 3]) * inv);
                }
            }
            if (row_valid) {
                if (partial) a.part_lse[prow] = m_used * c + log2f(l_run);
                else if (a.lse) a.lse[(size_t)tok * Hq + head] = (m_used * c + log2f(l_run)) * kLn2;
            }
            ptx::tc_fence_before();  // our reads of O precede the arrive that lets the next item's P V overwrite it
        }
    } else if (warp == C::NSW) {
        // ===================== TMA loader =====================
        uint32_t slot = 0, phase = 0, qcnt[2] = {0, 0};
        for (int idx = blockIdx.x; idx < num_items; idx += gridDim.x) {
            const PrefillItem it = fetch_item<MODE>(a, idx);
            TileView tv[2];
            int n_kv[2];
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                tv[t] = tile_view(a, it, t, tok_per_tile);
                n_kv[t] = (t < NT && tv[t].tok_valid > 0) ? (tv[t].npages + kTilePages - 1) / kTilePages : 0;
            }
            if (n_kv[0] == 0) continue;
#pragma unroll
            for (int t = 0; t < NT; ++t) {
                if (n_kv[t] == 0) continue;
                ptx::mbar_wait(&q_empty[t], (qcnt[t] & 1) ^ 1);
                ++qcnt[t];
                if (lane == 0) {
                    ptx::mbar_expect_tx(&q_full[t], C::Q_BYTES);
                    for (int h = 0; h < C::KH; ++h)
                        ptx::tma_load_3d(sQ + t * C::Q_BYTES + h * C::HALF, &maps.q, h * 64, it.kv_head * G,
                                         tv[t].q_row0, &q_full[t]);
                }
            }
            // one K (is_v = false) or V tile of tile slot t's stream into the next ring slot
            auto load_tile = [&](int t, int j, bool is_v) {
                const int pages_here = min(kTilePages, tv[t].npages - j * kTilePages);
                int row0 = 0;
                if (lane < pages_here) {
                    const int pid = a.page_ids[tv[t].pbeg + j * kTilePages + lane];
                    row0 = a.layer_row0 + (pid * a.num_kv_heads + it.kv_head) * kPage;
                }
                ptx::mbar_wait(&kv_empty[slot], phase ^ 1);
                unsigned char *dst = sKV + slot * C::SLOT;
                if (lane == 0)
                    ptx::mbar_expect_tx(&kv_full[slot], (uint32_t)pages_here * kPage * (is_v ? DV : DQK) * 2);
                __syncwarp();
                if (CL > 1) {  // this CTA's share of the pages, into both CTAs' slots
                    if (lane < pages_here && (lane % CL) == (int)cta_rank) {
                        const CUtensorMap *m = is_v ? &maps.v : &maps.k;
                        for (int h = 0; h < (is_v ? C::VH : C::KH); ++h)
                            ptx::tma_load_2d_multicast(dst + h * C::HALF + lane * 2048, m, h * 64, row0, &kv_full[slot],
                                                       kClusterMask);
                    }
                } else if (lane < pages_here) {
                    if (!is_v) {
#pragma unroll
                        for (int h = 0; h < C::KH; ++h)
                            ptx::tma_load_2d(dst + h * C::HALF + lane * 2048, &maps.k, h * 64, row0, &kv_full[slot]);
                    } else {
#pragma unroll
                        for (int h = 0; h < C::VH; ++h)
                            ptx::tma_load_2d(dst + h * C::HALF + lane * 2048, &maps.v, h * 64, row0, &kv_full[slot]);
                    }
                }
                if (++slot == C::NSLOT) { slot = 0; phase ^= 1; }
            };
            for (int j = 0; j < n_kv[0]; ++j) {  // both tile slots read the same stream: K_0 V_0 K_1 V_1 ...
                load_tile(0, j, false);
                load_tile(0, j, true);
            }
        }
    } else if (warp == C::NSW + 1) {
        // ===================== MMA issuer =====================
        // The whole warp runs the control flow (so descriptors and barrier addresses stay in uniform registers and
        // no per-instruction waterfall loop is needed); one elected lane issues the tcgen05 instructions.
        const bool leader = ptx::elect_one();
        constexpr uint32_t idesc_s = ptx::umma_idesc_bf16(kTileM, kTileN, false);
        constexpr uint32_t idesc_o = ptx::umma_idesc_bf16(kTileM, DV, true);
        // descriptors advance by adding (byte offset >> 4) to the 14-bit start-address field
        const uint64_t dq0 = ptx::umma_desc_sw128(ptx::smem_u32(sQ), 16, 1024);
        const uint64_t dk0 = ptx::umma_desc_sw128(ptx::smem_u32(sKV), 16, 1024);
        const uint64_t dv0 = ptx::umma_desc_sw128(ptx::smem_u32(sKV), C::HALF, 1024);
        uint32_t slot = 0, phase = 0, qcnt[2] = {0, 0}, pcnt[2] = {0, 0};
        auto release_slot = [&](uint32_t sl) {  // the slot is free when the MMAs issued so far have read it
            if (CL > 1) ptx::mma_commit_multicast(&kv_empty[sl], kClusterMask);
            else ptx::mma_commit(&kv_empty[sl]);
        };
        auto issue_s = [&](int t, uint32_t kslot) {
            const uint64_t dq = dq0 + (uint64_t)((t * C::Q_BYTES) >> 4), dk = dk0 + (uint64_t)((kslot * C::SLOT) >> 4);
#pragma unroll
            for (int kk = 0; kk < DQK / 16; ++kk) {
                const uint64_t off = (uint64_t)(((kk / 4) * C::HALF + (kk % 4) * 32) >> 4);
                if (leader) ptx::mma_ss(tmem + t * 128, dq + off, dk + off, idesc_s, kk > 0);
            }
        };
        for (int idx = blockIdx.x; idx < num_items; idx += gridDim.x) {
            const PrefillItem it = fetch_item<MODE>(a, idx);
            const int npages = item_kv(a, it).npages;
            const int n_kv = (npages + kTilePages - 1) / kTilePages;
            if (n_kv == 0) continue;
            const int nq = it.q_rows > tok_per_tile ? 2 : 1;
            // prologue: S_t = Q_t K_0^T
            uint32_t kslot = slot;
            ptx::mbar_wait(&kv_full[kslot], phase);
            if (++slot == C::NSLOT) { slot = 0; phase ^= 1; }
            for (int t = 0; t < nq; ++t) {
                ptx::mbar_wait(&q_full[t], qcnt[t] & 1);
                ++qcnt[t];
                ptx::tc_fence_after();
                issue_s(t, kslot);
                if (leader) ptx::mma_commit(&s_full[t]);
                if (n_kv == 1) if (leader) ptx::mma_commit(&q_empty[t]);
            }
            if (leader) release_slot(kslot);
            for (int j = 0; j < n_kv; ++j) {
                const int pages_here = min(kTilePages, npages - j * kTilePages);
                const bool more = j + 1 < n_kv;
                const uint32_t vslot = slot;
                ptx::mbar_wait(&kv_full[vslot], phase);
                if (++slot == C::NSLOT) { slot = 0; phase ^= 1; }
                const uint32_t kphase = phase;
                kslot = slot;
                if (more && ++slot == C::NSLOT) { slot = 0; phase ^= 1; }
                for (int t = 0; t < nq; ++t) {
#pragma unroll
                    for (int half = 0; half < 2; ++half) {  // O_t += P_t V_j, one k-step of 16 keys per page
                        if (half == 0) COMB_TR_MMA(t, pcnt[t], 0);
                        ptx::mbar_wait(&p_full[t * 2 + half], pcnt[t] & 1);
                        COMB_TR_MMA(t, pcnt[t], 1 + half);
                        ptx::tc_fence_after();
                        for (int ks = half * 4; ks < min(pages_here, half * 4 + 4); ++ks)
                            if (leader) ptx::mma_ts(tmem + 128 * NT + t * DV, tmem + t * 128 + ks * 8,
                                                    dv0 + (uint64_t)((vslot * C::SLOT + ks * 2048) >> 4), idesc_o,
                                                    (j > 0 || ks > 0) ? 1u : 0u);
                    }
                    COMB_TR_MMA(t, pcnt[t], 3);
                    ++pcnt[t];
                    if (t == nq - 1) if (leader) release_slot(vslot);  // V_j is free once its last P V is done
                    if (!more) if (leader) ptx::mma_commit(&o_done[t]);
                    if (more) {
                        if (t == 0) {
                            ptx::mbar_wait(&kv_full[kslot], kphase);
                            ptx::tc_fence_after();
                        }
                        COMB_TR_MMA(t, pcnt[t] - 1, 5);
                        issue_s(t, kslot);
                        COMB_TR_MMA(t, pcnt[t] - 1, 6);
                        if (leader) ptx::mma_commit(&s_full[t]);
                        if (j + 2 == n_kv) if (leader) ptx::mma_commit(&q_empty[t]);
                    }
                }
                if (more) if (leader) release_slot(kslot);
            }
        }
    }

    COMB_TR_CTA(2);
    ptx::tc_fence_before();
    __syncthreads();
    if (CL > 1) ptx::cluster_sync();  // no CTA leaves while its peer may still write into its ring or barriers
    ptx::tc_fence_after();
    if (warp == C::NSW) ptx::tmem_dealloc(tmem, C::TMEM_COLS);
    COMB_TR_CTA(3);
}

}  // namespace
}  // namespace comb
