// cascade_kernel.cu — (f1) chunk-major ("cascade") decode cross-attention.
//
// PICaches are position-independent: a chunk's K/V is the same bytes for every request that links it, in any order
// (§1 "in any order/position"), and retrieval workloads re-use a few hot chunks heavily
// (PAPER.md:297).  So instead of streaming a chunk once per linking request (GEMV-shaped, CUDA cores, up to 99 reads
// of the hottest chunk in BASELINE configs[1]), the batch is inverted at link time and every DISTINCT chunk is
// streamed from HBM once; the query rows of all the requests that link it attend to it together.
//
// Decode has few query rows per chunk (entries x G, mostly 4..32) and many keys, so the contraction is issued with
// the operands swapped: the 128 KEYS of a KV tile are the M dimension of the tcgen05 MMA and the query rows the N
// dimension (16 or 32):
//   S^T[key][row] = K_tile[128 x Dqk] . Q^T          A = K tile (smem, K-major, as TMA wrote the pages), B = Q rows
//   O^T[d][row]  += V_tile^T[Dv x 128] . P^T         A = V tile (smem, MN-major, straight from its page layout), B = P
// One softmax thread owns one KEY (TMEM lane) and the 16/32 rows are its columns: 8x fewer exponentials and TMEM reads
// per tile than a 128-row tile needs, and the per-tile dependency chain is ~500 clk, so the kernel is bound by the
// HBM stream alone.  The row maximum (over keys = across threads) is a CREDUX per row and warp plus one exchange
// through shared memory; the reference maximum only moves when it grows by more than 2^8 (lazy rescale of O^T).
// Work items (tile of entries, KV range of the chunk, kv-head) are handed out through an atomic counter (the tail of a
// static assignment cost 16 % on configs[1]); long chunks are cut into KV ranges when the batch has too few items.
// Each (entry, range, head) gets a normalised fp32 partial row and a log2-domain LSE; cascade_merge_kernel combines a
// request's partials by identity P8:  O = sum_e w_e O_e / sum_e w_e,  w_e = 2^(lse2_e - max),
// LSE = ln 2 (max + log2 sum_e w_e).  One joint softmax over the concatenation, as Eq. 7-8 with PAPER.md:149 demand.
//
// Warp roles (256 threads, one CTA per SM): 0-3 softmax + epilogue (thread = key / output column d), 4 K/V TMA loader,
// 5 tcgen05.mma issuer, 6 scheduler (atomic item fetch) + gather of the items' Q rows, 7 idle.
#include "kernels.h"
#include "ptx.cuh"

#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_fp8.h>
#include <cstring>

namespace comb {
namespace {

constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;
constexpr int kRowsMax = 32;       // query rows (N of the MMA) per item: 16 or 32
constexpr int kItemRing = 3;       // items the scheduler may be ahead

struct CascadeArgs {
    const CascadeItem *items;
    unsigned int *counter;
    int num_items;  // units x kv-heads
    const int32_t *cas_page_indptr, *cas_page_ids, *cas_tile_indptr;
    const uint64_t *cas_tile_ntok;
    const int32_t *cas_row_req, *cas_row_entry;
    const char *q;  // bf16 [R][Hq][Dqk]
    float *part_o, *part_lse;
    int4 *ent_info;
    int num_q_heads, num_kv_heads, group, group_shift;
    int layer_row0;
    float scale_log2;
    // fp8 pools: this layer's scale tables, fp32 [num_pages][Hkv]
    const float *k_scale, *v_scale;
};

struct KvMaps {
    CUtensorMap k, v;
};

// Timeline of CTA 0 of the bf16 chunk-major kernel (profiling aid, compiled only with -DCOMB_TRACE; build.py --trace):
// clock64() per KV tile t of the CTA.  softmax thread 0: [0] before / [1] after the s_full wait, [2] S read, [3] the
// rescale vote done, [4] P buffer free, [5] P handed over.  issuer: [0] before the K / s_empty waits, [1] S issued,
// [2] P seen, [3] P V issued (stamps of tile t - 1's P V are stored under t - 1).
#ifdef COMB_TRACE
__device__ unsigned long long g_trace_cas[2][256][8];
#define COMB_TRC(w, t, k)                                                                              \
    do {                                                                                               \
        if (blockIdx.x == 0 && (threadIdx.x & 31) == 0 && (t) < 256u) g_trace_cas[w][t][k] = clock64(); \
    } while (0)
#else
#define COMB_TRC(w, t, k)
#endif

// what the scheduler hands to the other warps (shared memory)
struct ItemEntry {
    int32_t valid, kvh, nrows, ncols;
    int32_t pbeg, npages, tile0, row0;
    int32_t part0, stride, range_nr, pad;
};
static_assert(sizeof(ItemEntry) == 48, "ItemEntry is copied as three 16-byte words");

template <int DQK, int DV>
struct CasCfg {
    static constexpr int KH = DQK / 64, VH = DV / 64;
    static constexpr int HALF = 128 * 128;               // [128 keys][64 bf16] of a K or V tile
    static constexpr int K_BYTES = KH * HALF, V_BYTES = VH * HALF;
    static constexpr int SLOT = K_BYTES > V_BYTES ? K_BYTES : V_BYTES;
    static constexpr int QH = kRowsMax * 128;             // [32 rows][64 bf16] of a Q or P tile
    static constexpr int Q_BYTES = KH * QH;
    static constexpr int P_BYTES = 2 * QH;                // 32 rows x 128 keys
    static constexpr int MISC = 3072;
    static constexpr int SMEM_MAX = 232448;
    static constexpr int NSLOT_RAW = (SMEM_MAX - 1024 - MISC - 2 * Q_BYTES - P_BYTES) / SLOT;
    static constexpr int NSLOT = NSLOT_RAW > 8 ? 8 : NSLOT_RAW;
    static constexpr int SMEM = 1024 + 2 * Q_BYTES + P_BYTES + NSLOT * SLOT + MISC;
    static constexpr int THREADS = 256;
    static constexpr int TMEM_COLS = 128;                 // S^T x2 @0,32; O^T x2 @64,96
};

struct Misc {
    uint64_t item_full[kItemRing], item_empty[kItemRing];
    uint64_t q_full[2], q_empty[2], s_full[2], s_empty[2], o_full[2], o_empty[2];
    uint64_t p_full, p_empty;
    uint64_t kv_full[8], kv_empty[8];
    uint64_t sc_full[8];  // fp8 kernel: the scales / tile mask of ring entry t & 7 are written
    float wmax[4][kRowsMax];
    float wsum[4][kRowsMax];
    float mref[kRowsMax], inv_l[kRowsMax];
    // fp8 pools: scales of the 8 pages of the last 8 tiles (written by the loader), the items' Q scale, and the warps'
    // largest V scale of a tile
    float kscale[8][8], vscale[8][8], qscale[2], wvs[4];
    unsigned long long tntok[8];  // fp8 kernel: tile_ntok of the last 8 tiles (written by the K loader)
    alignas(16) int32_t srow[2][kRowsMax];
    ItemEntry items[kItemRing];
    uint32_t tmem_slot;
};
static_assert(sizeof(Misc) <= 3072, "Misc must fit its reservation");

__device__ __forceinline__ float warp_max(float x) {
    float y;
    asm volatile("redux.sync.max.f32 %0, %1, 0xffffffff;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ void named_bar_sync(int id, int threads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory");
}
// kind::f16 instruction descriptor, bf16 x bf16 -> fp32, with either operand MN-major
__host__ __device__ constexpr uint32_t idesc_bf16(int m, int n, bool a_mn, bool b_mn) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((a_mn ? 1u : 0u) << 15) | ((b_mn ? 1u : 0u) << 16) |
           ((uint32_t)(n >> 3) << 17) | ((uint32_t)(m >> 4) << 24);
}

// Named barrier over `threads` threads that also ORs a predicate across them (one instruction: no flag in shared
// memory, no vote).
__device__ __forceinline__ bool named_bar_or(int id, int threads, bool pred) {
    uint32_t r;
    asm volatile(
        "{\n\t.reg .pred p, q;\n\tsetp.ne.u32 p, %1, 0;\n\t"
        "bar.red.or.pred q, %2, %3, p;\n\tselp.u32 %0, 1, 0, q;\n\t}"
        : "=r"(r)
        : "r"((uint32_t)pred), "r"(id), "r"(threads)
        : "memory");
    return r != 0;
}

// One stage of a butterfly reduce-scatter over the lanes of a warp: every lane holds 2 CNT values, keeps CNT of them
// (the upper half if its `OFF` bit is set) and adds the partner's copies of those.
template <int CNT, int OFF>
__device__ __forceinline__ void scatter_stage(float *v, int lane) {
    const bool hi = (lane & OFF) != 0;
#pragma unroll
    for (int i = 0; i < CNT; ++i) {
        const float a = v[i], b = v[i + CNT];
        v[i] = (hi ? b : a) + __shfl_xor_sync(0xffffffffu, hi ? a : b, OFF);
    }
}
// v[n] = this lane's value for row n.  Returns the sum over the 32 lanes for row (lane & (NC - 1)).
template <int NC>
__device__ __forceinline__ float warp_row_sums(float (&v)[NC], int lane) {
    if constexpr (NC == 32) {
        scatter_stage<16, 16>(v, lane);
    } else {
#pragma unroll
        for (int i = 0; i < NC; ++i) v[i] += __shfl_xor_sync(0xffffffffu, v[i], 16);
    }
    if constexpr (NC >= 16) {
        scatter_stage<8, 8>(v, lane);
    } else {
#pragma unroll
        for (int i = 0; i < NC; ++i) v[i] += __shfl_xor_sync(0xffffffffu, v[i], 8);
    }
    scatter_stage<4, 4>(v, lane);
    scatter_stage<2, 2>(v, lane);
    scatter_stage<1, 1>(v, lane);
    return v[0];
}

// ---- softmax + epilogue of one item, NC = 16 or 32 query rows (columns of S^T / O^T) ----
// A thread owns one key of the tile.  mc[n] is the reference maximum of row n in the log2 domain (max * scale_log2),
// identical in all 128 threads.  The exact row maxima (CREDUX per warp + an exchange through shared memory) are only
// computed for an item's first tile and when some score exceeds its row's reference by more than 2^8 (one barrier
// with an OR reduction decides that for all 128 threads); otherwise the reference stays and O^T needs no rescale.
template <int DQK, int DV, int NC>
__device__ __forceinline__ void softmax_item(const CascadeArgs &a, Misc *mi, unsigned char *sP, uint32_t tmem,
                                             const ItemEntry &it, const int k, uint32_t &t) {
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t lane_base = (uint32_t)(warp * 32) << 16;
    const int ip = k & 1;
    const int n_kv = (it.npages + kTilePages - 1) / kTilePages;
    const float c = a.scale_log2;
    float mc[NC], l_part[NC];
#pragma unroll
    for (int n = 0; n < NC; ++n) { mc[n] = -INFINITY; l_part[n] = 0.f; }
    // this thread's key inside a tile: page kp, slot ks; where its P goes (row n adds n * 128 and the swizzle)
    const int kp = tid >> 4, ks = tid & 15;
    unsigned char *p_dst = sP + (tid >> 6) * CasCfg<DQK, DV>::QH + (tid & 7) * 2;
    const uint32_t p_unit = (uint32_t)((tid & 63) >> 3);
    for (int j = 0; j < n_kv; ++j, ++t) {
        const uint64_t ntok8 = a.cas_tile_ntok[it.tile0 + j];
        const bool key_valid = ks < (int)((ntok8 >> (8 * kp)) & 0xffu);
        const int sb = t & 1;
        if (warp == 0) COMB_TRC(0, t, 0);
        ptx::mbar_wait(&mi->s_full[sb], (t >> 1) & 1);
        if (warp == 0) COMB_TRC(0, t, 1);
        ptx::tc_fence_after();
        uint32_t r[NC];
#pragma unroll
        for (int q = 0; q < NC / 16; ++q)
            ptx::tmem_ld16(tmem + lane_base + sb * kRowsMax + q * 16, *reinterpret_cast<uint32_t(*)[16]>(&r[q * 16]));
        ptx::tmem_wait_ld();
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(&mi->s_empty[sb]);
        if (warp == 0) COMB_TRC(0, t, 2);
        if (!key_valid) {  // slots past a chunk's length / pages the tile does not have
#pragma unroll
            for (int n = 0; n < NC; ++n) r[n] = 0xff800000u;
        }
        float x[NC];  // exponent of every weight: s * c - mc
        bool exact = j == 0;
        if (j > 0) {
            float over = -INFINITY;
#pragma unroll
            for (int n = 0; n < NC; ++n) {
                x[n] = fmaf(__uint_as_float(r[n]), c, -mc[n]);
                over = fmaxf(over, x[n]);
            }
            exact = named_bar_or(1, 128, over > 8.f);
        }
        if (warp == 0) COMB_TRC(0, t, 3);
        if (exact) {  // the same decision in all 128 threads
            float wm[NC];
#pragma unroll
            for (int n = 0; n < NC; ++n) wm[n] = warp_max(__uint_as_float(r[n]));
            if (lane == 0) {
#pragma unroll
                for (int n = 0; n < NC; n += 4)
                    *reinterpret_cast<float4 *>(&mi->wmax[warp][n]) = make_float4(wm[n], wm[n + 1], wm[n + 2], wm[n + 3]);
            }
            named_bar_sync(1, 128);
#pragma unroll
            for (int n = 0; n < NC; n += 4) {
                const float4 w0 = *reinterpret_cast<const float4 *>(&mi->wmax[0][n]);
                const float4 w1 = *reinterpret_cast<const float4 *>(&mi->wmax[1][n]);
                const float4 w2 = *reinterpret_cast<const float4 *>(&mi->wmax[2][n]);
                const float4 w3 = *reinterpret_cast<const float4 *>(&mi->wmax[3][n]);
                wm[n] = fmaxf(fmaxf(w0.x, w1.x), fmaxf(w2.x, w3.x)) * c;
                wm[n + 1] = fmaxf(fmaxf(w0.y, w1.y), fmaxf(w2.y, w3.y)) * c;
                wm[n + 2] = fmaxf(fmaxf(w0.z, w1.z), fmaxf(w2.z, w3.z)) * c;
                wm[n + 3] = fmaxf(fmaxf(w0.w, w1.w), fmaxf(w2.w, w3.w)) * c;
            }
            // P V_{t-1} has completed: the P tile may be overwritten and O^T is up to date
            ptx::mbar_wait(&mi->p_empty, (t & 1) ^ 1);
            if (j > 0) {  // move the reference of every row that grew, rescale O^T and the partial row sums
                ptx::tc_fence_after();
                uint32_t o[NC];
#pragma unroll
                for (int q = 0; q < NC / 16; ++q)
                    ptx::tmem_ld16(tmem + lane_base + 64 + ip * kRowsMax + q * 16, *reinterpret_cast<uint32_t(*)[16]>(&o[q * 16]));
                ptx::tmem_wait_ld();
#pragma unroll
                for (int n = 0; n < NC; ++n) {
                    const float m_new = fmaxf(mc[n], wm[n]);
                    const float alpha = ptx::ex2(mc[n] - m_new);
                    o[n] = __float_as_uint(__uint_as_float(o[n]) * alpha);
                    l_part[n] *= alpha;
                    mc[n] = m_new;
                }
#pragma unroll
                for (int q = 0; q < NC / 16; ++q)
                    ptx::tmem_st16(tmem + lane_base + 64 + ip * kRowsMax + q * 16, *reinterpret_cast<uint32_t(*)[16]>(&o[q * 16]));
                ptx::tmem_wait_st();
                ptx::tc_fence_before();
            } else {
#pragma unroll
                for (int n = 0; n < NC; ++n) mc[n] = wm[n];
            }
#pragma unroll
            for (int n = 0; n < NC; ++n) x[n] = fmaf(__uint_as_float(r[n]), c, -mc[n]);
        } else {
            ptx::mbar_wait(&mi->p_empty, (t & 1) ^ 1);
        }
        if (warp == 0) COMB_TRC(0, t, 4);
#pragma unroll
        for (int n = 0; n < NC; ++n) {
            const float p = ptx::ex2(x[n]);
            l_part[n] += p;
            *reinterpret_cast<__nv_bfloat16 *>(p_dst + n * 128 + ((p_unit ^ (uint32_t)(n & 7)) << 4)) = __float2bfloat16_rn(p);
        }
        ptx::fence_proxy_async_smem();  // generic-proxy stores -> visible to the tensor core's shared-memory reads
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(&mi->p_full);
        if (warp == 0) COMB_TRC(0, t, 5);
    }
    // ---- epilogue: row sums across the 128 keys, then O^T / l -> fp32 partial rows ----
    const float lsum = warp_row_sums<NC>(l_part, lane);
    if (lane < NC) mi->wsum[warp][lane] = lsum;
    if (tid == 0) {
#pragma unroll
        for (int n = 0; n < NC; n += 4)
            *reinterpret_cast<float4 *>(&mi->mref[n]) = make_float4(mc[n], mc[n + 1], mc[n + 2], mc[n + 3]);
    }
    ptx::mbar_wait(&mi->o_full[ip], (k >> 1) & 1);
    ptx::tc_fence_after();
    uint32_t o[NC];
#pragma unroll
    for (int q = 0; q < NC / 16; ++q)
        ptx::tmem_ld16(tmem + lane_base + 64 + ip * kRowsMax + q * 16, *reinterpret_cast<uint32_t(*)[16]>(&o[q * 16]));
    ptx::tmem_wait_ld();
    ptx::tc_fence_before();
    __syncwarp();
    if (lane == 0) ptx::mbar_arrive(&mi->o_empty[ip]);
    named_bar_sync(1, 128);
    if (tid < NC) {  // thread n finishes row n: 1 / l for the scaling below, and the row's log2-domain LSE
        const float l = (mi->wsum[0][tid] + mi->wsum[1][tid]) + (mi->wsum[2][tid] + mi->wsum[3][tid]);
        mi->inv_l[tid] = 1.f / l;
        const int prow = mi->srow[ip][tid];
        if (prow >= 0) a.part_lse[prow] = mi->mref[tid] + log2f(l);
    }
    named_bar_sync(1, 128);
    if (tid < DV) {
#pragma unroll
        for (int n = 0; n < NC; n += 4) {
            const int4 pr = *reinterpret_cast<const int4 *>(&mi->srow[ip][n]);
            const float4 iv = *reinterpret_cast<const float4 *>(&mi->inv_l[n]);
            if (pr.x >= 0) a.part_o[(size_t)pr.x * DV + tid] = __uint_as_float(o[n]) * iv.x;
            if (pr.y >= 0) a.part_o[(size_t)pr.y * DV + tid] = __uint_as_float(o[n + 1]) * iv.y;
            if (pr.z >= 0) a.part_o[(size_t)pr.z * DV + tid] = __uint_as_float(o[n + 2]) * iv.z;
            if (pr.w >= 0) a.part_o[(size_t)pr.w * DV + tid] = __uint_as_float(o[n + 3]) * iv.w;
        }
    }
}

template <int DQK, int DV>
__global__ void __launch_bounds__(256, 1)
cascade_decode_kernel(const CascadeArgs a, const __grid_constant__ KvMaps maps) {
    using C = CasCfg<DQK, DV>;
    extern __shared__ unsigned char smem_raw[];
    unsigned char *smem = ptx::align_smem_1024(smem_raw);
    unsigned char *sQ = smem;                       // 2 x [KH][32 rows][64]
    unsigned char *sP = sQ + 2 * C::Q_BYTES;        // [2][32 rows][64 keys]
    unsigned char *sKV = sP + C::P_BYTES;           // ring of NSLOT K / V tiles
    Misc *mi = reinterpret_cast<Misc *>(sKV + C::NSLOT * C::SLOT);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (tid == 0) {
        for (int i = 0; i < kItemRing; ++i) {
            ptx::mbar_init(&mi->item_full[i], 1);
            ptx::mbar_init(&mi->item_empty[i], 6);  // loader, issuer, four softmax warps
        }
        for (int i = 0; i < 2; ++i) {
            ptx::mbar_init(&mi->q_full[i], 1);
            ptx::mbar_init(&mi->q_empty[i], 1);
            ptx::mbar_init(&mi->s_full[i], 1);
            ptx::mbar_init(&mi->s_empty[i], 4);
            ptx::mbar_init(&mi->o_full[i], 1);
            ptx::mbar_init(&mi->o_empty[i], 4);
        }
        ptx::mbar_init(&mi->p_full, 4);
        ptx::mbar_init(&mi->p_empty, 1);
        for (int s = 0; s < C::NSLOT; ++s) {
            ptx::mbar_init(&mi->kv_full[s], 1);
            ptx::mbar_init(&mi->kv_empty[s], 1);
        }
        ptx::fence_barrier_init();
        ptx::tma_prefetch_desc(&maps.k);
        ptx::tma_prefetch_desc(&maps.v);
    }
    if (warp == 5) {
        ptx::tmem_alloc(&mi->tmem_slot, C::TMEM_COLS);
        ptx::tmem_relinquish();
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem = mi->tmem_slot;
    const int G = a.group, Hq = a.num_q_heads, Hkv = a.num_kv_heads;

    if (warp < 4) {
        // ===================== softmax + epilogue: thread = key of the tile / output column d =====================
        uint32_t t = 0;
        for (int k = 0;; ++k) {
            const int ir = k % kItemRing;
            ptx::mbar_wait(&mi->item_full[ir], (k / kItemRing) & 1);
            const ItemEntry it = mi->items[ir];
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(&mi->item_empty[ir]);
            if (!it.valid) break;
            if (tid < kRowsMax) {  // where the rows of this item go
                const int e_pos = tid >> a.group_shift, head = tid & (G - 1);
                const bool valid = e_pos < it.nrows;
                mi->srow[k & 1][tid] = valid ? (it.part0 + e_pos) * Hq + it.kvh * G + head : -1;
            }
            // (srow is read after the barrier syncs of the tile loop below)
            if (it.ncols == 16) softmax_item<DQK, DV, 16>(a, mi, sP, tmem, it, k, t);
            else softmax_item<DQK, DV, 32>(a, mi, sP, tmem, it, k, t);
        }
    } else if (warp == 4) {
        // ===================== K/V TMA loader: K_t, then V_{t-1}, through one ring =====================
        uint32_t slot = 0, phase = 0;
        bool have_prev = false;
        int prev_row0 = 0, prev_pages = 0;
        auto issue = [&](bool is_v, int row0, int pages_here) {
            ptx::mbar_wait(&mi->kv_empty[slot], phase ^ 1);
            unsigned char *dst = sKV + slot * C::SLOT;
            if (lane == 0) ptx::mbar_expect_tx(&mi->kv_full[slot], (uint32_t)pages_here * kPage * (is_v ? DV : DQK) * 2);
            __syncwarp();
            if (lane < pages_here) {
                if (!is_v) {
#pragma unroll
                    for (int h = 0; h < C::KH; ++h)
                        ptx::tma_load_2d(dst + h * C::HALF + lane * 2048, &maps.k, h * 64, row0, &mi->kv_full[slot]);
                } else {
#pragma unroll
                    for (int h = 0; h < C::VH; ++h)
                        ptx::tma_load_2d(dst + h * C::HALF + lane * 2048, &maps.v, h * 64, row0, &mi->kv_full[slot]);
                }
            }
            if (++slot == C::NSLOT) { slot = 0; phase ^= 1; }
        };
        for (int k = 0;; ++k) {
            const int ir = k % kItemRing;
            ptx::mbar_wait(&mi->item_full[ir], (k / kItemRing) & 1);
            const ItemEntry it = mi->items[ir];
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(&mi->item_empty[ir]);
            if (!it.valid) break;
            const int n_kv = (it.npages + kTilePages - 1) / kTilePages;
            int ids = 0;
            for (int j = 0; j < n_kv; ++j) {
                if ((j & 3) == 0)  // page ids of the next four tiles, one load
                    ids = (j * kTilePages + lane < it.npages) ? a.cas_page_ids[it.pbeg + j * kTilePages + lane] : 0;
                const int pages_here = min(kTilePages, it.npages - j * kTilePages);
                const int pid = __shfl_sync(0xffffffffu, ids, (j & 3) * kTilePages + (lane & 7));
                const int row0 = a.layer_row0 + (pid * Hkv + it.kvh) * kPage;
                issue(false, row0, pages_here);
                if (have_prev) issue(true, prev_row0, prev_pages);
                prev_row0 = row0;
                prev_pages = pages_here;
                have_prev = true;
            }
            // the item's last V tile follows at once (the issuer runs the last P V before the next item's first S^T)
            if (have_prev) issue(true, prev_row0, prev_pages);
            have_prev = false;
        }
    } else if (warp == 5) {
        // ===================== MMA issuer: inside an item S^T_t is issued before P V_{t-1} =====================
        const bool leader = ptx::elect_one();
        const uint64_t dq0 = ptx::umma_desc_sw128(ptx::smem_u32(sQ), 16, 1024);
        const uint64_t dp0 = ptx::umma_desc_sw128(ptx::smem_u32(sP), 16, 1024);
        const uint64_t dk0 = ptx::umma_desc_sw128(ptx::smem_u32(sKV), 16, 1024);
        const uint64_t dv0 = ptx::umma_desc_sw128(ptx::smem_u32(sKV), C::VH > 1 ? C::HALF : 0, 1024);
        uint32_t slot = 0, phase = 0, t = 0;
        struct Pend { bool on, first, last; int pages, ip, k; uint32_t t, idesc; } pd{false, false, false, 0, 0, 0, 0, 0};
        auto do_pv = [&]() {
            ptx::mbar_wait(&mi->kv_full[slot], phase);
            ptx::mbar_wait(&mi->p_full, pd.t & 1);
            COMB_TRC(1, pd.t, 2);
            if (pd.first) ptx::mbar_wait(&mi->o_empty[pd.ip], ((pd.k >> 1) & 1) ^ 1);
            ptx::tc_fence_after();
            for (int ks = 0; ks < pd.pages; ++ks)  // one k-step of 16 keys per page the tile has
                if (leader)
                    ptx::mma_ss(tmem + 64 + pd.ip * kRowsMax, dv0 + (uint64_t)((slot * C::SLOT + ks * 2048) >> 4),
                                dp0 + (uint64_t)(((ks >> 2) * C::QH + (ks & 3) * 32) >> 4), pd.idesc,
                                (pd.first && ks == 0) ? 0u : 1u);
            COMB_TRC(1, pd.t, 3);
            if (leader) {
                ptx::mma_commit(&mi->p_empty);
                ptx::mma_commit(&mi->kv_empty[slot]);
                if (pd.last) ptx::mma_commit(&mi->o_full[pd.ip]);
            }
            if (++slot == C::NSLOT) { slot = 0; phase ^= 1; }
            pd.on = false;
        };
        for (int k = 0;; ++k) {
            const int ir = k % kItemRing;
            ptx::mbar_wait(&mi->item_full[ir], (k / kItemRing) & 1);
            const ItemEntry it = mi->items[ir];
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(&mi->item_empty[ir]);
            if (!it.valid) break;
            const int ip = k & 1;
            const int n_kv = (it.npages + kTilePages - 1) / kTilePages;
            const uint32_t idesc_s = idesc_bf16(128, it.ncols, false, false);
            const uint32_t idesc_o = idesc_bf16(128, it.ncols, true, false);
            ptx::mbar_wait(&mi->q_full[ip], (k >> 1) & 1);
            for (int j = 0; j < n_kv; ++j, ++t) {
                const int sb = t & 1;
                COMB_TRC(1, t, 0);
                ptx::mbar_wait(&mi->kv_full[slot], phase);
                ptx::mbar_wait(&mi->s_empty[sb], ((t >> 1) & 1) ^ 1);
                ptx::tc_fence_after();
                const uint64_t dk = dk0 + (uint64_t)((slot * C::SLOT) >> 4), dq = dq0 + (uint64_t)((ip * C::Q_BYTES) >> 4);
#pragma unroll
                for (int kk = 0; kk < DQK / 16; ++kk)
                    if (leader)
                        ptx::mma_ss(tmem + sb * kRowsMax, dk + (uint64_t)(((kk / 4) * C::HALF + (kk % 4) * 32) >> 4),
                                    dq + (uint64_t)(((kk / 4) * C::QH + (kk % 4) * 32) >> 4), idesc_s, kk > 0);
                COMB_TRC(1, t, 1);
                if (leader) {
                    ptx::mma_commit(&mi->s_full[sb]);
                    ptx::mma_commit(&mi->kv_empty[slot]);
                    if (j + 1 == n_kv) ptx::mma_commit(&mi->q_empty[ip]);
                }
                if (++slot == C::NSLOT) { slot = 0; phase ^= 1; }
                if (pd.on) do_pv();
                pd = Pend{true, j == 0, j + 1 == n_kv, min(kTilePages, it.npages - j * kTilePages), ip, k, t, idesc_o};
            }
            // the item's last P V is not deferred behind the next item's first S^T: the softmax threads wait for it
            // (o_full) before their epilogue, and cannot start the next item earlier anyway
            if (pd.on) do_pv();
        }
    } else if (warp == 6) {
        // ===================== scheduler + Q gather =====================
        constexpr int UPR = DQK / 8;  // 16-byte units per Q row
        unsigned int idx = 0;
        if (lane == 0) idx = atomicAdd(a.counter, 1u);
        for (int k = 0;; ++k) {
            const int ir = k % kItemRing;
            ptx::mbar_wait(&mi->item_empty[ir], ((k / kItemRing) & 1) ^ 1);
            idx = __shfl_sync(0xffffffffu, idx, 0);
            if (idx >= (unsigned int)a.num_items) {
                if (lane == 0) {
                    mi->items[ir].valid = 0;
                    ptx::mbar_arrive(&mi->item_full[ir]);
                }
                break;
            }
            const int unit = (int)idx / Hkv, kvh = (int)idx - unit * Hkv;
            const CascadeItem ci = a.items[unit];
            // the next item's index is fetched now, so the atomic's round trip runs under this item's Q gather
            if (lane == 0) idx = atomicAdd(a.counter, 1u);
            const int rows_valid = ci.nrows * G;
            const int ncols = rows_valid <= 16 ? 16 : 32;
            if (lane == 0) {
                ItemEntry e;
                e.valid = 1;
                e.kvh = kvh;
                e.nrows = ci.nrows;
                e.ncols = ncols;
                e.pbeg = ci.pbeg;
                e.npages = ci.npages;
                e.tile0 = ci.tile0;
                e.row0 = ci.row0;
                e.part0 = ci.part0;
                e.stride = ci.part_stride;
                e.range_nr = ci.range_nr;
                e.pad = 0;
                mi->items[ir] = e;
                ptx::mbar_arrive(&mi->item_full[ir]);
            }
            // where the merge finds an entry's partials (once per entry: first kv-head, first range); written here so
            // that the dependent load of the entry index is not on the softmax threads' path
            if (lane < ci.nrows && kvh == 0 && (ci.range_nr & 0xff) == 0)
                a.ent_info[a.cas_row_entry[ci.row0 + lane]] = make_int4(ci.part0 + lane, ci.part_stride, ci.range_nr >> 8, 0);
            // ---- Q rows of the item: entry e_pos of the tile, head hh of the kv-head -> row e_pos * G + hh, laid out
            // as the SWIZZLE_128B K-major tile TMA would have written (unit j of row r at unit j ^ (r & 7)); rows up
            // to ncols are zero-filled
            const int req_lane = lane < ci.nrows ? a.cas_row_req[ci.row0 + lane] : 0;
            const int qb = k & 1;
            ptx::mbar_wait(&mi->q_empty[qb], ((k >> 1) & 1) ^ 1);
            unsigned char *dstq = sQ + qb * C::Q_BYTES;
            const int units = ncols * UPR;
            for (int u0 = 0; u0 < units; u0 += 128) {
                uint4 val[4];
                uint32_t dst[4];
#pragma unroll
                for (int x = 0; x < 4; ++x) {
                    const int u = u0 + x * 32 + lane;
                    const int row = u / UPR, j = u - row * UPR;
                    const int e_pos = row >> a.group_shift, hh = row & (G - 1);
                    const int qrow = __shfl_sync(0xffffffffu, req_lane, e_pos & 31);
                    val[x] = make_uint4(0u, 0u, 0u, 0u);
                    dst[x] = 0xffffffffu;
                    if (u < units) {
                        if (row < rows_valid)
                            val[x] = __ldg(reinterpret_cast<const uint4 *>(
                                a.q + (((size_t)qrow * Hq + kvh * G + hh) * DQK) * 2 + (size_t)j * 16));
                        dst[x] = (uint32_t)((j >> 3) * C::QH + row * 128 + (((j & 7) ^ (row & 7)) << 4));
                    }
                }
#pragma unroll
                for (int x = 0; x < 4; ++x)
                    if (dst[x] != 0xffffffffu) *reinterpret_cast<uint4 *>(dstq + dst[x]) = val[x];
            }
            ptx::fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(&mi->q_full[qb]);
        }
    }

    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    if (warp == 5) ptx::tmem_dealloc(tmem, C::TMEM_COLS);
}

// =====================================================================================================================
// fp8 pools (include/comb.h "fp8 pools"; DESIGN.md §2 I31-I33, §4.4): the same kernel over e4m3 pages, Dqk = Dv = 128.
//   K and V codes go to the tensor cores as they are (kind::f8f6f4); a (page, kv-head) block's power-of-two scale is
//   applied by the softmax thread that owns the key: to its score column entries (K) and to its weights (V).
//   Both operands of kind::f8f6f4 must be 8-bit, so the SMALL operands are split into two e4m3 terms each:
//     Q rows   q / qs = hi + lo / 16   (qs: one power-of-two scale per item; lo = e4m3(16 (q / qs - hi)))
//     weights  p vs / vref = hi + lo / 16
//   which keeps 7-8 significant bits on that side (bf16 has 8).  hi and lo are extra COLUMNS of the same MMAs:
//   S^T has 2 N columns (hi | lo), O^T likewise; the thread combines hi + lo / 16 after tcgen05.ld.
//   vref, the reference V scale of the accumulator, is the largest V scale met so far in the item; it moves (with a
//   rescale of O^T) through the same rare path as the reference maximum.
// =====================================================================================================================
struct F8Cfg {
    static constexpr int SLOT = 128 * 128;                  // [128 keys][128 bytes] of a K or V tile
    static constexpr int ROWS = 16;                         // query rows per item (8 or 16): N = 16 / 32 MMA columns
    static constexpr int NSLOT = 4;                         // per CTA; two CTAs share an SM
    static constexpr int Q_BYTES = 2 * ROWS * 128;          // [hi 16 rows | lo 16 rows][128 bytes]
    static constexpr int P_BYTES = 128 * 128;               // [128 keys][hi rows | lo rows, 128-byte pitch]: MN-major B
    static constexpr int MISC = 3072;
    static constexpr int SMEM = 1024 + 2 * Q_BYTES + P_BYTES + NSLOT * SLOT + MISC;
    static constexpr int THREADS = 256;
    static constexpr int TMEM_COLS = 128;                   // S^T x2 @0,32; O^T x2 @64,96 (2 N columns each)
    // Two CTAs per SM (their per-item bubbles — Q split, first loads, epilogue — hide under each other's tiles):
    // 128 registers per thread on average, moved by setmaxnreg: 128 x 168 (softmax) + 128 x 88 (the rest) = 256 x 128
    static constexpr int REG_SOFTMAX = 168, REG_OTHER = 88;
};

__device__ __forceinline__ float pow2_scale_for(float amax) {  // smallest 2^e with amax <= 448 * 2^e, e in [-100, 100]
    if (!(amax > 0.f)) return 1.f;
    const uint32_t bits = __float_as_uint(amax);
    int e = (int)(bits >> 23) - 127 - 8 + ((bits & 0x7fffffu) > 0x600000u ? 1 : 0);
    if ((bits >> 23) == 0) e = -100;
    e = e < -100 ? -100 : (e > 100 ? 100 : e);
    return __uint_as_float((uint32_t)(e + 127) << 23);
}
// two values -> (hi codes, lo codes), each two e4m3 bytes (first value in the low byte): v = hi + lo / 16
__device__ __forceinline__ void split_e4m3x2(float v0, float v1, uint32_t &hi, uint32_t &lo) {
    hi = (uint32_t)__nv_cvt_float2_to_fp8x2(make_float2(v0, v1), __NV_SATFINITE, __NV_E4M3);
    const __half2_raw hr = __nv_cvt_fp8x2_to_halfraw2((__nv_fp8x2_storage_t)hi, __NV_E4M3);
    const float2 b = __half22float2(*reinterpret_cast<const __half2 *>(&hr));
    lo = (uint32_t)__nv_cvt_float2_to_fp8x2(make_float2((v0 - b.x) * 16.f, (v1 - b.y) * 16.f), __NV_SATFINITE, __NV_E4M3);
}

template <int NC>
__device__ __forceinline__ void softmax_item_f8(const CascadeArgs &a, Misc *mi, unsigned char *sP, uint32_t tmem,
                                                const ItemEntry &it, const int k, uint32_t &t) {
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t lane_base = (uint32_t)(warp * 32) << 16;
    const int ip = k & 1;
    const int n_kv = (it.npages + kTilePages - 1) / kTilePages;
    const float c = a.scale_log2;
    float mc[NC], l_part[NC];
#pragma unroll
    for (int n = 0; n < NC; ++n) { mc[n] = -INFINITY; l_part[n] = 0.f; }
    float vref = 0.f, inv_vref = 0.f;  // reference V scale of O^T (identical in all 128 threads) and 1 / vref
    // this thread's key inside a tile: page kp, slot ks; its weights are row `tid` of the P tile (MN-major B operand:
    // the 2 NC codes of a key are contiguous, [hi rows | lo rows], in 16-byte units swizzled by the row)
    const int kp = tid >> 4, ks = tid & 15;
    unsigned char *p_dst = sP + tid * 128;
    const float qs = mi->qscale[ip];
    for (int j = 0; j < n_kv; ++j, ++t) {
        const int sb = t & 1;
        ptx::mbar_wait(&mi->s_full[sb], (t >> 1) & 1);
        ptx::tc_fence_after();
        ptx::mbar_wait(&mi->sc_full[t & 7], (t >> 3) & 1);  // the K loader has written this tile's mask and scales
        const uint64_t ntok8 = mi->tntok[t & 7];
        const bool key_valid = ks < (int)((ntok8 >> (8 * kp)) & 0xffu);
        uint32_t r[2 * NC];
#pragma unroll
        for (int q = 0; q < 2 * NC / 16; ++q)
            ptx::tmem_ld16(tmem + lane_base + sb * 32 + q * 16, *reinterpret_cast<uint32_t(*)[16]>(&r[q * 16]));
        const float ksc = mi->kscale[t & 7][kp], vsc = key_valid ? mi->vscale[t & 7][kp] : 0.f;
        ptx::tmem_wait_ld();
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(&mi->s_empty[sb]);
        // log2-domain scores of this key: (hi + lo / 16) * (K scale * Q scale * scale_log2)
        const float f = ksc * qs * c;
        float y[NC];
#pragma unroll
        for (int n = 0; n < NC; ++n)
            y[n] = key_valid ? fmaf(__uint_as_float(r[NC + n]), 0.0625f, __uint_as_float(r[n])) * f : -INFINITY;
        bool exact = j == 0;
        if (j > 0) {
            float over = -INFINITY;
#pragma unroll
            for (int n = 0; n < NC; ++n) over = fmaxf(over, y[n] - mc[n]);
            exact = named_bar_or(1, 128, over > 8.f || vsc > vref);
        }
        if (exact) {  // the same decision in all 128 threads
            float wm[NC];
#pragma unroll
            for (int n = 0; n < NC; ++n) wm[n] = warp_max(y[n]);
            const float wv = warp_max(vsc);
            if (lane == 0) {
#pragma unroll
                for (int n = 0; n < NC; n += 4)
                    *reinterpret_cast<float4 *>(&mi->wmax[warp][n]) = make_float4(wm[n], wm[n + 1], wm[n + 2], wm[n + 3]);
                mi->wvs[warp] = wv;
            }
            named_bar_sync(1, 128);
#pragma unroll
            for (int n = 0; n < NC; n += 4) {
                const float4 w0 = *reinterpret_cast<const float4 *>(&mi->wmax[0][n]);
                const float4 w1 = *reinterpret_cast<const float4 *>(&mi->wmax[1][n]);
                const float4 w2 = *reinterpret_cast<const float4 *>(&mi->wmax[2][n]);
                const float4 w3 = *reinterpret_cast<const float4 *>(&mi->wmax[3][n]);
                wm[n] = fmaxf(fmaxf(w0.x, w1.x), fmaxf(w2.x, w3.x));
                wm[n + 1] = fmaxf(fmaxf(w0.y, w1.y), fmaxf(w2.y, w3.y));
                wm[n + 2] = fmaxf(fmaxf(w0.z, w1.z), fmaxf(w2.z, w3.z));
                wm[n + 3] = fmaxf(fmaxf(w0.w, w1.w), fmaxf(w2.w, w3.w));
            }
            const float vnew = fmaxf(vref, fmaxf(fmaxf(mi->wvs[0], mi->wvs[1]), fmaxf(mi->wvs[2], mi->wvs[3])));
            ptx::mbar_wait(&mi->p_empty, (t & 1) ^ 1);  // P V_{t-1} has completed
            if (j > 0) {  // move the references, rescale O^T (hi and lo columns) and the partial row sums
                ptx::tc_fence_after();
                const float av = vref / vnew;  // exact: powers of two
                uint32_t o[2 * NC];
#pragma unroll
                for (int q = 0; q < 2 * NC / 16; ++q)
                    ptx::tmem_ld16(tmem + lane_base + 64 + ip * 32 + q * 16, *reinterpret_cast<uint32_t(*)[16]>(&o[q * 16]));
                ptx::tmem_wait_ld();
#pragma unroll
                for (int n = 0; n < NC; ++n) {
                    const float m_new = fmaxf(mc[n], wm[n]);
                    const float alpha = ptx::ex2(mc[n] - m_new);
                    o[n] = __float_as_uint(__uint_as_float(o[n]) * (alpha * av));
                    o[NC + n] = __float_as_uint(__uint_as_float(o[NC + n]) * (alpha * av));
                    l_part[n] *= alpha;
                    mc[n] = m_new;
                }
#pragma unroll
                for (int q = 0; q < 2 * NC / 16; ++q)
                    ptx::tmem_st16(tmem + lane_base + 64 + ip * 32 + q * 16, *reinterpret_cast<uint32_t(*)[16]>(&o[q * 16]));
                ptx::tmem_wait_st();
                ptx::tc_fence_before();
            } else {
#pragma unroll
                for (int n = 0; n < NC; ++n) mc[n] = wm[n];
            }
            vref = vnew;
            inv_vref = 1.f / vnew;
        } else {
            ptx::mbar_wait(&mi->p_empty, (t & 1) ^ 1);
        }
        const float vw = vsc * inv_vref;  // <= 1, exact (0 for a masked key)
        uint32_t ph[NC / 4], pl[NC / 4];  // codes of rows 4 i .. 4 i + 3, hi and lo
#pragma unroll
        for (int n = 0; n < NC; n += 4) {
            const float p0 = ptx::ex2(y[n] - mc[n]), p1 = ptx::ex2(y[n + 1] - mc[n + 1]);
            const float p2 = ptx::ex2(y[n + 2] - mc[n + 2]), p3 = ptx::ex2(y[n + 3] - mc[n + 3]);
            l_part[n] += p0;
            l_part[n + 1] += p1;
            l_part[n + 2] += p2;
            l_part[n + 3] += p3;
            uint32_t h0, l0, h1, l1;
            split_e4m3x2(p0 * vw, p1 * vw, h0, l0);
            split_e4m3x2(p2 * vw, p3 * vw, h1, l1);
            ph[n / 4] = h0 | (h1 << 16);
            pl[n / 4] = l0 | (l1 << 16);
        }
        uint32_t pc[NC / 2];  // the key's 2 NC codes: [hi rows | lo rows]
#pragma unroll
        for (int i = 0; i < NC / 4; ++i) { pc[i] = ph[i]; pc[NC / 4 + i] = pl[i]; }
#pragma unroll
        for (int u = 0; u < NC / 8; ++u)  // 16-byte units, swizzled by the row (= key)
            *reinterpret_cast<uint4 *>(p_dst + ((u ^ (tid & 7)) << 4)) = make_uint4(pc[4 * u], pc[4 * u + 1], pc[4 * u + 2], pc[4 * u + 3]);
        ptx::fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(&mi->p_full);
    }
    // ---- epilogue ----
    const float lsum = warp_row_sums<NC>(l_part, lane);
    if (lane < NC) mi->wsum[warp][lane] = lsum;
    if (tid == 0) {
#pragma unroll
        for (int n = 0; n < NC; n += 4)
            *reinterpret_cast<float4 *>(&mi->mref[n]) = make_float4(mc[n], mc[n + 1], mc[n + 2], mc[n + 3]);
    }
    ptx::mbar_wait(&mi->o_full[ip], (k >> 1) & 1);
    ptx::tc_fence_after();
    uint32_t o[2 * NC];
#pragma unroll
    for (int q = 0; q < 2 * NC / 16; ++q)
        ptx::tmem_ld16(tmem + lane_base + 64 + ip * 32 + q * 16, *reinterpret_cast<uint32_t(*)[16]>(&o[q * 16]));
    ptx::tmem_wait_ld();
    ptx::tc_fence_before();
    __syncwarp();
    if (lane == 0) ptx::mbar_arrive(&mi->o_empty[ip]);
    named_bar_sync(1, 128);
    if (tid < NC) {
        const float l = (mi->wsum[0][tid] + mi->wsum[1][tid]) + (mi->wsum[2][tid] + mi->wsum[3][tid]);
        mi->inv_l[tid] = vref / l;  // the accumulator is in units of vref
        const int prow = mi->srow[ip][tid];
        if (prow >= 0) a.part_lse[prow] = mi->mref[tid] + log2f(l);
    }
    named_bar_sync(1, 128);
#pragma unroll
    for (int n = 0; n < NC; n += 4) {
        const int4 pr = *reinterpret_cast<const int4 *>(&mi->srow[ip][n]);
        const float4 iv = *reinterpret_cast<const float4 *>(&mi->inv_l[n]);
        const int prow[4] = {pr.x, pr.y, pr.z, pr.w};
        const float inv[4] = {iv.x, iv.y, iv.z, iv.w};
#pragma unroll
        for (int e = 0; e < 4; ++e)
            if (prow[e] >= 0)
                a.part_o[(size_t)prow[e] * 128 + tid] =
                    fmaf(__uint_as_float(o[NC + n + e]), 0.0625f, __uint_as_float(o[n + e])) * inv[e];
    }
}

__global__ void __launch_bounds__(256, 2)
cascade_decode_f8_kernel(const CascadeArgs a, const __grid_constant__ KvMaps maps) {
    using C = F8Cfg;
    extern __shared__ unsigned char smem_raw[];
    unsigned char *smem = ptx::align_smem_1024(smem_raw);
    unsigned char *sQ = smem;                       // 2 x [64 rows][128 B]
    unsigned char *sP = sQ + 2 * C::Q_BYTES;        // [64 rows][128 keys]
    unsigned char *sKV = sP + C::P_BYTES;           // ring of NSLOT K / V tiles
    Misc *mi = reinterpret_cast<Misc *>(sKV + C::NSLOT * C::SLOT);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    // A k-step of the P V contraction spans 32 keys = two pages; when a tile has an odd number of pages the second
    // half is whatever the slot held before (weight 0).  Start from zeros so that no byte is ever a NaN code.
    for (int i = tid; i < C::NSLOT * C::SLOT / 16; i += C::THREADS) reinterpret_cast<uint4 *>(sKV)[i] = make_uint4(0, 0, 0, 0);
    ptx::fence_proxy_async_smem();
    if (tid == 0) {
        for (int i = 0; i < kItemRing; ++i) {
            ptx::mbar_init(&mi->item_full[i], 1);
            ptx::mbar_init(&mi->item_empty[i], 7);  // two loaders, issuer, four softmax warps
        }
        for (int i = 0; i < 2; ++i) {
            ptx::mbar_init(&mi->q_full[i], 1);
            ptx::mbar_init(&mi->q_empty[i], 1);
            ptx::mbar_init(&mi->s_full[i], 1);
            ptx::mbar_init(&mi->s_empty[i], 4);
            ptx::mbar_init(&mi->o_full[i], 1);
            ptx::mbar_init(&mi->o_empty[i], 4);
        }
        ptx::mbar_init(&mi->p_full, 4);
        ptx::mbar_init(&mi->p_empty, 1);
        for (int s = 0; s < C::NSLOT; ++s) {
            ptx::mbar_init(&mi->kv_full[s], 1);
            ptx::mbar_init(&mi->kv_empty[s], 1);
        }
        for (int s = 0; s < 8; ++s) ptx::mbar_init(&mi->sc_full[s], 1);
        ptx::fence_barrier_init();
        ptx::tma_prefetch_desc(&maps.k);
        ptx::tma_prefetch_desc(&maps.v);
    }
    if (warp == 5) {
        ptx::tmem_alloc(&mi->tmem_slot, C::TMEM_COLS);
        ptx::tmem_relinquish();
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem = mi->tmem_slot;
    const int G = a.group, Hq = a.num_q_heads, Hkv = a.num_kv_heads;
    if (warp < 4) {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(C::REG_SOFTMAX));
    } else {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(C::REG_OTHER));
    }

    if (warp < 4) {
        // ===================== softmax + epilogue =====================
        uint32_t t = 0;
        for (int k = 0;; ++k) {
            const int ir = k % kItemRing;
            ptx::mbar_wait(&mi->item_full[ir], (k / kItemRing) & 1);
            const ItemEntry it = mi->items[ir];
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(&mi->item_empty[ir]);
            if (!it.valid) break;
            if (tid < kRowsMax) {
                const int e_pos = tid >> a.group_shift, head = tid & (G - 1);
                const bool valid = e_pos < it.nrows;
                mi->srow[k & 1][tid] = valid ? (it.part0 + e_pos) * Hq + it.kvh * G + head : -1;
            }
            ptx::mbar_wait(&mi->q_full[k & 1], (k >> 1) & 1);  // the item's Q scale is written with its Q tile
            if (it.ncols == 8) softmax_item_f8<8>(a, mi, sP, tmem, it, k, t);
            else softmax_item_f8<16>(a, mi, sP, tmem, it, k, t);
        }
    } else if (warp == 4 || warp == 7) {
        // ===================== K/V TMA loaders + page scales =====================
        // Both warps walk the same slot sequence (K_t, then V_{t-1}); warp 4 issues the K tiles and writes the pages'
        // scales, warp 7 issues the V tiles: per byte an fp8 tile needs twice the TMA issues of a bf16 tile, and one
        // issuing warp was 75 % busy.
        const bool mine_v = warp == 7;
        uint32_t slot = 0, phase = 0, tt = 0;
        bool have_prev = false;
        int prev_row0 = 0, prev_pages = 0;
        auto issue = [&](bool is_v, int row0, int pages_here) {
            if (is_v == mine_v) {
                ptx::mbar_wait(&mi->kv_empty[slot], phase ^ 1);
                unsigned char *dst = sKV + slot * C::SLOT;
                if (lane == 0) ptx::mbar_expect_tx(&mi->kv_full[slot], (uint32_t)pages_here * kPage * 128);
                __syncwarp();
                if (lane < pages_here)
                    ptx::tma_load_2d(dst + lane * 2048, is_v ? &maps.v : &maps.k, 0, row0, &mi->kv_full[slot]);
            }
            if (++slot == C::NSLOT) { slot = 0; phase ^= 1; }
        };
        for (int k = 0;; ++k) {
            const int ir = k % kItemRing;
            ptx::mbar_wait(&mi->item_full[ir], (k / kItemRing) & 1);
            const ItemEntry it = mi->items[ir];
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(&mi->item_empty[ir]);
            if (!it.valid) break;
            const int n_kv = (it.npages + kTilePages - 1) / kTilePages;
            int ids = 0;
            float ksc = 1.f, vsc = 0.f;
            unsigned long long nt4 = 0;
            for (int j = 0; j < n_kv; ++j, ++tt) {
                if ((j & 3) == 0) {  // page ids (and, in the K warp, scales and tile masks) of the next four tiles
                    const bool have = j * kTilePages + lane < it.npages;
                    ids = have ? a.cas_page_ids[it.pbeg + j * kTilePages + lane] : 0;
                    if (!mine_v) {
                        if (lane < 4 && j + lane < n_kv) nt4 = a.cas_tile_ntok[it.tile0 + j + lane];
                        ksc = have ? a.k_scale[(size_t)ids * Hkv + it.kvh] : 1.f;
                        vsc = have ? a.v_scale[(size_t)ids * Hkv + it.kvh] : 0.f;
                    }
                }
                const int pages_here = min(kTilePages, it.npages - j * kTilePages);
                const int pid = __shfl_sync(0xffffffffu, ids, (j & 3) * kTilePages + (lane & 7));
                const int row0 = a.layer_row0 + (pid * Hkv + it.kvh) * kPage;
                issue(false, row0, pages_here);
                // The K warp publishes the tile's mask and scales AFTER it has issued the tile's loads (the scale loads
                // depend on the page ids: waiting for them first would put a memory round trip in front of every
                // item's first TMA).  Ring entry tt & 7 was last used by tile tt - 8, consumed long ago (the K/V ring
                // holds at most NSLOT / 2 tiles); the softmax threads wait on sc_full before they read.
                if (!mine_v) {
                    if ((lane >> 3) == (j & 3)) {
                        mi->kscale[tt & 7][lane & 7] = ksc;
                        mi->vscale[tt & 7][lane & 7] = vsc;
                    }
                    if (lane == (j & 3)) mi->tntok[tt & 7] = nt4;
                    __syncwarp();
                    if (lane == 0) ptx::mbar_arrive(&mi->sc_full[tt & 7]);
                }
                if (have_prev) issue(true, prev_row0, prev_pages);
                prev_row0 = row0;
                prev_pages = pages_here;
                have_prev = true;
            }
        }
        if (have_prev) issue(true, prev_row0, prev_pages);
    } else if (warp == 5) {
        // ===================== MMA issuer =====================
        const bool leader = ptx::elect_one();
        const uint64_t dq0 = ptx::umma_desc_sw128(ptx::smem_u32(sQ), 16, 1024);
        const uint64_t dk0 = ptx::umma_desc_sw128(ptx::smem_u32(sKV), 16, 1024);
        const uint64_t dv0 = ptx::umma_desc_sw128(ptx::smem_u32(sKV), 0, 1024);  // MN-major: one 128-byte block along d
        const uint64_t dpm = ptx::umma_desc_sw128(ptx::smem_u32(sP), 0, 1024);   // MN-major: a key's codes along the rows
        uint32_t slot = 0, phase = 0, t = 0;
        struct Pend { bool on, first, last; int pages, ip, k; uint32_t t, idesc; } pd{false, false, false, 0, 0, 0, 0, 0};
        auto do_pv = [&]() {
            ptx::mbar_wait(&mi->kv_full[slot], phase);
            ptx::mbar_wait(&mi->p_full, pd.t & 1);
            if (pd.first) ptx::mbar_wait(&mi->o_empty[pd.ip], ((pd.k >> 1) & 1) ^ 1);
            ptx::tc_fence_after();
            const int ksteps = (pd.pages + 1) >> 1;  // 32 keys (two pages) per k-step
            for (int ks = 0; ks < ksteps; ++ks)
                if (leader)
                    ptx::mma_ss_f8(tmem + 64 + pd.ip * 32, dv0 + (uint64_t)((slot * C::SLOT + ks * 4096) >> 4),
                                   dpm + (uint64_t)((ks * 4096) >> 4), pd.idesc, (pd.first && ks == 0) ? 0u : 1u);
            if (leader) {
                ptx::mma_commit(&mi->p_empty);
                ptx::mma_commit(&mi->kv_empty[slot]);
                if (pd.last) ptx::mma_commit(&mi->o_full[pd.ip]);
            }
            if (++slot == C::NSLOT) { slot = 0; phase ^= 1; }
            pd.on = false;
        };
        for (int k = 0;; ++k) {
            const int ir = k % kItemRing;
            ptx::mbar_wait(&mi->item_full[ir], (k / kItemRing) & 1);
            const ItemEntry it = mi->items[ir];
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(&mi->item_empty[ir]);
            if (!it.valid) break;
            const int ip = k & 1;
            const int n_kv = (it.npages + kTilePages - 1) / kTilePages;
            const uint32_t idesc_s = ptx::umma_idesc_e4m3(128, 2 * it.ncols, false, false);
            const uint32_t idesc_o = ptx::umma_idesc_e4m3(128, 2 * it.ncols, true, true);
            ptx::mbar_wait(&mi->q_full[ip], (k >> 1) & 1);
            for (int j = 0; j < n_kv; ++j, ++t) {
                const int sb = t & 1;
                ptx::mbar_wait(&mi->kv_full[slot], phase);
                ptx::mbar_wait(&mi->s_empty[sb], ((t >> 1) & 1) ^ 1);
                ptx::tc_fence_after();
                const uint64_t dk = dk0 + (uint64_t)((slot * C::SLOT) >> 4), dq = dq0 + (uint64_t)((ip * C::Q_BYTES) >> 4);
#pragma unroll
                for (int kk = 0; kk < 4; ++kk)  // 32 dims per k-step
                    if (leader)
                        ptx::mma_ss_f8(tmem + sb * 32, dk + (uint64_t)((kk * 32) >> 4), dq + (uint64_t)((kk * 32) >> 4),
                                       idesc_s, kk > 0);
                if (leader) {
                    ptx::mma_commit(&mi->s_full[sb]);
                    ptx::mma_commit(&mi->kv_empty[slot]);
                    if (j + 1 == n_kv) ptx::mma_commit(&mi->q_empty[ip]);
                }
                if (++slot == C::NSLOT) { slot = 0; phase ^= 1; }
                if (pd.on) do_pv();
                pd = Pend{true, j == 0, j + 1 == n_kv, min(kTilePages, it.npages - j * kTilePages), ip, k, t, idesc_o};
            }
        }
        if (pd.on) do_pv();
    } else if (warp == 6) {
        // ===================== scheduler + Q gather (rows quantised to hi + lo / 16 with one scale per item) =========
        unsigned int idx = 0;
        if (lane == 0) idx = atomicAdd(a.counter, 1u);
        for (int k = 0;; ++k) {
            const int ir = k % kItemRing;
            ptx::mbar_wait(&mi->item_empty[ir], ((k / kItemRing) & 1) ^ 1);
            idx = __shfl_sync(0xffffffffu, idx, 0);
            if (idx >= (unsigned int)a.num_items) {
                if (lane == 0) {
                    mi->items[ir].valid = 0;
                    ptx::mbar_arrive(&mi->item_full[ir]);
                }
                break;
            }
            const int unit = (int)idx / Hkv, kvh = (int)idx - unit * Hkv;
            const CascadeItem ci = a.items[unit];
            if (lane == 0) idx = atomicAdd(a.counter, 1u);
            const int rows_valid = ci.nrows * G;
            const int ncols = rows_valid <= 8 ? 8 : 16;
            if (lane == 0) {
                ItemEntry e;
                e.valid = 1;
                e.kvh = kvh;
                e.nrows = ci.nrows;
                e.ncols = ncols;
                e.pbeg = ci.pbeg;
                e.npages = ci.npages;
                e.tile0 = ci.tile0;
                e.row0 = ci.row0;
                e.part0 = ci.part0;
                e.stride = ci.part_stride;
                e.range_nr = ci.range_nr;
                e.pad = 0;
                mi->items[ir] = e;
                ptx::mbar_arrive(&mi->item_full[ir]);
            }
            // Q rows: 16 units of 8 bf16 per row; lane holds unit (x * 32 + lane) = row 2 x + (lane >> 4), unit lane & 15
            const int req_lane = lane < ci.nrows ? a.cas_row_req[ci.row0 + lane] : 0;
            // where the merge finds an entry's partials (once per entry: first kv-head, first range)
            if (lane < ci.nrows && kvh == 0 && (ci.range_nr & 0xff) == 0)
                a.ent_info[a.cas_row_entry[ci.row0 + lane]] = make_int4(ci.part0 + lane, ci.part_stride, ci.range_nr >> 8, 0);
            const int qb = k & 1;
            uint4 val[8];
            __nv_bfloat162 am2 = __floats2bfloat162_rn(0.f, 0.f);
#pragma unroll
            for (int x = 0; x < 8; ++x) {
                if (2 * x < ncols) {  // uniform: an item has 8 or 16 row slots
                    const int row = 2 * x + (lane >> 4), j = lane & 15;
                    const int e_pos = row >> a.group_shift, hh = row & (G - 1);
                    const int qrow = __shfl_sync(0xffffffffu, req_lane, e_pos & 31);
                    val[x] = make_uint4(0u, 0u, 0u, 0u);
                    if (row < rows_valid)
                        val[x] = __ldg(reinterpret_cast<const uint4 *>(a.q + (((size_t)qrow * Hq + kvh * G + hh) * 128) * 2 +
                                                                       (size_t)j * 16));
                    const __nv_bfloat162 *h2 = reinterpret_cast<const __nv_bfloat162 *>(&val[x]);
#pragma unroll
                    for (int e = 0; e < 4; ++e) am2 = __hmax2(am2, __habs2(h2[e]));
                }
            }
            float amax = fmaxf(__low2float(am2), __high2float(am2));
            amax = __uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(amax)));
            const float qs = pow2_scale_for(amax), qinv = 1.f / qs;
            ptx::mbar_wait(&mi->q_empty[qb], ((k >> 1) & 1) ^ 1);
            unsigned char *dstq = sQ + qb * F8Cfg::Q_BYTES;
#pragma unroll
            for (int x = 0; x < 8; ++x) {
                const int row = 2 * x + (lane >> 4), j = lane & 15;
                if (2 * x < ncols) {
                    const uint32_t w[4] = {val[x].x, val[x].y, val[x].z, val[x].w};
                    uint32_t hi[4], lo[4];
#pragma unroll
                    for (int e = 0; e < 4; ++e)
                        split_e4m3x2(__uint_as_float(w[e] << 16) * qinv, __uint_as_float(w[e] & 0xffff0000u) * qinv, hi[e], lo[e]);
                    // 8 bytes at byte j * 8 of the row: 16-byte unit j >> 1, half j & 1; SWIZZLE_128B on the unit
                    const uint32_t off_hi = (uint32_t)(row * 128 + ((((j >> 1) ^ (row & 7))) << 4) + (j & 1) * 8);
                    const int rl = ncols + row;
                    const uint32_t off_lo = (uint32_t)(rl * 128 + ((((j >> 1) ^ (rl & 7))) << 4) + (j & 1) * 8);
                    *reinterpret_cast<uint2 *>(dstq + off_hi) = make_uint2(hi[0] | (hi[1] << 16), hi[2] | (hi[3] << 16));
                    *reinterpret_cast<uint2 *>(dstq + off_lo) = make_uint2(lo[0] | (lo[1] << 16), lo[2] | (lo[3] << 16));
                }
            }
            if (lane == 0) mi->qscale[qb] = qs;
            ptx::fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(&mi->q_full[qb]);
        }
    }

    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    if (warp == 5) ptx::tmem_dealloc(tmem, C::TMEM_COLS);
}

// WPR warps per (request, q head) row, 8 warps per CTA; a lane owns DV/32 consecutive output columns.  The row's
// partials (one per (entry, KV range of the entry's chunk), found through ent_info = (first index, stride, count))
// are merged ONLINE by identity P8 — running maximum m, weight sum and weighted row, rescaled when m grows — so the
// LSE and the partial row of an entry are loaded together and four entries are in flight per warp: the dependent
// chain is entry_indptr -> ent_info -> (LSE, row), three round trips to L2 where the partials were just written.
// WPR = 1 when a request links a handful of chunks (cfg 2: 8); requests with many entries (cfg 4: 64, each with
// several KV ranges) deal them to 2, 4 or 8 warps whose (m, sum, row) triples meet in shared memory.
constexpr int kMergeWarps = 8;
template <int DV, int WPR>
__global__ void __launch_bounds__(32 * kMergeWarps) cascade_merge_kernel(const float *__restrict__ part_o,
                                                                         const float *__restrict__ part_lse,
                                                                         const int4 *__restrict__ ent_info,
                                                                         const int32_t *__restrict__ entry_indptr,
                                                                         __nv_bfloat16 *__restrict__ out,
                                                                         float *__restrict__ lse, int Hq, int rows) {
    constexpr int CPL = DV / 32, RPC = kMergeWarps / WPR;  // columns per lane, rows per CTA
    __shared__ float s_acc[WPR > 1 ? kMergeWarps : 1][WPR > 1 ? DV : 1];
    __shared__ float2 s_mw[kMergeWarps];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int sub = warp % WPR;                               // this warp's share of the row's entries
    const int row = blockIdx.x * RPC + warp / WPR;            // (request, head)
    const bool live = row < rows;
    const int r = live ? row / Hq : 0, h = live ? row - r * Hq : 0;
    const int e0 = live ? entry_indptr[r] : 0, e1 = live ? entry_indptr[r + 1] : 0;
    float m = -INFINITY, wsum = 0.f, acc[4] = {0.f, 0.f, 0.f, 0.f};
    auto load_row = [&](size_t prow) {
        const float *po = part_o + prow * DV + lane * CPL;
        if constexpr (CPL == 4) return *reinterpret_cast<const float4 *>(po);
        else { const float2 t = *reinterpret_cast<const float2 *>(po); return make_float4(t.x, t.y, 0.f, 0.f); }
    };
    auto fold = [&](float l2, float w, const float4 v) {  // a partial (weight sum w relative to 2^l2) into the merge
        if (l2 == -INFINITY) return;
        const float mn = fmaxf(m, l2);
        const float sa = ptx::ex2(m - mn), sb = ptx::ex2(l2 - mn);
        m = mn;
        wsum = wsum * sa + sb * w;
        acc[0] = acc[0] * sa + sb * v.x;
        acc[1] = acc[1] * sa + sb * v.y;
        acc[2] = acc[2] * sa + sb * v.z;
        acc[3] = acc[3] * sa + sb * v.w;
    };
    for (int e = e0 + 4 * sub; e < e1; e += 4 * WPR) {
        int4 inf[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) inf[u] = e + u < e1 ? ent_info[e + u] : make_int4(0, 0, 0, 0);
        float l2[4];
        float4 v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {  // the first range of four entries, all loads independent
            const bool ok = inf[u].z > 0;
            const size_t prow = (size_t)inf[u].x * Hq + h;
            l2[u] = ok ? part_lse[prow] : -INFINITY;
            v[u] = ok ? load_row(prow) : make_float4(0.f, 0.f, 0.f, 0.f);
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) fold(l2[u], 1.f, v[u]);
#pragma unroll
        for (int u = 0; u < 4; ++u)  // further KV ranges of a long chunk, two at a time
            for (int s0 = 1; s0 < inf[u].z; s0 += 2) {
                const bool two = s0 + 1 < inf[u].z;
                const size_t pa = (size_t)(inf[u].x + s0 * inf[u].y) * Hq + h;
                const size_t pb = two ? (size_t)(inf[u].x + (s0 + 1) * inf[u].y) * Hq + h : pa;
                const float la = part_lse[pa], lb = two ? part_lse[pb] : -INFINITY;
                const float4 va = load_row(pa), vb = load_row(pb);
                fold(la, 1.f, va);
                fold(lb, 1.f, vb);
            }
    }
    if constexpr (WPR > 1) {  // the row's warps meet: unnormalised rows, (m, sum) pairs
#pragma unroll
        for (int c = 0; c < CPL; ++c) s_acc[warp][lane * CPL + c] = acc[c];
        if (lane == 0) s_mw[warp] = make_float2(m, wsum);
        __syncthreads();
        if (sub != 0) return;
#pragma unroll
        for (int o = 1; o < WPR; ++o) {
            const float2 mw = s_mw[warp + o];
            float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
            v.x = s_acc[warp + o][lane * CPL];
            v.y = s_acc[warp + o][lane * CPL + 1];
            if constexpr (CPL == 4) { v.z = s_acc[warp + o][lane * CPL + 2]; v.w = s_acc[warp + o][lane * CPL + 3]; }
            fold(mw.x, mw.y, v);
        }
    }
    if (!live) return;
    __nv_bfloat16 *orow = out + (size_t)row * DV + lane * CPL;
    if (e0 == e1) {  // no contexts linked (reading I13)
        if constexpr (CPL == 4) *reinterpret_cast<uint2 *>(orow) = make_uint2(0u, 0u);
        else *reinterpret_cast<uint32_t *>(orow) = 0u;
        if (lane == 0 && lse) lse[row] = -INFINITY;
        return;
    }
    const float inv = 1.f / wsum;
    if constexpr (CPL == 4)
        *reinterpret_cast<uint2 *>(orow) = make_uint2(ptx::pack_bf16x2(acc[0] * inv, acc[1] * inv),
                                                      ptx::pack_bf16x2(acc[2] * inv, acc[3] * inv));
    else
        *reinterpret_cast<uint32_t *>(orow) = ptx::pack_bf16x2(acc[0] * inv, acc[1] * inv);
    if (lane == 0 && lse) lse[row] = (m + log2f(wsum)) * kLn2;
}

template <int DV>
void launch_cascade_merge(const CascadeArgs &a, const int32_t *entry_indptr, void *out, float *lse, int Hq, int rows,
                          int64_t num_partials, int num_requests, cudaStream_t stream) {
    const int64_t per_row = num_requests > 0 ? num_partials / num_requests : 0;  // partials an output row merges
#define COMB_MERGE_CASE(W)                                                                                         \
    cascade_merge_kernel<DV, W><<<(rows + kMergeWarps / W - 1) / (kMergeWarps / W), 32 * kMergeWarps, 0, stream>>>( \
        a.part_o, a.part_lse, a.ent_info, entry_indptr, (__nv_bfloat16 *)out, lse, Hq, rows)
    if (per_row <= 16) COMB_MERGE_CASE(1);
    else if (per_row <= 32) COMB_MERGE_CASE(2);
    else if (per_row <= 64) COMB_MERGE_CASE(4);
    else COMB_MERGE_CASE(8);
#undef COMB_MERGE_CASE
}

template <int DQK, int DV>
cudaError_t launch_cascade_t(const CascadeArgs &a, const KvMaps &maps, int num_sms, cudaStream_t st) {
    using C = CasCfg<DQK, DV>;
    static_assert(C::NSLOT >= 3, "the ring needs at least K_t, V_{t-1} and one tile in flight");
    auto kern = cascade_decode_kernel<DQK, DV>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM);
    if (e != cudaSuccess) return e;
    const int grid = a.num_items < num_sms ? a.num_items : num_sms;
    kern<<<grid, C::THREADS, C::SMEM, st>>>(a, maps);
    return cudaGetLastError();
}

}  // namespace

bool cascade_supported(int group, int dqk, int dv) {
    if (group < 1 || group > 16 || (group & (group - 1))) return false;
    return (dqk == 64 || dqk == 128 || dqk == 192) && (dv == 64 || dv == 128);
}

CascadeLayout cascade_layout(size_t num_units, int64_t total_entries, int64_t num_partials, int num_q_heads, int dv) {
    auto up = [](size_t x) { return (x + 255) / 256 * 256; };
    CascadeLayout L;
    L.off_items = kCascadeHeaderBytes;
    L.off_ent = up(L.off_items + (num_units > 0 ? num_units : 1) * sizeof(CascadeItem));
    L.off_part_o = up(L.off_ent + (size_t)(total_entries > 0 ? total_entries : 1) * sizeof(int4));
    L.off_part_lse = up(L.off_part_o + (size_t)num_partials * (size_t)num_q_heads * (size_t)dv * sizeof(float));
    L.bytes = up(L.off_part_lse + (size_t)num_partials * (size_t)num_q_heads * sizeof(float));
    L.num_partials = num_partials;
    return L;
}

cudaError_t launch_decode_cascade(const PoolGeom &g, int layer, const LinkView &lv, const PrefillMaps &pm,
                                  void *workspace, const CascadeLayout &lay, int num_units, int num_requests,
                                  int num_q_heads, const void *q, float scale, void *out, float *lse, int num_sms,
                                  cudaStream_t stream, int *launches, const LaunchHook *hook) {
    if (!workspace) return cudaErrorInvalidValue;
    char *ws = (char *)workspace;
    CascadeArgs a{};
    a.items = (const CascadeItem *)(ws + lay.off_items);
    a.counter = (unsigned int *)ws;
    a.num_items = num_units * g.num_kv_heads;
    a.cas_page_indptr = lv.cas_page_indptr;
    a.cas_page_ids = lv.cas_page_ids;
    a.cas_tile_indptr = lv.cas_tile_indptr;
    a.cas_tile_ntok = lv.cas_tile_ntok;
    a.cas_row_req = lv.cas_row_req;
    a.cas_row_entry = lv.cas_row_entry;
    a.q = (const char *)q;
    a.part_o = (float *)(ws + lay.off_part_o);
    a.part_lse = (float *)(ws + lay.off_part_lse);
    a.ent_info = (int4 *)(ws + lay.off_ent);
    a.num_q_heads = num_q_heads;
    a.num_kv_heads = g.num_kv_heads;
    a.group = num_q_heads / g.num_kv_heads;
    a.group_shift = 0;
    while ((1 << a.group_shift) < a.group) ++a.group_shift;
    a.layer_row0 = layer * g.num_pages * g.num_kv_heads * kPage;
    a.scale_log2 = scale * kLog2e;
    KvMaps maps;
    memcpy(&maps.k, &pm.k, sizeof(CUtensorMap));
    memcpy(&maps.v, &pm.v, sizeof(CUtensorMap));
    cudaError_t e = a.num_items > 0 ? cudaErrorInvalidValue : cudaSuccess;  // every request empty: only the merge runs
    if (hook && a.num_items > 0) hook->begin(hook->ctx, kKernelDecodeCascade, stream);
    if (g.kv_dtype == 1) {  // fp8 pool
        if (g.head_dim_qk != 128 || g.head_dim_v != 128 || !g.k_scale || !g.v_scale) return cudaErrorInvalidValue;
        const size_t blocks = (size_t)g.num_pages * g.num_kv_heads;
        a.k_scale = g.k_scale + (size_t)layer * blocks;
        a.v_scale = g.v_scale + (size_t)layer * blocks;
        if (a.num_items > 0) {
            e = cudaFuncSetAttribute(cascade_decode_f8_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, F8Cfg::SMEM);
            if (e == cudaSuccess) {
                const int grid = a.num_items < 2 * num_sms ? a.num_items : 2 * num_sms;  // two CTAs per SM
                cascade_decode_f8_kernel<<<grid, F8Cfg::THREADS, F8Cfg::SMEM, stream>>>(a, maps);
                e = cudaGetLastError();
            }
        }
    } else {
#define COMB_CASCADE_CASE(DQ, DVV)                                      \
    if (a.num_items > 0 && g.head_dim_qk == DQ && g.head_dim_v == DVV) \
        e = launch_cascade_t<DQ, DVV>(a, maps, num_sms, stream);
    COMB_CASCADE_CASE(128, 128)
    COMB_CASCADE_CASE(64, 64)
    COMB_CASCADE_CASE(192, 128)
    COMB_CASCADE_CASE(128, 64)
    COMB_CASCADE_CASE(64, 128)
    COMB_CASCADE_CASE(192, 64)
#undef COMB_CASCADE_CASE
    }
    if (hook && a.num_items > 0) hook->end(hook->ctx, stream);
    if (e != cudaSuccess) return e;
    *launches += a.num_items > 0 ? 1 : 0;
    const int rows = num_requests * num_q_heads;
    if (hook) hook->begin(hook->ctx, kKernelCascadeMerge, stream);
    if (g.head_dim_v == 128)
        launch_cascade_merge<128>(a, lv.entry_indptr, out, lse, num_q_heads, rows, lay.num_partials, num_requests, stream);
    else
        launch_cascade_merge<64>(a, lv.entry_indptr, out, lse, num_q_heads, rows, lay.num_partials, num_requests, stream);
    if (hook) hook->end(hook->ctx, stream);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    *launches += 1;
    return cudaSuccess;
}

}  // namespace comb

#ifdef COMB_TRACE
// libcomb_trace*.so only: the timeline of the most recent bf16 chunk-major decode launch, 2 x 256 x 8 uint64.
#pragma GCC visibility push(default)
extern "C" int32_t comb_trace_cascade_read(void *out) {
    if (cudaDeviceSynchronize() != cudaSuccess) return -6;
    if (cudaMemcpyFromSymbol(out, comb::g_trace_cas, sizeof(comb::g_trace_cas)) != cudaSuccess) return -6;
    return 0;
}
#pragma GCC visibility pop
#endif
