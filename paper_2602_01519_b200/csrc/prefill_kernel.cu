// prefill_kernel.cu — (a4) prefill cross-attention: a block of a request's query tokens attends, without
// mask, over the request's block-table-linked chunk KV (§4.2 Eq. 7-8: A = softmax(QK^T/sqrt d),
// H = AV; PAPER.md:119 + 149: one joint softmax over the concatenation of the linked chunks; Eq. 12 cost).
//
// Flash-style online softmax; both contractions run on tcgen05 tensor cores with TMEM accumulators:
//   S = Q K^T : A = Q tile (smem, K-major, SWIZZLE_128B), B = K tile (smem, K-major)      -> TMEM fp32 [128][128]
//   O += P V  : A = P (TMEM, bf16, written in place over S), B = V tile (smem, MN-major)  -> TMEM fp32 [128][Dv]
// K/V pages are gathered by block table with 2-D TMA boxes of {64 dims, 16 tokens} straight out of the paged
// arena ([page][Hkv][16][D] is a dense [rows][D] matrix), eight pages forming one 128-key tile.
// GQA: the 128 rows of a Q tile are (128/G tokens) x (G heads of one kv-head), one 3-D TMA box.
// Softmax statistics (running max in the log2 domain, running sum) are fp32 in registers; one thread owns one row.
#include "kernels.h"
#include "ptx.cuh"

#include <cuda.h>
#include <cuda_bf16.h>
#include <cstring>

namespace comb {
namespace {

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
};

struct Maps {
    CUtensorMap q, k, v;
};

// ============================================================================================
// v0: one CTA of 128 threads per work item, everything in sequence (load -> S -> softmax -> PV).
// Correct and simple; it pins descriptors, layouts and masks for the pipelined kernel.
// ============================================================================================
template <int DQK, int DV>
struct V0Cfg {
    static constexpr int KH = DQK / 64;  // 64-wide halves of the head dim (one SWIZZLE_128B row each)
    static constexpr int VH = DV / 64;
    static constexpr int HALF_BYTES = kTileM * 128;  // [128 rows][64 bf16]
    static constexpr int Q_BYTES = KH * HALF_BYTES;
    static constexpr int K_BYTES = KH * HALF_BYTES;
    static constexpr int V_BYTES = VH * HALF_BYTES;
    static constexpr int SMEM = Q_BYTES + K_BYTES + V_BYTES + 1024 /*align*/ + 64 /*barriers*/;
    static constexpr int TMEM_COLS = 256;  // S/P: 0..127, O: 128..128+DV
};

template <int DQK, int DV>
__global__ void __launch_bounds__(128, 1)
prefill_v0_kernel(const PrefillArgs a, const __grid_constant__ Maps maps) {
    using C = V0Cfg<DQK, DV>;
    extern __shared__ unsigned char smem_raw[];
    unsigned char *smem = reinterpret_cast<unsigned char *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    unsigned char *sQ = smem, *sK = sQ + C::Q_BYTES, *sV = sK + C::K_BYTES;
    uint64_t *bar_load = reinterpret_cast<uint64_t *>(sV + C::V_BYTES);
    uint64_t *bar_mma = bar_load + 1;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(bar_load + 2);

    const int tid = threadIdx.x, warp = tid >> 5;
    const PrefillItem it = a.items[blockIdx.x];
    const int G = a.group, Hq = a.num_q_heads;
    const int tok_per_tile = kTileM / G;
    const int pbeg = a.page_indptr[it.request], npages = a.page_indptr[it.request + 1] - pbeg;
    const int ntiles_kv = (npages + kTilePages - 1) / kTilePages;
    const int tile0 = a.tile_indptr[it.request];

    if (tid == 0) {
        ptx::mbar_init(bar_load, 1);
        ptx::mbar_init(bar_mma, 1);
        ptx::fence_barrier_init();
        ptx::tma_prefetch_desc(&maps.q);
        ptx::tma_prefetch_desc(&maps.k);
        ptx::tma_prefetch_desc(&maps.v);
    }
    if (warp == 0) {
        ptx::tmem_alloc(tmem_slot, C::TMEM_COLS);
        ptx::tmem_relinquish();
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const uint32_t lane_base = (uint32_t)(warp * 32) << 16;
    const uint32_t tS = tmem + lane_base, tO = tmem + lane_base + 128;
    uint32_t ph_load = 0, ph_mma = 0;

    constexpr uint32_t idesc_s = ptx::umma_idesc_bf16(kTileM, kTileN, false);
    constexpr uint32_t idesc_o = ptx::umma_idesc_bf16(kTileM, DV, true);

    const int q_tiles = (it.q_rows + tok_per_tile - 1) / tok_per_tile;
    for (int t = 0; t < q_tiles; ++t) {
        const int tok0 = it.q_row0 + t * tok_per_tile;
        const int tok_valid = min(tok_per_tile, it.q_rows - t * tok_per_tile);
        const int row = tid;                       // tile row owned by this thread
        const int tok = tok0 + row / G, head = it.kv_head * G + row % G;
        const bool row_valid = row / G < tok_valid;
        float m_run = -INFINITY, l_run = 0.f;

        for (int j = 0; j < ntiles_kv; ++j) {
            const int pages_here = min(kTilePages, npages - j * kTilePages);
            if (tid == 0) {
                uint32_t bytes = (uint32_t)pages_here * kPage * (DQK + DV) * 2;
                if (j == 0) bytes += C::Q_BYTES;
                ptx::mbar_expect_tx(bar_load, bytes);
                if (j == 0)
                    for (int h = 0; h < C::KH; ++h)
                        ptx::tma_load_3d(sQ + h * C::HALF_BYTES, &maps.q, h * 64, it.kv_head * G, tok0, bar_load);
                for (int p = 0; p < pages_here; ++p) {
                    const int pid = a.page_ids[pbeg + j * kTilePages + p];
                    const int row0 = a.layer_row0 + (pid * a.num_kv_heads + it.kv_head) * kPage;
                    for (int h = 0; h < C::KH; ++h)
                        ptx::tma_load_2d(sK + h * C::HALF_BYTES + p * 2048, &maps.k, h * 64, row0, bar_load);
                    for (int h = 0; h < C::VH; ++h)
                        ptx::tma_load_2d(sV + h * C::HALF_BYTES + p * 2048, &maps.v, h * 64, row0, bar_load);
                }
            }
            ptx::mbar_wait(bar_load, ph_load);
            ph_load ^= 1;
            // ---- S = Q K^T ----
            if (tid == 0) {
                ptx::tc_fence_after();
#pragma unroll
                for (int kk = 0; kk < DQK / 16; ++kk) {
                    const uint32_t off = (kk / 4) * C::HALF_BYTES + (kk % 4) * 32;
                    ptx::mma_ss(tmem, ptx::umma_desc_sw128(ptx::smem_u32(sQ) + off, 16, 1024),
                                ptx::umma_desc_sw128(ptx::smem_u32(sK) + off, 16, 1024), idesc_s, kk > 0);
                }
                ptx::mma_commit(bar_mma);
            }
            ptx::mbar_wait(bar_mma, ph_mma);
            ph_mma ^= 1;
            ptx::tc_fence_after();
            // ---- online softmax on this thread's row ----
            const uint64_t ntok8 = a.tile_ntok[tile0 + j];
            float s[kTileN];
#pragma unroll
            for (int c = 0; c < kTileN / 32; ++c) {
                uint32_t r[32];
                ptx::tmem_ld32(tS + c * 32, r);
                ptx::tmem_wait_ld();
#pragma unroll
                for (int e = 0; e < 32; ++e) s[c * 32 + e] = __uint_as_float(r[e]) * a.scale_log2;
            }
            if (ntok8 != kFullTile) {  // slots past a chunk's length (interior partial pages) and missing pages
#pragma unroll
                for (int c = 0; c < kTileN; ++c) {
                    const int nt = (int)((ntok8 >> (8 * (c / kPage))) & 0xffu);
                    if ((c % kPage) >= nt) s[c] = -INFINITY;
                }
            }
            float mx = m_run;
#pragma unroll
            for (int c = 0; c < kTileN; ++c) mx = fmaxf(mx, s[c]);
            const float alpha = ptx::ex2(m_run - mx);  // first tile: ex2(-inf) = 0
            m_run = mx;
            float sum = 0.f;
#pragma unroll
            for (int c = 0; c < kTileN; ++c) {
                s[c] = ptx::ex2(s[c] - mx);
                sum += s[c];
            }
            l_run = l_run * alpha + sum;
            if (j > 0) {  // rescale the accumulator (always, in v0)
#pragma unroll
                for (int c = 0; c < DV / 32; ++c) {
                    uint32_t r[32];
                    ptx::tmem_ld32(tO + c * 32, r);
                    ptx::tmem_wait_ld();
#pragma unroll
                    for (int e = 0; e < 32; ++e) r[e] = __float_as_uint(__uint_as_float(r[e]) * alpha);
                    ptx::tmem_st32(tO + c * 32, r);
                }
            }
#pragma unroll
            for (int c = 0; c < kTileN / 64; ++c) {  // P as bf16 pairs over the first 64 columns of S
                uint32_t r[32];
#pragma unroll
                for (int e = 0; e < 32; ++e) r[e] = ptx::pack_bf16x2(s[c * 64 + 2 * e], s[c * 64 + 2 * e + 1]);
                ptx::tmem_st32(tS + c * 32, r);
            }
            ptx::tmem_wait_st();
            ptx::tc_fence_before();
            __syncthreads();
            // ---- O += P V : one k-step of 16 keys per page ----
            if (tid == 0) {
                ptx::tc_fence_after();
                for (int ks = 0; ks < pages_here; ++ks)
                    ptx::mma_ts(tmem + 128, tmem + ks * 8,
                                ptx::umma_desc_sw128(ptx::smem_u32(sV) + ks * 2048, C::HALF_BYTES, 1024), idesc_o,
                                (j > 0 || ks > 0) ? 1u : 0u);
                ptx::mma_commit(bar_mma);
            }
            ptx::mbar_wait(bar_mma, ph_mma);
            ph_mma ^= 1;
            ptx::tc_fence_after();
        }

        // ---- epilogue: O / l -> bf16 ----
        __nv_bfloat16 *orow = a.out + ((size_t)tok * Hq + head) * DV;
        if (ntiles_kv == 0) {  // no contexts linked (reading I13): zero contribution, lse = -inf
            if (row_valid) {
                for (int c = 0; c < DV / 8; ++c) reinterpret_cast<uint4 *>(orow)[c] = make_uint4(0, 0, 0, 0);
                if (a.lse) a.lse[(size_t)tok * Hq + head] = -INFINITY;
            }
        } else {
            const float inv = 1.f / l_run;
#pragma unroll
            for (int c = 0; c < DV / 32; ++c) {
                uint32_t r[32];
                ptx::tmem_ld32(tO + c * 32, r);
                ptx::tmem_wait_ld();
                if (row_valid) {
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        uint4 w;
                        w.x = ptx::pack_bf16x2(__uint_as_float(r[8 * e + 0]) * inv, __uint_as_float(r[8 * e + 1]) * inv);
                        w.y = ptx::pack_bf16x2(__uint_as_float(r[8 * e + 2]) * inv, __uint_as_float(r[8 * e + 3]) * inv);
                        w.z = ptx::pack_bf16x2(__uint_as_float(r[8 * e + 4]) * inv, __uint_as_float(r[8 * e + 5]) * inv);
                        w.w = ptx::pack_bf16x2(__uint_as_float(r[8 * e + 6]) * inv, __uint_as_float(r[8 * e + 7]) * inv);
                        reinterpret_cast<uint4 *>(orow)[c * 4 + e] = w;
                    }
                }
            }
            if (row_valid && a.lse) a.lse[(size_t)tok * Hq + head] = (m_run + log2f(l_run)) * kLn2;
        }
        ptx::tc_fence_before();
        __syncthreads();  // the next Q tile reuses smem and TMEM
        ptx::tc_fence_after();
    }

    if (warp == 0) ptx::tmem_dealloc(tmem, C::TMEM_COLS);
}

// ---------------------------------------------------------------- TMA descriptor encoding (host)
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) != cudaSuccess ||
            qres != cudaDriverEntryPointSuccess)
            return nullptr;
        fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}

static_assert(sizeof(CUtensorMap) == sizeof(TensorMapBlob), "CUtensorMap is 128 bytes");

// arena [L][pages][Hkv][16][D] seen as a dense bf16 matrix [rows][D]; box = {64 dims, 16 tokens}
cudaError_t encode_arena_map(void *arena, int64_t rows, int d, TensorMapBlob *out) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return cudaErrorNotSupported;
    const cuuint64_t dims[2] = {(cuuint64_t)d, (cuuint64_t)rows};
    const cuuint64_t strides[1] = {(cuuint64_t)d * 2};
    const cuuint32_t box[2] = {64, (cuuint32_t)kPage};
    const cuuint32_t estr[2] = {1, 1};
    CUresult r = fn(reinterpret_cast<CUtensorMap *>(out), CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, arena, dims, strides, box,
                    estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

template <int DQK, int DV>
cudaError_t launch_v0(const PrefillArgs &a, const Maps &maps, int num_items, cudaStream_t st) {
    using C = V0Cfg<DQK, DV>;
    auto kern = prefill_v0_kernel<DQK, DV>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM);
    if (e != cudaSuccess) return e;
    kern<<<num_items, 128, C::SMEM, st>>>(a, maps);
    return cudaGetLastError();
}

}  // namespace

bool prefill_supported(int group, int dqk, int dv) {
    const bool dims = (dqk == 64 || dqk == 128 || dqk == 192) && (dv == 64 || dv == 128);
    return dims && group >= 1 && group <= 16 && (group & (group - 1)) == 0;
}

cudaError_t prefill_encode_kv_maps(const PoolGeom &g, TensorMapBlob *k_map, TensorMapBlob *v_map) {
    const int64_t rows = (int64_t)g.num_layers * g.num_pages * g.num_kv_heads * kPage;
    if (rows > INT32_MAX) return cudaErrorInvalidValue;
    cudaError_t e = encode_arena_map(g.k_arena, rows, g.head_dim_qk, k_map);
    if (e != cudaSuccess) return e;
    return encode_arena_map(g.v_arena, rows, g.head_dim_v, v_map);
}

// q [total_q][Hq][Dqk]; box = {64 dims, G heads of one kv-head, 128/G tokens} -> tile row = token * G + head
cudaError_t prefill_encode_q_map(const void *q, int64_t total_q, int num_q_heads, int group, int dqk,
                                 TensorMapBlob *q_map) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return cudaErrorNotSupported;
    const cuuint64_t dims[3] = {(cuuint64_t)dqk, (cuuint64_t)num_q_heads, (cuuint64_t)total_q};
    const cuuint64_t strides[2] = {(cuuint64_t)dqk * 2, (cuuint64_t)num_q_heads * dqk * 2};
    const cuuint32_t box[3] = {64, (cuuint32_t)group, (cuuint32_t)(kTileM / group)};
    const cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = fn(reinterpret_cast<CUtensorMap *>(q_map), CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void *>(q),
                    dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                    CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

cudaError_t launch_prefill(const PoolGeom &g, int layer, const LinkView &lv, const PrefillMaps &pm,
                           const PrefillItem *items_dev, int num_items, int num_q_heads, float scale, void *out,
                           float *lse, cudaStream_t stream) {
    PrefillArgs a;
    a.items = items_dev;
    a.page_indptr = lv.page_indptr;
    a.page_ids = lv.page_ids;
    a.tile_indptr = lv.tile_indptr;
    a.tile_ntok = lv.tile_ntok;
    a.out = (__nv_bfloat16 *)out;
    a.lse = lse;
    a.num_q_heads = num_q_heads;
    a.num_kv_heads = g.num_kv_heads;
    a.group = num_q_heads / g.num_kv_heads;
    a.layer_row0 = layer * g.num_pages * g.num_kv_heads * kPage;
    a.scale_log2 = scale * kLog2e;
    Maps maps;
    memcpy(&maps.q, &pm.q, sizeof(CUtensorMap));
    memcpy(&maps.k, &pm.k, sizeof(CUtensorMap));
    memcpy(&maps.v, &pm.v, sizeof(CUtensorMap));
#define COMB_PREFILL_CASE(DQ, DVV) \
    if (g.head_dim_qk == DQ && g.head_dim_v == DVV) return launch_v0<DQ, DVV>(a, maps, num_items, stream);
    COMB_PREFILL_CASE(128, 128)
    COMB_PREFILL_CASE(64, 64)
    COMB_PREFILL_CASE(192, 128)
    COMB_PREFILL_CASE(128, 64)
    COMB_PREFILL_CASE(64, 128)
    COMB_PREFILL_CASE(192, 64)
#undef COMB_PREFILL_CASE
    return cudaErrorInvalidValue;
}

}  // namespace comb
