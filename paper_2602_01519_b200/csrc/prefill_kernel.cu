// prefill_kernel.cu — (a4) prefill cross-attention: a block of a request's query tokens attends, without
// mask, over the request's block-table-linked chunk KV (§4.2 Eq. 7-8; PAPER.md:119 + 149: one
// joint softmax over the concatenation of the linked chunks; Eq. 12 cost).  The tcgen05 kernel itself is
// attn_core.cuh (modes kModeFinal / kModeRanges); here are the KV-range merge kernel, the TMA descriptor encoding
// and the launchers.
#include "attn_core.cuh"

#include <cstring>

namespace comb {
namespace {

// ============================================================================================
// Merge of KV ranges (SURVEY.md §8(c) pin P8): for the rows of every item with split == 0,
//   out = sum_s w_s O_s / sum_s w_s,  w_s = 2^(lse2_s - max_s lse2_s),  lse = ln 2 * (max + log2 sum_s w_s).
// Grid (item, row group): items with split != 0 return at once; a warp merges one row, a lane owns DV/32 columns.
// Every load of a row is independent of the others (all ranges' LSEs first, then all partial rows), so a row costs
// about two memory round trips.
// ============================================================================================
template <int DV>
__global__ void __launch_bounds__(128) prefill_merge_kernel(const PrefillArgs a, const int num_items) {
    const PrefillItem it = a.items[blockIdx.x];
    if (it.split != 0) return;
    const int G = a.group, Hq = a.num_q_heads;
    const int np = a.page_indptr[it.request + 1] - a.page_indptr[it.request];
    const int n_kv = (np + kTilePages - 1) / kTilePages;
    const int nsp = (n_kv + it.tps - 1) / it.tps;  // ranges of this request
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    constexpr int CPL = DV / 32;  // columns per lane (2 or 4)
    constexpr int kMaxSplits = kPrefillMaxSplits;
    const int row = blockIdx.y * 4 + warp;
    if (row < it.q_rows * G && nsp <= kMaxSplits) {
        const int tok = it.q_row0 + row / G, head = it.kv_head * G + row % G;
        const size_t r0 = (size_t)tok * Hq + head;                  // output row
        const size_t p0 = (size_t)it.part_base + (size_t)row;       // partial row of range 0 (row = t * 128 + tile row)
        constexpr size_t stride = 2 * kTileM;                       // partial rows per range
        float l2[kMaxSplits], m = -INFINITY;
#pragma unroll
        for (int s = 0; s < kMaxSplits; ++s) l2[s] = s < nsp ? a.part_lse[p0 + s * stride] : -INFINITY;
#pragma unroll
        for (int s = 0; s < kMaxSplits; ++s) m = fmaxf(m, l2[s]);
        float acc[CPL];
#pragma unroll
        for (int e = 0; e < CPL; ++e) acc[e] = 0.f;
        float wsum = 0.f;
#pragma unroll 4
        for (int s = 0; s < nsp; ++s) {
            const float w = ptx::ex2(l2[s] - m);
            wsum += w;
            // block layout [Dv/4][128 rows][4] (attn_core.cuh): this lane's CPL columns of tile row `row % 128`
            const float *po = a.part_o + (p0 - (size_t)(row % kTileM) + s * stride) * DV +
                              ((size_t)((lane * CPL) / 4) * kTileM + (size_t)(row % kTileM)) * 4 + (lane * CPL) % 4;
            if constexpr (CPL == 4) {
                const float4 v = *reinterpret_cast<const float4 *>(po);
                acc[0] += w * v.x; acc[1] += w * v.y; acc[2] += w * v.z; acc[3] += w * v.w;
            } else {
                const float2 v = *reinterpret_cast<const float2 *>(po);
                acc[0] += w * v.x; acc[1] += w * v.y;
            }
        }
        const float inv = 1.f / wsum;
        __nv_bfloat16 *orow = a.out + r0 * DV + lane * CPL;
#pragma unroll
        for (int e = 0; e < CPL; e += 2)
            *reinterpret_cast<uint32_t *>(orow + e) = ptx::pack_bf16x2(acc[e] * inv, acc[e + 1] * inv);
        if (lane == 0 && a.lse) a.lse[r0] = (m + log2f(wsum)) * kLn2;
    }
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

}  // namespace

// Dense row-major bf16 matrix [outer][inner] (row pitch given in bytes) -> 2-D tiled map, SWIZZLE_128B boxes.
cudaError_t encode_tma_2d_bf16(const void *base, uint64_t inner, uint64_t outer, uint64_t row_pitch_bytes,
                               uint32_t box_inner, uint32_t box_outer, TensorMapBlob *out) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return cudaErrorNotSupported;
    const cuuint64_t dims[2] = {(cuuint64_t)inner, (cuuint64_t)outer};
    const cuuint64_t strides[1] = {(cuuint64_t)row_pitch_bytes};
    const cuuint32_t box[2] = {box_inner, box_outer};
    const cuuint32_t estr[2] = {1, 1};
    CUresult r = fn(reinterpret_cast<CUtensorMap *>(out), CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void *>(base),
                    dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                    CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

// Dense row-major byte matrix [outer][inner bytes] -> 2-D tiled map of uint8, SWIZZLE_128B boxes (box_inner <= 128).
cudaError_t encode_tma_2d_u8(const void *base, uint64_t inner, uint64_t outer, uint64_t row_pitch_bytes,
                             uint32_t box_inner, uint32_t box_outer, TensorMapBlob *out) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return cudaErrorNotSupported;
    const cuuint64_t dims[2] = {(cuuint64_t)inner, (cuuint64_t)outer};
    const cuuint64_t strides[1] = {(cuuint64_t)row_pitch_bytes};
    const cuuint32_t box[2] = {box_inner, box_outer};
    const cuuint32_t estr[2] = {1, 1};
    CUresult r = fn(reinterpret_cast<CUtensorMap *>(out), CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<void *>(base),
                    dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                    CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

namespace {

// arena [L][pages][Hkv][16][D] seen as a dense bf16 matrix [rows][D]; box = {64 dims, 16 tokens}
// (fp8 pools: a byte matrix [rows][D], box = {128 bytes, 16 tokens})
cudaError_t encode_arena_map(void *arena, int64_t rows, int d, bool fp8, TensorMapBlob *out) {
    if (fp8) return encode_tma_2d_u8(arena, (uint64_t)d, (uint64_t)rows, (uint64_t)d, 128, (uint32_t)kPage, out);
    return encode_tma_2d_bf16(arena, (uint64_t)d, (uint64_t)rows, (uint64_t)d * 2, 64, (uint32_t)kPage, out);
}

// Two-tile kernel on clusters of two CTAs (attn_core.cuh, CL = 2): consecutive items (2i, 2i + 1) share their K/V
// stream.  cudaErrorNotSupported = the device cannot keep a cluster on every pair of SMs; the caller then takes the
// plain launch.
template <int DQK, int DV>
cudaError_t launch_v1_clusters(const PrefillArgs &a, const Maps &maps, int num_items, int num_sms, cudaStream_t st) {
    using C = V1Cfg<DQK, DV, 2>;
    if constexpr (!C::FITS) {
        return cudaErrorNotSupported;
    } else {
        auto kern = attn_core_kernel<DQK, DV, kModeFinal, 2, 2>;
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM);
        if (e != cudaSuccess) return e;
        const int pairs = num_items / 2, want = pairs < num_sms / 2 ? pairs : num_sms / 2;
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3(2 * (unsigned)want, 1, 1);
        cfg.blockDim = dim3(C::THREADS, 1, 1);
        cfg.dynamicSmemBytes = C::SMEM;
        cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = 2;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        static int max_clusters[64];  // per device: co-resident clusters of this kernel + 1 (0 = not asked yet)
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return cudaErrorNotSupported;
        if (max_clusters[dev] == 0) {
            int n = 0;
            if (cudaOccupancyMaxActiveClusters(&n, kern, &cfg) != cudaSuccess) {
                (void)cudaGetLastError();
                n = 0;
            }
            max_clusters[dev] = n + 1;
        }
        if (max_clusters[dev] - 1 < want) return cudaErrorNotSupported;  // a persistent grid must be co-resident
        return cudaLaunchKernelEx(&cfg, kern, a, maps, num_items);
    }
}

template <int DQK, int DV, int NT>
cudaError_t launch_v1(const PrefillArgs &a, const Maps &maps, int num_items, int num_sms, cudaStream_t st) {
    using C = V1Cfg<DQK, DV, NT>;
    if constexpr (!C::FITS) {
        return cudaErrorInvalidValue;
    } else {
        auto kern = a.nsplit > 1 ? attn_core_kernel<DQK, DV, kModeRanges, NT> : attn_core_kernel<DQK, DV, kModeFinal, NT>;
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM);
        if (e != cudaSuccess) return e;
        const int ctas = num_sms * C::CTAS_PER_SM;
        const int grid = num_items < ctas ? num_items : ctas;
        kern<<<grid, C::THREADS, C::SMEM, st>>>(a, maps, num_items);
        return cudaGetLastError();
    }
}

}  // namespace

bool prefill_supported(int group, int dqk, int dv) {
    const bool dims = (dqk == 64 || dqk == 128 || dqk == 192) && (dv == 64 || dv == 128);
    return dims && group >= 1 && group <= 16 && (group & (group - 1)) == 0;
}

cudaError_t prefill_encode_kv_maps(const PoolGeom &g, TensorMapBlob *k_map, TensorMapBlob *v_map) {
    const int64_t rows = (int64_t)g.num_layers * g.num_pages * g.num_kv_heads * kPage;
    if (rows > INT32_MAX) return cudaErrorInvalidValue;
    cudaError_t e = encode_arena_map(g.k_arena, rows, g.head_dim_qk, g.kv_dtype == 1, k_map);
    if (e != cudaSuccess) return e;
    return encode_arena_map(g.v_arena, rows, g.head_dim_v, g.kv_dtype == 1, v_map);
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

// Q tiles per CTA for a call whose longest request has `max_q_tokens` query tokens: 1 (two CTAs per SM) when every
// request fits one 128-row tile per kv-head and the shape's shared-memory budget allows it, else 2.
int prefill_tiles_per_cta(int group, int dqk, int dv, int64_t max_q_tokens, int64_t num_items, int num_sms) {
    if (max_q_tokens * group > kTileM) return 2;
    // Two single-tile CTAs per SM only pay when CTAs really share SMs; a lone CTA is better off with the two-tile
    // kernel's deeper K/V ring. The full-SM single-tile variant (Dqk = 192) has the deeper ring itself.
#define COMB_NT1_CASE(DQ, DVV)                                              \
    if (dqk == DQ && dv == DVV) {                                           \
        using C1 = V1Cfg<DQ, DVV, 1>;                                       \
        if (!C1::FITS) return 2;                                            \
        return (!C1::HALF_SM || num_items > num_sms) ? 1 : 2;               \
    }
    COMB_NT1_CASE(128, 128)
    COMB_NT1_CASE(64, 64)
    COMB_NT1_CASE(192, 128)
    COMB_NT1_CASE(128, 64)
    COMB_NT1_CASE(64, 128)
    COMB_NT1_CASE(192, 64)
#undef COMB_NT1_CASE
    return 2;
}

int prefill_ctas_per_sm(int tiles_per_cta, int dqk, int dv) {
    if (tiles_per_cta != 1) return 1;
#define COMB_CPS_CASE(DQ, DVV) \
    if (dqk == DQ && dv == DVV) return V1Cfg<DQ, DVV, 1>::CTAS_PER_SM;
    COMB_CPS_CASE(128, 128)
    COMB_CPS_CASE(64, 64)
    COMB_CPS_CASE(192, 128)
    COMB_CPS_CASE(128, 64)
    COMB_CPS_CASE(64, 128)
    COMB_CPS_CASE(192, 64)
#undef COMB_CPS_CASE
    return 1;
}

cudaError_t launch_prefill(const PoolGeom &g, int layer, const LinkView &lv, const PrefillMaps &pm,
                           const PrefillItem *items_dev, int num_items, int num_q_heads, float scale, void *out,
                           float *lse, int64_t total_q, void *partials, int64_t part_rows, int tiles_per_cta,
                           bool paired, int num_sms, cudaStream_t stream, int *launches, const LaunchHook *hook) {
    PrefillArgs a{};
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
    a.total_q = total_q;
    const bool ranges = part_rows > 0;
    a.nsplit = ranges ? 2 : 1;
    a.part_o = ranges ? (float *)partials : nullptr;
    a.part_lse = ranges ? a.part_o + (size_t)part_rows * g.head_dim_v : nullptr;
    if (ranges && !partials) return cudaErrorInvalidValue;
    Maps maps;
    memcpy(&maps.q, &pm.q, sizeof(CUtensorMap));
    memcpy(&maps.k, &pm.k, sizeof(CUtensorMap));
    memcpy(&maps.v, &pm.v, sizeof(CUtensorMap));
    cudaError_t e = cudaErrorInvalidValue;
    if (hook) hook->begin(hook->ctx, kKernelPrefill, stream);
    const bool clusters = paired && !ranges && tiles_per_cta == 2 && num_items % 2 == 0 && num_items >= num_sms;
#define COMB_PREFILL_CASE(DQ, DVV)                                                              \
    if (g.head_dim_qk == DQ && g.head_dim_v == DVV) {                                           \
        e = cudaErrorNotSupported;                                                              \
        if (clusters) e = launch_v1_clusters<DQ, DVV>(a, maps, num_items, num_sms, stream);     \
        if (e == cudaErrorNotSupported)                                                         \
            e = tiles_per_cta == 1 ? launch_v1<DQ, DVV, 1>(a, maps, num_items, num_sms, stream) \
                                   : launch_v1<DQ, DVV, 2>(a, maps, num_items, num_sms, stream); \
    }
    COMB_PREFILL_CASE(128, 128)
    COMB_PREFILL_CASE(64, 64)
    COMB_PREFILL_CASE(192, 128)
    COMB_PREFILL_CASE(128, 64)
    COMB_PREFILL_CASE(64, 128)
    COMB_PREFILL_CASE(192, 64)
#undef COMB_PREFILL_CASE
    if (hook) hook->end(hook->ctx, stream);
    if (e != cudaSuccess) return e;
    *launches += 1;
    if (ranges) {
        const dim3 mgrid(num_items, 2 * kTileM / 4);  // an item has at most 2 x 128 rows, a CTA merges 4
        if (hook) hook->begin(hook->ctx, kKernelPrefillMerge, stream);
        if (g.head_dim_v == 128) prefill_merge_kernel<128><<<mgrid, 128, 0, stream>>>(a, num_items);
        else prefill_merge_kernel<64><<<mgrid, 128, 0, stream>>>(a, num_items);
        if (hook) hook->end(hook->ctx, stream);
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
        *launches += 1;
    }
    return cudaSuccess;
}

}  // namespace comb

#ifdef COMB_TRACE
// libcomb_trace.so only (`build.py --trace`): copies the timeline of the most recent prefill launch to host arrays of
// 2 x 128 x 8 uint64 each (attn_core.cuh says what the stamps are).  Synchronises the device.
#pragma GCC visibility push(default)
extern "C" int32_t comb_trace_prefill_read(void *softmax, void *issuer) {
    if (cudaDeviceSynchronize() != cudaSuccess) return -6;
    if (cudaMemcpyFromSymbol(softmax, comb::g_trace_sm, sizeof(comb::g_trace_sm)) != cudaSuccess) return -6;
    if (cudaMemcpyFromSymbol(issuer, comb::g_trace_mma, sizeof(comb::g_trace_mma)) != cudaSuccess) return -6;
    return 0;
}
// per-CTA %globaltimer stamps of the most recent prefill launch: 1024 x 4 uint64 (entry, set-up done, loop end, exit)
extern "C" int32_t comb_trace_prefill_read_ctas(void *ctas) {
    if (cudaDeviceSynchronize() != cudaSuccess) return -6;
    if (cudaMemcpyFromSymbol(ctas, comb::g_trace_cta, sizeof(comb::g_trace_cta)) != cudaSuccess) return -6;
    return 0;
}
#pragma GCC visibility pop
#endif
