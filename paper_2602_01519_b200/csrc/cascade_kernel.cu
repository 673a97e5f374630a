// cascade_kernel.cu — (f1) chunk-major ("cascade") decode cross-attention.
//
// PICaches are position-independent: a chunk's K/V is the same bytes for every request that links it, in any order
// (§1 "in any order/position"), and retrieval workloads re-use a few hot chunks heavily
// (PAPER.md:297).  So instead of streaming a chunk once per linking request (GEMV-shaped, CUDA cores, up to 99 reads
// of the hottest chunk in BASELINE configs[1]), the batch is inverted at link time and every DISTINCT chunk is
// streamed once: the (entries x G) query rows that link it form the M tile of the tcgen05 contraction of
// attn_core.cuh (mode kModeCascade: Q rows gathered from the linking requests, KV = the chunk's own page list).  Each
// (entry, head) gets a normalised fp32 partial row and a log2-domain LSE; cascade_merge_kernel combines a request's
// entries by identity P8:  O = sum_e w_e O_e / sum_e w_e,  w_e = 2^(lse2_e - max),
// LSE = ln 2 (max + log2 sum_e w_e).  One joint softmax over the concatenation, as Eq. 7-8 with PAPER.md:149 demand.
#include "attn_core.cuh"

#include <cstring>

namespace comb {
namespace {

// One CTA of 4 warps per (request, q head): the request's entries are dealt round-robin to the warps, a lane owns
// DV/32 consecutive output columns, and the four warps' weighted sums meet in shared memory.  Every warp first reads
// ALL of the request's LSEs (one per lane per pass; they are few) to agree on the maximum, then streams its share of
// the partial rows with 4 independent loads in flight.
template <int DV>
__global__ void __launch_bounds__(128) cascade_merge_kernel(const float *__restrict__ part_o,
                                                            const float *__restrict__ part_lse,
                                                            const int32_t *__restrict__ entry_indptr,
                                                            __nv_bfloat16 *__restrict__ out, float *__restrict__ lse,
                                                            int Hq) {
    constexpr int CPL = DV / 32;
    __shared__ float s_acc[4][DV];
    __shared__ float s_w[4];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int row = blockIdx.x;  // (request, head)
    const int r = row / Hq, h = row - r * Hq;
    const int e0 = entry_indptr[r], e1 = entry_indptr[r + 1];
    __nv_bfloat16 *orow = out + (size_t)row * DV;
    if (e0 == e1) {  // no contexts linked (reading I13)
        if (threadIdx.x < DV / 2) reinterpret_cast<uint32_t *>(orow)[threadIdx.x] = 0u;
        if (threadIdx.x == 0 && lse) lse[row] = -INFINITY;
        return;
    }
    float m = -INFINITY;
    for (int e = e0 + lane; e < e1; e += 32) m = fmaxf(m, part_lse[(size_t)e * Hq + h]);
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, off));
    float acc[CPL];
#pragma unroll
    for (int c = 0; c < CPL; ++c) acc[c] = 0.f;
    float wsum = 0.f;
    for (int eb = e0 + warp; eb < e1; eb += 16) {  // this warp: entries eb, eb + 4, eb + 8, eb + 12
        float w[4];
        float4 v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int e = eb + 4 * u;
            const bool ok = e < e1;
            w[u] = ok ? ptx::ex2(part_lse[(size_t)e * Hq + h] - m) : 0.f;
            v[u] = make_float4(0.f, 0.f, 0.f, 0.f);
            if (ok) {
                const float *po = part_o + ((size_t)e * Hq + h) * DV + lane * CPL;
                if constexpr (CPL == 4) v[u] = *reinterpret_cast<const float4 *>(po);
                else { const float2 t = *reinterpret_cast<const float2 *>(po); v[u].x = t.x; v[u].y = t.y; }
            }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            wsum += w[u];
            acc[0] += w[u] * v[u].x;
            acc[1] += w[u] * v[u].y;
            if constexpr (CPL == 4) { acc[2] += w[u] * v[u].z; acc[3] += w[u] * v[u].w; }
        }
    }
#pragma unroll
    for (int c = 0; c < CPL; ++c) s_acc[warp][lane * CPL + c] = acc[c];
    if (lane == 0) s_w[warp] = wsum;
    __syncthreads();
    const float wtot = (s_w[0] + s_w[1]) + (s_w[2] + s_w[3]);
    if (threadIdx.x < DV / 2) {
        const int c = 2 * threadIdx.x;
        const float inv = 1.f / wtot;
        const float a0 = (s_acc[0][c] + s_acc[1][c]) + (s_acc[2][c] + s_acc[3][c]);
        const float a1 = (s_acc[0][c + 1] + s_acc[1][c + 1]) + (s_acc[2][c + 1] + s_acc[3][c + 1]);
        reinterpret_cast<uint32_t *>(orow)[threadIdx.x] = ptx::pack_bf16x2(a0 * inv, a1 * inv);
    }
    if (threadIdx.x == 0 && lse) lse[row] = (m + log2f(wtot)) * kLn2;
}

template <int DQK, int DV>
cudaError_t launch_cascade_t(const PrefillArgs &a, const Maps &maps, int num_items, int num_sms, cudaStream_t st) {
    using C = V1Cfg<DQK, DV, 1>;
    if constexpr (!C::FITS) {
        return cudaErrorInvalidValue;
    } else {
        auto kern = attn_core_kernel<DQK, DV, kModeCascade, 1>;
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM);
        if (e != cudaSuccess) return e;
        const int ctas = num_sms * C::CTAS_PER_SM;
        const int grid = num_items < ctas ? num_items : ctas;
        kern<<<grid, C::THREADS, C::SMEM, st>>>(a, maps, num_items);
        return cudaGetLastError();
    }
}

}  // namespace

size_t cascade_partial_bytes(int64_t total_entries, int num_q_heads, int dv) {
    return (size_t)total_entries * (size_t)num_q_heads * (size_t)(dv + 1) * sizeof(float);
}

cudaError_t launch_decode_cascade(const PoolGeom &g, int layer, const LinkView &lv, const PrefillMaps &pm,
                                  const CascadeTile *tiles_dev, int num_tiles, int num_requests, int num_q_heads,
                                  const void *q, float scale, void *out, float *lse, int64_t total_entries,
                                  void *partials, int num_sms, cudaStream_t stream, int *launches,
                                  const LaunchHook *hook) {
    PrefillArgs a{};
    a.items = nullptr;
    a.page_indptr = lv.cas_page_indptr;  // a "request" of the core kernel is a chunk slot
    a.page_ids = lv.cas_page_ids;
    a.tile_indptr = lv.cas_tile_indptr;
    a.tile_ntok = lv.cas_tile_ntok;
    a.out = (__nv_bfloat16 *)out;
    a.lse = lse;
    a.num_q_heads = num_q_heads;
    a.num_kv_heads = g.num_kv_heads;
    a.group = num_q_heads / g.num_kv_heads;
    a.layer_row0 = layer * g.num_pages * g.num_kv_heads * kPage;
    a.scale_log2 = scale * kLog2e;
    a.total_q = num_requests;
    a.nsplit = 1;
    a.part_o = (float *)partials;
    a.part_lse = a.part_o + (size_t)total_entries * num_q_heads * g.head_dim_v;
    a.cas_tiles = tiles_dev;
    a.cas_row_req = lv.cas_row_req;
    a.cas_row_entry = lv.cas_row_entry;
    a.q = (const char *)q;
    if (!partials) return cudaErrorInvalidValue;
    Maps maps;
    memcpy(&maps.q, &pm.k, sizeof(CUtensorMap));  // unused in this mode (Q rows are gathered); any valid map
    memcpy(&maps.k, &pm.k, sizeof(CUtensorMap));
    memcpy(&maps.v, &pm.v, sizeof(CUtensorMap));
    const int num_items = num_tiles * g.num_kv_heads;
    cudaError_t e = num_items > 0 ? cudaErrorInvalidValue : cudaSuccess;  // every request empty: only the merge runs
    if (hook && num_items > 0) hook->begin(hook->ctx, kKernelDecodeCascade, stream);
#define COMB_CASCADE_CASE(DQ, DVV)                                    \
    if (num_items > 0 && g.head_dim_qk == DQ && g.head_dim_v == DVV) \
        e = launch_cascade_t<DQ, DVV>(a, maps, num_items, num_sms, stream);
    COMB_CASCADE_CASE(128, 128)
    COMB_CASCADE_CASE(64, 64)
    COMB_CASCADE_CASE(192, 128)
    COMB_CASCADE_CASE(128, 64)
    COMB_CASCADE_CASE(64, 128)
    COMB_CASCADE_CASE(192, 64)
#undef COMB_CASCADE_CASE
    if (hook && num_items > 0) hook->end(hook->ctx, stream);
    if (e != cudaSuccess) return e;
    *launches += num_items > 0 ? 1 : 0;
    const int rows = num_requests * num_q_heads;
    if (hook) hook->begin(hook->ctx, kKernelCascadeMerge, stream);
    if (g.head_dim_v == 128)
        cascade_merge_kernel<128><<<rows, 128, 0, stream>>>(a.part_o, a.part_lse, lv.entry_indptr, a.out, lse, num_q_heads);
    else
        cascade_merge_kernel<64><<<rows, 128, 0, stream>>>(a.part_o, a.part_lse, lv.entry_indptr, a.out, lse, num_q_heads);
    if (hook) hook->end(hook->ctx, stream);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    *launches += 1;
    return cudaSuccess;
}

}  // namespace comb
