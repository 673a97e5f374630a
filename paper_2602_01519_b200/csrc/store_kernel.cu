// store_kernel.cu — (a2) paged store: scatter a chunk's K/V [T][Hkv][D] into 16-token pages
// [page][Hkv][16][D], zero-filling the tail of a chunk's last page.
// PAPER.md:62 §3 step 3 ("store the KV caches"), §4.2 (K^cross, V^cross are what is stored),
// PAPER.md:205 §5.3 (stored asynchronously -> enqueued on the caller's stream, no sync).
//
// HBM-bound byte permutation (bf16 bit copy). A unit = one destination page of K or of V, taken by one CTA of a
// persistent grid; one warp moves one (page, kv-head) block = 16 rows of D bf16, which is contiguous in the arena. Per block a
// lane issues all its 16-byte loads (4 to 12, groups of lanes reading whole source rows) before its stores, the
// stores of a warp are one contiguous run, and there is no integer division in the index math (VPR =
// 16-byte vectors per row is a template constant; an earlier one-CTA-per-page version spent ~90 instructions per
// vector on it). Algorithmic traffic: read + write 2 * T * Hkv * (Dqk + Dv) * 2 B.
#include "kernels.h"

namespace comb {
namespace {

constexpr int kStoreThreads = 256;
constexpr int kStoreWarps = kStoreThreads / 32;

__device__ __forceinline__ uint4 ld_stream(const uint4 *p) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(p));
    return r;
}

// One (page, head) block: dst [16][VPR] vectors contiguous; src row s at src + s * hkv * VPR.
template <int VPR>
__device__ __forceinline__ void store_block(uint4 *__restrict__ dst, const uint4 *__restrict__ src, int hkv, int ntok,
                                            int lane) {
    constexpr int NV = kPage * VPR / 32;  // vectors per lane (4, 8 or 12)
    uint4 r[NV];
#pragma unroll
    for (int i = 0; i < NV; ++i) {
        const int idx = i * 32 + lane;    // vector index inside the block
        const int s = idx / VPR, c = idx % VPR;  // VPR is a compile-time constant: multiply-shift, no division
        r[i] = make_uint4(0u, 0u, 0u, 0u);      // slots past the chunk's length are zero-filled
        if (s < ntok) r[i] = ld_stream(src + (size_t)s * hkv * VPR + c);
    }
#pragma unroll
    for (int i = 0; i < NV; ++i) dst[i * 32 + lane] = r[i];
}

template <int VPR>
__device__ __forceinline__ void store_page(uint4 *__restrict__ layer, const uint4 *__restrict__ src_all,
                                           const StorePageDesc d, int hkv) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    uint4 *dst = layer + (size_t)d.dst_page * hkv * (kPage * VPR);
    const uint4 *src = src_all + (size_t)d.src_tok * hkv * VPR;
    for (int h = warp; h < hkv; h += kStoreWarps)
        store_block<VPR>(dst + (size_t)h * (kPage * VPR), src + (size_t)h * VPR, hkv, d.ntok, lane);
}

// Persistent grid-stride over units u = 2 * page + tensor; the next unit's descriptor is fetched while the current
// unit's rows are in flight, so a CTA never sits on a dependent descriptor -> data round trip.
template <int VPR_K, int VPR_V>
__global__ void __launch_bounds__(kStoreThreads)
store_pages_kernel(const StorePageDesc *__restrict__ descs, int num_units, uint4 *__restrict__ k_layer,
                   uint4 *__restrict__ v_layer, const uint4 *__restrict__ k_src, const uint4 *__restrict__ v_src,
                   int hkv) {
    int u = blockIdx.x;
    if (u >= num_units) return;
    StorePageDesc d = descs[u >> 1];
    while (true) {
        const int un = u + gridDim.x;
        StorePageDesc dn = d;
        if (un < num_units) dn = descs[un >> 1];
        if ((u & 1) == 0) store_page<VPR_K>(k_layer, k_src, d, hkv);
        else store_page<VPR_V>(v_layer, v_src, d, hkv);
        if (un >= num_units) break;
        u = un;
        d = dn;
    }
}

// Read-only stream: every thread keeps 8 independent 16-byte loads in flight and folds them into one word; the
// measurement kernel behind comb_util_stream_read (bench.py's read-only HBM ceiling, SURVEY.md §8(d) "Denominators").
__global__ void __launch_bounds__(256) stream_read_kernel(const uint4 *__restrict__ src, size_t n_vec,
                                                          unsigned int *__restrict__ sink) {
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned int acc = 0;
    for (; i + 7 * stride < n_vec; i += 8 * stride) {
        uint4 v[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) v[u] = __ldcs(src + i + u * stride);
#pragma unroll
        for (int u = 0; u < 8; ++u) acc ^= v[u].x ^ v[u].y ^ v[u].z ^ v[u].w;
    }
    for (; i < n_vec; i += stride) {
        const uint4 v = __ldcs(src + i);
        acc ^= v.x ^ v.y ^ v.z ^ v.w;
    }
    if (acc == 0x9e3779b9u) atomicXor(sink, acc);  // practically never true: keeps the loads alive without a store stream
}

}  // namespace

cudaError_t launch_stream_read(const void *src, size_t bytes, void *sink, cudaStream_t stream) {
    if (!src || !sink || bytes < 16) return cudaErrorInvalidValue;
    stream_read_kernel<<<148 * 8, 256, 0, stream>>>((const uint4 *)src, bytes / 16, (unsigned int *)sink);
    return cudaGetLastError();
}

cudaError_t launch_store(const PoolGeom &g, int layer, const StorePageDesc *descs_dev, int num_descs, const void *k_src,
                         const void *v_src, cudaStream_t stream) {
    if (num_descs <= 0) return cudaSuccess;
    const int vpr_k = g.head_dim_qk / 8, vpr_v = g.head_dim_v / 8;
    const size_t layer_vec_k = (size_t)g.num_pages * g.num_kv_heads * kPage * vpr_k;
    const size_t layer_vec_v = (size_t)g.num_pages * g.num_kv_heads * kPage * vpr_v;
    uint4 *k_layer = (uint4 *)g.k_arena + (size_t)layer * layer_vec_k;
    uint4 *v_layer = (uint4 *)g.v_arena + (size_t)layer * layer_vec_v;
    const int num_units = 2 * num_descs;
    const int grid = num_units < 148 * 8 ? num_units : 148 * 8;  // <= 8 resident CTAs of 256 threads per SM
#define COMB_STORE_CASE(DQ, DVV)                                                                           \
    if (g.head_dim_qk == DQ && g.head_dim_v == DVV) {                                                      \
        store_pages_kernel<DQ / 8, DVV / 8><<<grid, kStoreThreads, 0, stream>>>(                           \
            descs_dev, num_units, k_layer, v_layer, (const uint4 *)k_src, (const uint4 *)v_src,            \
            g.num_kv_heads);                                                                               \
        return cudaGetLastError();                                                                         \
    }
    COMB_STORE_CASE(128, 128)
    COMB_STORE_CASE(64, 64)
    COMB_STORE_CASE(192, 128)
    COMB_STORE_CASE(128, 64)
    COMB_STORE_CASE(64, 128)
    COMB_STORE_CASE(192, 64)
#undef COMB_STORE_CASE
    return cudaErrorInvalidValue;
}

}  // namespace comb
