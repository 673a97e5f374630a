// store_kernel.cu — (a2) paged store: scatter a chunk's K/V [T][Hkv][D] into 16-token pages
// [page][Hkv][16][D], zero-filling the tail of a chunk's last page.
// PAPER.md:62 §3 step 3 ("store the KV caches"), §4.2 (K^cross, V^cross are what is stored),
// PAPER.md:205 §5.3 (stored asynchronously -> enqueued on the caller's stream, no sync).
//
// HBM-bound byte permutation (bf16 bit copy): one CTA per destination page, 16-byte vectors, all of a
// batch's loads issued before its stores so each thread keeps 8 x 16 B in flight. Algorithmic traffic:
// read + write 2 * T * Hkv * (Dqk + Dv) * 2 B.
#include "kernels.h"

namespace comb {
namespace {

constexpr int kStoreThreads = 256;
constexpr int kStoreBatch = 8;

__device__ __forceinline__ uint4 ld_stream(const uint4 *p) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(p));
    return r;
}

// Copies one page of one tensor. dst block: [Hkv][16][VPR] vectors; src rows: [(tok)][Hkv][VPR] vectors.
__device__ __forceinline__ void store_page(uint4 *__restrict__ dst, const uint4 *__restrict__ src, int hkv, int vpr,
                                           int ntok) {
    const int nvec = hkv * kPage * vpr;
    const int row_vecs = kPage * vpr;  // vectors per head inside the page
    for (int base = 0; base < nvec; base += kStoreThreads * kStoreBatch) {
        uint4 r[kStoreBatch];
#pragma unroll
        for (int j = 0; j < kStoreBatch; ++j) {
            const int idx = base + j * kStoreThreads + (int)threadIdx.x;
            r[j] = make_uint4(0u, 0u, 0u, 0u);
            if (idx < nvec) {
                const int h = idx / row_vecs;
                const int rem = idx - h * row_vecs;
                const int s = rem / vpr;
                const int c = rem - s * vpr;
                if (s < ntok) r[j] = ld_stream(src + ((size_t)s * hkv + h) * vpr + c);
            }
        }
#pragma unroll
        for (int j = 0; j < kStoreBatch; ++j) {
            const int idx = base + j * kStoreThreads + (int)threadIdx.x;
            if (idx < nvec) dst[idx] = r[j];
        }
    }
}

__global__ void __launch_bounds__(kStoreThreads)
store_pages_kernel(const StorePageDesc *__restrict__ descs, uint4 *__restrict__ k_layer, uint4 *__restrict__ v_layer,
                   const uint4 *__restrict__ k_src, const uint4 *__restrict__ v_src, int hkv, int vpr_k, int vpr_v) {
    const StorePageDesc d = descs[blockIdx.x];
    const size_t page_vec_k = (size_t)hkv * kPage * vpr_k;
    const size_t page_vec_v = (size_t)hkv * kPage * vpr_v;
    store_page(k_layer + (size_t)d.dst_page * page_vec_k, k_src + (size_t)d.src_tok * hkv * vpr_k, hkv, vpr_k, d.ntok);
    store_page(v_layer + (size_t)d.dst_page * page_vec_v, v_src + (size_t)d.src_tok * hkv * vpr_v, hkv, vpr_v, d.ntok);
}

}  // namespace

cudaError_t launch_store(const PoolGeom &g, int layer, const StorePageDesc *descs_dev, int num_descs, const void *k_src,
                         const void *v_src, cudaStream_t stream) {
    if (num_descs <= 0) return cudaSuccess;
    const int vpr_k = g.head_dim_qk / 8, vpr_v = g.head_dim_v / 8;
    const size_t layer_vec_k = (size_t)g.num_pages * g.num_kv_heads * kPage * vpr_k;
    const size_t layer_vec_v = (size_t)g.num_pages * g.num_kv_heads * kPage * vpr_v;
    uint4 *k_layer = (uint4 *)g.k_arena + (size_t)layer * layer_vec_k;
    uint4 *v_layer = (uint4 *)g.v_arena + (size_t)layer * layer_vec_v;
    store_pages_kernel<<<num_descs, kStoreThreads, 0, stream>>>(descs_dev, k_layer, v_layer, (const uint4 *)k_src,
                                                               (const uint4 *)v_src, g.num_kv_heads, vpr_k, vpr_v);
    return cudaGetLastError();
}

}  // namespace comb
