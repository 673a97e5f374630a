// fp8_kernel.cu — (f4) fp8 (e4m3) pages: the quantising store and the dequantising staging copy.
// SURVEY.md §8(f4) "fp8 (e4m3) pages with per-page scales to halve decode bytes"; PAPER.md:277 (KV memory bounds
// concurrency).  The quantisation rule is part of the bit-exact contract (include/comb.h "fp8 pools"; DESIGN.md §2
// I31-I33): per (page, kv-head) block, scale = the smallest power of two 2^e with amax <= 448 * 2^e, code =
// e4m3_rne(x / scale).  Dividing by a power of two is exact and value(code) * scale is exactly a bf16 number, so
// neither direction rounds anywhere but in the e4m3 conversion itself.
//
// Both kernels move one (page, kv-head) block per warp (16 rows x 128 elements, contiguous on the page side) on a
// persistent grid, like store_kernel.cu; both are HBM-bound byte streams (3 B per element: 2 in + 1 out, or 1 + 2).
#include "kernels.h"

#include <cuda_bf16.h>
#include <cuda_fp8.h>

namespace comb {
namespace {

constexpr int kThreads = 256, kWarps = kThreads / 32;
constexpr int kD = 128;                       // head dim of fp8 pools
constexpr int kVpr = kD / 8;                  // 16-byte bf16 vectors per row
constexpr int kNv = kPage * kVpr / 32;        // vectors per lane and block (8)

__device__ __forceinline__ uint4 ld_stream(const uint4 *p) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(p));
    return r;
}
__device__ __forceinline__ float bf16_lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t w) { return __uint_as_float(w & 0xffff0000u); }

// 2^e, e = the smallest integer with amax <= 448 * 2^e (448 = 1.75 * 2^8), clamped to [-100, 100]; amax > 0, finite.
__device__ __forceinline__ float block_scale(float amax) {
    const uint32_t bits = __float_as_uint(amax);
    int ex = (int)(bits >> 23) - 127;          // amax = m * 2^ex, m in [1, 2) (bf16 subnormals: handled by the loop)
    const uint32_t man = bits & 0x7fffffu;
    int e = ex - 8 + (man > 0x600000u ? 1 : 0);  // m <= 1.75 -> 2^(ex-8) suffices, else one more
    if ((bits >> 23) == 0) {                   // subnormal amax: far below the clamp
        e = -100;
    }
    e = e < -100 ? -100 : (e > 100 ? 100 : e);
    return __uint_as_float((uint32_t)(e + 127) << 23);
}

// One block: src rows s at src + s * hkv * kVpr (bf16 [T][Hkv][128]); dst 16 x 128 codes contiguous; one scale.
__device__ __forceinline__ void quantise_block(uint2 *__restrict__ dst, float *__restrict__ scale_out,
                                               const uint4 *__restrict__ src, int hkv, int ntok, int lane) {
    uint4 r[kNv];
#pragma unroll
    for (int i = 0; i < kNv; ++i) {
        const int idx = i * 32 + lane, s = idx / kVpr, c = idx % kVpr;
        r[i] = make_uint4(0u, 0u, 0u, 0u);     // slots past the chunk's length count as zeros
        if (s < ntok) r[i] = ld_stream(src + (size_t)s * hkv * kVpr + c);
    }
    float amax = 0.f;
#pragma unroll
    for (int i = 0; i < kNv; ++i) {
        const uint32_t w[4] = {r[i].x, r[i].y, r[i].z, r[i].w};
#pragma unroll
        for (int j = 0; j < 4; ++j) amax = fmaxf(amax, fmaxf(fabsf(bf16_lo(w[j])), fabsf(bf16_hi(w[j]))));
    }
    // non-negative floats order like their bit patterns
    amax = __uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(amax)));
    const float scale = amax > 0.f ? block_scale(amax) : 1.f;
    const float inv = 1.f / scale;             // exact: a power of two within [2^-100, 2^100]
    if (lane == 0) *scale_out = scale;
#pragma unroll
    for (int i = 0; i < kNv; ++i) {
        const uint32_t w[4] = {r[i].x, r[i].y, r[i].z, r[i].w};
        uint32_t q[4];
#pragma unroll
        for (int j = 0; j < 4; ++j)  // element 2j in the low byte, 2j + 1 in the high byte
            q[j] = (uint32_t)__nv_cvt_float2_to_fp8x2(make_float2(bf16_lo(w[j]) * inv, bf16_hi(w[j]) * inv),
                                                     __NV_SATFINITE, __NV_E4M3);
        dst[i * 32 + lane] = make_uint2(q[0] | (q[1] << 16), q[2] | (q[3] << 16));
    }
}

__global__ void __launch_bounds__(kThreads)
store_pages_fp8_kernel(const StorePageDesc *__restrict__ descs, int num_units, uint2 *__restrict__ k_layer,
                       uint2 *__restrict__ v_layer, float *__restrict__ k_scale, float *__restrict__ v_scale,
                       const uint4 *__restrict__ k_src, const uint4 *__restrict__ v_src, int hkv) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    constexpr int kBlk = kPage * kD / 8;       // uint2 per block
    for (int u = blockIdx.x; u < num_units; u += gridDim.x) {
        const StorePageDesc d = descs[u >> 1];
        const bool is_v = u & 1;
        uint2 *dst = (is_v ? v_layer : k_layer) + (size_t)d.dst_page * hkv * kBlk;
        float *sc = (is_v ? v_scale : k_scale) + (size_t)d.dst_page * hkv;
        const uint4 *src = (is_v ? v_src : k_src) + (size_t)d.src_tok * hkv * kVpr;
        for (int h = warp; h < hkv; h += kWarps)
            quantise_block(dst + (size_t)h * kBlk, sc + h, src + (size_t)h * kVpr, hkv, d.ntok, lane);
    }
}

// staging page i <- pool page page_ids[i]: bf16(value(code) * scale), exact
__global__ void __launch_bounds__(kThreads)
dequant_pages_kernel(const int32_t *__restrict__ page_ids, int num_units, const uint2 *__restrict__ k_layer,
                     const uint2 *__restrict__ v_layer, const float *__restrict__ k_scale,
                     const float *__restrict__ v_scale, uint4 *__restrict__ k_out, uint4 *__restrict__ v_out, int hkv) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    constexpr int kBlk = kPage * kD / 8;
    for (int u = blockIdx.x; u < num_units; u += gridDim.x) {
        const int i = u >> 1;
        const bool is_v = u & 1;
        const int page = page_ids[i];
        const uint2 *src = (is_v ? v_layer : k_layer) + (size_t)page * hkv * kBlk;
        const float *sc = (is_v ? v_scale : k_scale) + (size_t)page * hkv;
        uint4 *dst = (is_v ? v_out : k_out) + (size_t)i * hkv * kBlk;
        for (int h = warp; h < hkv; h += kWarps) {
            const float scale = sc[h];
            uint2 q[kNv];
#pragma unroll
            for (int j = 0; j < kNv; ++j) q[j] = src[(size_t)h * kBlk + j * 32 + lane];
#pragma unroll
            for (int j = 0; j < kNv; ++j) {
                const uint32_t w[2] = {q[j].x, q[j].y};
                uint32_t o[4];
#pragma unroll
                for (int t = 0; t < 4; ++t) {
                    const __half2_raw hr = __nv_cvt_fp8x2_to_halfraw2(
                        (__nv_fp8x2_storage_t)((w[t >> 1] >> (16 * (t & 1))) & 0xffffu), __NV_E4M3);
                    const float2 f = __half22float2(*reinterpret_cast<const __half2 *>(&hr));
                    const __nv_bfloat162 b = __floats2bfloat162_rn(f.x * scale, f.y * scale);
                    o[t] = *reinterpret_cast<const uint32_t *>(&b);
                }
                dst[(size_t)h * kBlk + j * 32 + lane] = make_uint4(o[0], o[1], o[2], o[3]);
            }
        }
    }
}

}  // namespace

cudaError_t launch_store_fp8(const PoolGeom &g, int layer, const StorePageDesc *descs_dev, int num_descs,
                             const void *k_src, const void *v_src, cudaStream_t stream) {
    if (num_descs <= 0) return cudaSuccess;
    if (g.kv_dtype != 1 || g.head_dim_qk != kD || g.head_dim_v != kD || !g.k_scale || !g.v_scale)
        return cudaErrorInvalidValue;
    const size_t blocks = (size_t)g.num_pages * g.num_kv_heads;
    uint2 *k_layer = (uint2 *)g.k_arena + (size_t)layer * blocks * (kPage * kD / 8);
    uint2 *v_layer = (uint2 *)g.v_arena + (size_t)layer * blocks * (kPage * kD / 8);
    const int num_units = 2 * num_descs;
    const int grid = num_units < 148 * 8 ? num_units : 148 * 8;
    store_pages_fp8_kernel<<<grid, kThreads, 0, stream>>>(descs_dev, num_units, k_layer, v_layer,
                                                         g.k_scale + (size_t)layer * blocks,
                                                         g.v_scale + (size_t)layer * blocks, (const uint4 *)k_src,
                                                         (const uint4 *)v_src, g.num_kv_heads);
    return cudaGetLastError();
}

cudaError_t launch_dequant_pages(const PoolGeom &g, int layer, const int32_t *page_ids_dev, int num_pages, void *k_out,
                                 void *v_out, cudaStream_t stream) {
    if (num_pages <= 0) return cudaSuccess;
    if (g.kv_dtype != 1 || g.head_dim_qk != kD || g.head_dim_v != kD || !page_ids_dev || !k_out || !v_out)
        return cudaErrorInvalidValue;
    const size_t blocks = (size_t)g.num_pages * g.num_kv_heads;
    const uint2 *k_layer = (const uint2 *)g.k_arena + (size_t)layer * blocks * (kPage * kD / 8);
    const uint2 *v_layer = (const uint2 *)g.v_arena + (size_t)layer * blocks * (kPage * kD / 8);
    const int num_units = 2 * num_pages;
    const int grid = num_units < 148 * 8 ? num_units : 148 * 8;
    dequant_pages_kernel<<<grid, kThreads, 0, stream>>>(page_ids_dev, num_units, k_layer, v_layer,
                                                       g.k_scale + (size_t)layer * blocks,
                                                       g.v_scale + (size_t)layer * blocks, (uint4 *)k_out,
                                                       (uint4 *)v_out, g.num_kv_heads);
    return cudaGetLastError();
}

}  // namespace comb
