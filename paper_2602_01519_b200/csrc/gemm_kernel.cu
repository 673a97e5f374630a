// gemm_kernel.cu — (f2)/(f3) the projections either side of the link-stage attention, C = A W^T on tcgen05:
//   K^cross = H^E W_K, V^cross = H^E W_V   (§4.2 Eq. 5-6) with an epilogue that writes bf16 straight
//                                          into the chunk's pages (K/V are what is stored)
//   Q = X^D W_Q                            (Eq. 4)
//   X^D + H W_O                            (output projection + residual)
//
// Persistent, warp-specialised: warp 0 = TMA producer (A tile 128 x 64, W tile 256 x 64, SWIZZLE_128B, 4-stage
// mbarrier ring), warp 1 = single-thread tcgen05.mma issuer (M 128, N 256, K 16 per instruction, fp32 accumulators in
// TMEM, two accumulator buffers of 256 columns so the epilogue of tile i runs under the main loop of tile i + 1),
// warps 2-5 = epilogue (tcgen05.ld of the warp's 32 TMEM lanes, bf16 pack, 64-byte stores).
#include "kernels.h"
#include "ptx.cuh"

#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_fp8.h>
#include <cstring>

namespace comb {
namespace {

constexpr int BM = 128, BK = 64;
constexpr int A_BYTES = BM * BK * 2;
constexpr int GEMM_THREADS = 192;
// N tile: 256 columns (4 stages of 48 KB), or 64 columns with an 8-stage ring of 24 KB for problems whose 256-column
// tiles would leave most SMs idle, or 32 columns with a 10-stage ring of 20 KB when 64-column tiles still would (a
// decode-phase projection: M <= 128 rows and N = 4096 give 128 tiles of 32 columns; the weights are the traffic and
// every SM should stream its share of them — a CTA's rate is set by the bytes its ring keeps in flight)
template <int BN>
struct GemmCfg {
    static constexpr int STAGES = BN == 256 ? 4 : BN == 64 ? 8 : 10;
    static constexpr int B_BYTES = BN * BK * 2, STAGE_BYTES = A_BYTES + B_BYTES;
    static constexpr int SMEM = 1024 + STAGES * STAGE_BYTES + 256;
};

enum { kEpiRowMajor = 0, kEpiPaged = 1, kEpiPagedF8 = 2 };

struct GemmArgs {
    int64_t M;
    int N, K;
    int num_m_tiles, num_n_tiles;
    // row-major epilogue
    __nv_bfloat16 *c;
    const __nv_bfloat16 *residual;
    // paged epilogue
    const GemmRowTile *row_tiles;
    char *k_layer, *v_layer;   // this layer's arenas: bf16 (or e4m3 bytes) [num_pages][Hkv][16][D]
    float *k_scale, *v_scale;  // fp8 pools: this layer's scale tables [num_pages][Hkv]
    int hkv, dqk, dv;
};

struct GemmMaps {
    CUtensorMap a, w;
};

template <int EPI, int BN>
__global__ void __launch_bounds__(GEMM_THREADS, 1)
gemm_bf16_kernel(const GemmArgs g, const __grid_constant__ GemmMaps maps) {
    constexpr int STAGES = GemmCfg<BN>::STAGES, STAGE_BYTES = GemmCfg<BN>::STAGE_BYTES;
    extern __shared__ unsigned char smem_raw[];
    unsigned char *smem = ptx::align_smem_1024(smem_raw);
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + STAGES * STAGE_BYTES);
    uint64_t *full = bars, *empty = bars + STAGES, *acc_full = bars + 2 * STAGES, *acc_empty = bars + 2 * STAGES + 2;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(bars + 2 * STAGES + 4);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) {
            ptx::mbar_init(&full[s], 1);
            ptx::mbar_init(&empty[s], 1);
        }
        for (int s = 0; s < 2; ++s) {
            ptx::mbar_init(&acc_full[s], 1);
            ptx::mbar_init(&acc_empty[s], 4);  // one arrival per epilogue warp
        }
        ptx::fence_barrier_init();
        ptx::tma_prefetch_desc(&maps.a);
        ptx::tma_prefetch_desc(&maps.w);
    }
    if (warp == 1) {
        ptx::tmem_alloc(tmem_slot, 512);
        ptx::tmem_relinquish();
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    const int num_tiles = g.num_m_tiles * g.num_n_tiles;
    const int num_kb = (g.K + BK - 1) / BK;

    if (warp == 0) {
        // ===================== TMA producer =====================
        uint32_t stage = 0, phase = 0;
        for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
            const int mt = tile / g.num_n_tiles, nt = tile - mt * g.num_n_tiles;
            int a_row0 = mt * BM;
            if constexpr (EPI != kEpiRowMajor) a_row0 = g.row_tiles[mt].a_row0;
            for (int kb = 0; kb < num_kb; ++kb) {
                ptx::mbar_wait(&empty[stage], phase ^ 1);
                if (lane == 0) {
                    unsigned char *sa = smem + stage * STAGE_BYTES, *sb = sa + A_BYTES;
                    ptx::mbar_expect_tx(&full[stage], STAGE_BYTES);
                    ptx::tma_load_2d(sa, &maps.a, kb * BK, a_row0, &full[stage]);
                    ptx::tma_load_2d(sb, &maps.w, kb * BK, nt * BN, &full[stage]);
                }
                if (++stage == STAGES) { stage = 0; phase ^= 1; }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer (whole warp runs the control flow, one lane issues) =====================
        const bool leader = ptx::elect_one();
        constexpr uint32_t idesc = ptx::umma_idesc_bf16(BM, BN, false);
        const uint64_t da0 = ptx::umma_desc_sw128(ptx::smem_u32(smem), 16, 1024);
        const uint64_t db0 = ptx::umma_desc_sw128(ptx::smem_u32(smem + A_BYTES), 16, 1024);
        uint32_t stage = 0, phase = 0, acc = 0, acc_phase = 0;
        for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
            ptx::mbar_wait(&acc_empty[acc], acc_phase ^ 1);  // the epilogue has drained this accumulator
            ptx::tc_fence_after();
            for (int kb = 0; kb < num_kb; ++kb) {
                ptx::mbar_wait(&full[stage], phase);
                ptx::tc_fence_after();
                const uint64_t so = (uint64_t)((stage * STAGE_BYTES) >> 4);
#pragma unroll
                for (int kk = 0; kk < BK / 16; ++kk)
                    if (leader)
                        ptx::mma_ss(tmem + acc * BN, da0 + so + (uint64_t)((kk * 32) >> 4), db0 + so + (uint64_t)((kk * 32) >> 4),
                                    idesc, (kb > 0 || kk > 0) ? 1u : 0u);
                if (leader) ptx::mma_commit(&empty[stage]);  // frees the smem stage when these MMAs have read it
                if (++stage == STAGES) { stage = 0; phase ^= 1; }
            }
            if (leader) ptx::mma_commit(&acc_full[acc]);
            if (++acc == 2) { acc = 0; acc_phase ^= 1; }
        }
    } else {
        // ===================== epilogue: warps 2..5 own TMEM lanes 32 (warp % 4) .. + 31 =====================
        const int quad = warp & 3;
        const int row = quad * 32 + lane;  // row of the tile
        const uint32_t lane_base = (uint32_t)(quad * 32) << 16;
        uint32_t acc = 0, acc_phase = 0;
        for (int tile = blockIdx.x; tile < num_tiles; tile += gridDim.x) {
            const int mt = tile / g.num_n_tiles, nt = tile - mt * g.num_n_tiles;
            // ---- where this thread's row goes ----
            bool store_row = false, zero_row = false;
            int page = -1;
            char *dst_k = nullptr, *dst_v = nullptr;           // paged: (page, head 0, slot) of the row in each arena
            __nv_bfloat16 *dst_c = nullptr;
            const __nv_bfloat16 *res = nullptr;
            if constexpr (EPI == kEpiRowMajor) {
                const int64_t grow = (int64_t)mt * BM + row;
                store_row = grow < g.M;
                dst_c = g.c + grow * g.N;
                res = g.residual ? g.residual + grow * g.N : nullptr;
            } else {
                const GemmRowTile rt = g.row_tiles[mt];
                page = rt.pages[row >> 4];
                zero_row = row >= rt.rows_valid && row < rt.rows_zero_to;
                store_row = (row < rt.rows_valid || zero_row) && page >= 0;
                const int slot = row & 15;
                constexpr size_t ELT = EPI == kEpiPagedF8 ? 1 : 2;
                dst_k = g.k_layer + (((size_t)page * g.hkv) * kPage + slot) * (size_t)g.dqk * ELT;
                dst_v = g.v_layer + (((size_t)page * g.hkv) * kPage + slot) * (size_t)g.dv * ELT;
            }
            ptx::mbar_wait(&acc_full[acc], acc_phase);
            ptx::tc_fence_after();
            const uint32_t tacc = tmem + lane_base + acc * BN;
            if constexpr (EPI == kEpiPagedF8) {
                // fp8 pool (include/comb.h "fp8 pools"): a 128-column group is one head; the 16 rows of a page sit in
                // one half-warp.  Per (page, head) block: the values the bf16 pool would hold (bf16_rne of the
                // accumulators; rows past the chunk's length count as zero), their amax over the half-warp, the
                // power-of-two scale, e4m3 codes, 128-byte rows.
#pragma unroll 1
                for (int hb = 0; hb < BN / 128; ++hb) {
                    uint32_t r[128];
#pragma unroll
                    for (int q = 0; q < 4; ++q)
                        ptx::tmem_ld32(tacc + hb * 128 + q * 32, *reinterpret_cast<uint32_t(*)[32]>(&r[q * 32]));
                    ptx::tmem_wait_ld();
                    const int col0 = nt * BN + hb * 128;
                    const bool live = store_row && !zero_row && col0 < g.N;
                    float amax = 0.f;
#pragma unroll
                    for (int e = 0; e < 128; ++e) {
                        const float x = live ? __bfloat162float(__float2bfloat16_rn(__uint_as_float(r[e]))) : 0.f;
                        r[e] = __float_as_uint(x);
                        amax = fmaxf(amax, fabsf(x));
                    }
#pragma unroll
                    for (int off = 8; off >= 1; off >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, off));
                    float scale = 1.f;
                    if (amax > 0.f) {  // smallest 2^e with amax <= 448 * 2^e, e in [-100, 100]
                        const uint32_t bits = __float_as_uint(amax);
                        int e = (int)(bits >> 23) - 127 - 8 + ((bits & 0x7fffffu) > 0x600000u ? 1 : 0);
                        if ((bits >> 23) == 0) e = -100;
                        e = e < -100 ? -100 : (e > 100 ? 100 : e);
                        scale = __uint_as_float((uint32_t)(e + 127) << 23);
                    }
                    const float inv = 1.f / scale;
                    if (store_row && col0 < g.N) {
                        const int nk = g.hkv * g.dqk;
                        const bool is_k = col0 < nk;
                        const int head = is_k ? col0 / g.dqk : (col0 - nk) / g.dv;
                        uint4 *dst = reinterpret_cast<uint4 *>((is_k ? dst_k : dst_v) + (size_t)head * kPage * 128);
#pragma unroll
                        for (int v = 0; v < 8; ++v) {
                            uint32_t w[4];
#pragma unroll
                            for (int j = 0; j < 4; ++j) {
                                const int e = v * 16 + j * 4;
                                const uint32_t a = (uint32_t)__nv_cvt_float2_to_fp8x2(
                                    make_float2(__uint_as_float(r[e]) * inv, __uint_as_float(r[e + 1]) * inv), __NV_SATFINITE, __NV_E4M3);
                                const uint32_t b = (uint32_t)__nv_cvt_float2_to_fp8x2(
                                    make_float2(__uint_as_float(r[e + 2]) * inv, __uint_as_float(r[e + 3]) * inv), __NV_SATFINITE, __NV_E4M3);
                                w[j] = a | (b << 16);
                            }
                            dst[v] = make_uint4(w[0], w[1], w[2], w[3]);
                        }
                        if ((lane & 15) == 0) (is_k ? g.k_scale : g.v_scale)[(size_t)page * g.hkv + head] = scale;
                    }
                    __syncwarp();
                }
            } else {
#pragma unroll 1
            for (int cb = 0; cb < BN / 32; ++cb) {
                uint32_t r[32];
                ptx::tmem_ld32(tacc + cb * 32, r);
                ptx::tmem_wait_ld();
                const int col0 = nt * BN + cb * 32;  // first output column of these 32
                if (store_row && col0 < g.N) {
                uint4 *dst;
                if constexpr (EPI == kEpiRowMajor) {
                    dst = reinterpret_cast<uint4 *>(dst_c + col0);
                    if (res) {
                        const uint4 *rs = reinterpret_cast<const uint4 *>(res + col0);
#pragma unroll
                        for (int v = 0; v < 4; ++v) {
                            const uint4 x = rs[v];
                            const uint32_t xs[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
                            for (int e = 0; e < 4; ++e) {
                                const float2 f = ptx::bf16x2_to_f2(xs[e]);
                                r[v * 8 + 2 * e] = __float_as_uint(__uint_as_float(r[v * 8 + 2 * e]) + f.x);
                                r[v * 8 + 2 * e + 1] = __float_as_uint(__uint_as_float(r[v * 8 + 2 * e + 1]) + f.y);
                            }
                        }
                    }
                } else {
                    // columns [0, Hkv Dqk) are K heads, then V heads; 32 columns never straddle a head (D % 32 == 0)
                    const int nk = g.hkv * g.dqk;
                    if (col0 < nk) {
                        const int head = col0 / g.dqk, dim = col0 - head * g.dqk;
                        dst = reinterpret_cast<uint4 *>(dst_k + ((size_t)head * kPage * g.dqk + dim) * 2);
                    } else {
                        const int c2 = col0 - nk;
                        const int head = c2 / g.dv, dim = c2 - head * g.dv;
                        dst = reinterpret_cast<uint4 *>(dst_v + ((size_t)head * kPage * g.dv + dim) * 2);
                    }
                }
#pragma unroll
                for (int v = 0; v < 4; ++v) {
                    uint4 w;
                    w.x = ptx::pack_bf16x2(__uint_as_float(r[v * 8 + 0]), __uint_as_float(r[v * 8 + 1]));
                    w.y = ptx::pack_bf16x2(__uint_as_float(r[v * 8 + 2]), __uint_as_float(r[v * 8 + 3]));
                    w.z = ptx::pack_bf16x2(__uint_as_float(r[v * 8 + 4]), __uint_as_float(r[v * 8 + 5]));
                    w.w = ptx::pack_bf16x2(__uint_as_float(r[v * 8 + 6]), __uint_as_float(r[v * 8 + 7]));
                    if (EPI == kEpiPaged && zero_row) w = make_uint4(0u, 0u, 0u, 0u);
                    dst[v] = w;
                }
                }
                __syncwarp();  // the next tcgen05.ld is warp-collective
            }
            }
            ptx::tc_fence_before();  // our TMEM reads precede the arrive that lets the next tile overwrite the buffer
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(&acc_empty[acc]);
            if (++acc == 2) { acc = 0; acc_phase ^= 1; }
        }
    }

    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    if (warp == 1) ptx::tmem_dealloc(tmem, 512);
}

template <int EPI, int BN>
cudaError_t launch_bn(const GemmArgs &g, const GemmMaps &maps, int num_sms, cudaStream_t st) {
    auto kern = gemm_bf16_kernel<EPI, BN>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, GemmCfg<BN>::SMEM);
    if (e != cudaSuccess) return e;
    const int tiles = g.num_m_tiles * g.num_n_tiles;
    if (tiles <= 0) return cudaSuccess;
    const int grid = tiles < num_sms ? tiles : num_sms;
    kern<<<grid, GEMM_THREADS, GemmCfg<BN>::SMEM, st>>>(g, maps);
    return cudaGetLastError();
}

// 64-column tiles when 256-column tiles would occupy fewer than half of the SMs, 32-column tiles when 64-column tiles
// still would
int pick_bn(int num_m_tiles, int N, int num_sms) {
    if ((int64_t)num_m_tiles * ((N + 63) / 64) * 2 <= num_sms) return 32;
    return (int64_t)num_m_tiles * ((N + 255) / 256) * 2 <= num_sms ? 64 : 256;
}

template <int EPI>
cudaError_t launch_t(GemmArgs &g, const GemmMaps &maps, int bn, int num_sms, cudaStream_t st) {
    g.num_n_tiles = (g.N + bn - 1) / bn;
    if (bn == 32) return launch_bn<EPI, 32>(g, maps, num_sms, st);
    return bn == 64 ? launch_bn<EPI, 64>(g, maps, num_sms, st) : launch_bn<EPI, 256>(g, maps, num_sms, st);
}

cudaError_t encode_maps(const GemmProblem &p, int bn, GemmMaps *maps) {
    TensorMapBlob a, w;
    cudaError_t e = encode_tma_2d_bf16(p.a, (uint64_t)p.K, (uint64_t)p.M, (uint64_t)p.K * 2, BK, BM, &a);
    if (e != cudaSuccess) return e;
    e = encode_tma_2d_bf16(p.w, (uint64_t)p.K, (uint64_t)p.N, (uint64_t)p.K * 2, BK, (uint32_t)bn, &w);
    if (e != cudaSuccess) return e;
    static_assert(sizeof(CUtensorMap) == sizeof(TensorMapBlob), "CUtensorMap is 128 bytes");
    memcpy(&maps->a, &a, sizeof(CUtensorMap));
    memcpy(&maps->w, &w, sizeof(CUtensorMap));
    return cudaSuccess;
}

}  // namespace

// K and N: 16-byte row pitches for TMA (K % 8) and whole 64-byte epilogue stores (N % 32)
bool gemm_shape_ok(int64_t M, int32_t N, int32_t K) { return M > 0 && M < (int64_t)INT32_MAX && N > 0 && K > 0 && K % 8 == 0 && N % 32 == 0; }

cudaError_t launch_gemm_rowmajor(const GemmProblem &p, void *c, const void *residual, int num_sms, cudaStream_t stream) {
    if (!gemm_shape_ok(p.M, p.N, p.K) || !p.a || !p.w || !c) return cudaErrorInvalidValue;
    const int num_m_tiles = (int)((p.M + BM - 1) / BM);
    const int bn = pick_bn(num_m_tiles, p.N, num_sms);
    GemmMaps maps;
    cudaError_t e = encode_maps(p, bn, &maps);
    if (e != cudaSuccess) return e;
    GemmArgs g{};
    g.M = p.M;
    g.N = p.N;
    g.K = p.K;
    g.num_m_tiles = num_m_tiles;
    g.c = (__nv_bfloat16 *)c;
    g.residual = (const __nv_bfloat16 *)residual;
    return launch_t<kEpiRowMajor>(g, maps, bn, num_sms, stream);
}

cudaError_t launch_gemm_paged(const GemmProblem &p, const PoolGeom &pg, int layer, const GemmRowTile *tiles_dev,
                              int num_tiles, int num_sms, cudaStream_t stream) {
    if (!gemm_shape_ok(p.M, p.N, p.K) || !p.a || !p.w || !tiles_dev) return cudaErrorInvalidValue;
    if (p.N != pg.num_kv_heads * (pg.head_dim_qk + pg.head_dim_v)) return cudaErrorInvalidValue;
    // fp8 pools: a head's 128 columns must sit in one N tile (its amax spans them) -> 256-column tiles only
    const int bn = pg.kv_dtype == 1 ? 256 : pick_bn(num_tiles, p.N, num_sms);
    if (pg.kv_dtype == 1 && (pg.head_dim_qk != 128 || pg.head_dim_v != 128)) return cudaErrorInvalidValue;
    GemmMaps maps;
    cudaError_t e = encode_maps(p, bn, &maps);
    if (e != cudaSuccess) return e;
    GemmArgs g{};
    g.M = p.M;
    g.N = p.N;
    g.K = p.K;
    g.num_m_tiles = num_tiles;
    g.row_tiles = tiles_dev;
    const size_t kb = (size_t)kPage * pg.head_dim_qk * pg.elt_bytes(), vb = (size_t)kPage * pg.head_dim_v * pg.elt_bytes();
    g.k_layer = (char *)pg.k_arena + (size_t)layer * pg.num_pages * pg.num_kv_heads * kb;
    g.v_layer = (char *)pg.v_arena + (size_t)layer * pg.num_pages * pg.num_kv_heads * vb;
    g.hkv = pg.num_kv_heads;
    g.dqk = pg.head_dim_qk;
    g.dv = pg.head_dim_v;
    if (pg.kv_dtype == 1) {
        const size_t blocks = (size_t)pg.num_pages * pg.num_kv_heads;
        g.k_scale = pg.k_scale + (size_t)layer * blocks;
        g.v_scale = pg.v_scale + (size_t)layer * blocks;
        g.num_n_tiles = (g.N + 255) / 256;
        return launch_bn<kEpiPagedF8, 256>(g, maps, num_sms, stream);
    }
    return launch_t<kEpiPaged>(g, maps, bn, num_sms, stream);
}

}  // namespace comb
