// decode_kernel.cu — (a5) decode cross-attention: one query row per request attends, without mask, over
// the request's block-table-linked chunk KV (§4 "newly generated tokens are ... treated
// identically to the initial query tokens"; Eq. 7-8; PAPER.md:119 concatenation).
//
// HBM-bound (4 flop/B at GQA 4, 1 flop/B at G = 1): no tensor cores, the math is GEMV-shaped.
//   pass 1  decode_split_kernel: grid (split, kv-head, request). Each of the CTA's 4 warps streams its own
//           pages through a private ring of shared-memory stages filled by 1-D TMA bulk copies (one
//           contiguous 16 x D burst per (page, kv-head) for K and for V, completion on an mbarrier), so
//           ~100 KB of loads are in flight per SM with no register staging. 8 lanes share a key (128-bit
//           conflict-free LDS), FFMA2 dot products, a reduce-scatter butterfly of warp shuffles, online
//           softmax in the log2 domain with lazy rescale, then P.V. Warps merge through shared memory.
//   pass 2  decode_merge_kernel: LSE-merge of the splits (SURVEY.md §8(c) pin P8).
// Algorithmic bytes: 2 B * Hkv * (Dqk + Dv) per linked key, read once.
#include "kernels.h"
#include "ptx.cuh"

#include <algorithm>
#include <cuda_bf16.h>

namespace comb {
namespace {

constexpr int kWarps = 4;
constexpr int kThreads = kWarps * 32;
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;

struct DecodeArgs {
    const char *k_layer;  // bf16 [num_pages][Hkv][16][Dqk]
    const char *v_layer;  // bf16 [num_pages][Hkv][16][Dv]
    const int32_t *page_indptr, *page_ids;
    const uint8_t *page_ntok;
    const uint16_t *q;  // bf16 [R][Hq][Dqk]
    __nv_bfloat16 *out;  // [R][Hq][Dv]
    float *lse;          // [R][Hq] or null
    float *part_o;       // [R][Hq][S][Dv]
    float *part_ml;      // [R][Hq][S][2]  (m in log2 units, l)
    int num_q_heads, num_kv_heads, chunk_pages, num_splits;
    int group;   // Hq / Hkv (q heads per kv head)
    int hsub;    // head sub-groups per kv head: a CTA owns G = group / hsub consecutive q heads (hsub > 1 for group 8, 16)
    float scale_log2;  // scale * log2(e)
};

template <int G, int DQK, int DV>
struct Cfg {
    static constexpr int CK = DQK / 64;  // 16-byte chunks of a K row per lane (8 lanes per key)
    static constexpr int CV = DV / 64;
    static constexpr int KB = kPage * DQK * 2;  // bytes of one (page, kv-head) K block
    static constexpr int VB = kPage * DV * 2;
    static constexpr int NSTAGE = (KB + VB > 8192) ? 2 : 3;
    static constexpr int HPL = (G >= 2) ? G / 2 : 1;  // heads per lane after the reduce-scatter
    static constexpr int N = 4 * G;                   // partial dot products per lane per page (4 passes)
    static constexpr size_t RING = (size_t)kWarps * NSTAGE * (KB + VB);
    static constexpr size_t MERGE = (size_t)kWarps * 4 * G * DV * sizeof(float);
    static constexpr size_t BODY = RING > MERGE ? RING : MERGE;
    static constexpr size_t TAIL = 128 + (size_t)kWarps * kPage * G * sizeof(float);  // mbarriers + P staging
    static constexpr size_t SMEM = BODY + TAIL;
};

// Sum N per-lane values over the 8 lanes that share a key; afterwards lane `sub` holds max(1, N/8) sums:
// for N >= 8 the values idx = sub*(N/8) + t, for N = 4 the value idx = sub/2 (lane pairs hold copies).
template <int NCUR, int OFF, int N>
__device__ __forceinline__ void reduce_scatter_step(float (&v)[N], int sub) {
    if constexpr (OFF >= 1) {
        if constexpr (NCUR >= 2) {
            constexpr int half = NCUR / 2;
            const bool upper = (sub & OFF) != 0;
#pragma unroll
            for (int t = 0; t < half; ++t) {
                const float send = upper ? v[t] : v[t + half];
                const float keep = upper ? v[t + half] : v[t];
                v[t] = keep + __shfl_xor_sync(0xffffffffu, send, OFF);
            }
            reduce_scatter_step<half, OFF / 2>(v, sub);
        } else {
            v[0] += __shfl_xor_sync(0xffffffffu, v[0], OFF);
            reduce_scatter_step<1, OFF / 2>(v, sub);
        }
    }
}
template <int N>
__device__ __forceinline__ void reduce_scatter8(float (&v)[N], int sub) {
    reduce_scatter_step<N, 4>(v, sub);
}

template <int G, int DQK, int DV>
__global__ void __launch_bounds__(kThreads, 2) decode_split_kernel(const DecodeArgs a) {
    using C = Cfg<G, DQK, DV>;
    extern __shared__ __align__(128) unsigned char smem[];
    // 1-D grid over (request, kv-head, head sub-group, split), split fastest (no 65535 limit on any factor)
    const int split = blockIdx.x % a.num_splits;
    const int gy = (blockIdx.x / a.num_splits) % (a.num_kv_heads * a.hsub);
    const int r = blockIdx.x / (a.num_splits * a.num_kv_heads * a.hsub);
    const int g = gy / a.hsub;                          // kv head: whose K/V blocks are streamed
    const int head0 = g * a.group + (gy % a.hsub) * G;  // first of this CTA's G query heads
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int sub = lane & 7, kg = lane >> 3;
    const int Hq = a.num_q_heads;

    const int pbeg_r = a.page_indptr[r], pend_r = a.page_indptr[r + 1];
    const int npages_r = pend_r - pbeg_r;
    if (npages_r == 0) {  // no contexts linked: zero contribution, lse = -inf (reading I13)
        if (split == 0) {
            for (int e = tid; e < G * DV; e += kThreads)
                a.out[((size_t)r * Hq + head0 + e / DV) * DV + e % DV] = __float2bfloat16_rn(0.f);
            if (a.lse && tid < G) a.lse[(size_t)r * Hq + head0 + tid] = -INFINITY;
        }
        return;
    }
    const int nsplit_r = (npages_r + a.chunk_pages - 1) / a.chunk_pages;
    if (split >= nsplit_r) return;
    const int pb = pbeg_r + split * a.chunk_pages;
    const int pe = min(pend_r, pb + a.chunk_pages);
    const int n_w = (pe - pb > warp) ? (pe - pb - warp + kWarps - 1) / kWarps : 0;  // pages of this warp

    unsigned char *ring = smem + (size_t)warp * C::NSTAGE * (C::KB + C::VB);
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + C::BODY) + warp * C::NSTAGE;
    float *pbuf = reinterpret_cast<float *>(smem + C::BODY + 128) + warp * (kPage * G);
    static_assert(kWarps * C::NSTAGE * 8 <= 128, "mbarriers fit the first 128 bytes of the tail");

    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < C::NSTAGE; ++s) ptx::mbar_init(&bars[s], 1);
        ptx::fence_barrier_init();
        ptx::fence_proxy_async_smem();
    }
    __syncwarp();

    // ---- q for the G heads of this kv-head, this lane's dims, pre-scaled into the log2 domain ----
    float2 q2[G][C::CK * 4];
#pragma unroll
    for (int h = 0; h < G; ++h) {
        const uint4 *qrow = reinterpret_cast<const uint4 *>(a.q + ((size_t)r * Hq + head0 + h) * DQK);
#pragma unroll
        for (int cc = 0; cc < C::CK; ++cc) {
            const uint4 w = qrow[cc * 8 + sub];
            const uint32_t ww[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                float2 f = ptx::bf16x2_to_f2(ww[e]);
                q2[h][cc * 4 + e] = make_float2(f.x * a.scale_log2, f.y * a.scale_log2);
            }
        }
    }

    // ---- block-table caches: lane i holds the entry of this warp's (blk*32 + i)-th page ----
    int iss_blk = -1, iss_id = 0, cmp_blk = -1, cmp_nt = 0;
    auto issue = [&](int i) {
        const int blk = i >> 5;
        if (blk != iss_blk) {
            const int mine = blk * 32 + lane;
            iss_id = (mine < n_w) ? a.page_ids[pb + warp + kWarps * mine] : 0;
            iss_blk = blk;
        }
        const int pid = __shfl_sync(0xffffffffu, iss_id, i & 31);
        if (lane == 0) {
            const int s = i % C::NSTAGE;
            unsigned char *dst = ring + (size_t)s * (C::KB + C::VB);
            const size_t blk_idx = (size_t)pid * a.num_kv_heads + g;
            ptx::fence_proxy_async_smem();  // order this warp's earlier reads of the stage before the refill
            ptx::mbar_expect_tx(&bars[s], C::KB + C::VB);
            ptx::bulk_g2s(dst, a.k_layer + blk_idx * C::KB, C::KB, &bars[s]);
            ptx::bulk_g2s(dst + C::KB, a.v_layer + blk_idx * C::VB, C::VB, &bars[s]);
        }
    };

#pragma unroll 1
    for (int i = 0; i < C::NSTAGE && i < n_w; ++i) issue(i);

    float m_run[G];
    float l_part[C::HPL];
    float2 o2[G][C::CV * 4];
#pragma unroll
    for (int h = 0; h < G; ++h) {
        m_run[h] = -INFINITY;
#pragma unroll
        for (int e = 0; e < C::CV * 4; ++e) o2[h][e] = make_float2(0.f, 0.f);
    }
#pragma unroll
    for (int t = 0; t < C::HPL; ++t) l_part[t] = 0.f;

#pragma unroll 1
    for (int i = 0; i < n_w; ++i) {
        const int s = i % C::NSTAGE;
        {
            const int blk = i >> 5;
            if (blk != cmp_blk) {
                const int mine = blk * 32 + lane;
                cmp_nt = (mine < n_w) ? a.page_ntok[pb + warp + kWarps * mine] : 0;
                cmp_blk = blk;
            }
        }
        const int ntok = __shfl_sync(0xffffffffu, cmp_nt, i & 31);
        ptx::mbar_wait(&bars[s], (uint32_t)(i / C::NSTAGE) & 1u);
        const unsigned char *ks = ring + (size_t)s * (C::KB + C::VB);
        const unsigned char *vs = ks + C::KB;

        // ---- scores: 4 passes x 4 keys; this lane's partial dot products for its 8*CK dims ----
        float acc[C::N];
#pragma unroll
        for (int ip = 0; ip < 4; ++ip) {
            const uint4 *krow = reinterpret_cast<const uint4 *>(ks + (size_t)(ip * 4 + kg) * (DQK * 2));
            float2 a2[G];
#pragma unroll
            for (int h = 0; h < G; ++h) a2[h] = make_float2(0.f, 0.f);
#pragma unroll
            for (int cc = 0; cc < C::CK; ++cc) {
                const uint4 w = krow[cc * 8 + sub];
                const uint32_t ww[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const float2 kf = ptx::bf16x2_to_f2(ww[e]);
#pragma unroll
                    for (int h = 0; h < G; ++h) a2[h] = ptx::ffma2(q2[h][cc * 4 + e], kf, a2[h]);
                }
            }
#pragma unroll
            for (int h = 0; h < G; ++h) acc[ip * G + h] = a2[h].x + a2[h].y;
        }
        reduce_scatter8<C::N>(acc, sub);
        // now: key j = (sub/2)*4 + kg, heads h0 .. h0+HPL-1 with h0 = (sub&1)*HPL (G = 1: h0 = 0, pairs hold copies)
        const int j = (sub >> 1) * 4 + kg;
        const bool odd = (sub & 1) != 0;
        float sc[C::HPL], mx[C::HPL];
#pragma unroll
        for (int t = 0; t < C::HPL; ++t) {
            sc[t] = (j < ntok) ? acc[t] : -INFINITY;  // slots past the chunk's length are masked (reading I12)
            mx[t] = sc[t];
        }
#pragma unroll
        for (int off = 2; off <= 16; off <<= 1)
#pragma unroll
            for (int t = 0; t < C::HPL; ++t) mx[t] = fmaxf(mx[t], __shfl_xor_sync(0xffffffffu, mx[t], off));
        float mall[G];
        if constexpr (G == 1) {
            mall[0] = mx[0];
        } else {
#pragma unroll
            for (int t = 0; t < C::HPL; ++t) {
                const float other = __shfl_xor_sync(0xffffffffu, mx[t], 1);
                mall[t] = odd ? other : mx[t];
                mall[C::HPL + t] = odd ? mx[t] : other;
            }
        }
        bool changed = false;
#pragma unroll
        for (int h = 0; h < G; ++h) changed |= mall[h] > m_run[h];
        if (changed) {  // warp-uniform: every lane holds the same mall / m_run
            float corr[G];
#pragma unroll
            for (int h = 0; h < G; ++h) {
                const float mn = fmaxf(m_run[h], mall[h]);
                corr[h] = ptx::ex2(m_run[h] - mn);  // ex2(-inf) = 0 on the first page
                m_run[h] = mn;
                const float2 c2 = make_float2(corr[h], corr[h]);
#pragma unroll
                for (int e = 0; e < C::CV * 4; ++e) o2[h][e] = ptx::fmul2(o2[h][e], c2);
            }
#pragma unroll
            for (int t = 0; t < C::HPL; ++t) {
                if constexpr (G == 1) l_part[t] *= corr[0];
                else l_part[t] *= odd ? corr[C::HPL + t] : corr[t];
            }
        }
        float p[C::HPL];
#pragma unroll
        for (int t = 0; t < C::HPL; ++t) {
            float mine;
            if constexpr (G == 1) mine = m_run[0];
            else mine = odd ? m_run[C::HPL + t] : m_run[t];
            p[t] = ptx::ex2(sc[t] - mine);
            l_part[t] += (G == 1 && odd) ? 0.f : p[t];
            pbuf[j * G + ((G == 1) ? 0 : (odd ? C::HPL : 0)) + t] = p[t];
        }
        __syncwarp();

        // ---- O += P V : same lane/key mapping, this lane's 8*CV output dims ----
#pragma unroll
        for (int ip = 0; ip < 4; ++ip) {
            const int jj = ip * 4 + kg;
            float pv[G];
#pragma unroll
            for (int h = 0; h < G; ++h) pv[h] = pbuf[jj * G + h];
            const uint4 *vrow = reinterpret_cast<const uint4 *>(vs + (size_t)jj * (DV * 2));
#pragma unroll
            for (int cc = 0; cc < C::CV; ++cc) {
                const uint4 w = vrow[cc * 8 + sub];
                const uint32_t ww[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const float2 vf = ptx::bf16x2_to_f2(ww[e]);
#pragma unroll
                    for (int h = 0; h < G; ++h)
                        o2[h][cc * 4 + e] = ptx::ffma2(make_float2(pv[h], pv[h]), vf, o2[h][cc * 4 + e]);
                }
            }
        }
        __syncwarp();
        if (i + C::NSTAGE < n_w) issue(i + C::NSTAGE);
    }

    // ---- merge the 4 warps (and the 4 key groups inside each warp) through shared memory ----
#pragma unroll
    for (int off = 2; off <= 16; off <<= 1)
#pragma unroll
        for (int t = 0; t < C::HPL; ++t) l_part[t] += __shfl_xor_sync(0xffffffffu, l_part[t], off);
    __syncthreads();  // every warp is done with its ring: the merge buffers alias it
    float *o_part = reinterpret_cast<float *>(smem);                       // [warp][kg][G][DV]
    float *m_w = pbuf - warp * (kPage * G);                                // reuse pbuf area: [warp][G] m, then l
    float *l_w = m_w + kWarps * G;
    static_assert(2 * kWarps * G <= kWarps * kPage * G, "m/l scratch fits the P staging area");
#pragma unroll
    for (int h = 0; h < G; ++h)
#pragma unroll
        for (int cc = 0; cc < C::CV; ++cc)
#pragma unroll
            for (int e = 0; e < 4; ++e)
                *reinterpret_cast<float2 *>(o_part + ((size_t)(warp * 4 + kg) * G + h) * DV + (cc * 8 + sub) * 8 + 2 * e) =
                    o2[h][cc * 4 + e];
    if (lane == 0)
#pragma unroll
        for (int h = 0; h < G; ++h) m_w[warp * G + h] = m_run[h];
    if (kg == 0 && sub < 2 && (G > 1 || sub == 0))
#pragma unroll
        for (int t = 0; t < C::HPL; ++t) l_w[warp * G + ((G == 1) ? 0 : sub * C::HPL) + t] = l_part[t];
    __syncthreads();

    for (int e = tid; e < G * DV; e += kThreads) {
        const int h = e / DV, d = e - h * DV;
        float m = -INFINITY;
#pragma unroll
        for (int w = 0; w < kWarps; ++w) m = fmaxf(m, m_w[w * G + h]);
        float o = 0.f, l = 0.f;
#pragma unroll
        for (int w = 0; w < kWarps; ++w) {
            const float mw = m_w[w * G + h];
            const float wt = (mw == -INFINITY) ? 0.f : ptx::ex2(mw - m);
            float x = 0.f;
#pragma unroll
            for (int k4 = 0; k4 < 4; ++k4) x += o_part[((size_t)(w * 4 + k4) * G + h) * DV + d];
            o += wt * x;
            l += wt * l_w[w * G + h];
        }
        const int hq = head0 + h;
        if (nsplit_r == 1) {
            a.out[((size_t)r * Hq + hq) * DV + d] = __float2bfloat16_rn(o / l);
            if (a.lse && d == 0) a.lse[(size_t)r * Hq + hq] = (m + log2f(l)) * kLn2;
        } else {
            const size_t slot = ((size_t)r * Hq + hq) * a.num_splits + split;
            a.part_o[slot * DV + d] = o;
            if (d == 0) {
                a.part_ml[slot * 2 + 0] = m;
                a.part_ml[slot * 2 + 1] = l;
            }
        }
    }
}

// pass 2: out = sum_s e^{m_s - m} o_s / sum_s e^{m_s - m} l_s ; lse = ln2 * (m + log2 l)
template <int DV>
__global__ void __launch_bounds__(DV) decode_merge_kernel(const DecodeArgs a) {
    const int hq = blockIdx.x % a.num_q_heads, r = blockIdx.x / a.num_q_heads, d = threadIdx.x;
    const int npages_r = a.page_indptr[r + 1] - a.page_indptr[r];
    const int nsplit_r = (npages_r + a.chunk_pages - 1) / a.chunk_pages;
    if (nsplit_r <= 1) return;  // written by pass 1
    const size_t base = ((size_t)r * a.num_q_heads + hq) * a.num_splits;
    float m = -INFINITY;
    for (int s = 0; s < nsplit_r; ++s) m = fmaxf(m, a.part_ml[(base + s) * 2]);
    float o = 0.f, l = 0.f;
    for (int s = 0; s < nsplit_r; ++s) {
        const float wt = ptx::ex2(a.part_ml[(base + s) * 2] - m);
        o += wt * a.part_o[(base + s) * DV + d];
        l += wt * a.part_ml[(base + s) * 2 + 1];
    }
    a.out[((size_t)r * a.num_q_heads + hq) * DV + d] = __float2bfloat16_rn(o / l);
    if (a.lse && d == 0) a.lse[(size_t)r * a.num_q_heads + hq] = (m + log2f(l)) * kLn2;
}

template <int G, int DQK, int DV>
cudaError_t launch_t(const DecodeArgs &a, int R, bool merge, cudaStream_t st, int *launches, const LaunchHook *hook) {
    using C = Cfg<G, DQK, DV>;
    auto kern = decode_split_kernel<G, DQK, DV>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);
    if (e != cudaSuccess) return e;
    const unsigned grid = (unsigned)((size_t)a.num_splits * a.num_kv_heads * a.hsub * R);
    if (hook) hook->begin(hook->ctx, kKernelDecodeSplit, st);
    kern<<<grid, kThreads, C::SMEM, st>>>(a);
    if (hook) hook->end(hook->ctx, st);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    *launches += 1;
    if (merge) {
        if (hook) hook->begin(hook->ctx, kKernelDecodeMerge, st);
        decode_merge_kernel<DV><<<(unsigned)((size_t)a.num_q_heads * R), DV, 0, st>>>(a);
        if (hook) hook->end(hook->ctx, st);
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
        *launches += 1;
    }
    return cudaSuccess;
}

}  // namespace

// Every group size prefill accepts (powers of two up to 16): groups of 8 and 16 heads run as 2 or 4 sub-groups of
// 4 heads, each its own CTA streaming the same K/V blocks (the second read is an L2 hit).
bool decode_supported(int group, int dqk, int dv) {
    const bool dims = (dqk == 64 || dqk == 128 || dqk == 192) && (dv == 64 || dv == 128);
    return dims && group >= 1 && group <= 16 && (group & (group - 1)) == 0;
}
int decode_head_subgroups(int group) { return group > 4 ? group / 4 : 1; }

// `Hkv` here counts the CTA columns per request: kv heads x head sub-groups.
DecodePlan make_decode_plan(int R, int Hkv, int max_pages, int num_sms) {
    DecodePlan p;
    if (max_pages <= 0 || R <= 0) {
        p.chunk_pages = kWarps;
        p.num_splits = 1;
        return p;
    }
    // aim for ~4 waves of 2 CTAs per SM, but never fewer than 16 pages (4 per warp) per split; around that target
    // take the split count whose CTA total fills its last wave best (8 requests x 8 kv-heads x 19 splits would run
    // 4.1 waves, x 18 splits 3.9)
    const long units = (long)R * Hkv;
    const long wave = (long)num_sms * 2;
    const long target = wave * 4;
    const long cap = std::max(1L, (long)(max_pages + 15) / 16);
    const long ns0 = std::max(1L, std::min((target + units - 1) / units, cap));
    long best = ns0;
    double best_eff = 0.0;
    for (long ns = std::max(1L, ns0 - ns0 / 4); ns <= std::min(cap, ns0 + ns0 / 4); ++ns) {
        int chunk = (int)((max_pages + ns - 1) / ns);
        chunk = (chunk + kWarps - 1) / kWarps * kWarps;
        const long eff_ns = (max_pages + chunk - 1) / chunk;  // splits the longest request really gets
        const long ctas = units * eff_ns;
        const double eff = (double)ctas / (double)((ctas + wave - 1) / wave * wave);
        if (eff > best_eff + 1e-9) { best_eff = eff; best = ns; }
    }
    int chunk = (int)((max_pages + best - 1) / best);
    chunk = (chunk + kWarps - 1) / kWarps * kWarps;
    p.chunk_pages = chunk;
    p.num_splits = (max_pages + chunk - 1) / chunk;
    return p;
}

size_t decode_workspace_bytes(int R, int Hq, int dv, const DecodePlan &p) {
    if (p.num_splits <= 1) return 0;
    return (size_t)R * Hq * p.num_splits * (dv + 2) * sizeof(float);
}

cudaError_t launch_decode(const PoolGeom &g, int layer, const LinkView &lv, int R, int Hq, const void *q, float scale,
                          void *out, float *lse, void *workspace, const DecodePlan &p, cudaStream_t stream,
                          int *launches, const LaunchHook *hook) {
    DecodeArgs a;
    const size_t kb = (size_t)kPage * g.head_dim_qk * 2, vb = (size_t)kPage * g.head_dim_v * 2;
    a.k_layer = (const char *)g.k_arena + (size_t)layer * g.num_pages * g.num_kv_heads * kb;
    a.v_layer = (const char *)g.v_arena + (size_t)layer * g.num_pages * g.num_kv_heads * vb;
    a.page_indptr = lv.page_indptr;
    a.page_ids = lv.page_ids;
    a.page_ntok = lv.page_ntok;
    a.q = (const uint16_t *)q;
    a.out = (__nv_bfloat16 *)out;
    a.lse = lse;
    a.num_q_heads = Hq;
    a.num_kv_heads = g.num_kv_heads;
    a.group = Hq / g.num_kv_heads;
    a.hsub = decode_head_subgroups(a.group);
    a.chunk_pages = p.chunk_pages;
    a.num_splits = p.num_splits;
    a.scale_log2 = scale * kLog2e;
    a.part_o = (float *)workspace;
    a.part_ml = a.part_o ? a.part_o + (size_t)R * Hq * p.num_splits * g.head_dim_v : nullptr;
    const bool merge = p.num_splits > 1;
    const int G = a.group / a.hsub;  // heads per CTA
#define COMB_DECODE_CASE(GG, DQ, DVV) \
    if (G == GG && g.head_dim_qk == DQ && g.head_dim_v == DVV) return launch_t<GG, DQ, DVV>(a, R, merge, stream, launches, hook);
    COMB_DECODE_CASE(4, 128, 128)
    COMB_DECODE_CASE(4, 64, 64)
    COMB_DECODE_CASE(1, 192, 128)
    COMB_DECODE_CASE(1, 128, 128)
    COMB_DECODE_CASE(1, 64, 64)
    COMB_DECODE_CASE(2, 128, 128)
    COMB_DECODE_CASE(2, 64, 64)
    COMB_DECODE_CASE(4, 192, 128)
    COMB_DECODE_CASE(2, 192, 128)
    COMB_DECODE_CASE(1, 128, 64)
    COMB_DECODE_CASE(2, 128, 64)
    COMB_DECODE_CASE(4, 128, 64)
    COMB_DECODE_CASE(1, 64, 128)
    COMB_DECODE_CASE(2, 64, 128)
    COMB_DECODE_CASE(4, 64, 128)
    COMB_DECODE_CASE(1, 192, 64)
    COMB_DECODE_CASE(2, 192, 64)
    COMB_DECODE_CASE(4, 192, 64)
#undef COMB_DECODE_CASE
    return cudaErrorInvalidValue;
}

}  // namespace comb
