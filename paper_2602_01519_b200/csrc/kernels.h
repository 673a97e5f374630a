// kernels.h — host-side launch interface between the C-ABI runtime (comb_host.cu) and the sm_100a
// kernels (store_kernel.cu, decode_kernel.cu, prefill_kernel.cu).  Internal; not part of the ABI.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

namespace comb {

constexpr int kPage = 16;            // tokens per page (BASELINE.json)
constexpr int kTilePages = 8;        // pages per 128-slot KV tile
constexpr int kTileSlots = kPage * kTilePages;

// One destination page of a (batched) store.  16 bytes, read once per CTA.
struct StorePageDesc {
    int32_t dst_page;   // page id inside the layer
    int32_t src_tok;    // first token row of this page in the packed source tensors
    int32_t ntok;       // valid tokens in this page (1..16); slots beyond are zero-filled
    int32_t pad;
};

// Optional bracket around a kernel launch (per-kernel CUDA-event timing, comb_profile_*).
struct LaunchHook {
    void (*begin)(void *ctx, int kernel_id, cudaStream_t st);
    void (*end)(void *ctx, cudaStream_t st);
    void *ctx;
};
enum { kKernelStore = 0, kKernelDecodeSplit = 1, kKernelDecodeMerge = 2, kKernelPrefill = 3, kKernelDecodeCascade = 4,
       kKernelCascadeMerge = 5, kKernelPrefillMerge = 6, kKernelGemm = 7, kNumKernelIds = 8 };

struct PoolGeom {
    int32_t num_layers, num_kv_heads, head_dim_qk, head_dim_v, num_pages;
    void *k_arena, *v_arena;
    // fp8 pools (include/comb.h "fp8 pools"): one byte per element, fp32 power-of-two scale per (page, kv-head) block
    int32_t kv_dtype = 0;   // 0 bf16, 1 e4m3
    float *k_scale = nullptr, *v_scale = nullptr;
    size_t elt_bytes() const { return kv_dtype == 1 ? 1 : 2; }
};

// Device pointers of a link (see comb_link_t in include/comb.h).
struct LinkView {
    const int32_t *page_indptr, *page_ids, *kv_len, *tile_indptr;
    const uint8_t *page_ntok;
    const uint64_t *tile_ntok;
    // chunk-major view (distinct chunks as slots) + the entries of every request
    const int32_t *entry_indptr, *cas_page_indptr, *cas_page_ids, *cas_tile_indptr;
    const uint64_t *cas_tile_ntok;
    const int32_t *cas_row_indptr, *cas_row_req, *cas_row_entry;
};

// ---- (a2) store -------------------------------------------------------------------------------
cudaError_t launch_store(const PoolGeom &g, int layer, const StorePageDesc *descs_dev, int num_descs,
                         const void *k_src, const void *v_src, cudaStream_t stream);

// fp8 pool: quantising store (same descriptors; bf16 source, e4m3 codes + scales out). D = 128 only.
cudaError_t launch_store_fp8(const PoolGeom &g, int layer, const StorePageDesc *descs_dev, int num_descs,
                             const void *k_src, const void *v_src, cudaStream_t stream);
// fp8 pool: dequantise `num_pages` pages (ids in page_ids_dev, e.g. the distinct pages of a link) of `layer` into compact
// bf16 staging arenas k_out / v_out [num_pages][Hkv][16][128] (page i of the staging = page_ids[i] of the pool).
cudaError_t launch_dequant_pages(const PoolGeom &g, int layer, const int32_t *page_ids_dev, int num_pages, void *k_out,
                                 void *v_out, cudaStream_t stream);

// read-only HBM stream over `bytes` bytes (measurement utility; `sink` = 4 device bytes)
cudaError_t launch_stream_read(const void *src, size_t bytes, void *sink, cudaStream_t stream);

// ---- (a5) decode ------------------------------------------------------------------------------
struct DecodePlan {
    int chunk_pages;   // table entries per split (multiple of the warps per CTA)
    int num_splits;    // splits of the longest request
};
DecodePlan make_decode_plan(int num_requests, int cta_columns /* Hkv x head sub-groups */, int max_pages_per_request,
                            int num_sms);
size_t decode_workspace_bytes(int num_requests, int num_q_heads, int head_dim_v, const DecodePlan &p);
bool decode_supported(int group, int dqk, int dv);
int decode_head_subgroups(int group);  // CTAs per (request, kv-head, split): 1 for G <= 4, G/4 above
// launches the split kernel and (if num_splits > 1) the merge kernel; *launches += kernels launched
cudaError_t launch_decode(const PoolGeom &g, int layer, const LinkView &lv, int num_requests, int num_q_heads,
                          const void *q, float scale, void *out, float *lse, void *workspace, const DecodePlan &p,
                          cudaStream_t stream, int *launches, const LaunchHook *hook);

// ---- (a4) prefill -----------------------------------------------------------------------------
// One CTA work item: up to two consecutive 128-row Q tiles of one (request, kv-head) against a range of the
// request's 128-slot KV tiles. A request's KV is cut into `nsplit` ranges when there are too few items to fill the
// GPU (low-parallelism shapes: few requests, few query tokens); the ranges' partial results are merged by LSE.
struct PrefillItem {
    int32_t request;
    int32_t kv_head;
    int32_t q_row0;     // first query token row (absolute row in q) of tile 0
    int32_t q_rows;     // valid query tokens in this item (1 .. 2*128/G)
    int32_t kv_tile0;   // first KV tile of this item (index inside the request)
    int32_t kv_tiles;   // KV tiles of this item (clamped to the request's on the device; the last range is open-ended)
    int32_t split;      // -1: the item sees all of the request's KV and writes the final output; else its range index
    int32_t tps;        // split >= 0: tiles per range of this request (the merge derives the range count from it)
    int32_t part_base;  // split >= 0: first partial row of this item's ranges; range s, tile slot t, tile row i lives
                        // at part_base + s * 256 + t * 128 + i
    int32_t pad;
};
constexpr int kPrefillMaxSplits = 16;
// Splits of a request with n_kv tiles when the call uses `nsplit` ranges: ceil(n_kv / ceil(n_kv / nsplit)).
inline int prefill_tiles_per_split(int n_kv, int nsplit) { return (n_kv + nsplit - 1) / nsplit; }
// Q tiles per CTA (1 or 2) for a call whose longest request has max_q_tokens query tokens and that would have
// num_items single-tile items; an item then covers up to that many 128-row tiles.
int prefill_tiles_per_cta(int group, int dqk, int dv, int64_t max_q_tokens, int64_t num_items, int num_sms);
int prefill_ctas_per_sm(int tiles_per_cta, int dqk, int dv);  // resident CTAs per SM of the kernel that choice selects
bool prefill_supported(int group, int dqk, int dv);
// CUtensorMap is 128 bytes, 64-byte aligned; kept opaque here so the runtime needs no cuda.h.
struct alignas(64) TensorMapBlob { unsigned char bytes[128]; };
struct PrefillMaps { TensorMapBlob q, k, v; };
// Encodes the TMA maps (k/v depend on pool + layer-independent geometry; q on the call).
cudaError_t prefill_encode_kv_maps(const PoolGeom &g, TensorMapBlob *k_map, TensorMapBlob *v_map);
cudaError_t prefill_encode_q_map(const void *q, int64_t total_q, int num_q_heads, int group, int dqk,
                                 TensorMapBlob *q_map);
// part_rows > 0: some items are KV ranges; `partials` holds part_rows x (Dv + 1) floats and a second kernel merges
// the ranges (*launches += 1).  paired: items (2i, 2i + 1) have the same (request, kv-head) and see all of its KV, so a
// cluster of two CTAs may share their K/V stream (TMA multicast).
cudaError_t launch_prefill(const PoolGeom &g, int layer, const LinkView &lv, const PrefillMaps &maps,
                           const PrefillItem *items_dev, int num_items, int num_q_heads, float scale, void *out,
                           float *lse, int64_t total_q, void *partials, int64_t part_rows, int tiles_per_cta,
                           bool paired, int num_sms, cudaStream_t stream, int *launches, const LaunchHook *hook);

// Dense row-major bf16 matrix [outer][inner] -> 2-D TMA map with SWIZZLE_128B boxes {box_inner (<= 64), box_outer}.
cudaError_t encode_tma_2d_bf16(const void *base, uint64_t inner, uint64_t outer, uint64_t row_pitch_bytes,
                               uint32_t box_inner, uint32_t box_outer, TensorMapBlob *out);

cudaError_t encode_tma_2d_u8(const void *base, uint64_t inner, uint64_t outer, uint64_t row_pitch_bytes,
                             uint32_t box_inner, uint32_t box_outer, TensorMapBlob *out);

// ---- (f1) chunk-major ("cascade") decode --------------------------------------------------------
// One work unit of the chunk-major decode: up to 32/G consecutive entries (query tokens) of chunk slot `slot`, starting
// at position row0 of cas_row_req / cas_row_entry (each entry contributes the G rows of one kv-head), against KV tiles
// [kv_tile0, kv_tile0 + kv_tiles) of the chunk. A work item of the kernel is (unit, kv-head).
// Every (entry, KV range) pair owns one partial result; entry i of the slot at range s has partial index
// part_base + s * part_stride + i, and `part0` is that index for the unit's first entry and its own range.
struct CascadeItem {
    int32_t slot, row0, nrows;
    int32_t kv_tile0, kv_tiles;
    int32_t part0;        // partial index of entry row0 at this unit's range
    int32_t part_stride;  // entries of the slot (distance between the ranges of one entry)
    int32_t range_nr;     // (number of ranges of the slot << 8) | this unit's range index
    // where the unit's KV lives in the chunk-major tables (filled by the planner from the host mirror, so the kernel's
    // scheduler needs no dependent table lookups): first entry of cas_page_ids, number of pages, first cas_tile_ntok
    int32_t pbeg, npages, tile0, pad;
};
// device workspace of one chunk-major decode call:
//   [0, 16)  header (uint32 item counter, zero)   [16, ..) CascadeItem[num_units]     -- one H2D copy
//   then int4 ent_info[E] (written by the kernel: where the merge finds an entry's partials),
//   then float part_o[P][Hq][Dv], float part_lse[P][Hq]        (P = partial indices in all)
constexpr size_t kCascadeHeaderBytes = 16;
struct CascadeLayout {
    size_t off_items, off_ent, off_part_o, off_part_lse, bytes;
    int64_t num_partials;  // (entry, KV range) partials of the call: the merge picks its warps per row from it
};
CascadeLayout cascade_layout(size_t num_units, int64_t total_entries, int64_t num_partials, int num_q_heads, int dv);
bool cascade_supported(int group, int dqk, int dv);
// tcgen05 kernel over (unit, kv-head) items writing per-(entry, range) partials, then the per-request LSE merge.
cudaError_t launch_decode_cascade(const PoolGeom &g, int layer, const LinkView &lv, const PrefillMaps &maps,
                                  void *workspace, const CascadeLayout &lay, int num_units, int num_requests,
                                  int num_q_heads, const void *q, float scale, void *out, float *lse, int num_sms,
                                  cudaStream_t stream, int *launches, const LaunchHook *hook);

// ---- (f2)/(f3) projections: C = A W^T on tcgen05 ---------------------------------------------------
// A bf16 [M][K] row-major, W bf16 [N][K] row-major (the nn.Linear layout: row n holds the weights of output n),
// fp32 accumulation in TMEM. Two epilogues:
//   row-major : C bf16 [M][N] = bf16(acc (+ residual[M][N]))                                (Eq. 4; output projection)
//   paged     : the columns are [K heads | V heads] of a chunk-KV pool layer; row t of a chunk goes straight into
//               slot t % 16 of the chunk's page t / 16, tail slots of the last page are zero-filled   (Eq. 5-6 + store)
// One M tile of the paged epilogue: 128 rows of A starting at a_row0; rows < rows_valid are tokens, rows in
// [rows_valid, rows_zero_to) are the zero-filled tail of the chunk's last page, the rest is not written.
struct GemmRowTile {
    int32_t a_row0, rows_valid, rows_zero_to, pad;
    int32_t pages[8];  // destination page of rows 16 i .. 16 i + 15 (-1: none)
};
struct GemmProblem {
    const void *a;
    const void *w;
    int64_t M;
    int32_t N, K;
};
cudaError_t launch_gemm_rowmajor(const GemmProblem &p, void *c, const void *residual, int num_sms, cudaStream_t stream);
cudaError_t launch_gemm_paged(const GemmProblem &p, const PoolGeom &g, int layer, const GemmRowTile *tiles_dev,
                              int num_tiles, int num_sms, cudaStream_t stream);
bool gemm_shape_ok(int64_t M, int32_t N, int32_t K);

}  // namespace comb
