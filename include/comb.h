/*
 * comb.h — C ABI of the COMB link-stage hot path on B200 (sm_100a).
 *
 * The calls follow the paper's compile/link statement of the problem (arxiv 2602.01519;
 * PAPER.md = the text under /root/reference at authoring time):
 *   lookup -> (miss) allocate -> compile -> store -> update table -> fetch/link -> attend with the
 *   query tokens -> attend with every generated token   (§3 steps 1-8, §5.3,
 *   PAPER.md:66 §4).
 *
 * Conventions
 *   - Every function returns int32_t: COMB_OK (0) or a negative comb_status_t. No exception or abort
 *     crosses the ABI.
 *   - "device" pointers are CUDA device pointers on the current device; "host" pointers are ordinary
 *     host memory. `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).
 *   - NO function synchronises the device. Kernels and copies are enqueued on `stream`. (A call may
 *     block the host on an event only when its staging ring of 4 slots is full, i.e. the GPU is four
 *     calls behind.)
 *   - The library allocates NO device memory: arenas, scratch, link buffers, Q/O and workspace are
 *     allocated by the caller (PyTorch) and stay caller-owned; they must outlive their use on the
 *     stream. Host metadata (directory, free list, pinned staging) belongs to the pool and is freed by
 *     comb_pool_destroy.
 *   - A pool is not thread-safe; callers serialise. The paper stores PICaches "asynchronously":
 *     a store may run on any stream; comb_link orders its own stream after the stores of the chunks it names
 *     (see (f4) "ready"), so an attention call that follows a comb_link on the same stream reads complete pages.
 *     A caller that writes link tables itself orders streams itself.
 *   - dtype: bf16 storage for Q, K, V and O (bit patterns, 2 bytes); fp32 statistics (lse).
 *
 * Layout of the chunk-KV pool (part of the bit-exact contract)
 *   K arena  bf16 [num_layers][num_pages][num_kv_heads][16][head_dim_qk]
 *   V arena  bf16 [num_layers][num_pages][num_kv_heads][16][head_dim_v]
 *   One (page, kv-head) block is a contiguous 16 x D burst. Slots of a chunk's last page beyond its
 *   length are zero-filled by the store. Pages owned by no chunk are never touched.
 *
 * Allocation policy (part of the contract, so block tables are reproducible)
 *   FIFO free list, initially 0,1,...,num_pages-1 (or the seeded permutation below); a chunk of T
 *   tokens takes ceil(T/16) ids from the head; comb_chunk_free appends a chunk's ids to the tail in
 *   page-list order. Page ids are shared by all layers (a chunk has one page list).
 */
#ifndef COMB_H_
#define COMB_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    COMB_OK = 0,
    COMB_ERR_INVALID = -1,       /* null pointer, page_size != 16, head dims outside {64,128,192}x{64,128},
                                    Hq % Hkv != 0 or an unsupported group size, num_tokens <= 0, layer out of
                                    range, non-monotone indptr */
    COMB_ERR_NO_SPACE = -2,      /* store/alloc needs more pages than are free; nothing allocated */
    COMB_ERR_EXISTS = -3,        /* chunk id already present with a different length */
    COMB_ERR_UNKNOWN_CHUNK = -4, /* link/free/query names an id that is not in the directory (the caller
                                    must compile + store first, PAPER.md:62 step 2); nothing is written */
    COMB_ERR_CAPACITY = -5,      /* link buffer, scratch or workspace too small */
    COMB_ERR_CUDA = -6,          /* a CUDA call failed; cudaGetLastError() is preserved for the caller */
    COMB_ERR_BUSY = -7,          /* comb_chunk_free of a pinned chunk */
    COMB_ERR_READ_ONLY = -8      /* alloc / store / free on a pool opened with comb_pool_import */
} comb_status_t;

typedef struct comb_pool comb_pool_t; /* opaque */

/* (a1) chunk-KV pool + chunk directory — PAPER.md:205 "reserves a portion ... of GPU memory, initializes
 * the PIC allocator"; PAPER.md:62 step 1/4 the hash table context -> PICache. */
typedef struct {
    int32_t num_layers;    /* cross-attention layers sharing one page-id space (>= 1) */
    int32_t num_kv_heads;  /* Hkv */
    int32_t head_dim_qk;   /* Dqk in {64, 128, 192} */
    int32_t head_dim_v;    /* Dv  in {64, 128} */
    int32_t page_size;     /* must be 16 */
    int32_t num_pages;     /* pages per layer */
    void *k_arena;         /* device, bf16 (or e4m3 bytes), comb_pool_bytes().k_bytes, 1024-byte aligned */
    void *v_arena;         /* device, bf16 (or e4m3 bytes), comb_pool_bytes().v_bytes, 1024-byte aligned */
    void *scratch;         /* device, comb_pool_bytes().scratch_bytes: store page / tile descriptors (ring of 4) */
    uint64_t free_list_shuffle_seed; /* 0: ascending ids. Else: Fisher-Yates (i = n-1..1, j = next() mod
                                        (i+1), swap) driven by splitmix64(seed) — scatters a chunk's pages
                                        over the arena like a long-running server would */
    /* (f4) fp8 pages — see "fp8 pools" below. Zero-initialised = a bf16 pool. */
    int32_t kv_dtype;      /* COMB_KV_BF16 (0) or COMB_KV_E4M3 (1) */
    int32_t reserved;      /* must be 0 */
    void *k_scale;         /* device fp32 [num_layers][num_pages][num_kv_heads], comb_pool_scale_bytes(); E4M3 only */
    void *v_scale;         /* likewise for V */
} comb_pool_config_t;
enum { COMB_KV_BF16 = 0, COMB_KV_E4M3 = 1 };

/* fp8 pools (SURVEY.md §8(f4) "fp8 (e4m3) pages with per-page scales to halve decode bytes"; KV memory is
 * what bounds concurrency).  The paper has no quantised cache; this is DESIGN.md §2 readings I31-I33.
 *   layout   K arena u8 [L][pages][Hkv][16][Dqk], V arena u8 [L][pages][Hkv][16][Dv]: the bf16 layout with one byte per
 *            element (OCP E4M3: 1-4-3, bias 7, max 448, no infinity); scales fp32 [L][pages][Hkv], one per (page,
 *            kv-head) block of K and of V.  head_dim_qk = head_dim_v = 128 only (INVALID otherwise).
 *   store    the caller still hands bf16 K/V.  Per block: amax = max |x| over its 16 x D values (slots past the chunk's
 *            length count as zero), scale = 2^e with e the smallest integer such that amax <= 448 * 2^e (clamped to
 *            [-100, 100]; 1 for an all-zero block), code = e4m3(x / scale) round-to-nearest-even; tail slots are byte 0.
 *            The page image (codes and scales) is part of the bit-exact contract.
 *   attend   attention over an fp8 pool is Eq. 7-8 over the dequantised values value(code) * scale (exactly bf16
 *            numbers, because the scale is a power of two).  comb_cross_attn_decode always takes the chunk-major path
 *            (the link needs its host mirror): K and V codes feed tcgen05 kind::f8f6f4 directly; the query rows and the
 *            softmax weights, the small operands, are each split into two e4m3 terms (hi + lo) so that side keeps
 *            bf16-level accuracy.  comb_cross_attn_prefill dequantises the batch's DISTINCT pages into bf16 staging in
 *            the workspace and runs the bf16 kernel on it (correct, not fast: prefill runs once per request, decode
 *            once per generated token); its workspace must be sized with comb_attn_workspace_bytes (the staging holds
 *            link->distinct_pages pages).  comb_project_store_chunks quantises in the GEMM's epilogue (the values a bf16
 *            pool would hold, bf16_rne of the fp32 accumulators, go through the store's rule; 256-column tiles so that
 *            a head's 128 columns and a page's 16 rows meet in one half-warp); comb_pool_export carries the scale
 *            tables along. */
size_t comb_pool_scale_bytes(const comb_pool_config_t *cfg); /* bytes of k_scale (= of v_scale); 0 for a bf16 pool */

/* Sizes the caller must allocate for a config (pointers in cfg are ignored). */
int32_t comb_pool_bytes(const comb_pool_config_t *cfg, size_t *k_bytes, size_t *v_bytes, size_t *scratch_bytes);

/* Validates cfg, builds the free list and an empty directory. Touches no device memory. */
int32_t comb_pool_create(const comb_pool_config_t *cfg, comb_pool_t **out);
int32_t comb_pool_destroy(comb_pool_t *pool);
int32_t comb_pool_free_pages(const comb_pool_t *pool); /* pages currently on the free list (>= 0) */

/* (f4) pool lifecycle — PAPER.md:205 (the PIC manager "reserves a portion ... of GPU memory", the allocator hands
 * out free memory, PICaches are "stored asynchronously"), PAPER.md:277 (memory is what bounds concurrency)
 * step 4 (the manager updates its table).  The paper does not say what happens when the reserved memory is full;
 * reading I16: explicit comb_chunk_free always works; with COMB_OPT_EVICT_LRU the pool also makes room
 * by itself.
 *   pins      comb_chunk_pin raises a chunk's reference count, comb_chunk_unpin lowers it (INVALID below zero). A
 *             pinned chunk is never evicted and comb_chunk_free on it returns COMB_ERR_BUSY. A serving loop pins the
 *             chunks of a request from lookup until the request's last attention call has completed.
 *   use stamp comb_chunk_alloc / a store stamps the chunk with a fresh tick; every comb_link draws ONE fresh tick and
 *             stamps all chunks it names (comb_link_plan stamps nothing).
 *   eviction  (only with comb_pool_set_option(pool, COMB_OPT_EVICT_LRU, 1)) when an alloc/store needs more pages
 *             than are free, unpinned chunks that are not part of the call are evicted in ascending (use stamp,
 *             creation order) until it fits; each evicted chunk's pages go to the free-list tail in page-list order,
 *             exactly as comb_chunk_free would put them. If even that cannot make room: NO_SPACE, nothing evicted.
 *             comb_pool_evicted() lists what the most recent alloc/store call evicted, so the caller can update its
 *             own table. Kernels in flight are NOT tracked: unpin only what the GPU is done with.
 *   ready     a store records an event on its stream; comb_link makes ITS stream wait for the stores of the chunks
 *             it names that have not completed yet (cudaStreamWaitEvent; no host wait). So a store may run on a side
 *             stream ("asynchronously") and the link + attention calls that follow on another stream are ordered
 *             after it without the caller handling events. */
int32_t comb_chunk_pin(comb_pool_t *pool, uint64_t chunk_id);
int32_t comb_chunk_unpin(comb_pool_t *pool, uint64_t chunk_id);
/* Writes up to `cap` ids evicted by the most recent alloc/store call (in eviction order); returns how many were. */
int32_t comb_pool_evicted(const comb_pool_t *pool, uint64_t *chunk_ids, int32_t cap);
int64_t comb_pool_eviction_count(const comb_pool_t *pool); /* chunks evicted since the pool was created */

/* (f4) export to another process — PAPER.md:205 §5.3: the PIC manager is its own component that "reserves a portion
 * ... of GPU memory" and hands PICaches to the inference engine; PAPER.md:229 (vLLM engine processes).  The manager
 * process owns the arenas and the directory; an engine process opens them READ-ONLY through CUDA IPC and runs
 * comb_link + the attention calls on the same bytes (zero copy, as the link itself).
 *   comb_pool_export  writes a self-contained blob (host memory): geometry, the directory (every chunk's id, length
 *       and page list, in creation order) and — unless COMB_EXPORT_DIRECTORY_ONLY — the cudaIpcMemHandle_t of the
 *       allocations that hold the K and V arenas (plus the arenas' offsets inside them: the arenas may be
 *       sub-allocations of a caching allocator) and the handle of an interprocess event recorded on `stream` after
 *       every store enqueued so far (`stream` is first made to wait for the pending store events).  The arenas must
 *       come from cudaMalloc (legacy IPC does not cover cuMemCreate / expandable segments).  *written = bytes used;
 *       CAPACITY if cap < comb_pool_export_bytes().  A directory-only export needs no GPU.
 *   comb_pool_import  (another process, same GPU) opens the handles, rebuilds the directory and makes `stream` wait
 *       for the exporter's event.  The pool it returns is read-only: comb_link, comb_link_plan, comb_chunk_query/
 *       pin/unpin, both attention calls and comb_cross_layer_forward work; comb_chunk_alloc/free and the stores
 *       return COMB_ERR_READ_ONLY.  Its free list is empty.  comb_pool_destroy closes the handles.
 *   comb_pool_refresh replaces an imported pool's directory by the one in a newer blob of the same exporter (full or
 *       directory-only; geometry must match: INVALID otherwise) and, when the blob carries an event, orders `stream`
 *       after it.  Chunks the exporter has evicted since disappear; what they were pinned for is the caller's
 *       protocol (the exporter must not reuse pages an importer may still read: pin on the exporter side).
 * Errors: INVALID (null, malformed or truncated blob, geometry mismatch), CAPACITY, CUDA. */
enum { COMB_EXPORT_DIRECTORY_ONLY = 1 };
size_t comb_pool_export_bytes(const comb_pool_t *pool);
int32_t comb_pool_export(comb_pool_t *pool, uint32_t flags, void *stream, void *blob, size_t cap, size_t *written);
int32_t comb_pool_import(const void *blob, size_t bytes, void *stream, comb_pool_t **out);
int32_t comb_pool_refresh(comb_pool_t *pool, const void *blob, size_t bytes, void *stream);

/* Directory-only half of a store: insert chunk_id with num_tokens and take ceil(T/16) pages from the head
 * of the free list; no data moves (a fused producer may write the pages itself). Idempotent for an
 * existing id with the same length; COMB_ERR_EXISTS for a different length. */
int32_t comb_chunk_alloc(comb_pool_t *pool, uint64_t chunk_id, int32_t num_tokens);
/* Remove the chunk; its pages go to the free-list tail in page-list order. */
int32_t comb_chunk_free(comb_pool_t *pool, uint64_t chunk_id);
/* Lookup (PAPER.md:62 step 1). Writes num_tokens and up to `cap` page ids (host); returns the number of
 * pages (>= 0) or COMB_ERR_UNKNOWN_CHUNK. `pages` may be NULL when cap == 0. */
int32_t comb_chunk_query(const comb_pool_t *pool, uint64_t chunk_id, int32_t *num_tokens, int32_t *pages,
                         int32_t cap);

/* (a2) paged store of one chunk's K/V — PAPER.md:62 step 3, "stored asynchronously",
 * PAPER.md:119 (store K^cross and V^cross, not H^E; Eq. 5-6 produce them as [T][H][D]).
 *   k  device bf16 [num_tokens][Hkv][Dqk] contiguous;  v  device bf16 [num_tokens][Hkv][Dv] contiguous
 * For t < T, head h:  Kpage[layer][pages[t/16]][h][t%16][:] = k[t][h][:]  (same for V); slots T%16..15 of
 * the last page are zero-filled. Allocates the page list on the first store of chunk_id (any layer);
 * stores on other layers reuse it. Errors: INVALID, NO_SPACE, EXISTS, CUDA. */
int32_t comb_store_chunk(comb_pool_t *pool, int32_t layer, uint64_t chunk_id, int32_t num_tokens, const void *k,
                         const void *v, void *stream);
/* Batched form, one kernel launch: chunk i has tokens tok_indptr[i]..tok_indptr[i+1] (host int32 [n+1]) of the
 * packed device tensors k_packed [sum T][Hkv][Dqk], v_packed [sum T][Hkv][Dv]. All-or-nothing: on any error
 * (including a CUDA failure) the directory and the free list are as before the call — except that chunks evicted
 * to make room (COMB_OPT_EVICT_LRU) stay evicted and are listed by comb_pool_evicted(). The same id twice in one
 * batch is INVALID. Storing an id that already exists with the same length overwrites its pages (that is how
 * the other layers of a chunk are filled); ordering against attention calls in flight that read those pages is
 * the caller's, as for any store. */
int32_t comb_store_chunks(comb_pool_t *pool, int32_t layer, int32_t n, const uint64_t *chunk_ids,
                          const int32_t *tok_indptr, const void *k_packed, const void *v_packed, void *stream);

/* (f2) compile-side producer fused into the store — PAPER.md:105-109 §4.2 Eq. 5-6: K^cross = H^E W_K,
 * V^cross = H^E W_V, and PAPER.md:119 / 205: what is stored is K^cross and V^cross.  One tcgen05 GEMM whose epilogue
 * writes bf16 straight into the chunks' pages (tail slots of a last page zero-filled): the [T][Hkv][D] K/V tensors
 * of comb_store_chunks never exist in HBM.
 *   h_packed  device bf16 [sum T][d_model]   encoder hidden states of the n chunks, packed as tok_indptr says
 *   w_kv      device bf16 [Hkv*Dqk + Hkv*Dv][d_model]: row (h*Dqk + d) holds column (h, d) of W_K, then the rows of
 *             W_V likewise (the nn.Linear layout, i.e. the paper's W transposed); d_model % 8 == 0
 * Page image afterwards: Kpage[layer][pages[t/16]][h][t%16][d] = bf16_rne(sum_c h[t][c] * W_K[c][(h,d)]) with the
 * sum accumulated in fp32 (same for V).  Directory semantics, all-or-nothing and errors as comb_store_chunks. */
int32_t comb_project_store_chunks(comb_pool_t *pool, int32_t layer, int32_t n, const uint64_t *chunk_ids,
                                  const int32_t *tok_indptr, const void *h_packed, int32_t d_model, const void *w_kv,
                                  void *stream);

/* (a3) link — PAPER.md:24 "loads and concatenates needed KV vectors (in any order/position)",
 * PAPER.md:119, PAPER.md:62 step 5.  Zero-copy: builds the request's block table from an ORDERED
 * chunk-id list; no kernel touches K/V.
 *
 * The caller provides device_buf (comb_link_bytes() bytes, 16-byte aligned) and, optionally, host_buf
 * (comb_link_host_bytes() bytes of ordinary host memory). comb_link lays the tables out inside device_buf, fills
 * the pointers below and enqueues ONE host->device copy on `stream`.  An "entry" is one (request, linked chunk)
 * pair, numbered in the order of chunk_ids.
 *
 * Request-major view (what prefill and the per-request decode read):
 *   page_indptr int32 [R+1]      page range of request r in page_ids / page_ntok
 *   page_ids    int32 [total]    pages(c_0) || ... || pages(c_{m-1}) in the caller's order
 *   page_ntok   uint8 [total]    16, except the last page of each chunk = T - 16*(npages-1)
 *   kv_len      int32 [R]        sum of the linked chunks' lengths
 *   tile_indptr int32 [R+1]      tile range of request r in tile_ntok (a tile = 8 consecutive table
 *                                entries of the request, i.e. 128 slots, counted from its first page)
 *   tile_ntok   uint64 [tiles]   byte j = page_ntok of entry 8*t+j, 0 past the request's last page
 *                                (derived from page_ntok; lets kernels skip the slot mask on full tiles)
 *   entry_indptr int32 [R+1]     entries of request r (= chunk_indptr)
 * Chunk-major ("cascade") view — the same batch inverted, so that every DISTINCT chunk is streamed once and all
 * the query rows that link it attend to it together (possible because PICaches carry no per-request position:
 * PAPER.md:24, 119).  Distinct chunks get slots u = 0..U-1, ordered by descending number of entries, ties by
 * first appearance in chunk_ids:
 *   cas_page_indptr int32 [U+1], cas_page_ids int32 [distinct pages]    page list of slot u
 *   cas_tile_indptr int32 [U+1], cas_tile_ntok uint64 [..]              as tile_indptr / tile_ntok, per slot
 *   cas_row_indptr  int32 [U+1]                                         entries that link slot u
 *   cas_row_req     int32 [E]    request of the entry;   cas_row_entry int32 [E]   the entry's number
 *                                (inside a slot, entries are in ascending entry number)
 * Host mirror (only when host_buf != NULL; plain host memory the caller owns — a caller that builds its own
 * tables fills these three arrays itself):
 *   host_req_pages int32 [R]     page_indptr[r+1] - page_indptr[r]  (the prefill planner cuts KV ranges with it)
 *   host_cas_rows  int32 [U]     cas_row_indptr[u+1] - cas_row_indptr[u]  (the chunk-major decode groups rows with it)
 *   host_cas_pages int32 [U]     cas_page_indptr[u+1] - cas_page_indptr[u] (... and cuts long chunks into KV ranges)
 * Without a host mirror both attention calls still work: prefill does not cut KV ranges, decode runs per request.
 * A request with zero chunks is legal (kv_len 0). Duplicate ids inside a request are taken literally (two entries).
 * Errors: INVALID, UNKNOWN_CHUNK (nothing written), CAPACITY, CUDA. */
typedef struct {
    /* in: caller-owned memory */
    void *device_buf;
    size_t device_bytes;
    void *host_buf;      /* nullable */
    size_t host_bytes;
    /* out: device pointers into device_buf */
    int32_t *page_indptr;
    int32_t *page_ids;
    uint8_t *page_ntok;
    int32_t *kv_len;
    int32_t *tile_indptr;
    uint64_t *tile_ntok;
    int32_t *entry_indptr;
    int32_t *cas_page_indptr;
    int32_t *cas_page_ids;
    int32_t *cas_tile_indptr;
    uint64_t *cas_tile_ntok;
    int32_t *cas_row_indptr;
    int32_t *cas_row_req;
    int32_t *cas_row_entry;
    int32_t *page_ids_compact;   /* fp8 pools only (NULL otherwise): int32 [total], entry i of page_ids as an index into
                                    cas_page_ids (the batch's distinct pages) — the page table of the bf16 staging
                                    that comb_cross_attn_prefill dequantises those pages into */
    /* out: host pointers into host_buf (NULL without one) */
    int32_t *host_req_pages;
    int32_t *host_cas_rows;
    int32_t *host_cas_pages;
    /* out: host-side summary */
    int32_t num_requests;
    int32_t max_pages_per_request;
    int64_t total_pages;
    int64_t total_tiles;
    int64_t total_kv_tokens;
    int64_t total_entries;        /* E */
    int32_t num_distinct_chunks;  /* U */
    int32_t max_rows_per_chunk;   /* entries of slot 0 */
    int64_t distinct_pages;       /* pages of the U distinct chunks */
    int64_t distinct_kv_tokens;   /* their tokens: what a chunk-major pass reads once */
    size_t bytes_used; /* bytes of device_buf written = size of the single H2D copy */
} comb_link_t;

/* Bytes of device_buf / host_buf that suffice for num_requests requests with total_entries (request, chunk)
 * pairs naming total_pages table entries. */
size_t comb_link_bytes(int32_t num_requests, int64_t total_entries, int64_t total_pages);
size_t comb_link_host_bytes(int32_t num_requests, int64_t total_entries);
int32_t comb_link(comb_pool_t *pool, int32_t num_requests, const int32_t *chunk_indptr /* host [R+1] */,
                  const uint64_t *chunk_ids /* host, link order */, comb_link_t *link, void *stream);
/* Same tables written into HOST memory `staging` (link->device_bytes bytes available); the pointers in
 * `link` are laid out as if staging were device_buf. No CUDA call, and the pool is not modified (no use stamps,
 * no waiting for stores) — used by host tests and by callers that plan ahead. */
int32_t comb_link_plan(const comb_pool_t *pool, int32_t num_requests, const int32_t *chunk_indptr,
                       const uint64_t *chunk_ids, comb_link_t *link, void *staging);

/* (a4) prefill cross-attention — PAPER.md:112-115 §4.2 Eq. 7-8 (softmax(QK^T/sqrt d) V, NO mask), over the
 * concatenation of the linked chunks; cost O(l_query * l_doc) per layer (Eq. 12).
 *   q         device bf16 [sum lq][Hq][Dqk];   q_indptr  HOST int32 [R+1] (rows of request r)
 *   out       device bf16 [sum lq][Hq][Dv];    lse       device fp32 [sum lq][Hq] or NULL
 *   scale     multiplies q.k before the softmax (the paper's 1/sqrt(d), per head: 1/sqrt(Dqk)); must be a
 *             finite positive number (INVALID otherwise)
 *   workspace device, comb_attn_workspace_bytes() bytes, 16-byte aligned
 * q-head h reads kv-head h / (Hq/Hkv); Hq/Hkv must be a power of two <= 16. kv_len == 0 gives out = 0,
 * lse = -inf. tcgen05/TMEM/TMA kernel.
 * When the call has fewer work items than the GPU has SMs (few requests with few query tokens — the paper's
 * regime) and link->host_req_pages is given, every request's KV is cut into ranges that run on
 * different SMs; their fp32 partial rows live in `workspace` and are merged by LSE.
 * The result is the same function; only fp32 summation order differs. host_req_pages is checked against the
 * link's summary (sum = total_pages, max = max_pages_per_request): INVALID if it disagrees.
 * Errors: INVALID, CAPACITY (workspace smaller than comb_attn_workspace_bytes() for this call, or not 16-byte
 * aligned), CUDA. */
int32_t comb_cross_attn_prefill(comb_pool_t *pool, int32_t layer, const comb_link_t *link, int32_t num_requests,
                                const void *q, const int32_t *q_indptr, int32_t num_q_heads, float scale, void *out,
                                float *lse, void *workspace, size_t workspace_bytes, void *stream);

/* (a5) decode cross-attention — the same function with exactly one query row per request (PAPER.md:66:
 * generated tokens are "treated identically to the initial query tokens").
 *   q device bf16 [R][Hq][Dqk];  out device bf16 [R][Hq][Dv];  lse device fp32 [R][Hq] or NULL
 * Two paths compute it (same result up to fp32 summation order and, on the second, bf16 rounding of the softmax
 * weights fed to the tensor cores, as in prefill):
 *   per-request : split-KV kernel on CUDA cores (HBM-bound, GEMV-shaped) + LSE-merge kernel;
 *   chunk-major : every distinct chunk of the batch is streamed from HBM ONCE; the (entries x Hq/Hkv) query rows that
 *                 link it are the N dimension (16 or 32 columns) of a tcgen05 contraction whose M dimension is the
 *                 128 keys of a KV tile; per-(entry, KV range) fp32 partials are merged by LSE per request
 *                 (needs link->host_cas_rows and host_cas_pages; Hq/Hkv <= 16).
 * COMB_OPT_DECODE_PATH picks one (default: chunk-major when the batch shares chunks, see comb_pool_set_option).
 * Errors as above. */
int32_t comb_cross_attn_decode(comb_pool_t *pool, int32_t layer, const comb_link_t *link, int32_t num_requests,
                               const void *q, int32_t num_q_heads, float scale, void *out, float *lse,
                               void *workspace, size_t workspace_bytes, void *stream);

/* (a5) decode for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): the SAME function as comb_cross_attn_decode (Eq. 7-8 at one query row per request)
 * on its per-request path (split-KV kernel + LSE merge), with the split partials in a fixed device array that is part
 * of the library image instead of a caller workspace.  The call allocates nothing — no cudaMalloc / cudaFree /
 * cudaMallocHost, no host containers, no pinned staging (it copies nothing) — and takes no workspace argument; q, out
 * and lse are the caller's as before and the link must already be resident (comb_link).
 *   limit    the array is comb_noalloc_scratch_bytes() = 8 MiB, held by every GPU that loads the library until
 *            the process exits.  A call whose partials need more — num_requests x num_q_heads x splits x (Dv + 2)
 *            floats, splits chosen as in comb_cross_attn_decode (cfg 2: 4.3 MB, cfg 4 decode: 2.5 MB; the plan aims
 *            at ~4 waves of CTAs, so on a 148-SM B200 no call needs more than ~5 MB) — returns COMB_ERR_CAPACITY
 *            and launches nothing: use comb_cross_attn_decode with a workspace.
 *   sharing  every call on a device uses the same array, whatever pool or stream: calls that overlap on the GPU
 *            (different streams without an ordering between them) RACE on it.  The array keeps the previous call's
 *            contents; nothing in it must start at zero (every partial the merge reads is written by the same call).
 *   scope    bf16 pools only (an fp8 pool has no per-request kernel): INVALID.  COMB_OPT_DECODE_PATH is ignored.
 *            comb_profile_* does not see these launches.
 * Errors: INVALID, CAPACITY, CUDA. */
int32_t comb_cross_attn_decode_noalloc(comb_pool_t *pool, int32_t layer, const comb_link_t *link,
                                       int32_t num_requests, const void *q, int32_t num_q_heads, float scale,
                                       void *out, float *lse, void *stream);
size_t comb_noalloc_scratch_bytes(void);

/* Workspace that suffices for either attention call on THIS link: num_q_heads heads, total_q query rows (decode:
 * total_q = num_requests). Holds the decode split partials or the chunk-major tiles and per-entry partials, or the
 * prefill work-item list plus the partial rows of its KV ranges. */
size_t comb_attn_workspace_bytes(const comb_pool_t *pool, const comb_link_t *link, int32_t num_q_heads,
                                 int64_t total_q);
/* Link-independent bound for callers that size the workspace before linking: num_requests requests, total_q query
 * rows, max_pages_per_request table entries in the longest request. Covers prefill and the per-request decode;
 * a decode whose workspace is too small for the chunk-major path quietly takes the per-request one (unless
 * COMB_OPT_DECODE_PATH forces chunk-major: CAPACITY). */
size_t comb_workspace_bytes(const comb_pool_t *pool, int32_t num_requests, int32_t num_q_heads, int64_t total_q,
                            int32_t max_pages_per_request);

/* (f3) the cross-attention sub-layer around the attention — PAPER.md:102-105 Eq. 4 (Q = X^D W_Q), Eq. 7-8, and the
 * output projection whose result "is then passed through the standard decoder pathway via residual connections"
 * (PAPER.md:117):   x_out = x + Attn(x W_Q ; linked K, V) W_O      (no norm, gate or bias: none is in Eq. 4-8)
 *   x, x_out  device bf16 [rows][d_model]  (rows = sum lq for prefill, = num_requests for decode); x_out may alias x
 *             only if the caller does not need x afterwards (each row is read before it is written)
 *   w_q       device bf16 [Hq*Dqk][d_model]   row (h*Dqk + d) = column (h, d) of W_Q
 *   w_o       device bf16 [d_model][Hq*Dv]    row c = the weights producing output feature c
 *   q_indptr  HOST int32 [R+1] for prefill; NULL selects decode (one row per request)
 *   workspace device, comb_layer_workspace_bytes() bytes, 16-byte aligned: Q and attention-output staging + the
 *             attention call's own workspace
 * Three launches on `stream`: GEMM (tcgen05) -> comb_cross_attn_prefill/decode -> GEMM with the residual added in
 * its epilogue.  Q and the attention output are rounded to bf16 between the steps (they are the inputs of the next
 * tensor-core contraction).  A model's L cross layers (8 in the paper's Llama instance) are L calls,
 * layer = 0..L-1, each with its own weights, over one link (page ids are shared by all layers).
 * Errors: INVALID, CAPACITY, CUDA. */
int32_t comb_cross_layer_forward(comb_pool_t *pool, int32_t layer, const comb_link_t *link, int32_t num_requests,
                                 const void *x, const int32_t *q_indptr, int32_t d_model, int32_t num_q_heads,
                                 const void *w_q, const void *w_o, float scale, void *x_out, void *workspace,
                                 size_t workspace_bytes, void *stream);
size_t comb_layer_workspace_bytes(const comb_pool_t *pool, const comb_link_t *link, int32_t num_q_heads, int64_t rows);
/* The projection alone: c[M][N] = bf16(a[M][K] w[N][K]^T (+ residual[M][N])), fp32 accumulation on tcgen05.
 * K % 8 == 0, N % 32 == 0. (pool is only used for the device's SM count and profiling.) Errors: INVALID, CUDA. */
int32_t comb_gemm_bf16(comb_pool_t *pool, const void *a, const void *w, const void *residual, void *c, int64_t M,
                       int32_t N, int32_t K, void *stream);

/* Pool options. COMB_OPT_DECODE_PATH: 0 = automatic (chunk-major when total_entries >= 1.25 x distinct chunks,
 * i.e. the batch re-reads at least a fifth of its KV), 1 = always per-request, 2 = always chunk-major.
 * Errors: INVALID (unknown option or value). */
/* COMB_OPT_PREFILL_CLUSTERS: 1 (default) = a prefill call whose work items come in pairs that share their K/V stream
 * (two Q-tile pairs of one (request, kv-head), whole KV each, at least one item per SM) runs on thread-block clusters
 * of two CTAs that fetch each K/V tile once and TMA-multicast it to both; 0 = always one CTA per item. Same result
 * bit for bit (same arithmetic in the same order); falls back by itself when the device cannot co-schedule the clusters. */
enum { COMB_OPT_DECODE_PATH = 1, COMB_OPT_EVICT_LRU = 2 /* 0 (default) = never evict, 1 = LRU eviction, see (f4) */,
       COMB_OPT_PREFILL_CLUSTERS = 3 };
enum { COMB_DECODE_AUTO = 0, COMB_DECODE_PER_REQUEST = 1, COMB_DECODE_CHUNK_MAJOR = 2 };
int32_t comb_pool_set_option(comb_pool_t *pool, int32_t option, int64_t value);

/* Kernels launched by this library since the pool was created (store/attention/reduce; copies excluded). */
int64_t comb_pool_launch_count(const comb_pool_t *pool);

/* Optional per-kernel device timing (bench.py uses it for the roofline of the dominant kernel). While enabled,
 * every kernel this pool launches is bracketed by two CUDA events recorded on the launching stream.
 * comb_profile_read synchronises on the recorded events (the one call here that waits for the device), adds up
 * the elapsed times of kernel class `kernel` (COMB_KERNEL_*), reports them and forgets those records.
 * Errors: INVALID, CUDA. */
enum { COMB_KERNEL_STORE = 0, COMB_KERNEL_DECODE_SPLIT = 1, COMB_KERNEL_DECODE_MERGE = 2, COMB_KERNEL_PREFILL = 3,
       COMB_KERNEL_DECODE_CASCADE = 4, COMB_KERNEL_CASCADE_MERGE = 5, COMB_KERNEL_PREFILL_MERGE = 6, COMB_KERNEL_GEMM = 7 };
int32_t comb_profile_enable(comb_pool_t *pool, int32_t on);
int32_t comb_profile_read(comb_pool_t *pool, int32_t kernel, double *total_ms, int64_t *launches);
/* Same, but hands back the elapsed time of every recorded launch of that class (oldest first, at most `cap`
 * values into host array `ms`; the rest are dropped) so a caller can report median and minimum. */
int32_t comb_profile_read_samples(comb_pool_t *pool, int32_t kernel, float *ms, int64_t cap, int64_t *launches);

/* Measurement utility (bench.py's read-only HBM ceiling): one kernel that reads `bytes` bytes of
 * device memory at `src` (16-byte aligned) with streaming 128-bit loads and writes nothing; `sink` = 4 device
 * bytes. Enqueued on `stream`; timed by the caller. Errors: INVALID, CUDA. */
int32_t comb_util_stream_read(const void *src, size_t bytes, void *sink, void *stream);

const char *comb_strerror(int32_t status);
const char *comb_version(void);

#ifdef __cplusplus
}
#endif
#endif /* COMB_H_ */
