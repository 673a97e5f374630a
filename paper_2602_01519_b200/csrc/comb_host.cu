// comb_host.cu — host runtime behind the C ABI of include/comb.h: page allocator (FIFO free list),
// chunk directory (hash map chunk_id -> page list), block-table builder, pinned staging ring, and the
// five entry points. No device memory is allocated here; kernels live in *_kernel.cu.
//
// Paper anchors: §3 steps 1-8 (lookup / store / update table / fetch), §5.3
// (PIC manager, allocator, asynchronous store), PAPER.md:24 + 119 (link = concatenate in any order).
#include "../../include/comb.h"
#include "kernels.h"

#include <algorithm>
#include <cstdlib>
#include <cstring>
#include <new>
#include <type_traits>
#include <unordered_map>
#include <vector>

using namespace comb;

namespace {

constexpr int kRingSlots = 4;
// scratch per page and slot: one StorePageDesc (16 B) for a store, or at worst one GemmRowTile (48 B) when every
// chunk of a fused projection store is a single page
constexpr size_t kScratchBytesPerPage = 48;

struct Chunk {
    int32_t num_tokens;
    std::vector<int32_t> pages;
    // lifecycle
    int32_t pins = 0;        // reference count: a pinned chunk is never evicted or freed
    uint64_t last_use = 0;   // tick of the last alloc / store / comb_link that named it
    uint64_t seq = 0;        // creation order (tie-break of the LRU order)
    int32_t ready = -1;      // index of the event its last store recorded, -1 once known complete
    // scratch of the link planner: which link call saw this chunk last, and its distinct index there (so that
    // finding the distinct chunks of a batch needs no second hash map)
    mutable uint64_t link_mark = 0;
    mutable int32_t link_index = 0;
};

// Event recorded by a store on its stream; comb_link makes its stream wait for it while it is pending.
struct ReadyEvent {
    cudaEvent_t ev = nullptr;
    int32_t users = 0;  // chunks that still reference it
};

// Pinned host staging, reused round-robin; an event per slot marks when the GPU is done with it.
struct StagingSlot {
    void *host = nullptr;
    size_t cap = 0;
    cudaEvent_t ev = nullptr;
    bool busy = false;
};

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

}  // namespace

struct comb_pool {
    comb_pool_config_t cfg;
    PoolGeom geom;
    std::vector<int32_t> free_list;  // FIFO: [head, size) are free
    size_t free_head = 0;
    std::unordered_map<uint64_t, Chunk> dir;
    StagingSlot ring[kRingSlots];
    int ring_next = 0;
    int num_sms = 148;
    bool device_probed = false;
    bool kv_maps_ready = false;
    TensorMapBlob k_map, v_map;
    int64_t launches = 0;
    int64_t opt_decode_path = COMB_DECODE_AUTO;
    bool opt_prefill_clusters = true;
    bool opt_evict_lru = false;
    uint64_t tick = 0, next_seq = 0;
    std::vector<uint64_t> last_evicted;
    int64_t evictions = 0;
    std::vector<ReadyEvent> ready_events;
    mutable uint64_t link_calls = 0;  // stamps Chunk::link_mark
    // (f4) CUDA IPC: an imported pool is read-only and owns the mappings it opened; an exporting pool owns one
    // interprocess event
    bool imported = false;
    std::vector<std::pair<cudaIpcMemHandle_t, void *>> ipc_maps;  // allocations opened by comb_pool_import
    cudaEvent_t ipc_event = nullptr;
    void drop_ready(Chunk &c) {
        if (c.ready >= 0 && ready_events[(size_t)c.ready].users > 0) ready_events[(size_t)c.ready].users -= 1;
        c.ready = -1;
    }
    // an event slot nobody references any more (or a new one); -1 on CUDA failure
    int take_ready_event() {
        for (size_t i = 0; i < ready_events.size(); ++i)
            if (ready_events[i].users == 0 && ready_events[i].ev) return (int)i;
        ReadyEvent e;
        if (cudaEventCreateWithFlags(&e.ev, cudaEventDisableTiming) != cudaSuccess) return -1;
        ready_events.push_back(e);
        return (int)ready_events.size() - 1;
    }
    // per-kernel timing (comb_profile_*)
    struct ProfRec { int id; cudaEvent_t a, b; };
    bool prof_on = false;
    std::vector<ProfRec> prof_recs;
    std::vector<cudaEvent_t> prof_free;
    LaunchHook hook{};

    cudaEvent_t prof_event() {
        if (!prof_free.empty()) { cudaEvent_t e = prof_free.back(); prof_free.pop_back(); return e; }
        cudaEvent_t e = nullptr;
        if (cudaEventCreate(&e) != cudaSuccess) return nullptr;
        return e;
    }
    static void hook_begin(void *ctx, int id, cudaStream_t st) {
        comb_pool *p = (comb_pool *)ctx;
        ProfRec r{id, p->prof_event(), p->prof_event()};
        if (r.a && r.b) { cudaEventRecord(r.a, st); p->prof_recs.push_back(r); }
    }
    static void hook_end(void *ctx, cudaStream_t st) {
        comb_pool *p = (comb_pool *)ctx;
        if (!p->prof_recs.empty()) cudaEventRecord(p->prof_recs.back().b, st);
    }
    const LaunchHook *active_hook() { return prof_on ? &hook : nullptr; }

    size_t scratch_slot_bytes() const { return align_up((size_t)cfg.num_pages * kScratchBytesPerPage, 256); }

    void probe_device() {
        if (device_probed) return;
        int dev = 0, sms = 0;
        if (cudaGetDevice(&dev) == cudaSuccess &&
            cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0)
            num_sms = sms;
        else
            (void)cudaGetLastError();
        device_probed = true;
    }

    // Returns slot index with at least `bytes` of pinned memory, or -1 on CUDA failure.
    int acquire(size_t bytes) {
        int i = ring_next;
        ring_next = (ring_next + 1) % kRingSlots;
        StagingSlot &s = ring[i];
        if (!s.ev && cudaEventCreateWithFlags(&s.ev, cudaEventDisableTiming) != cudaSuccess) return -1;
        if (s.busy) {
            if (cudaEventSynchronize(s.ev) != cudaSuccess) return -1;
            s.busy = false;
        }
        if (s.cap < bytes) {
            if (s.host) cudaFreeHost(s.host);
            s.host = nullptr;
            s.cap = 0;
            size_t want = std::max(align_up(bytes, 4096), (size_t)65536);
            if (cudaHostAlloc(&s.host, want, cudaHostAllocDefault) != cudaSuccess) return -1;
            s.cap = want;
        }
        return i;
    }
    bool release(int i, cudaStream_t st) {
        if (cudaEventRecord(ring[i].ev, st) != cudaSuccess) return false;
        ring[i].busy = true;
        return true;
    }
};

namespace {

uint64_t splitmix64_next(uint64_t &state) {
    state += 0x9E3779B97F4A7C15ull;
    uint64_t z = state;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

bool dims_ok(int dqk, int dv) {
    return (dqk == 64 || dqk == 128 || dqk == 192) && (dv == 64 || dv == 128);
}

int32_t validate_cfg(const comb_pool_config_t *c) {
    if (!c) return COMB_ERR_INVALID;
    if (c->page_size != kPage || c->num_layers < 1 || c->num_kv_heads < 1 || c->num_pages < 1)
        return COMB_ERR_INVALID;
    if (!dims_ok(c->head_dim_qk, c->head_dim_v)) return COMB_ERR_INVALID;
    if (c->kv_dtype != COMB_KV_BF16 && c->kv_dtype != COMB_KV_E4M3) return COMB_ERR_INVALID;
    if (c->reserved != 0) return COMB_ERR_INVALID;
    if (c->kv_dtype == COMB_KV_E4M3 && (c->head_dim_qk != 128 || c->head_dim_v != 128)) return COMB_ERR_INVALID;
    return COMB_OK;
}

void dir_free(comb_pool_t *p, std::unordered_map<uint64_t, Chunk>::iterator it) {
    // compact the consumed prefix now and then so the vector does not grow without bound
    if (p->free_head > 65536 && p->free_head * 2 > p->free_list.size()) {
        p->free_list.erase(p->free_list.begin(), p->free_list.begin() + p->free_head);
        p->free_head = 0;
    }
    p->free_list.insert(p->free_list.end(), it->second.pages.begin(), it->second.pages.end());
    p->drop_ready(it->second);
    p->dir.erase(it);
}

// LRU eviction (policy stated in include/comb.h): make `need` pages available by evicting unpinned
// chunks that are not in `keep`, in ascending (use stamp, creation order). All or nothing.
bool evict_for(comb_pool_t *p, size_t need, const std::unordered_map<uint64_t, int32_t> *keep) {
    size_t have = p->free_list.size() - p->free_head;
    if (have >= need) return true;
    if (!p->opt_evict_lru) return false;
    struct Cand { uint64_t use, seq, id; size_t pages; };
    std::vector<Cand> cands;
    for (auto &kv : p->dir)
        if (kv.second.pins == 0 && !(keep && keep->count(kv.first)))
            cands.push_back(Cand{kv.second.last_use, kv.second.seq, kv.first, kv.second.pages.size()});
    std::sort(cands.begin(), cands.end(),
              [](const Cand &a, const Cand &b) { return a.use != b.use ? a.use < b.use : a.seq < b.seq; });
    size_t n = 0;
    while (n < cands.size() && have < need) have += cands[n++].pages;
    if (have < need) return false;
    for (size_t i = 0; i < n; ++i) {
        dir_free(p, p->dir.find(cands[i].id));
        p->last_evicted.push_back(cands[i].id);
        p->evictions += 1;
    }
    return true;
}

// take ceil(T/16) pages from the head of the free list (or find the existing entry)
int32_t dir_alloc(comb_pool_t *p, uint64_t id, int32_t T, const Chunk **out, bool *created) {
    if (T <= 0) return COMB_ERR_INVALID;
    auto it = p->dir.find(id);
    if (it != p->dir.end()) {
        if (it->second.num_tokens != T) return COMB_ERR_EXISTS;
        it->second.last_use = ++p->tick;
        if (out) *out = &it->second;
        if (created) *created = false;
        return COMB_OK;
    }
    const size_t n = (size_t)(T + kPage - 1) / kPage;
    if (n > p->free_list.size() - p->free_head) return COMB_ERR_NO_SPACE;
    Chunk c;
    c.num_tokens = T;
    c.pages.assign(p->free_list.begin() + p->free_head, p->free_list.begin() + p->free_head + n);
    c.last_use = ++p->tick;
    c.seq = p->next_seq++;
    p->free_head += n;
    auto ins = p->dir.emplace(id, std::move(c));
    if (out) *out = &ins.first->second;
    if (created) *created = true;
    return COMB_OK;
}

struct LinkLayout {
    size_t off_page_indptr, off_kv_len, off_tile_indptr, off_entry_indptr, off_cas_page_indptr, off_cas_tile_indptr,
        off_cas_row_indptr, off_tile_ntok, off_cas_tile_ntok, off_page_ids, off_page_ntok, off_cas_page_ids,
        off_cas_row_req, off_cas_row_entry, off_page_ids_compact, bytes;
};

// R requests, E entries, U distinct chunks with Pd pages and Tc tiles in all, P table entries, T tiles
LinkLayout link_layout(int32_t R, int64_t E, int64_t U, int64_t P, int64_t T, int64_t Pd, int64_t Tc,
                       bool compact = false) {
    LinkLayout L;
    size_t o = 0;
    auto take = [&](size_t elem, int64_t n) {
        const size_t at = o;
        o = align_up(o + elem * (size_t)std::max<int64_t>(n, 1), 16);
        return at;
    };
    L.off_page_indptr = take(4, R + 1);
    L.off_kv_len = take(4, R);
    L.off_tile_indptr = take(4, R + 1);
    L.off_entry_indptr = take(4, R + 1);
    L.off_cas_page_indptr = take(4, U + 1);
    L.off_cas_tile_indptr = take(4, U + 1);
    L.off_cas_row_indptr = take(4, U + 1);
    L.off_tile_ntok = take(8, T);
    L.off_cas_tile_ntok = take(8, Tc);
    L.off_page_ids = take(4, P);
    L.off_page_ntok = take(1, P);  // one byte per entry (1..16): a third less table to copy than int32 counts
    L.off_cas_page_ids = take(4, Pd);
    L.off_cas_row_req = take(4, E);
    L.off_cas_row_entry = take(4, E);
    L.off_page_ids_compact = o;
    if (compact) L.off_page_ids_compact = take(4, P);  // fp8 pools: the page table of the dequantised staging
    L.bytes = o;
    return L;
}

// byte j = page_ntok of table entry t + j, 0 past `end`
uint64_t pack_tile_ntok(const uint8_t *page_ntok, int64_t t, int64_t end) {
    uint64_t packed = 0;
    const int lim = (int)std::min<int64_t>(kTilePages, end - t);
    for (int j = 0; j < lim; ++j) packed |= (uint64_t)page_ntok[t + j] << (8 * j);
    return packed;
}

// KV ranges per request for a prefill call that has `num_items` unsplit work items and whose longest request has
// `max_tiles` 128-slot tiles. Ranges are only worth their fixed cost (pipeline fill per item, fp32 partial rows,
// the merge pass) when the items cannot fill even one wave of the persistent grid: measured on B200, cutting a
// 1.7-wave or 3.5-wave problem into ranges gained nothing (profiles/r01_bench.md). So: no ranges once there is an
// item per SM; otherwise the largest count that still fits one wave, every range keeping at least two tiles.
int plan_prefill_splits(size_t num_items, int max_tiles, int num_sms) {
    static const int cands[] = {1, 2, 3, 4, 6, 8, 12, 16};
    if (num_items == 0 || num_items >= (size_t)num_sms) return 1;
    int best = 1;
    for (int ns : cands) {
        if (ns > kPrefillMaxSplits) break;
        if (ns > 1 && prefill_tiles_per_split(max_tiles, ns) < 2) break;
        if (num_items * (size_t)ns > (size_t)num_sms) break;
        best = ns;
    }
    return best;
}

LinkView view_of(const comb_link_t *l) {
    LinkView v;
    v.page_indptr = l->page_indptr;
    v.page_ids = l->page_ids;
    v.page_ntok = l->page_ntok;
    v.kv_len = l->kv_len;
    v.tile_indptr = l->tile_indptr;
    v.tile_ntok = l->tile_ntok;
    v.entry_indptr = l->entry_indptr;
    v.cas_page_indptr = l->cas_page_indptr;
    v.cas_page_ids = l->cas_page_ids;
    v.cas_tile_indptr = l->cas_tile_indptr;
    v.cas_tile_ntok = l->cas_tile_ntok;
    v.cas_row_indptr = l->cas_row_indptr;
    v.cas_row_req = l->cas_row_req;
    v.cas_row_entry = l->cas_row_entry;
    return v;
}

// ---------------------------------------------------------------- prefill planning (one place: the workspace bound
// and the call agree by construction)
constexpr int kPartRowsPerRange = 2 * 128;  // partial rows reserved per (split item): two 128-row tile slots

struct PrefillPlan {
    std::vector<PrefillItem> items;
    int tiles_per_cta = 2;
    int64_t part_rows = 0;  // fp32 partial rows of the KV ranges (0: no item is split)
};
size_t prefill_items_bytes(size_t n) { return align_up(n * sizeof(PrefillItem), 256); }
size_t prefill_part_bytes(int64_t rows, int dv) { return (size_t)rows * (size_t)(dv + 1) * sizeof(float); }

// Upper bounds over every plan a call with these sizes can produce: the split items of a call never number more
// than two waves of CTAs (uniform ranges: items x ranges <= #SM; last-wave ranges: tail x factor <= CTAs), each with
// kPartRowsPerRange partial rows.
void prefill_bounds(const comb_pool *p, int32_t Hq, int64_t total_q, size_t *max_items, int64_t *max_part_rows) {
    const int Hkv = p->cfg.num_kv_heads;
    const int G = std::max(1, Hq / Hkv);
    const int tok_per_tile = std::max(1, 128 / std::min(G, 128));
    // one item per (request, kv-head, 1-2 tiles): at most one more item per request than full tiles, and no more
    // requests with rows than rows
    const size_t base_hi = ((size_t)total_q / tok_per_tile + (size_t)total_q + 1) * Hkv;
    const size_t ctas_hi = (size_t)p->num_sms * 2;
    *max_items = base_hi + ctas_hi;
    *max_part_rows = (int64_t)ctas_hi * kPartRowsPerRange;
}

int32_t plan_prefill(comb_pool *p, const comb_link_t *link, int32_t R, const int32_t *q_indptr, int32_t Hq,
                     PrefillPlan *out) {
    const int Hkv = p->cfg.num_kv_heads, G = Hq / Hkv;
    int64_t max_lq = 0, nonempty = 0;
    for (int32_t r = 0; r < R; ++r) {
        max_lq = std::max<int64_t>(max_lq, q_indptr[r + 1] - q_indptr[r]);
        nonempty += q_indptr[r + 1] > q_indptr[r];
    }
    // per-request page counts: the caller-visible host mirror of the link (checked against its summary so that a
    // stale or foreign array cannot silently drop KV tiles)
    const int32_t *req_pages = link->host_req_pages;
    if (req_pages) {
        int64_t sum = 0;
        int32_t mx = 0;
        for (int32_t r = 0; r < R; ++r) {
            if (req_pages[r] < 0) return COMB_ERR_INVALID;
            sum += req_pages[r];
            mx = std::max(mx, req_pages[r]);
        }
        if (sum != link->total_pages || mx != link->max_pages_per_request) return COMB_ERR_INVALID;
    }
    out->tiles_per_cta = prefill_tiles_per_cta(G, p->cfg.head_dim_qk, p->cfg.head_dim_v, max_lq, nonempty * Hkv,
                                               p->num_sms);
    const int tok_per_tile = 128 / G, tok_per_item = out->tiles_per_cta * tok_per_tile;
    // ---- work items: (request, kv-head, one or two Q tiles) against the request's KV, or against a range of it.
    // Requests are ordered by work (query rows x KV tiles when the page counts are known on the host, else query
    // rows) so the tail of the persistent grid is made of short items.
    auto tiles_of = [&](int32_t r) { return req_pages ? (req_pages[r] + kTilePages - 1) / kTilePages : 1; };
    struct Req { int32_t r; int64_t rows, cost; };
    std::vector<Req> order;
    order.reserve(R);
    for (int32_t r = 0; r < R; ++r) {
        const int64_t rows = (int64_t)q_indptr[r + 1] - q_indptr[r];
        order.push_back(Req{r, rows, rows * std::max(1, tiles_of(r))});
    }
    std::stable_sort(order.begin(), order.end(), [](const Req &a, const Req &b) { return a.cost > b.cost; });
    // kv-head-major: the items in flight at any time (one per CTA, consecutive in this list) then belong to one or two
    // kv-heads across ALL requests, so requests that link the same chunk read its (page, head) blocks within the same
    // window and the later readers hit L2 (Zipf / few-shot reuse); the Q tile groups of one (request, kv-head) are
    // adjacent and share their K/V stream as before.
    std::vector<PrefillItem> base;
    for (int g = 0; g < Hkv; ++g)
        for (const Req &x : order)
            for (int64_t t = 0; t < x.rows; t += tok_per_item)
                base.push_back(PrefillItem{x.r, g, q_indptr[x.r] + (int32_t)t,
                                           (int32_t)std::min<int64_t>(tok_per_item, x.rows - t), 0,
                                           INT32_MAX / kTilePages, -1, 0, 0, 0});
    out->items.clear();
    out->part_rows = 0;
    if (base.empty()) return COMB_OK;
    // ---- KV ranges (need the page counts): (1) fewer items than SMs: every request is cut so that items x ranges
    // fill one wave; (2) several waves with a last wave at most half full: only the items of that last wave are cut
    // (by up to 4), so it takes a fraction of an item's time instead of a whole one (cfg 4: 512 items on 148 SMs).
    const int max_tiles = (link->max_pages_per_request + kTilePages - 1) / kTilePages;
    const size_t ctas = (size_t)p->num_sms *
                        (size_t)prefill_ctas_per_sm(out->tiles_per_cta, p->cfg.head_dim_qk, p->cfg.head_dim_v);
    int uniform = 1, tail_factor = 1;
    size_t tail_from = base.size();
    if (req_pages) {
        // (one item per SM is the target even when two single-tile CTAs share an SM: measured, 256 ranges on 148
        // SMs were slower than 128)
        uniform = plan_prefill_splits(base.size(), max_tiles, p->num_sms);
        const size_t tail = base.size() % ctas;
        if (uniform == 1 && base.size() > ctas && tail > 0 && 2 * tail <= ctas) {
            tail_factor = (int)std::min<size_t>(4, ctas / tail);
            tail_from = base.size() - tail;
        }
    }
    out->items.reserve(base.size() * (size_t)std::max(uniform, 1) + (base.size() - tail_from) * (size_t)tail_factor);
    for (size_t i = 0; i < base.size(); ++i) {
        const int want = i >= tail_from ? tail_factor : uniform;
        const int n_kv = want > 1 ? tiles_of(base[i].request) : 0;
        const int tps = want > 1 ? std::max(2, prefill_tiles_per_split(n_kv, want)) : 0;  // >= 2 tiles per range
        const int eff = tps > 0 ? (n_kv + tps - 1) / tps : 1;
        if (eff <= 1) {
            out->items.push_back(base[i]);
            continue;
        }
        for (int sidx = 0; sidx < eff; ++sidx) {
            PrefillItem it = base[i];
            it.kv_tile0 = sidx * tps;
            it.kv_tiles = sidx + 1 < eff ? tps : INT32_MAX / kTilePages;  // the last range is open-ended
            it.split = sidx;
            it.tps = tps;
            it.part_base = (int32_t)out->part_rows;
            out->items.push_back(it);
        }
        out->part_rows += (int64_t)eff * kPartRowsPerRange;
    }
    return COMB_OK;
}

// fp8 pools: bytes of the bf16 staging (K then V) that prefill dequantises `pages` distinct pages into
size_t fp8_staging_bytes(const comb_pool *p, int64_t pages) {
    const size_t per_page = (size_t)p->cfg.num_kv_heads * kPage * 2;
    return align_up((size_t)std::max<int64_t>(pages, 1) * per_page * p->cfg.head_dim_qk, 1024) +
           align_up((size_t)std::max<int64_t>(pages, 1) * per_page * p->cfg.head_dim_v, 1024);
}

// ---------------------------------------------------------------- chunk-major decode planning
// Units of the chunk-major decode: slot u's entries in groups of 32/G (each entry = G query rows = G columns of the
// swapped-operand MMA), times the KV ranges of the slot.  A long chunk is cut into ranges when the batch would
// otherwise give an SM fewer than ~4 items' worth of work (few chunks, few requests): the item size aimed at is
// a quarter of an SM's share of all KV tiles, never below 2 tiles.  Units are handed out by an atomic counter in the
// order written here: longest first (stable, so the units that stream the same bytes stay adjacent and the second
// and later readers hit L2; slots arrive ordered by descending entry count from comb_link).
constexpr int kCascadeRows = 32;
constexpr int kCascadeMaxRanges = 64;

// units == nullptr: sizes only (what comb_attn_workspace_bytes needs).
int32_t plan_cascade(const comb_link_t *link, int G, int Hkv, int num_sms, std::vector<CascadeItem> *units,
                     size_t *num_units, int64_t *num_partials, int rows_per_item = kCascadeRows) {
    const int32_t U = link->num_distinct_chunks;
    const int32_t *rows = link->host_cas_rows, *pages = link->host_cas_pages;
    if (!rows || !pages || G < 1 || G > rows_per_item) return COMB_ERR_INVALID;
    const int per_unit = rows_per_item / G;  // 32 query rows per item (16 in the fp8 kernel)
    int64_t sum = 0, psum = 0, work = 0;
    int32_t mx = 0;
    for (int32_t u = 0; u < U; ++u) {
        if (rows[u] <= 0 || pages[u] <= 0) return COMB_ERR_INVALID;
        sum += rows[u];
        psum += pages[u];
        mx = std::max(mx, rows[u]);
        work += (int64_t)((rows[u] + per_unit - 1) / per_unit) * ((pages[u] + kTilePages - 1) / kTilePages);
    }
    if (sum != link->total_entries || mx != link->max_rows_per_chunk || psum != link->distinct_pages)
        return COMB_ERR_INVALID;
    work *= Hkv;
    const int64_t share = (int64_t)std::max(num_sms, 1) * 4;
    const int64_t aim = std::max<int64_t>(2, (work + share - 1) / share);
    if (units) units->clear();
    size_t n_units = 0;
    int64_t partials = 0;
    int32_t row0 = 0;
    int64_t page0 = 0, tile0 = 0;  // prefix sums = cas_page_indptr[u], cas_tile_indptr[u]
    for (int32_t u = 0; u < U; ++u) {
        const int32_t tiles = (pages[u] + kTilePages - 1) / kTilePages;
        int32_t nr = (int32_t)std::min<int64_t>((tiles + aim - 1) / aim, kCascadeMaxRanges);
        const int32_t tps = (tiles + nr - 1) / nr;
        nr = (tiles + tps - 1) / tps;
        n_units += (size_t)((rows[u] + per_unit - 1) / per_unit) * (size_t)nr;
        if (units) {
            for (int32_t s = 0; s < nr; ++s)
                for (int32_t t = 0; t < rows[u]; t += per_unit) {
                    CascadeItem it;
                    it.slot = u;
                    it.row0 = row0 + t;
                    it.nrows = std::min<int32_t>(per_unit, rows[u] - t);
                    it.kv_tile0 = s * tps;
                    it.kv_tiles = std::min(tps, tiles - s * tps);
                    it.part0 = (int32_t)(partials + (int64_t)s * rows[u] + t);
                    it.part_stride = rows[u];
                    it.range_nr = (nr << 8) | s;
                    const int32_t skip = std::min(pages[u], it.kv_tile0 * kTilePages);
                    it.pbeg = (int32_t)page0 + skip;
                    it.npages = std::min(pages[u] - skip, it.kv_tiles * kTilePages);
                    it.tile0 = (int32_t)tile0 + it.kv_tile0;
                    it.pad = 0;
                    units->push_back(it);
                }
        }
        partials += (int64_t)rows[u] * nr;
        row0 += rows[u];
        page0 += pages[u];
        tile0 += tiles;
        if (partials > INT32_MAX / 2 || n_units > (size_t)INT32_MAX / 64) return COMB_ERR_CAPACITY;
    }
    if (units)
        std::stable_sort(units->begin(), units->end(),
                         [](const CascadeItem &a, const CascadeItem &b) { return a.kv_tiles > b.kv_tiles; });
    *num_units = n_units;
    *num_partials = partials;
    return COMB_OK;
}

}  // namespace

#pragma GCC visibility push(default)
extern "C" {

const char *comb_version(void) { return "comb-link-b200 0.1 (sm_100a)"; }

const char *comb_strerror(int32_t s) {
    switch (s) {
        case COMB_OK: return "ok";
        case COMB_ERR_INVALID: return "invalid argument";
        case COMB_ERR_NO_SPACE: return "not enough free pages";
        case COMB_ERR_EXISTS: return "chunk exists with a different length";
        case COMB_ERR_UNKNOWN_CHUNK: return "unknown chunk id (compile + store it first)";
        case COMB_ERR_CAPACITY: return "buffer too small";
        case COMB_ERR_CUDA: return "CUDA error (see cudaGetLastError)";
        case COMB_ERR_BUSY: return "chunk is pinned";
        case COMB_ERR_READ_ONLY: return "pool was imported read-only";
        default: return "unknown status";
    }
}

int32_t comb_pool_bytes(const comb_pool_config_t *cfg, size_t *k_bytes, size_t *v_bytes, size_t *scratch_bytes) {
    int32_t rc = validate_cfg(cfg);
    if (rc != COMB_OK) return rc;
    const size_t blocks = (size_t)cfg->num_layers * cfg->num_pages * cfg->num_kv_heads * kPage;
    const size_t elt = cfg->kv_dtype == COMB_KV_E4M3 ? 1 : 2;
    if (k_bytes) *k_bytes = blocks * cfg->head_dim_qk * elt;
    if (v_bytes) *v_bytes = blocks * cfg->head_dim_v * elt;
    if (scratch_bytes)
        *scratch_bytes = kRingSlots * align_up((size_t)cfg->num_pages * kScratchBytesPerPage, 256);
    return COMB_OK;
}

size_t comb_pool_scale_bytes(const comb_pool_config_t *cfg) {
    if (validate_cfg(cfg) != COMB_OK || cfg->kv_dtype != COMB_KV_E4M3) return 0;
    return (size_t)cfg->num_layers * cfg->num_pages * cfg->num_kv_heads * sizeof(float);
}

int32_t comb_pool_create(const comb_pool_config_t *cfg, comb_pool_t **out) {
    if (!out) return COMB_ERR_INVALID;
    *out = nullptr;
    int32_t rc = validate_cfg(cfg);
    if (rc != COMB_OK) return rc;
    if (!cfg->k_arena || !cfg->v_arena || !cfg->scratch) return COMB_ERR_INVALID;
    if (((uintptr_t)cfg->k_arena | (uintptr_t)cfg->v_arena) & 1023) return COMB_ERR_INVALID;
    if (cfg->kv_dtype == COMB_KV_E4M3 &&
        (!cfg->k_scale || !cfg->v_scale || (((uintptr_t)cfg->k_scale | (uintptr_t)cfg->v_scale) & 3)))
        return COMB_ERR_INVALID;
    comb_pool_t *p = new (std::nothrow) comb_pool();
    if (!p) return COMB_ERR_INVALID;
    p->cfg = *cfg;
    p->geom = PoolGeom{cfg->num_layers, cfg->num_kv_heads, cfg->head_dim_qk, cfg->head_dim_v, cfg->num_pages,
                       cfg->k_arena, cfg->v_arena};
    p->geom.kv_dtype = cfg->kv_dtype;
    p->geom.k_scale = (float *)cfg->k_scale;
    p->geom.v_scale = (float *)cfg->v_scale;
    p->free_list.resize(cfg->num_pages);
    for (int32_t i = 0; i < cfg->num_pages; ++i) p->free_list[i] = i;
    if (cfg->free_list_shuffle_seed) {
        uint64_t st = cfg->free_list_shuffle_seed;
        for (int64_t i = cfg->num_pages - 1; i >= 1; --i) {
            const uint64_t j = splitmix64_next(st) % (uint64_t)(i + 1);
            std::swap(p->free_list[i], p->free_list[j]);
        }
    }
    *out = p;
    return COMB_OK;
}

int32_t comb_pool_destroy(comb_pool_t *p) {
    if (!p) return COMB_ERR_INVALID;
    for (auto &r : p->prof_recs) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
    for (auto &e : p->prof_free) cudaEventDestroy(e);
    for (auto &e : p->ready_events)
        if (e.ev) cudaEventDestroy(e.ev);
    if (p->ipc_event) cudaEventDestroy(p->ipc_event);
    for (auto &m : p->ipc_maps) cudaIpcCloseMemHandle(m.second);
    for (auto &s : p->ring) {
        if (s.busy) cudaEventSynchronize(s.ev);
        if (s.ev) cudaEventDestroy(s.ev);
        if (s.host) cudaFreeHost(s.host);
    }
    delete p;
    return COMB_OK;
}

int32_t comb_pool_free_pages(const comb_pool_t *p) {
    if (!p) return COMB_ERR_INVALID;
    return (int32_t)(p->free_list.size() - p->free_head);
}

int64_t comb_pool_launch_count(const comb_pool_t *p) { return p ? p->launches : 0; }

int32_t comb_profile_enable(comb_pool_t *p, int32_t on) {
    if (!p) return COMB_ERR_INVALID;
    p->hook = LaunchHook{&comb_pool::hook_begin, &comb_pool::hook_end, p};
    p->prof_on = on != 0;
    return COMB_OK;
}

int32_t comb_profile_read(comb_pool_t *p, int32_t kernel, double *total_ms, int64_t *launches) {
    if (!p || kernel < 0 || kernel >= kNumKernelIds) return COMB_ERR_INVALID;
    double tot = 0.0;
    int64_t n = 0;
    std::vector<comb_pool::ProfRec> keep;
    for (auto &r : p->prof_recs) {
        if (r.id != kernel) { keep.push_back(r); continue; }
        float ms = 0.f;
        if (cudaEventSynchronize(r.b) != cudaSuccess || cudaEventElapsedTime(&ms, r.a, r.b) != cudaSuccess)
            return COMB_ERR_CUDA;
        tot += ms;
        ++n;
        p->prof_free.push_back(r.a);
        p->prof_free.push_back(r.b);
    }
    p->prof_recs.swap(keep);
    if (total_ms) *total_ms = tot;
    if (launches) *launches = n;
    return COMB_OK;
}

int32_t comb_profile_read_samples(comb_pool_t *p, int32_t kernel, float *ms_out, int64_t cap, int64_t *launches) {
    if (!p || kernel < 0 || kernel >= kNumKernelIds || cap < 0 || (cap > 0 && !ms_out)) return COMB_ERR_INVALID;
    int64_t n = 0;
    std::vector<comb_pool::ProfRec> keep;
    for (auto &r : p->prof_recs) {
        if (r.id != kernel) { keep.push_back(r); continue; }
        float ms = 0.f;
        if (cudaEventSynchronize(r.b) != cudaSuccess || cudaEventElapsedTime(&ms, r.a, r.b) != cudaSuccess)
            return COMB_ERR_CUDA;
        if (n < cap) ms_out[n] = ms;
        ++n;
        p->prof_free.push_back(r.a);
        p->prof_free.push_back(r.b);
    }
    p->prof_recs.swap(keep);
    if (launches) *launches = n;
    return COMB_OK;
}

int32_t comb_util_stream_read(const void *src, size_t bytes, void *sink, void *stream) {
    if (!src || !sink || bytes < 16 || (((uintptr_t)src) & 15)) return COMB_ERR_INVALID;
    return launch_stream_read(src, bytes, sink, (cudaStream_t)stream) == cudaSuccess ? COMB_OK : COMB_ERR_CUDA;
}

int32_t comb_chunk_alloc(comb_pool_t *p, uint64_t id, int32_t T) {
    if (!p) return COMB_ERR_INVALID;
    if (p->imported) return COMB_ERR_READ_ONLY;
    p->last_evicted.clear();
    if (T > 0 && p->dir.find(id) == p->dir.end()) {
        std::unordered_map<uint64_t, int32_t> keep;
        if (!evict_for(p, (size_t)(T + kPage - 1) / kPage, &keep)) return COMB_ERR_NO_SPACE;
    }
    return dir_alloc(p, id, T, nullptr, nullptr);
}

int32_t comb_chunk_pin(comb_pool_t *p, uint64_t id) {
    if (!p) return COMB_ERR_INVALID;
    auto it = p->dir.find(id);
    if (it == p->dir.end()) return COMB_ERR_UNKNOWN_CHUNK;
    it->second.pins += 1;
    return COMB_OK;
}

int32_t comb_chunk_unpin(comb_pool_t *p, uint64_t id) {
    if (!p) return COMB_ERR_INVALID;
    auto it = p->dir.find(id);
    if (it == p->dir.end()) return COMB_ERR_UNKNOWN_CHUNK;
    if (it->second.pins <= 0) return COMB_ERR_INVALID;
    it->second.pins -= 1;
    return COMB_OK;
}

int32_t comb_pool_evicted(const comb_pool_t *p, uint64_t *ids, int32_t cap) {
    if (!p || cap < 0 || (cap > 0 && !ids)) return COMB_ERR_INVALID;
    const int32_t n = (int32_t)p->last_evicted.size();
    for (int32_t i = 0; i < std::min(n, cap); ++i) ids[i] = p->last_evicted[(size_t)i];
    return n;
}

int64_t comb_pool_eviction_count(const comb_pool_t *p) { return p ? p->evictions : 0; }

int32_t comb_chunk_free(comb_pool_t *p, uint64_t id) {
    if (!p) return COMB_ERR_INVALID;
    if (p->imported) return COMB_ERR_READ_ONLY;
    auto it = p->dir.find(id);
    if (it == p->dir.end()) return COMB_ERR_UNKNOWN_CHUNK;
    if (it->second.pins > 0) return COMB_ERR_BUSY;
    dir_free(p, it);
    return COMB_OK;
}

int32_t comb_chunk_query(const comb_pool_t *p, uint64_t id, int32_t *num_tokens, int32_t *pages, int32_t cap) {
    if (!p || cap < 0 || (cap > 0 && !pages)) return COMB_ERR_INVALID;
    auto it = p->dir.find(id);
    if (it == p->dir.end()) return COMB_ERR_UNKNOWN_CHUNK;
    if (num_tokens) *num_tokens = it->second.num_tokens;
    const int32_t n = (int32_t)it->second.pages.size();
    for (int32_t i = 0; i < std::min(n, cap); ++i) pages[i] = it->second.pages[i];
    return n;
}

}  // extern "C"
#pragma GCC visibility pop

namespace {

// After a store's kernel has been enqueued on `st`: one event for the batch; every chunk of the batch points at it.
bool mark_ready(comb_pool_t *p, const std::vector<const Chunk *> &chunks, const uint64_t *ids, cudaStream_t st) {
    const int ei = p->take_ready_event();
    if (ei < 0) return false;
    if (cudaEventRecord(p->ready_events[(size_t)ei].ev, st) != cudaSuccess) return false;
    for (size_t i = 0; i < chunks.size(); ++i) {
        Chunk &c = p->dir.find(ids[i])->second;
        p->drop_ready(c);
        c.ready = ei;
        p->ready_events[(size_t)ei].users += 1;
    }
    return true;
}

// The directory half of a batched store: validates everything first so an error allocates nothing, then takes the
// pages. `undo` restores the directory and the free list exactly (pages are taken from the head in order).
struct StoreBatch {
    std::vector<const Chunk *> chunks;  // per batch entry
    std::vector<uint64_t> created;
    size_t head_before = 0;
    size_t total_pages = 0;             // page descriptors of the batch (existing chunks included)
};
int32_t store_begin(comb_pool_t *p, int32_t layer, int32_t n, const uint64_t *ids, const int32_t *tok_indptr,
                    StoreBatch *sb) {
    if (!p || n < 0 || (n > 0 && (!ids || !tok_indptr))) return COMB_ERR_INVALID;
    if (p->imported) return COMB_ERR_READ_ONLY;
    if (layer < 0 || layer >= p->cfg.num_layers) return COMB_ERR_INVALID;
    if (n == 0) return COMB_OK;
    if (tok_indptr[0] != 0) return COMB_ERR_INVALID;
    size_t need_pages = 0;
    {
        std::unordered_map<uint64_t, int32_t> seen;
        for (int32_t i = 0; i < n; ++i) {
            const int64_t T = (int64_t)tok_indptr[i + 1] - tok_indptr[i];
            if (T <= 0) return COMB_ERR_INVALID;
            const size_t np = (size_t)(T + kPage - 1) / kPage;
            sb->total_pages += np;
            if (!seen.emplace(ids[i], (int32_t)T).second) return COMB_ERR_INVALID;  // the same id twice in one batch
            auto it = p->dir.find(ids[i]);
            if (it != p->dir.end()) {
                if (it->second.num_tokens != T) return COMB_ERR_EXISTS;
            } else {
                need_pages += np;
            }
        }
    }
    if (sb->total_pages > (size_t)p->cfg.num_pages) return COMB_ERR_CAPACITY;
    p->last_evicted.clear();
    if (need_pages > p->free_list.size() - p->free_head) {
        std::unordered_map<uint64_t, int32_t> keep;
        for (int32_t i = 0; i < n; ++i) keep.emplace(ids[i], 0);
        if (!evict_for(p, need_pages, &keep)) return COMB_ERR_NO_SPACE;
    }
    sb->head_before = p->free_head;
    sb->chunks.reserve((size_t)n);
    for (int32_t i = 0; i < n; ++i) {
        const Chunk *c = nullptr;
        bool made = false;
        const int32_t rc = dir_alloc(p, ids[i], tok_indptr[i + 1] - tok_indptr[i], &c, &made);
        if (rc != COMB_OK) return rc;  // cannot happen after validation
        if (made) sb->created.push_back(ids[i]);
        sb->chunks.push_back(c);
    }
    return COMB_OK;
}
void store_undo(comb_pool_t *p, const StoreBatch &sb) {
    for (uint64_t id : sb.created) p->dir.erase(id);
    p->free_head = sb.head_before;
}

}  // namespace

#pragma GCC visibility push(default)
extern "C" {

int32_t comb_store_chunks(comb_pool_t *p, int32_t layer, int32_t n, const uint64_t *ids, const int32_t *tok_indptr,
                          const void *k_packed, const void *v_packed, void *stream) {
    if (n > 0 && (!k_packed || !v_packed)) return COMB_ERR_INVALID;
    StoreBatch sb;
    int32_t rc = store_begin(p, layer, n, ids, tok_indptr, &sb);
    if (rc != COMB_OK || n == 0) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const int slot = p->acquire(sb.total_pages * sizeof(StorePageDesc));
    if (slot < 0) { store_undo(p, sb); return COMB_ERR_CUDA; }
    StorePageDesc *h = (StorePageDesc *)p->ring[slot].host;
    size_t at = 0;
    for (int32_t i = 0; i < n; ++i) {
        const Chunk *c = sb.chunks[(size_t)i];
        const int32_t T = c->num_tokens;
        for (size_t j = 0; j < c->pages.size(); ++j) {
            StorePageDesc d;
            d.dst_page = c->pages[j];
            d.src_tok = tok_indptr[i] + (int32_t)j * kPage;
            d.ntok = std::min<int32_t>(kPage, T - (int32_t)j * kPage);
            d.pad = 0;
            h[at++] = d;
        }
    }
    StorePageDesc *dev = (StorePageDesc *)((char *)p->cfg.scratch + (size_t)slot * p->scratch_slot_bytes());
    if (cudaMemcpyAsync(dev, h, at * sizeof(StorePageDesc), cudaMemcpyHostToDevice, st) != cudaSuccess) {
        store_undo(p, sb);
        return COMB_ERR_CUDA;
    }
    if (p->prof_on) p->hook.begin(p, kKernelStore, st);
    const cudaError_t se = p->geom.kv_dtype == COMB_KV_E4M3
                               ? launch_store_fp8(p->geom, layer, dev, (int)at, k_packed, v_packed, st)
                               : launch_store(p->geom, layer, dev, (int)at, k_packed, v_packed, st);
    if (p->prof_on) p->hook.end(p, st);
    if (se != cudaSuccess) {
        store_undo(p, sb);
        return COMB_ERR_CUDA;
    }
    p->launches += 1;
    if (!mark_ready(p, sb.chunks, ids, st)) return COMB_ERR_CUDA;
    if (!p->release(slot, st)) return COMB_ERR_CUDA;
    return COMB_OK;
}

int32_t comb_project_store_chunks(comb_pool_t *p, int32_t layer, int32_t n, const uint64_t *ids,
                                  const int32_t *tok_indptr, const void *h_packed, int32_t d_model, const void *w_kv,
                                  void *stream) {
    if (n > 0 && (!h_packed || !w_kv)) return COMB_ERR_INVALID;
    if (!p || d_model <= 0 || d_model % 8) return COMB_ERR_INVALID;
    const int32_t N = p->cfg.num_kv_heads * (p->cfg.head_dim_qk + p->cfg.head_dim_v);
    StoreBatch sb;
    int32_t rc = store_begin(p, layer, n, ids, tok_indptr, &sb);
    if (rc != COMB_OK || n == 0) return rc;
    const int64_t M = tok_indptr[n];
    if (!gemm_shape_ok(M, N, d_model)) { store_undo(p, sb); return COMB_ERR_INVALID; }
    // M tiles: 128 tokens (8 pages) of ONE chunk each, so a tile's rows map to whole pages of that chunk
    std::vector<GemmRowTile> tiles;
    tiles.reserve(sb.total_pages / kTilePages + (size_t)n);
    for (int32_t i = 0; i < n; ++i) {
        const Chunk *c = sb.chunks[(size_t)i];
        const int32_t T = c->num_tokens, np = (int32_t)c->pages.size();
        for (int32_t t0 = 0; t0 < T; t0 += 128) {
            GemmRowTile rt;
            rt.a_row0 = tok_indptr[i] + t0;
            rt.rows_valid = std::min(128, T - t0);
            rt.rows_zero_to = std::min(128, np * kPage - t0);  // up to the end of the chunk's last page
            rt.pad = 0;
            for (int j = 0; j < 8; ++j) rt.pages[j] = (t0 / kPage + j < np) ? c->pages[(size_t)(t0 / kPage + j)] : -1;
            tiles.push_back(rt);
        }
    }
    p->probe_device();
    cudaStream_t st = (cudaStream_t)stream;
    const size_t bytes = tiles.size() * sizeof(GemmRowTile);
    if (bytes > p->scratch_slot_bytes()) { store_undo(p, sb); return COMB_ERR_CAPACITY; }
    const int slot = p->acquire(bytes);
    if (slot < 0) { store_undo(p, sb); return COMB_ERR_CUDA; }
    memcpy(p->ring[slot].host, tiles.data(), bytes);
    GemmRowTile *dev = (GemmRowTile *)((char *)p->cfg.scratch + (size_t)slot * p->scratch_slot_bytes());
    if (cudaMemcpyAsync(dev, p->ring[slot].host, bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) {
        store_undo(p, sb);
        return COMB_ERR_CUDA;
    }
    GemmProblem gp{h_packed, w_kv, M, N, d_model};
    if (p->prof_on) p->hook.begin(p, kKernelGemm, st);
    const cudaError_t ge = launch_gemm_paged(gp, p->geom, layer, dev, (int)tiles.size(), p->num_sms, st);
    if (p->prof_on) p->hook.end(p, st);
    if (ge != cudaSuccess) {
        store_undo(p, sb);
        return COMB_ERR_CUDA;
    }
    p->launches += 1;
    if (!mark_ready(p, sb.chunks, ids, st)) return COMB_ERR_CUDA;
    if (!p->release(slot, st)) return COMB_ERR_CUDA;
    return COMB_OK;
}

int32_t comb_gemm_bf16(comb_pool_t *p, const void *a, const void *w, const void *residual, void *c, int64_t M, int32_t N,
                       int32_t K, void *stream) {
    if (!p || !a || !w || !c || !gemm_shape_ok(M, N, K)) return COMB_ERR_INVALID;
    p->probe_device();
    cudaStream_t st = (cudaStream_t)stream;
    GemmProblem gp{a, w, M, N, K};
    if (p->prof_on) p->hook.begin(p, kKernelGemm, st);
    const cudaError_t e = launch_gemm_rowmajor(gp, c, residual, p->num_sms, st);
    if (p->prof_on) p->hook.end(p, st);
    if (e != cudaSuccess) return COMB_ERR_CUDA;
    p->launches += 1;
    return COMB_OK;
}

int32_t comb_store_chunk(comb_pool_t *p, int32_t layer, uint64_t id, int32_t T, const void *k, const void *v,
                         void *stream) {
    if (T <= 0) return COMB_ERR_INVALID;
    const int32_t indptr[2] = {0, T};
    return comb_store_chunks(p, layer, 1, &id, indptr, k, v, stream);
}

size_t comb_link_bytes(int32_t R, int64_t E, int64_t total_pages) {
    if (R < 0 || E < 0 || total_pages < 0) return 0;
    // U <= E distinct chunks; their pages <= total_pages; a chunk's / request's last tile may be partly filled
    return link_layout(R, E, E, total_pages, total_pages / kTilePages + R + 1, total_pages,
                       total_pages / kTilePages + E + 1, true).bytes;
}

size_t comb_link_host_bytes(int32_t R, int64_t E) {
    if (R < 0 || E < 0) return 0;
    return align_up(sizeof(int32_t) * (size_t)std::max(R, 1), 16) +
           2 * align_up(sizeof(int32_t) * (size_t)std::max<int64_t>(E, 1), 16);
}

}  // extern "C"
#pragma GCC visibility pop

namespace {

// PoolT = const comb_pool_t: pure planning. PoolT = comb_pool_t (comb_link): additionally stamps every named chunk
// with `tick` (LRU order) and collects the store events that are still pending for them.
template <class PoolT>
int32_t link_plan_impl(PoolT *p, int32_t R, const int32_t *chunk_indptr, const uint64_t *chunk_ids, comb_link_t *link,
                       void *staging, uint64_t tick, std::vector<int32_t> *pending_events) {
    constexpr bool kTouch = !std::is_const<PoolT>::value;
    if (!p || !link || R < 0 || !chunk_indptr || !staging || !link->device_buf) return COMB_ERR_INVALID;
    if (chunk_indptr[0] != 0) return COMB_ERR_INVALID;
    for (int32_t r = 0; r < R; ++r)
        if (chunk_indptr[r + 1] < chunk_indptr[r]) return COMB_ERR_INVALID;
    const int64_t E = chunk_indptr[R];
    if (E > 0 && !chunk_ids) return COMB_ERR_INVALID;
    // pass 1: lookups + sizes (nothing is written if any id is unknown); distinct chunks in order of first appearance
    int64_t total_pages = 0, total_tiles = 0, total_tok = 0;
    int32_t max_pages = 0;
    std::vector<const Chunk *> found((size_t)E);  // one directory lookup per entry
    std::vector<int32_t> ent_slot((size_t)E);     // entry -> distinct index (first-appearance order for now)
    std::vector<const Chunk *> distinct;
    std::vector<uint64_t> distinct_ids;
    std::vector<int32_t> drows;
    {
        const uint64_t mark = ++p->link_calls;
        for (int32_t r = 0; r < R; ++r) {
            int64_t pr = 0;
            for (int32_t e = chunk_indptr[r]; e < chunk_indptr[r + 1]; ++e) {
                auto it = p->dir.find(chunk_ids[e]);
                if (it == p->dir.end()) return COMB_ERR_UNKNOWN_CHUNK;
                const Chunk *c = &it->second;
                found[(size_t)e] = c;
                pr += (int64_t)c->pages.size();
                total_tok += c->num_tokens;
                if (c->link_mark != mark) {  // first appearance in this batch
                    c->link_mark = mark;
                    c->link_index = (int32_t)distinct.size();
                    distinct.push_back(c);
                    distinct_ids.push_back(chunk_ids[e]);
                    drows.push_back(0);
                }
                (void)tick;
                ent_slot[(size_t)e] = c->link_index;
                drows[(size_t)c->link_index] += 1;
            }
            if (pr > INT32_MAX / kPage) return COMB_ERR_CAPACITY;
            total_pages += pr;
            total_tiles += (pr + kTilePages - 1) / kTilePages;
            max_pages = std::max<int32_t>(max_pages, (int32_t)pr);
        }
    }
    if (total_pages > INT32_MAX) return COMB_ERR_CAPACITY;
    // slots: distinct chunks by descending entry count, ties by first appearance
    const int32_t U = (int32_t)distinct.size();
    std::vector<int32_t> slot_of((size_t)U), by_slot((size_t)U);
    for (int32_t i = 0; i < U; ++i) by_slot[(size_t)i] = i;
    std::stable_sort(by_slot.begin(), by_slot.end(),
                     [&](int32_t a, int32_t b) { return drows[(size_t)a] > drows[(size_t)b]; });
    int64_t distinct_pages = 0, distinct_tiles = 0, distinct_tok = 0;
    for (int32_t u = 0; u < U; ++u) {
        slot_of[(size_t)by_slot[(size_t)u]] = u;
        const Chunk *c = distinct[(size_t)by_slot[(size_t)u]];
        distinct_pages += (int64_t)c->pages.size();
        distinct_tiles += ((int64_t)c->pages.size() + kTilePages - 1) / kTilePages;
        distinct_tok += c->num_tokens;
    }
    const bool compact = p->geom.kv_dtype == COMB_KV_E4M3;
    const LinkLayout L = link_layout(R, E, U, total_pages, total_tiles, distinct_pages, distinct_tiles, compact);
    if (L.bytes > link->device_bytes) return COMB_ERR_CAPACITY;
    const size_t host_need = comb_link_host_bytes(R, U);
    if (link->host_buf && link->host_bytes < host_need) return COMB_ERR_CAPACITY;
    // pass 2: write the tables
    char *hb = (char *)staging;
    int32_t *page_indptr = (int32_t *)(hb + L.off_page_indptr);
    int32_t *kv_len = (int32_t *)(hb + L.off_kv_len);
    int32_t *tile_indptr = (int32_t *)(hb + L.off_tile_indptr);
    int32_t *entry_indptr = (int32_t *)(hb + L.off_entry_indptr);
    uint64_t *tile_ntok = (uint64_t *)(hb + L.off_tile_ntok);
    int32_t *page_ids = (int32_t *)(hb + L.off_page_ids);
    uint8_t *page_ntok = (uint8_t *)(hb + L.off_page_ntok);
    int64_t at = 0, tile_at = 0;
    page_indptr[0] = 0;
    tile_indptr[0] = 0;
    for (int32_t r = 0; r < R; ++r) {
        const int64_t begin = at;
        int64_t kv = 0;
        for (int32_t e = chunk_indptr[r]; e < chunk_indptr[r + 1]; ++e) {
            const Chunk &c = *found[(size_t)e];
            const int32_t np = (int32_t)c.pages.size();
            memcpy(page_ids + at, c.pages.data(), (size_t)np * sizeof(int32_t));
            memset(page_ntok + at, kPage, (size_t)np);
            page_ntok[at + np - 1] = (uint8_t)(c.num_tokens - kPage * (np - 1));  // the chunk's last page may be partly filled
            at += np;
            kv += c.num_tokens;
        }
        kv_len[r] = (int32_t)kv;
        page_indptr[r + 1] = (int32_t)at;
        for (int64_t t = begin; t < at; t += kTilePages) tile_ntok[tile_at++] = pack_tile_ntok(page_ntok, t, at);
        tile_indptr[r + 1] = (int32_t)tile_at;
    }
    memcpy(entry_indptr, chunk_indptr, sizeof(int32_t) * (size_t)(R + 1));
    // chunk-major view
    int32_t *cas_page_indptr = (int32_t *)(hb + L.off_cas_page_indptr);
    int32_t *cas_tile_indptr = (int32_t *)(hb + L.off_cas_tile_indptr);
    int32_t *cas_row_indptr = (int32_t *)(hb + L.off_cas_row_indptr);
    uint64_t *cas_tile_ntok = (uint64_t *)(hb + L.off_cas_tile_ntok);
    int32_t *cas_page_ids = (int32_t *)(hb + L.off_cas_page_ids);
    int32_t *cas_row_req = (int32_t *)(hb + L.off_cas_row_req);
    int32_t *cas_row_entry = (int32_t *)(hb + L.off_cas_row_entry);
    cas_page_indptr[0] = cas_tile_indptr[0] = cas_row_indptr[0] = 0;
    int32_t max_rows = 0;
    {
        int64_t pat = 0, tat = 0;
        std::vector<uint8_t> ntok_tmp;
        for (int32_t u = 0; u < U; ++u) {
            const Chunk &c = *distinct[(size_t)by_slot[(size_t)u]];
            const int32_t np = (int32_t)c.pages.size();
            memcpy(cas_page_ids + pat, c.pages.data(), (size_t)np * sizeof(int32_t));
            ntok_tmp.assign((size_t)np, (uint8_t)kPage);
            ntok_tmp[(size_t)np - 1] = (uint8_t)(c.num_tokens - kPage * (np - 1));
            for (int64_t t = 0; t < np; t += kTilePages) cas_tile_ntok[tat++] = pack_tile_ntok(ntok_tmp.data(), t, np);
            pat += np;
            cas_page_indptr[u + 1] = (int32_t)pat;
            cas_tile_indptr[u + 1] = (int32_t)tat;
            const int32_t rows = drows[(size_t)by_slot[(size_t)u]];
            cas_row_indptr[u + 1] = cas_row_indptr[u] + rows;
            max_rows = std::max(max_rows, rows);
        }
        // entries of a slot in ascending entry number (counting sort over the slots)
        std::vector<int32_t> fill(cas_row_indptr, cas_row_indptr + U);
        for (int32_t r = 0; r < R; ++r)
            for (int32_t e = chunk_indptr[r]; e < chunk_indptr[r + 1]; ++e) {
                const int32_t u = slot_of[(size_t)ent_slot[(size_t)e]];
                cas_row_req[fill[(size_t)u]] = r;
                cas_row_entry[fill[(size_t)u]] = e;
                fill[(size_t)u] += 1;
            }
    }
    if (compact) {  // entry e's pages are pages cas_page_indptr[slot(e)] .. of the distinct-page list, in order
        int32_t *pc = (int32_t *)(hb + L.off_page_ids_compact);
        int64_t w = 0;
        for (int64_t e = 0; e < E; ++e) {
            const int32_t u = slot_of[(size_t)ent_slot[(size_t)e]];
            const int32_t base = cas_page_indptr[u], np = cas_page_indptr[u + 1] - base;
            for (int32_t j = 0; j < np; ++j) pc[w++] = base + j;
        }
    }
    char *db = (char *)link->device_buf;
    link->page_ids_compact = compact ? (int32_t *)(db + L.off_page_ids_compact) : nullptr;
    link->page_indptr = (int32_t *)(db + L.off_page_indptr);
    link->kv_len = (int32_t *)(db + L.off_kv_len);
    link->tile_indptr = (int32_t *)(db + L.off_tile_indptr);
    link->entry_indptr = (int32_t *)(db + L.off_entry_indptr);
    link->tile_ntok = (uint64_t *)(db + L.off_tile_ntok);
    link->page_ids = (int32_t *)(db + L.off_page_ids);
    link->page_ntok = (uint8_t *)(db + L.off_page_ntok);
    link->cas_page_indptr = (int32_t *)(db + L.off_cas_page_indptr);
    link->cas_tile_indptr = (int32_t *)(db + L.off_cas_tile_indptr);
    link->cas_row_indptr = (int32_t *)(db + L.off_cas_row_indptr);
    link->cas_tile_ntok = (uint64_t *)(db + L.off_cas_tile_ntok);
    link->cas_page_ids = (int32_t *)(db + L.off_cas_page_ids);
    link->cas_row_req = (int32_t *)(db + L.off_cas_row_req);
    link->cas_row_entry = (int32_t *)(db + L.off_cas_row_entry);
    link->host_req_pages = nullptr;
    link->host_cas_rows = nullptr;
    link->host_cas_pages = nullptr;
    if (link->host_buf) {  // the host mirror: what the planners of the two attention calls read
        link->host_req_pages = (int32_t *)link->host_buf;
        link->host_cas_rows = (int32_t *)((char *)link->host_buf + align_up(sizeof(int32_t) * (size_t)std::max(R, 1), 16));
        for (int32_t r = 0; r < R; ++r) link->host_req_pages[r] = page_indptr[r + 1] - page_indptr[r];
        link->host_cas_pages = (int32_t *)((char *)link->host_cas_rows + align_up(sizeof(int32_t) * (size_t)std::max(U, 1), 16));
        for (int32_t u = 0; u < U; ++u) {
            link->host_cas_rows[u] = cas_row_indptr[u + 1] - cas_row_indptr[u];
            link->host_cas_pages[u] = cas_page_indptr[u + 1] - cas_page_indptr[u];
        }
    }
    link->num_requests = R;
    link->max_pages_per_request = max_pages;
    link->total_pages = total_pages;
    link->total_tiles = total_tiles;
    link->total_kv_tokens = total_tok;
    link->total_entries = E;
    link->num_distinct_chunks = U;
    link->max_rows_per_chunk = max_rows;
    link->distinct_pages = distinct_pages;
    link->distinct_kv_tokens = distinct_tok;
    link->bytes_used = L.bytes;
    if constexpr (kTouch) {  // the link succeeded: stamp its chunks, note whose stores may still be in flight
        for (int32_t u = 0; u < U; ++u) {
            auto it = p->dir.find(distinct_ids[(size_t)u]);
            it->second.last_use = tick;
            if (it->second.ready >= 0 && pending_events) pending_events->push_back(it->second.ready);
        }
    }
    return COMB_OK;
}

}  // namespace

#pragma GCC visibility push(default)
extern "C" {

int32_t comb_link_plan(const comb_pool_t *p, int32_t R, const int32_t *chunk_indptr, const uint64_t *chunk_ids,
                       comb_link_t *link, void *staging) {
    return link_plan_impl<const comb_pool_t>(p, R, chunk_indptr, chunk_ids, link, staging, 0, nullptr);
}


int32_t comb_link(comb_pool_t *p, int32_t R, const int32_t *chunk_indptr, const uint64_t *chunk_ids,
                  comb_link_t *link, void *stream) {
    if (!p || !link || !link->device_buf) return COMB_ERR_INVALID;
    if (((uintptr_t)link->device_buf) & 15) return COMB_ERR_INVALID;
    const int slot = p->acquire(link->device_bytes);
    if (slot < 0) return COMB_ERR_CUDA;
    std::vector<int32_t> pending;
    int32_t rc = link_plan_impl<comb_pool_t>(p, R, chunk_indptr, chunk_ids, link, p->ring[slot].host, p->tick + 1, &pending);
    if (rc != COMB_OK) return rc;
    p->tick += 1;
    cudaStream_t st = (cudaStream_t)stream;
    // "stored asynchronously": order this stream after the stores of the named chunks that are still
    // in flight (usually none: an event found complete is forgotten for good)
    if (!pending.empty()) {
        std::sort(pending.begin(), pending.end());
        pending.erase(std::unique(pending.begin(), pending.end()), pending.end());
        for (int32_t ei : pending) {
            ReadyEvent &re = p->ready_events[(size_t)ei];
            const cudaError_t q = cudaEventQuery(re.ev);
            if (q == cudaSuccess) {
                for (auto &kv : p->dir)
                    if (kv.second.ready == ei) kv.second.ready = -1;
                re.users = 0;
            } else if (q == cudaErrorNotReady) {
                (void)cudaGetLastError();
                if (cudaStreamWaitEvent(st, re.ev, 0) != cudaSuccess) return COMB_ERR_CUDA;
            } else {
                return COMB_ERR_CUDA;
            }
        }
    }
    // the ONLY data movement of the link stage: the tables. K/V are never touched.
    if (cudaMemcpyAsync(link->device_buf, p->ring[slot].host, link->bytes_used, cudaMemcpyHostToDevice, st) !=
        cudaSuccess)
        return COMB_ERR_CUDA;
    if (!p->release(slot, st)) return COMB_ERR_CUDA;
    return COMB_OK;
}

int32_t comb_pool_set_option(comb_pool_t *p, int32_t option, int64_t value) {
    if (!p) return COMB_ERR_INVALID;
    if (option == COMB_OPT_DECODE_PATH) {
        if (value != COMB_DECODE_AUTO && value != COMB_DECODE_PER_REQUEST && value != COMB_DECODE_CHUNK_MAJOR)
            return COMB_ERR_INVALID;
        p->opt_decode_path = value;
        return COMB_OK;
    }
    if (option == COMB_OPT_EVICT_LRU) {
        if (value != 0 && value != 1) return COMB_ERR_INVALID;
        p->opt_evict_lru = value == 1;
        return COMB_OK;
    }
    if (option == COMB_OPT_PREFILL_CLUSTERS) {
        if (value != 0 && value != 1) return COMB_ERR_INVALID;
        p->opt_prefill_clusters = value == 1;
        return COMB_OK;
    }
    return COMB_ERR_INVALID;
}

size_t comb_workspace_bytes(const comb_pool_t *p, int32_t R, int32_t Hq, int64_t total_q, int32_t max_pages) {
    if (!p || R < 0 || Hq <= 0 || total_q < 0 || max_pages < 0) return 0;
    const_cast<comb_pool_t *>(p)->probe_device();  // caches the SM count; the directory and free list are untouched
    const int G = std::max(1, Hq / p->cfg.num_kv_heads);
    const DecodePlan plan =
        make_decode_plan(R, p->cfg.num_kv_heads * decode_head_subgroups(G), max_pages, p->num_sms);
    const size_t dec = decode_workspace_bytes(R, Hq, p->cfg.head_dim_v, plan);
    size_t max_items = 0;
    int64_t max_rows = 0;
    prefill_bounds(p, Hq, total_q, &max_items, &max_rows);
    const size_t pre = prefill_items_bytes(max_items) + prefill_part_bytes(max_rows, p->cfg.head_dim_v);
    return align_up(std::max(dec, pre), 256) + 256;
}

size_t comb_attn_workspace_bytes(const comb_pool_t *p, const comb_link_t *link, int32_t Hq, int64_t total_q) {
    if (!p || !link || Hq <= 0 || total_q < 0) return 0;
    size_t need = comb_workspace_bytes(p, link->num_requests, Hq, total_q, link->max_pages_per_request);
    if (p->geom.kv_dtype == COMB_KV_E4M3)  // prefill: bf16 staging of the batch's distinct pages behind the rest
        need = align_up(need, 1024) + fp8_staging_bytes(p, link->distinct_pages);
    const int G = std::max(1, Hq / p->cfg.num_kv_heads);
    if (link->host_cas_rows && link->host_cas_pages && cascade_supported(G, p->cfg.head_dim_qk, p->cfg.head_dim_v)) {
        size_t units = 0;
        int64_t partials = 0;
        if (plan_cascade(link, G, p->cfg.num_kv_heads, p->num_sms, nullptr, &units, &partials,
                         p->geom.kv_dtype == COMB_KV_E4M3 ? 16 : kCascadeRows) == COMB_OK)
            need = std::max(need, cascade_layout(units, link->total_entries, partials, Hq, p->cfg.head_dim_v).bytes + 256);
    }
    return need;
}

int32_t comb_cross_attn_decode(comb_pool_t *p, int32_t layer, const comb_link_t *link, int32_t R, const void *q,
                               int32_t Hq, float scale, void *out, float *lse, void *ws, size_t ws_bytes,
                               void *stream) {
    if (!p || !link || R < 0 || Hq <= 0) return COMB_ERR_INVALID;
    if (!(scale > 0.f) || scale > 3.0e38f) return COMB_ERR_INVALID;  // also rejects NaN
    if (layer < 0 || layer >= p->cfg.num_layers) return COMB_ERR_INVALID;
    if (Hq % p->cfg.num_kv_heads) return COMB_ERR_INVALID;
    if (R != link->num_requests) return COMB_ERR_INVALID;
    if (R == 0) return COMB_OK;
    if (!q || !out || !link->page_indptr) return COMB_ERR_INVALID;
    const int G = Hq / p->cfg.num_kv_heads;
    if (!decode_supported(G, p->cfg.head_dim_qk, p->cfg.head_dim_v)) return COMB_ERR_INVALID;
    p->probe_device();
    cudaStream_t st = (cudaStream_t)stream;
    // ---- which path: chunk-major when the batch shares chunks (or when told to), else per request
    const bool can_cascade = link->host_cas_rows && link->host_cas_pages && link->cas_page_indptr &&
                             link->entry_indptr && cascade_supported(G, p->cfg.head_dim_qk, p->cfg.head_dim_v);
    bool cascade = false;
    const bool fp8 = p->geom.kv_dtype == COMB_KV_E4M3;  // fp8 pools: the chunk-major kernel is the only decode kernel
    if (p->opt_decode_path == COMB_DECODE_CHUNK_MAJOR || fp8) {
        if (!can_cascade) return COMB_ERR_INVALID;
        cascade = true;
    } else if (p->opt_decode_path == COMB_DECODE_AUTO && can_cascade) {
        cascade = link->total_entries * 4 >= (int64_t)link->num_distinct_chunks * 5 && link->total_entries > 0;
    }
    if (cascade) {
        std::vector<CascadeItem> units;
        size_t num_units = 0;
        int64_t partials = 0;
        int32_t rc = plan_cascade(link, G, p->cfg.num_kv_heads, p->num_sms, &units, &num_units, &partials,
                                  fp8 ? 16 : kCascadeRows);
        if (rc != COMB_OK) return rc;
        const CascadeLayout lay = cascade_layout(num_units, link->total_entries, partials, Hq, p->cfg.head_dim_v);
        if (!ws || ws_bytes < lay.bytes || (((uintptr_t)ws) & 15)) {
            if (p->opt_decode_path == COMB_DECODE_CHUNK_MAJOR || fp8) return COMB_ERR_CAPACITY;
            cascade = false;  // a workspace sized by the link-independent bound: take the per-request path
        } else {
            if (!p->kv_maps_ready) {
                if (prefill_encode_kv_maps(p->geom, &p->k_map, &p->v_map) != cudaSuccess) return COMB_ERR_CUDA;
                p->kv_maps_ready = true;
            }
            PrefillMaps maps;
            maps.k = p->k_map;
            maps.v = p->v_map;
            maps.q = p->k_map;
            // header (the kernel's item counter, zero) + the units, one copy
            const size_t head_bytes = kCascadeHeaderBytes + num_units * sizeof(CascadeItem);
            const int slot = p->acquire(head_bytes);
            if (slot < 0) return COMB_ERR_CUDA;
            memset(p->ring[slot].host, 0, kCascadeHeaderBytes);
            if (num_units) memcpy((char *)p->ring[slot].host + lay.off_items, units.data(), num_units * sizeof(CascadeItem));
            if (cudaMemcpyAsync(ws, p->ring[slot].host, head_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess)
                return COMB_ERR_CUDA;
            if (!p->release(slot, st)) return COMB_ERR_CUDA;
            int launches = 0;
            cudaError_t e = launch_decode_cascade(p->geom, layer, view_of(link), maps, ws, lay, (int)num_units, R, Hq, q,
                                                  scale, out, lse, p->num_sms, st, &launches, p->active_hook());
            p->launches += launches;
            return e == cudaSuccess ? COMB_OK : COMB_ERR_CUDA;
        }
    }
    const DecodePlan plan = make_decode_plan(R, p->cfg.num_kv_heads * decode_head_subgroups(G),
                                             link->max_pages_per_request, p->num_sms);
    const size_t need = decode_workspace_bytes(R, Hq, p->cfg.head_dim_v, plan);
    if (need > 0 && (!ws || ws_bytes < need)) return COMB_ERR_CAPACITY;
    int launches = 0;
    cudaError_t e = launch_decode(p->geom, layer, view_of(link), R, Hq, q, scale, out, lse, ws, plan, st, &launches,
                                  p->active_hook());
    p->launches += launches;
    return e == cudaSuccess ? COMB_OK : COMB_ERR_CUDA;
}

int32_t comb_cross_attn_prefill(comb_pool_t *p, int32_t layer, const comb_link_t *link, int32_t R, const void *q,
                                const int32_t *q_indptr, int32_t Hq, float scale, void *out, float *lse, void *ws,
                                size_t ws_bytes, void *stream) {
    if (!p || !link || R < 0 || Hq <= 0) return COMB_ERR_INVALID;
    if (!(scale > 0.f) || scale > 3.0e38f) return COMB_ERR_INVALID;  // also rejects NaN
    if (layer < 0 || layer >= p->cfg.num_layers) return COMB_ERR_INVALID;
    if (Hq % p->cfg.num_kv_heads) return COMB_ERR_INVALID;
    if (R != link->num_requests) return COMB_ERR_INVALID;
    if (R == 0) return COMB_OK;
    if (!q_indptr || q_indptr[0] != 0) return COMB_ERR_INVALID;
    for (int32_t r = 0; r < R; ++r)
        if (q_indptr[r + 1] < q_indptr[r]) return COMB_ERR_INVALID;
    const int64_t total_q = q_indptr[R];
    if (total_q == 0) return COMB_OK;
    if (!q || !out || !link->page_indptr) return COMB_ERR_INVALID;
    const int Hkv = p->cfg.num_kv_heads, G = Hq / Hkv;
    if (!prefill_supported(G, p->cfg.head_dim_qk, p->cfg.head_dim_v)) return COMB_ERR_INVALID;
    const bool fp8 = p->geom.kv_dtype == COMB_KV_E4M3;
    if (fp8 && (!link->page_ids_compact || !link->cas_page_ids)) return COMB_ERR_INVALID;
    p->probe_device();
    PrefillPlan plan;
    int32_t rc = plan_prefill(p, link, R, q_indptr, Hq, &plan);
    if (rc != COMB_OK) return rc;
    const size_t num_items = plan.items.size();
    if (num_items == 0) return COMB_OK;
    if (num_items > (size_t)INT32_MAX) return COMB_ERR_CAPACITY;
    const size_t items_bytes = prefill_items_bytes(num_items);
    size_t need = items_bytes + prefill_part_bytes(plan.part_rows, p->cfg.head_dim_v);
    const size_t stage_off = align_up(need, 1024);
    if (fp8) need = stage_off + fp8_staging_bytes(p, link->distinct_pages);
    if (!ws || ws_bytes < need || (((uintptr_t)ws) & 15)) return COMB_ERR_CAPACITY;
    cudaStream_t st = (cudaStream_t)stream;
    PrefillMaps maps;
    PoolGeom geom = p->geom;
    LinkView lv = view_of(link);
    int run_layer = layer;
    if (fp8) {
        // fp8 pool: dequantise the batch's distinct pages (exactly: the scales are powers of two) into a compact bf16
        // pool in the workspace and attend over that through the link's compact page table
        char *kst = (char *)ws + stage_off;
        char *vst = kst + align_up((size_t)std::max<int64_t>(link->distinct_pages, 1) * p->cfg.num_kv_heads * kPage * 2 *
                                   p->cfg.head_dim_qk, 1024);
        if (launch_dequant_pages(p->geom, layer, link->cas_page_ids, (int)link->distinct_pages, kst, vst, st) != cudaSuccess)
            return COMB_ERR_CUDA;
        p->launches += 1;
        geom.kv_dtype = 0;
        geom.k_scale = geom.v_scale = nullptr;
        geom.num_layers = 1;
        geom.num_pages = (int32_t)std::max<int64_t>(link->distinct_pages, 1);
        geom.k_arena = kst;
        geom.v_arena = vst;
        run_layer = 0;
        lv.page_ids = link->page_ids_compact;
        if (prefill_encode_kv_maps(geom, &maps.k, &maps.v) != cudaSuccess) return COMB_ERR_CUDA;
    } else {
        if (!p->kv_maps_ready) {
            if (prefill_encode_kv_maps(p->geom, &p->k_map, &p->v_map) != cudaSuccess) return COMB_ERR_CUDA;
            p->kv_maps_ready = true;
        }
        maps.k = p->k_map;
        maps.v = p->v_map;
    }
    if (prefill_encode_q_map(q, total_q, Hq, G, p->cfg.head_dim_qk, &maps.q) != cudaSuccess) return COMB_ERR_CUDA;
    const int slot = p->acquire(num_items * sizeof(PrefillItem));
    if (slot < 0) return COMB_ERR_CUDA;
    PrefillItem *h = (PrefillItem *)p->ring[slot].host;
    memcpy(h, plan.items.data(), num_items * sizeof(PrefillItem));
    if (cudaMemcpyAsync(ws, h, num_items * sizeof(PrefillItem), cudaMemcpyHostToDevice, st) != cudaSuccess)
        return COMB_ERR_CUDA;
    int launches = 0;
    // consecutive items that share their K/V stream (two Q-tile pairs of one (request, kv-head), whole KV each) may
    // run on a cluster of two CTAs
    bool paired = p->opt_prefill_clusters && plan.part_rows == 0 && num_items % 2 == 0;
    for (size_t i = 0; paired && i < num_items; i += 2)
        paired = plan.items[i].request == plan.items[i + 1].request && plan.items[i].kv_head == plan.items[i + 1].kv_head &&
                 plan.items[i].split < 0 && plan.items[i + 1].split < 0;
    cudaError_t e = launch_prefill(geom, run_layer, lv, maps, (const PrefillItem *)ws, (int)num_items, Hq,
                                   scale, out, lse, total_q, (char *)ws + items_bytes, plan.part_rows,
                                   plan.tiles_per_cta, paired, p->num_sms, st, &launches, p->active_hook());
    if (e != cudaSuccess) return COMB_ERR_CUDA;
    p->launches += launches;
    if (!p->release(slot, st)) return COMB_ERR_CUDA;
    return COMB_OK;
}

size_t comb_layer_workspace_bytes(const comb_pool_t *p, const comb_link_t *link, int32_t Hq, int64_t rows) {
    if (!p || !link || Hq <= 0 || rows < 0) return 0;
    const size_t qb = align_up((size_t)rows * Hq * p->cfg.head_dim_qk * 2, 256);
    const size_t ob = align_up((size_t)rows * Hq * p->cfg.head_dim_v * 2, 256);
    return qb + ob + comb_attn_workspace_bytes(p, link, Hq, rows);
}

int32_t comb_cross_layer_forward(comb_pool_t *p, int32_t layer, const comb_link_t *link, int32_t R, const void *x,
                                 const int32_t *q_indptr, int32_t d_model, int32_t Hq, const void *w_q, const void *w_o,
                                 float scale, void *x_out, void *ws, size_t ws_bytes, void *stream) {
    if (!p || !link || R < 0 || Hq <= 0 || d_model <= 0) return COMB_ERR_INVALID;
    if (R == 0) return COMB_OK;
    if (!x || !x_out || !w_q || !w_o) return COMB_ERR_INVALID;
    const int64_t rows = q_indptr ? (int64_t)q_indptr[R] : (int64_t)R;
    if (rows < 0) return COMB_ERR_INVALID;
    if (rows == 0) return COMB_OK;
    const int Dqk = p->cfg.head_dim_qk, Dv = p->cfg.head_dim_v;
    if (!gemm_shape_ok(rows, Hq * Dqk, d_model) || !gemm_shape_ok(rows, d_model, Hq * Dv)) return COMB_ERR_INVALID;
    const size_t qb = align_up((size_t)rows * Hq * Dqk * 2, 256), ob = align_up((size_t)rows * Hq * Dv * 2, 256);
    const size_t attn_ws = comb_attn_workspace_bytes(p, link, Hq, rows);
    if (!ws || (((uintptr_t)ws) & 15) || ws_bytes < qb + ob + attn_ws) return COMB_ERR_CAPACITY;
    char *qbuf = (char *)ws, *obuf = qbuf + qb, *aws = obuf + ob;
    // Eq. 4: Q = X W_Q
    int32_t rc = comb_gemm_bf16(p, x, w_q, nullptr, qbuf, rows, Hq * Dqk, d_model, stream);
    if (rc != COMB_OK) return rc;
    // Eq. 7-8 over the linked chunks
    rc = q_indptr ? comb_cross_attn_prefill(p, layer, link, R, qbuf, q_indptr, Hq, scale, obuf, nullptr, aws, attn_ws,
                                            stream)
                  : comb_cross_attn_decode(p, layer, link, R, qbuf, Hq, scale, obuf, nullptr, aws, attn_ws, stream);
    if (rc != COMB_OK) return rc;
    // output projection, residual added in the epilogue
    return comb_gemm_bf16(p, obuf, w_o, x, x_out, rows, d_model, Hq * Dv, stream);
}

}  // extern "C"
#pragma GCC visibility pop

// ---------------------------------------------------------------- (f4) export / import over CUDA IPC
namespace {

constexpr uint64_t kExportMagic = 0x31435049424d4f43ull;  // "COMBIPC1"
constexpr uint32_t kExportHasDevice = 1u;

// Fixed-size head of an export blob (little-endian, natural alignment, no pointers); the directory follows:
// per chunk {uint64 id; int32 num_tokens; int32 num_pages; int32 pages[num_pages]} padded to 8 bytes, creation order.
struct ExportHeader {
    uint64_t magic;
    uint32_t version, flags;
    int32_t num_layers, num_kv_heads, head_dim_qk, head_dim_v, page_size, num_pages;
    uint64_t k_bytes, v_bytes, k_offset, v_offset;
    unsigned char k_handle[64], v_handle[64], ev_handle[64];
    uint64_t num_chunks, dir_bytes;
    // fp8 pools: element type and the scale tables
    int32_t kv_dtype, pad;
    uint64_t ks_offset, vs_offset;
    unsigned char ks_handle[64], vs_handle[64];
};
static_assert(sizeof(cudaIpcMemHandle_t) == 64 && sizeof(cudaIpcEventHandle_t) == 64, "CUDA IPC handles are 64 bytes");

size_t export_dir_bytes(const comb_pool_t *p) {
    size_t b = 0;
    for (auto &kv : p->dir) b += 16 + align_up(kv.second.pages.size() * sizeof(int32_t), 8);
    return b;
}

// base address of the allocation that contains ptr (cuMemGetAddressRange through the runtime's driver entry point)
bool allocation_base(const void *ptr, void **base) {
    typedef int (*Fn)(unsigned long long *, size_t *, unsigned long long);
    static Fn fn = nullptr;
    if (!fn) {
        void *f = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuMemGetAddressRange", &f, cudaEnableDefault, &q) != cudaSuccess ||
            q != cudaDriverEntryPointSuccess)
            return false;
        fn = reinterpret_cast<Fn>(f);
    }
    unsigned long long b = 0;
    size_t sz = 0;
    if (fn(&b, &sz, (unsigned long long)(uintptr_t)ptr) != 0) return false;
    *base = (void *)(uintptr_t)b;
    return true;
}

// Parses and checks a blob; on success *h points into it and *dir at the first directory record.
int32_t parse_blob(const void *blob, size_t bytes, const ExportHeader **h, const unsigned char **dir) {
    if (!blob || bytes < sizeof(ExportHeader) || (((uintptr_t)blob) & 7)) return COMB_ERR_INVALID;
    const ExportHeader *x = (const ExportHeader *)blob;
    if (x->magic != kExportMagic || x->version != 1) return COMB_ERR_INVALID;
    if (x->dir_bytes > bytes - sizeof(ExportHeader)) return COMB_ERR_INVALID;
    comb_pool_config_t c{};
    c.num_layers = x->num_layers;
    c.num_kv_heads = x->num_kv_heads;
    c.head_dim_qk = x->head_dim_qk;
    c.head_dim_v = x->head_dim_v;
    c.page_size = x->page_size;
    c.num_pages = x->num_pages;
    c.kv_dtype = x->kv_dtype;
    if (validate_cfg(&c) != COMB_OK) return COMB_ERR_INVALID;
    *h = x;
    *dir = (const unsigned char *)blob + sizeof(ExportHeader);
    return COMB_OK;
}

// Rebuilds a directory from the records of a blob (validating every page id); `out` replaces the pool's on success.
int32_t read_directory(const ExportHeader *h, const unsigned char *dir, std::unordered_map<uint64_t, Chunk> *out) {
    size_t at = 0;
    std::vector<unsigned char> used((size_t)h->num_pages, 0);
    for (uint64_t i = 0; i < h->num_chunks; ++i) {
        if (at + 16 > h->dir_bytes) return COMB_ERR_INVALID;
        uint64_t id;
        int32_t T, np;
        memcpy(&id, dir + at, 8);
        memcpy(&T, dir + at + 8, 4);
        memcpy(&np, dir + at + 12, 4);
        at += 16;
        if (T <= 0 || np != (T + kPage - 1) / kPage) return COMB_ERR_INVALID;
        const size_t pb = align_up((size_t)np * sizeof(int32_t), 8);
        if (at + pb > h->dir_bytes) return COMB_ERR_INVALID;
        Chunk c;
        c.num_tokens = T;
        c.pages.resize((size_t)np);
        memcpy(c.pages.data(), dir + at, (size_t)np * sizeof(int32_t));
        at += pb;
        for (int32_t pg : c.pages) {
            if (pg < 0 || pg >= h->num_pages || used[(size_t)pg]) return COMB_ERR_INVALID;  // out of range / shared
            used[(size_t)pg] = 1;
        }
        c.seq = i;
        if (!out->emplace(id, std::move(c)).second) return COMB_ERR_INVALID;  // the same id twice
    }
    return COMB_OK;
}

int32_t wait_remote_event(const ExportHeader *h, cudaStream_t st) {
    cudaIpcEventHandle_t eh;
    memcpy(&eh, h->ev_handle, sizeof(eh));
    cudaEvent_t ev = nullptr;
    if (cudaIpcOpenEventHandle(&ev, eh) != cudaSuccess) return COMB_ERR_CUDA;
    const cudaError_t e = cudaStreamWaitEvent(st, ev, 0);
    cudaEventDestroy(ev);
    return e == cudaSuccess ? COMB_OK : COMB_ERR_CUDA;
}

}  // namespace

#pragma GCC visibility push(default)
extern "C" {

size_t comb_pool_export_bytes(const comb_pool_t *p) {
    if (!p) return 0;
    return sizeof(ExportHeader) + export_dir_bytes(p);
}

int32_t comb_pool_export(comb_pool_t *p, uint32_t flags, void *stream, void *blob, size_t cap, size_t *written) {
    if (!p || !blob || (flags & ~(uint32_t)COMB_EXPORT_DIRECTORY_ONLY) || (((uintptr_t)blob) & 7)) return COMB_ERR_INVALID;
    const size_t dir_bytes = export_dir_bytes(p);
    if (cap < sizeof(ExportHeader) + dir_bytes) return COMB_ERR_CAPACITY;
    ExportHeader h;
    memset(&h, 0, sizeof(h));
    h.magic = kExportMagic;
    h.version = 1;
    h.num_layers = p->cfg.num_layers;
    h.num_kv_heads = p->cfg.num_kv_heads;
    h.head_dim_qk = p->cfg.head_dim_qk;
    h.head_dim_v = p->cfg.head_dim_v;
    h.page_size = p->cfg.page_size;
    h.num_pages = p->cfg.num_pages;
    size_t kb = 0, vb = 0;
    comb_pool_bytes(&p->cfg, &kb, &vb, nullptr);
    h.k_bytes = kb;
    h.v_bytes = vb;
    h.num_chunks = p->dir.size();
    h.dir_bytes = dir_bytes;
    h.kv_dtype = p->cfg.kv_dtype;
    if (!(flags & COMB_EXPORT_DIRECTORY_ONLY)) {
        if (p->imported) return COMB_ERR_READ_ONLY;  // only the owner of the arenas hands them out
        cudaStream_t st = (cudaStream_t)stream;
        void *kbase = nullptr, *vbase = nullptr;
        if (!allocation_base(p->cfg.k_arena, &kbase) || !allocation_base(p->cfg.v_arena, &vbase)) return COMB_ERR_CUDA;
        cudaIpcMemHandle_t kh, vh;
        if (cudaIpcGetMemHandle(&kh, kbase) != cudaSuccess || cudaIpcGetMemHandle(&vh, vbase) != cudaSuccess)
            return COMB_ERR_CUDA;
        memcpy(h.k_handle, &kh, 64);
        memcpy(h.v_handle, &vh, 64);
        h.k_offset = (uint64_t)((char *)p->cfg.k_arena - (char *)kbase);
        h.v_offset = (uint64_t)((char *)p->cfg.v_arena - (char *)vbase);
        if (p->cfg.kv_dtype == COMB_KV_E4M3) {
            void *ksb = nullptr, *vsb = nullptr;
            if (!allocation_base(p->cfg.k_scale, &ksb) || !allocation_base(p->cfg.v_scale, &vsb)) return COMB_ERR_CUDA;
            cudaIpcMemHandle_t ksh, vsh;
            if (cudaIpcGetMemHandle(&ksh, ksb) != cudaSuccess || cudaIpcGetMemHandle(&vsh, vsb) != cudaSuccess)
                return COMB_ERR_CUDA;
            memcpy(h.ks_handle, &ksh, 64);
            memcpy(h.vs_handle, &vsh, 64);
            h.ks_offset = (uint64_t)((char *)p->cfg.k_scale - (char *)ksb);
            h.vs_offset = (uint64_t)((char *)p->cfg.v_scale - (char *)vsb);
        }
        // every store enqueued so far precedes the event the importer waits for
        for (auto &re : p->ready_events)
            if (re.ev && re.users > 0 && cudaStreamWaitEvent(st, re.ev, 0) != cudaSuccess) return COMB_ERR_CUDA;
        if (!p->ipc_event &&
            cudaEventCreateWithFlags(&p->ipc_event, cudaEventDisableTiming | cudaEventInterprocess) != cudaSuccess)
            return COMB_ERR_CUDA;
        if (cudaEventRecord(p->ipc_event, st) != cudaSuccess) return COMB_ERR_CUDA;
        cudaIpcEventHandle_t eh;
        if (cudaIpcGetEventHandle(&eh, p->ipc_event) != cudaSuccess) return COMB_ERR_CUDA;
        memcpy(h.ev_handle, &eh, 64);
        h.flags |= kExportHasDevice;
    }
    memcpy(blob, &h, sizeof(h));
    // directory in creation order (deterministic blobs; the importer keeps the order as its own creation order)
    std::vector<std::pair<uint64_t, uint64_t>> order;  // (seq, id)
    order.reserve(p->dir.size());
    for (auto &kv : p->dir) order.emplace_back(kv.second.seq, kv.first);
    std::sort(order.begin(), order.end());
    unsigned char *d = (unsigned char *)blob + sizeof(ExportHeader);
    size_t at = 0;
    for (auto &o : order) {
        const Chunk &c = p->dir.find(o.second)->second;
        const int32_t np = (int32_t)c.pages.size();
        memcpy(d + at, &o.second, 8);
        memcpy(d + at + 8, &c.num_tokens, 4);
        memcpy(d + at + 12, &np, 4);
        at += 16;
        const size_t pb = align_up((size_t)np * sizeof(int32_t), 8);
        memset(d + at, 0, pb);
        memcpy(d + at, c.pages.data(), (size_t)np * sizeof(int32_t));
        at += pb;
    }
    if (written) *written = sizeof(ExportHeader) + at;
    return COMB_OK;
}

int32_t comb_pool_import(const void *blob, size_t bytes, void *stream, comb_pool_t **out) {
    if (!out) return COMB_ERR_INVALID;
    *out = nullptr;
    const ExportHeader *h = nullptr;
    const unsigned char *dir = nullptr;
    int32_t rc = parse_blob(blob, bytes, &h, &dir);
    if (rc != COMB_OK) return rc;
    if (!(h->flags & kExportHasDevice)) return COMB_ERR_INVALID;  // a directory-only blob cannot open the arenas
    std::unordered_map<uint64_t, Chunk> d;
    if ((rc = read_directory(h, dir, &d)) != COMB_OK) return rc;
    comb_pool_t *p = new (std::nothrow) comb_pool();
    if (!p) return COMB_ERR_INVALID;
    // open every distinct allocation once (several tables may live in one allocation of a caching allocator)
    auto open = [&](const unsigned char *handle, uint64_t offset, void **out_ptr) -> bool {
        for (auto &m : p->ipc_maps)
            if (memcmp(&m.first, handle, 64) == 0) { *out_ptr = (char *)m.second + offset; return true; }
        cudaIpcMemHandle_t mh;
        memcpy(&mh, handle, 64);
        void *base = nullptr;
        if (cudaIpcOpenMemHandle(&base, mh, cudaIpcMemLazyEnablePeerAccess) != cudaSuccess) return false;
        p->ipc_maps.emplace_back(mh, base);
        *out_ptr = (char *)base + offset;
        return true;
    };
    void *ka = nullptr, *va = nullptr, *ksa = nullptr, *vsa = nullptr;
    bool ok = open(h->k_handle, h->k_offset, &ka) && open(h->v_handle, h->v_offset, &va);
    if (ok && h->kv_dtype == COMB_KV_E4M3)
        ok = open(h->ks_handle, h->ks_offset, &ksa) && open(h->vs_handle, h->vs_offset, &vsa);
    if (!ok) {
        comb_pool_destroy(p);
        return COMB_ERR_CUDA;
    }
    p->imported = true;
    p->cfg.num_layers = h->num_layers;
    p->cfg.num_kv_heads = h->num_kv_heads;
    p->cfg.head_dim_qk = h->head_dim_qk;
    p->cfg.head_dim_v = h->head_dim_v;
    p->cfg.page_size = h->page_size;
    p->cfg.num_pages = h->num_pages;
    p->cfg.k_arena = ka;
    p->cfg.v_arena = va;
    p->cfg.scratch = nullptr;
    p->cfg.free_list_shuffle_seed = 0;
    p->cfg.kv_dtype = h->kv_dtype;
    p->cfg.reserved = 0;
    p->cfg.k_scale = ksa;
    p->cfg.v_scale = vsa;
    p->geom = PoolGeom{h->num_layers, h->num_kv_heads, h->head_dim_qk, h->head_dim_v, h->num_pages, p->cfg.k_arena,
                       p->cfg.v_arena};
    p->geom.kv_dtype = h->kv_dtype;
    p->geom.k_scale = (float *)ksa;
    p->geom.v_scale = (float *)vsa;
    p->dir.swap(d);
    p->next_seq = h->num_chunks;
    if ((rc = wait_remote_event(h, (cudaStream_t)stream)) != COMB_OK) {
        comb_pool_destroy(p);
        return rc;
    }
    *out = p;
    return COMB_OK;
}

int32_t comb_pool_refresh(comb_pool_t *p, const void *blob, size_t bytes, void *stream) {
    if (!p || !p->imported) return COMB_ERR_INVALID;
    const ExportHeader *h = nullptr;
    const unsigned char *dir = nullptr;
    int32_t rc = parse_blob(blob, bytes, &h, &dir);
    if (rc != COMB_OK) return rc;
    if (h->num_layers != p->cfg.num_layers || h->num_kv_heads != p->cfg.num_kv_heads ||
        h->head_dim_qk != p->cfg.head_dim_qk || h->head_dim_v != p->cfg.head_dim_v || h->num_pages != p->cfg.num_pages ||
        h->kv_dtype != p->cfg.kv_dtype)
        return COMB_ERR_INVALID;
    std::unordered_map<uint64_t, Chunk> d;
    if ((rc = read_directory(h, dir, &d)) != COMB_OK) return rc;
    for (auto &kv : d) {  // local pins and use stamps survive for the chunks that are still there
        auto old = p->dir.find(kv.first);
        if (old != p->dir.end() && old->second.num_tokens == kv.second.num_tokens) {
            kv.second.pins = old->second.pins;
            kv.second.last_use = old->second.last_use;
        }
    }
    if ((h->flags & kExportHasDevice) && (rc = wait_remote_event(h, (cudaStream_t)stream)) != COMB_OK) return rc;
    p->dir.swap(d);
    p->next_seq = h->num_chunks;
    return COMB_OK;
}

}  // extern "C"
#pragma GCC visibility pop

// ============================================================================================
// Decode without any allocation (comb_cross_attn_decode_noalloc, include/comb.h): the per-request split-KV path
// with its split partials in a file-scope device array instead of a caller workspace.
// ============================================================================================
namespace comb {
namespace {

// 8 MiB, held by every GPU that loads the library. The decode plan aims at ~4 waves of 2 CTAs per SM, so on a
// 148-SM B200 the partials never exceed ~5 MB (R x Hq x splits <= ~9.5 K rows of Dv + 2 floats); the bound below only
// rejects calls on devices with more SMs (or a future plan that splits further).
constexpr size_t kNoAllocScratchBytes = (size_t)8 << 20;
static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocScratchBytes];

// In host code `g_noalloc_scratch` is a host-side stand-in, not a device address: the address the kernels get comes
// from cudaGetSymbolAddress, asked once per device with that device current.
constexpr int kNoAllocMaxDevices = 64;
void *g_noalloc_ptr[kNoAllocMaxDevices];  // written once per device (a benign race writes the same value twice)

int32_t noalloc_scratch(void **ptr) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return COMB_ERR_CUDA;
    if (dev < 0 || dev >= kNoAllocMaxDevices) return COMB_ERR_INVALID;
    void *p = g_noalloc_ptr[dev];
    if (!p) {
        if (cudaGetSymbolAddress(&p, g_noalloc_scratch) != cudaSuccess || !p) return COMB_ERR_CUDA;
        g_noalloc_ptr[dev] = p;
    }
    *ptr = p;
    return COMB_OK;
}

}  // namespace
}  // namespace comb

#pragma GCC visibility push(default)
extern "C" {

size_t comb_noalloc_scratch_bytes(void) { return comb::kNoAllocScratchBytes; }

int32_t comb_cross_attn_decode_noalloc(comb_pool_t *p, int32_t layer, const comb_link_t *link, int32_t R,
                                       const void *q, int32_t Hq, float scale, void *out, float *lse, void *stream) {
    using namespace comb;
    if (!p || !link || R < 0 || Hq <= 0) return COMB_ERR_INVALID;
    if (!(scale > 0.f) || scale > 3.0e38f) return COMB_ERR_INVALID;  // also rejects NaN
    if (layer < 0 || layer >= p->cfg.num_layers) return COMB_ERR_INVALID;
    if (Hq % p->cfg.num_kv_heads) return COMB_ERR_INVALID;
    if (R != link->num_requests) return COMB_ERR_INVALID;
    if (p->geom.kv_dtype == COMB_KV_E4M3) return COMB_ERR_INVALID;  // fp8 pools have no per-request kernel
    if (R == 0) return COMB_OK;
    if (!q || !out || !link->page_indptr) return COMB_ERR_INVALID;
    const int G = Hq / p->cfg.num_kv_heads;
    if (!decode_supported(G, p->cfg.head_dim_qk, p->cfg.head_dim_v)) return COMB_ERR_INVALID;
    p->probe_device();
    const DecodePlan plan = make_decode_plan(R, p->cfg.num_kv_heads * decode_head_subgroups(G),
                                             link->max_pages_per_request, p->num_sms);
    const size_t need = decode_workspace_bytes(R, Hq, p->cfg.head_dim_v, plan);
    if (need > kNoAllocScratchBytes) return COMB_ERR_CAPACITY;  // beyond the fixed array: use comb_cross_attn_decode
    void *scratch = nullptr;
    const int32_t rc = noalloc_scratch(&scratch);
    if (rc != COMB_OK) return rc;
    // Nothing in the array must start at zero: the split kernel writes every (request, head, split) partial the
    // merge kernel reads (the merge derives a request's split count from its page count), so the previous call's
    // contents are never seen.
    int launches = 0;
    cudaError_t e = launch_decode(p->geom, layer, view_of(link), R, Hq, q, scale, out, lse, scratch, plan,
                                  (cudaStream_t)stream, &launches, nullptr);
    p->launches += launches;
    return e == cudaSuccess ? COMB_OK : COMB_ERR_CUDA;
}

}  // extern "C"
#pragma GCC visibility pop
