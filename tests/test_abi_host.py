"""CPU-only tests of the C-ABI library: it loads without a GPU, exports every symbol include/comb.h declares,
and its host logic (allocator, directory, block-table builder, error paths) agrees bit-exactly with the
oracle's independent table model O3 (oracle.PoolModel).  No compute call is made here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import oracle
import paper_2602_01519_b200 as comb
from paper_2602_01519_b200 import _lib

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
FAKE_K, FAKE_V, FAKE_S = 0x7000_0000_0000, 0x7100_0000_0000, 0x7200_0000_0000  # never dereferenced on the host


def make_pool(num_pages=64, Hkv=2, Dqk=64, Dv=64, seed=0, layers=1):
    cfg = comb.PoolConfig(layers, Hkv, Dqk, Dv, 16, num_pages, FAKE_K, FAKE_V, FAKE_S, seed)
    return comb.comb_pool_create(cfg)


def plan(pool, lists, host_mirror=True):
    indptr = np.zeros(len(lists) + 1, np.int32)
    np.cumsum([len(x) for x in lists], out=indptr[1:])
    ids = np.array([c for l in lists for c in l], np.uint64)
    total = sum(len(comb.comb_chunk_query(pool, int(c))[1]) for c in ids)
    nbytes = comb.comb_link_bytes(len(lists), len(ids), total)
    host = np.zeros(nbytes, np.uint8)
    mirror = np.zeros(comb.comb_link_host_bytes(len(lists), len(ids)), np.uint8) if host_mirror else None
    link = comb.Link()
    link.device_buf = 0x10000  # layout base only; comb_link_plan writes into the staging array
    link.device_bytes = nbytes
    if host_mirror:
        link.host_buf, link.host_bytes = mirror.ctypes.data, mirror.nbytes
    comb.comb_link_plan(pool, indptr, ids, link, host)

    def view(ptr, n, dt):
        off = ptr - 0x10000
        return host[off:off + n * np.dtype(dt).itemsize].view(dt).copy()
    R, U, E = len(lists), int(link.num_distinct_chunks), int(link.total_entries)
    tabs = {
        "page_indptr": view(link.page_indptr, R + 1, np.int32),
        "page_ids": view(link.page_ids, int(link.total_pages), np.int32),
        "page_ntok": view(link.page_ntok, int(link.total_pages), np.uint8),
        "kv_len": view(link.kv_len, R, np.int32),
        "tile_indptr": view(link.tile_indptr, R + 1, np.int32),
        "tile_ntok": view(link.tile_ntok, int(link.total_tiles), np.uint64),
        "entry_indptr": view(link.entry_indptr, R + 1, np.int32),
        "cas_page_indptr": view(link.cas_page_indptr, U + 1, np.int32),
        "cas_page_ids": view(link.cas_page_ids, int(link.distinct_pages), np.int32),
        "cas_tile_indptr": view(link.cas_tile_indptr, U + 1, np.int32),
        "cas_row_indptr": view(link.cas_row_indptr, U + 1, np.int32),
        "cas_row_req": view(link.cas_row_req, E, np.int32),
        "cas_row_entry": view(link.cas_row_entry, E, np.int32),
    }
    tabs["cas_tile_ntok"] = view(link.cas_tile_ntok, int(tabs["cas_tile_indptr"][-1]), np.uint64)
    if host_mirror:
        o1, o2 = link.host_req_pages - mirror.ctypes.data, link.host_cas_rows - mirror.ctypes.data
        tabs["host_req_pages"] = mirror[o1:o1 + 4 * R].view(np.int32).copy()
        tabs["host_cas_rows"] = mirror[o2:o2 + 4 * U].view(np.int32).copy()
        o3 = link.host_cas_pages - mirror.ctypes.data
        tabs["host_cas_pages"] = mirror[o3:o3 + 4 * U].view(np.int32).copy()
    link._keepalive = (host, mirror)
    return link, tabs


def check_tiles(indptr, ntok, tile_indptr, tile_ntok):
    """tile_ntok is page_ntok regrouped by 8 (derived; checked against its definition in comb.h)."""
    for r in range(len(indptr) - 1):
        pn = ntok[indptr[r]:indptr[r + 1]]
        tiles = tile_ntok[tile_indptr[r]:tile_indptr[r + 1]]
        assert len(tiles) == (len(pn) + 7) // 8
        for t, packed in enumerate(tiles):
            want = [int(x) for x in pn[8 * t:8 * t + 8]] + [0] * (8 - len(pn[8 * t:8 * t + 8]))
            assert [(int(packed) >> (8 * j)) & 0xff for j in range(8)] == want


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "comb.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(comb_[a-z0-9_]+)\s*\(", hdr))
    assert {"comb_pool_create", "comb_store_chunk", "comb_link", "comb_cross_attn_prefill",
            "comb_cross_attn_decode"} <= declared
    lib = C.CDLL(_lib.LIB_PATH)
    for name in sorted(declared):
        assert hasattr(lib, name), "libcomb.so does not export %s" % name
    assert declared == set(_lib.EXPORTS), "binding and header disagree: %s" % (declared ^ set(_lib.EXPORTS))
    assert "sm_100a" in comb.comb_version()


def test_pool_bytes_and_layer_saving():
    k, v, s = comb.comb_pool_bytes(8, 8, 128, 128, 64)  # 8 cross layers, 1024 tokens
    per_layer_tok = 8 * 128 * 2
    assert k == 8 * 1024 * per_layer_tok and v == k and s > 0
    # PAPER.md:277 (Fig. 9): 8 cross layers instead of 32 decoder layers of the same head shape => 75 % saved
    k32, v32, _ = comb.comb_pool_bytes(32, 8, 128, 128, 64)
    assert 1.0 - (k + v) / (k32 + v32) == 0.75
    k, v, _ = comb.comb_pool_bytes(1, 16, 192, 128, 10)  # MLA-shaped: Dqk != Dv
    assert (k, v) == (10 * 16 * 16 * 192 * 2, 10 * 16 * 16 * 128 * 2)


def test_config_validation():
    for bad in [dict(page=8), dict(Dqk=96), dict(Dv=192), dict(pages=0), dict(Hkv=0)]:
        cfg = comb.PoolConfig(1, bad.get("Hkv", 2), bad.get("Dqk", 64), bad.get("Dv", 64), bad.get("page", 16),
                              bad.get("pages", 8), FAKE_K, FAKE_V, FAKE_S, 0)
        with pytest.raises(comb.CombError) as e:
            comb.comb_pool_create(cfg)
        assert e.value.status == comb.COMB_ERR_INVALID
    cfg = comb.PoolConfig(1, 2, 64, 64, 16, 8, FAKE_K + 16, FAKE_V, FAKE_S, 0)  # misaligned arena
    with pytest.raises(comb.CombError):
        comb.comb_pool_create(cfg)


@pytest.mark.parametrize("seed", [0, 12345])
def test_allocator_and_tables_match_oracle_model(seed):
    rng = np.random.default_rng(seed + 1)
    pool, model = make_pool(200, seed=seed), oracle.PoolModel(200, seed)
    lens = {}
    for cid in range(20):
        T = int(rng.integers(1, 100))
        comb.comb_chunk_alloc(pool, cid, T)
        model.store(cid, T)
        lens[cid] = T
    for cid in (3, 11, 7):  # freed pages go to the tail, in page-list order
        comb.comb_chunk_free(pool, cid)
        model.release(cid)
        del lens[cid]
    for cid in range(20, 30):
        T = int(rng.integers(1, 60))
        comb.comb_chunk_alloc(pool, cid, T)
        model.store(cid, T)
        lens[cid] = T
    assert _lib.lib.comb_pool_free_pages(pool) == model.free_pages()
    for cid, T in lens.items():
        nt, pages = comb.comb_chunk_query(pool, cid)
        assert nt == T and pages.tolist() == model.dir[cid][1]
    ids = sorted(lens)
    lists = [list(rng.choice(ids, size=int(rng.integers(0, 9)), replace=False)) for _ in range(7)]
    lists[2] = []                     # a request with no contexts
    lists[4] = [ids[0], ids[0]]       # duplicates are taken literally (reading I14)
    link, got = plan(pool, lists)
    exp = model.link(lists)
    for key in ("page_indptr", "page_ids", "page_ntok", "kv_len"):
        assert np.array_equal(got[key], exp[key]), key
    check_tiles(exp["page_indptr"], exp["page_ntok"], got["tile_indptr"], got["tile_ntok"])
    # chunk-major view of the same batch, bit-exact against the model's independent inversion
    cm = model.link_chunk_major(lists)
    for key in ("entry_indptr", "cas_page_indptr", "cas_page_ids", "cas_row_indptr", "cas_row_req", "cas_row_entry"):
        assert np.array_equal(got[key], cm[key]), key
    check_tiles(cm["cas_page_indptr"], cm["cas_page_ntok"], got["cas_tile_indptr"], got["cas_tile_ntok"])
    assert link.num_distinct_chunks == len(cm["slot_chunks"]) and link.total_entries == len(cm["cas_row_req"])
    assert link.distinct_pages == len(cm["cas_page_ids"])
    assert link.distinct_kv_tokens == sum(lens[int(c)] for c in cm["slot_chunks"])
    assert link.max_rows_per_chunk == (int(np.diff(cm["cas_row_indptr"]).max()) if len(cm["slot_chunks"]) else 0)
    # every entry appears exactly once, under the slot of its chunk, with its request
    flat = [int(c) for l in lists for c in l]
    assert sorted(got["cas_row_entry"].tolist()) == list(range(len(flat)))
    for u, c in enumerate(cm["slot_chunks"]):
        for x in range(cm["cas_row_indptr"][u], cm["cas_row_indptr"][u + 1]):
            e = int(got["cas_row_entry"][x])
            assert flat[e] == int(c) and got["entry_indptr"][got["cas_row_req"][x]] <= e < got["entry_indptr"][got["cas_row_req"][x] + 1]
    # host mirror = what the planners read
    assert np.array_equal(got["host_req_pages"], np.diff(exp["page_indptr"]))
    assert np.array_equal(got["host_cas_rows"], np.diff(cm["cas_row_indptr"]))
    assert np.array_equal(got["host_cas_pages"], np.diff(got["cas_page_indptr"]))
    assert link.total_kv_tokens == int(exp["kv_len"].sum())
    assert link.max_pages_per_request == int(np.diff(exp["page_indptr"]).max())
    comb.comb_pool_destroy(pool)


def test_error_paths():
    pool = make_pool(4)
    comb.comb_chunk_alloc(pool, 1, 33)                     # 3 pages
    comb.comb_chunk_alloc(pool, 1, 33)                     # idempotent
    with pytest.raises(comb.CombError) as e:
        comb.comb_chunk_alloc(pool, 1, 34)
    assert e.value.status == comb.COMB_ERR_EXISTS
    with pytest.raises(comb.CombError) as e:
        comb.comb_chunk_alloc(pool, 2, 17)                 # needs 2 pages, 1 free; nothing allocated
    assert e.value.status == comb.COMB_ERR_NO_SPACE
    assert _lib.lib.comb_pool_free_pages(pool) == 1
    with pytest.raises(comb.CombError) as e:
        comb.comb_chunk_alloc(pool, 3, 0)
    assert e.value.status == comb.COMB_ERR_INVALID
    with pytest.raises(comb.CombError) as e:
        comb.comb_chunk_query(pool, 99)
    assert e.value.status == comb.COMB_ERR_UNKNOWN_CHUNK
    with pytest.raises(comb.CombError) as e:
        comb.comb_chunk_free(pool, 99)
    assert e.value.status == comb.COMB_ERR_UNKNOWN_CHUNK
    # link before store: UNKNOWN_CHUNK, nothing written (PAPER.md:62 step 2: a miss must compile + store first)
    link = comb.Link()
    link.device_buf, link.device_bytes = 0x10000, 4096
    host = np.full(4096, 0xAB, np.uint8)
    mirror = np.full(64, 0xCD, np.uint8)
    link.host_buf, link.host_bytes = mirror.ctypes.data, mirror.nbytes
    with pytest.raises(comb.CombError) as e:
        comb.comb_link_plan(pool, np.array([0, 2], np.int32), np.array([1, 42], np.uint64), link, host)
    assert e.value.status == comb.COMB_ERR_UNKNOWN_CHUNK and np.all(host == 0xAB) and np.all(mirror == 0xCD)
    link.device_bytes = 16                                  # too small
    with pytest.raises(comb.CombError) as e:
        comb.comb_link_plan(pool, np.array([0, 1], np.int32), np.array([1], np.uint64), link, host)
    assert e.value.status == comb.COMB_ERR_CAPACITY
    with pytest.raises(comb.CombError) as e:                # non-monotone indptr
        link.device_bytes = 4096
        comb.comb_link_plan(pool, np.array([0, 1, 0], np.int32), np.array([1], np.uint64), link, host)
    assert e.value.status == comb.COMB_ERR_INVALID
    comb.comb_pool_destroy(pool)


def test_product_does_not_import_oracle():
    """The product path must not reach into oracle/ (or _work/)."""
    pkg = os.path.join(ROOT, "paper_2602_01519_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), f
                assert "comb_oracle" not in src and "_work/" not in src, f


def _prefill_status(pool, Hq, lists, lq, lens, ws_bytes=None, mirror=True):
    """Plans a link on the host and calls comb_cross_attn_prefill with fake device pointers: without a GPU the call
    stops at its first CUDA call (COMB_ERR_CUDA), but only after planning and the capacity check."""
    R = len(lists)
    q_indptr = np.zeros(R + 1, np.int32)
    np.cumsum(lq, out=q_indptr[1:])
    link, tabs = plan(pool, lists, host_mirror=mirror)
    link.device_buf = 0x7300_0000_0000
    total_q = int(q_indptr[-1])
    bound_any = comb.comb_workspace_bytes(pool, R, Hq, total_q, int(link.max_pages_per_request))
    bound_link = comb.comb_attn_workspace_bytes(pool, link, Hq, total_q)
    assert bound_link >= bound_any > 0
    st = _lib.lib.comb_cross_attn_prefill(pool, 0, C.byref(link), R, 0x7400_0000_0000, q_indptr.ctypes.data, Hq,
                                          C.c_float(0.1), 0x7500_0000_0000, None, 0x7600_0000_0000,
                                          bound_any if ws_bytes is None else ws_bytes, None)
    return st, total_q


def test_workspace_bound_covers_every_prefill_plan():
    """comb_workspace_bytes() must suffice for whatever the prefill planner decides (KV ranges for sub-wave calls,
    last-wave ranges, one or two Q tiles per CTA): COMB_ERR_CAPACITY here means the bound is too small."""
    rng = np.random.default_rng(123)
    shapes = [(32, 8, 128, 128), (16, 16, 192, 128), (8, 2, 64, 64), (8, 8, 128, 64)]
    for trial in range(60):
        Hq, Hkv, Dqk, Dv = shapes[trial % len(shapes)]
        n_chunks = int(rng.integers(1, 40))
        lens = rng.integers(1, 1200, size=n_chunks)
        pages = int(((lens + 15) // 16).sum())
        pool = make_pool(num_pages=pages, Hkv=Hkv, Dqk=Dqk, Dv=Dv, seed=trial)
        for c in range(n_chunks):
            comb.comb_chunk_alloc(pool, c, int(lens[c]))
        R = int(rng.integers(1, 48))
        lists = [list(rng.choice(n_chunks, size=int(rng.integers(0, min(n_chunks, 12) + 1)), replace=False))
                 for _ in range(R)]
        lq = rng.choice([0, 1, 7, 32, 33, 64, 128, 129, 300, 512], size=R)
        st, total_q = _prefill_status(pool, Hq, lists, lq, lens)
        assert st != comb.COMB_ERR_CAPACITY, "trial %d: workspace bound too small" % trial
        assert st in (comb.COMB_OK, comb.COMB_ERR_CUDA)
        if total_q > 0:  # and the check is really reached: a 16-byte workspace is refused
            st, _ = _prefill_status(pool, Hq, lists, lq, lens, ws_bytes=16)
            assert st == comb.COMB_ERR_CAPACITY
        comb.comb_pool_destroy(pool)


@pytest.mark.parametrize("case", [(5, 256, 300), (20, 64, 300), (10, 128, 260), (5, 256, 500), (5, 256, 600),
                                  (37, 256, 300), (39, 128, 520)])
def test_workspace_bound_last_wave_ranges_short_requests(case):
    """Requests of 3-5 KV tiles whose item count leaves a last wave at most half full are cut in two by the planner;
    the bound used to reserve partial rows only from 4 tiles up (round-1 ADVICE). One planner now serves both."""
    R, lq, T = case
    pool = make_pool(num_pages=R * ((T + 15) // 16), Hkv=8, Dqk=128, Dv=128)
    for c in range(R):
        comb.comb_chunk_alloc(pool, c, T)
    st, _ = _prefill_status(pool, 32, [[r] for r in range(R)], [lq] * R, None)
    assert st in (comb.COMB_OK, comb.COMB_ERR_CUDA), st
    comb.comb_pool_destroy(pool)


def test_prefill_rejects_a_host_mirror_that_disagrees_with_the_link():
    pool = make_pool(num_pages=64, Hkv=2, Dqk=64, Dv=64)
    comb.comb_chunk_alloc(pool, 0, 400)
    comb.comb_chunk_alloc(pool, 1, 300)
    lists, lq = [[0, 1], [1]], [4, 4]
    link, tabs = plan(pool, lists)
    q_indptr = np.array([0, 4, 8], np.int32)
    mirror = link._keepalive[1]
    off = link.host_req_pages - mirror.ctypes.data
    mirror[off:off + 8].view(np.int32)[:] = [10, 10]  # stale counts (e.g. from another link)
    ws = comb.comb_attn_workspace_bytes(pool, link, 8, 8)
    st = _lib.lib.comb_cross_attn_prefill(pool, 0, C.byref(link), 2, 0x7400_0000_0000, q_indptr.ctypes.data, 8,
                                          C.c_float(0.1), 0x7500_0000_0000, None, 0x7600_0000_0000, ws, None)
    assert st == comb.COMB_ERR_INVALID
    comb.comb_pool_destroy(pool)


def test_options_and_decode_group_sizes():
    pool = make_pool(num_pages=64, Hkv=1, Dqk=64, Dv=128)
    comb.comb_pool_set_option(pool, comb.OPT_DECODE_PATH, comb.DECODE_CHUNK_MAJOR)
    comb.comb_pool_set_option(pool, comb.OPT_DECODE_PATH, comb.DECODE_AUTO)
    for bad in ((comb.OPT_DECODE_PATH, 7), (99, 0)):
        with pytest.raises(comb.CombError) as e:
            comb.comb_pool_set_option(pool, *bad)
        assert e.value.status == comb.COMB_ERR_INVALID
    comb.comb_chunk_alloc(pool, 0, 40)
    link, _ = plan(pool, [[0]])
    # every group size prefill takes is taken by decode too (G = 8, 16 used to be INVALID); 3 and 32 are not
    for Hq, ok in ((1, True), (2, True), (4, True), (8, True), (16, True), (3, False), (32, False)):
        ws = comb.comb_attn_workspace_bytes(pool, link, Hq, 1)
        st = _lib.lib.comb_cross_attn_decode(pool, 0, C.byref(link), 1, 0x7400_0000_0000, Hq, C.c_float(0.1),
                                             0x7500_0000_0000, None, 0x7600_0000_0000, ws, None)
        assert (st != comb.COMB_ERR_INVALID) == ok, (Hq, st)
    # the prefill cluster option takes 0 / 1 only
    comb.comb_pool_set_option(pool, comb.OPT_PREFILL_CLUSTERS, 0)
    comb.comb_pool_set_option(pool, comb.OPT_PREFILL_CLUSTERS, 1)
    with pytest.raises(comb.CombError) as e:
        comb.comb_pool_set_option(pool, comb.OPT_PREFILL_CLUSTERS, 2)
    assert e.value.status == comb.COMB_ERR_INVALID
    # comb_cross_attn_decode_noalloc: the same argument checks, no workspace argument, a fixed 8 MiB array
    assert comb.comb_noalloc_scratch_bytes() == 8 << 20
    na = _lib.lib.comb_cross_attn_decode_noalloc
    q, o = 0x7400_0000_0000, 0x7500_0000_0000
    assert na(None, 0, C.byref(link), 1, q, 4, C.c_float(0.1), o, None, None) == comb.COMB_ERR_INVALID
    assert na(pool, 0, C.byref(link), 1, q, 3, C.c_float(0.1), o, None, None) == comb.COMB_ERR_INVALID      # Hq % Hkv, G
    assert na(pool, 0, C.byref(link), 1, q, 4, C.c_float(-1.0), o, None, None) == comb.COMB_ERR_INVALID    # scale
    assert na(pool, 1, C.byref(link), 1, q, 4, C.c_float(0.1), o, None, None) == comb.COMB_ERR_INVALID     # layer
    assert na(pool, 0, C.byref(link), 2, q, 4, C.c_float(0.1), o, None, None) == comb.COMB_ERR_INVALID     # R != link's
    assert na(pool, 0, C.byref(link), 1, None, 4, C.c_float(0.1), o, None, None) == comb.COMB_ERR_INVALID  # q
    comb.comb_pool_destroy(pool)


def test_pins_and_lru_eviction_match_oracle_model():
    """(f4) reference counts and LRU eviction: a random trace of alloc / link / pin / unpin / free on a small pool,
    the library against the oracle's independent restatement of the policy (page lists and eviction order bit-exact)."""
    rng = np.random.default_rng(7)
    pool, model = make_pool(40, seed=3), oracle.PoolModel(40, 3, evict_lru=True)
    comb.comb_pool_set_option(pool, comb.OPT_EVICT_LRU, 1)
    nxt, evicted_total = 0, 0
    for step in range(400):
        live = sorted(model.dir)
        op = rng.integers(0, 10)
        if op <= 3 or not live:                                   # a new chunk (may evict)
            T = int(rng.integers(1, 120))
            try:
                want = model.store(nxt, T)
            except MemoryError:
                with pytest.raises(comb.CombError) as e:
                    comb.comb_chunk_alloc(pool, nxt, T)
                assert e.value.status == comb.COMB_ERR_NO_SPACE
                assert comb.comb_pool_evicted(pool) == []
            else:
                comb.comb_chunk_alloc(pool, nxt, T)
                assert comb.comb_chunk_query(pool, nxt)[1].tolist() == want
                assert comb.comb_pool_evicted(pool) == model.evicted
                evicted_total += len(model.evicted)
            nxt += 1
        elif op <= 5:                                             # a link refreshes the use stamps (real comb_link
            lists = [list(rng.choice(live, size=int(rng.integers(1, min(4, len(live)) + 1)), replace=False))
                     for _ in range(2)]                           # needs CUDA; the stamps are host state: alloc of an
            for lst in lists:                                     # existing id stamps too, one tick per call)
                for c in lst:
                    comb.comb_chunk_alloc(pool, int(c), model.dir[int(c)][0])
                    model.store(int(c), model.dir[int(c)][0])
        elif op == 6:
            c = int(rng.choice(live))
            comb.comb_chunk_pin(pool, c)
            model.pin(c)
        elif op == 7:
            pinned = [c for c in live if model.pins.get(c, 0) > 0]
            if pinned:
                c = int(rng.choice(pinned))
                comb.comb_chunk_unpin(pool, c)
                model.unpin(c)
        else:
            c = int(rng.choice(live))
            if model.pins.get(c, 0) > 0:
                with pytest.raises(comb.CombError) as e:
                    comb.comb_chunk_free(pool, c)
                assert e.value.status == comb.COMB_ERR_BUSY
            else:
                comb.comb_chunk_free(pool, c)
                model.release(c)
        assert _lib.lib.comb_pool_free_pages(pool) == model.free_pages()
    assert evicted_total > 10 and comb.comb_pool_eviction_count(pool) == evicted_total
    for c in sorted(model.dir):
        assert comb.comb_chunk_query(pool, c)[1].tolist() == model.dir[c][1]
    with pytest.raises(comb.CombError) as e:
        comb.comb_chunk_unpin(pool, sorted(c for c in model.dir if model.pins.get(c, 0) == 0)[0])
    assert e.value.status == comb.COMB_ERR_INVALID
    comb.comb_pool_destroy(pool)


def test_eviction_is_off_by_default_and_all_or_nothing():
    pool = make_pool(4)
    comb.comb_chunk_alloc(pool, 1, 33)
    with pytest.raises(comb.CombError) as e:
        comb.comb_chunk_alloc(pool, 2, 17)
    assert e.value.status == comb.COMB_ERR_NO_SPACE and comb.comb_pool_eviction_count(pool) == 0
    comb.comb_pool_set_option(pool, comb.OPT_EVICT_LRU, 1)
    comb.comb_chunk_pin(pool, 1)
    with pytest.raises(comb.CombError) as e:                        # the only candidate is pinned
        comb.comb_chunk_alloc(pool, 2, 17)
    assert e.value.status == comb.COMB_ERR_NO_SPACE and comb.comb_chunk_query(pool, 1)[0] == 33
    comb.comb_chunk_unpin(pool, 1)
    comb.comb_chunk_alloc(pool, 2, 17)
    assert comb.comb_pool_evicted(pool) == [1]
    with pytest.raises(comb.CombError) as e:
        comb.comb_chunk_query(pool, 1)
    assert e.value.status == comb.COMB_ERR_UNKNOWN_CHUNK
    comb.comb_pool_destroy(pool)


def parse_export(blob: bytes):
    """Independent reader of the export blob format documented in include/comb.h / comb_host.cu."""
    magic, version, flags = np.frombuffer(blob[:16], dtype=[("m", "<u8"), ("v", "<u4"), ("f", "<u4")])[0]
    geom = np.frombuffer(blob[16:40], dtype="<i4")
    n_chunks, dir_bytes = np.frombuffer(blob[264:280], dtype="<u8")
    HEAD = 280 + 8 + 16 + 128    # + kv_dtype, pad, two scale-table offsets and handles (fp8 pools)
    at, chunks = HEAD, []
    for _ in range(int(n_chunks)):
        cid = int(np.frombuffer(blob[at:at + 8], "<u8")[0])
        T, npg = (int(x) for x in np.frombuffer(blob[at + 8:at + 16], "<i4"))
        pages = np.frombuffer(blob[at + 16:at + 16 + 4 * npg], "<i4").copy()
        at += 16 + (4 * npg + 7) // 8 * 8
        chunks.append((cid, T, pages))
    assert at == HEAD + int(dir_bytes) == len(blob)
    return {"magic": int(magic), "version": int(version), "flags": int(flags), "geom": geom, "chunks": chunks}


def test_directory_export_matches_oracle_model_and_rejects_bad_blobs():
    """(f4) the host half of the CUDA-IPC export: the blob carries the geometry and every chunk's id, length and page
    list in creation order, equal to the oracle's independent PoolModel after a trace of stores and frees."""
    pool = make_pool(num_pages=40, Hkv=2, Dqk=64, Dv=128, seed=9, layers=3)
    model = oracle.PoolModel(40, shuffle_seed=9)
    rng = np.random.default_rng(3)
    live = []
    for step in range(60):
        if live and rng.random() < 0.35:
            cid = live.pop(int(rng.integers(len(live))))
            comb.comb_chunk_free(pool, cid)
            model.release(cid)
        else:
            cid, T = 1000 + step, int(rng.integers(1, 70))
            if model.free_pages() < (T + 15) // 16:
                continue
            comb.comb_chunk_alloc(pool, cid, T)
            model.store(cid, T)
            live.append(cid)
    blob = comb.comb_pool_export(pool, directory_only=True).tobytes()
    ex = parse_export(blob)
    assert ex["magic"] == int.from_bytes(b"COMBIPC1", "little") and ex["version"] == 1 and ex["flags"] == 0
    assert list(ex["geom"]) == [3, 2, 64, 128, 16, 40]
    assert [c[0] for c in ex["chunks"]] == sorted(live, key=lambda c: c)  # ids grow with creation order in this trace
    for cid, T, pages in ex["chunks"]:
        assert (T, list(pages)) == (model.dir[cid][0], list(model.dir[cid][1]))
    # a directory-only blob cannot open arenas; malformed blobs are INVALID; nothing here needs a GPU
    aligned = np.zeros((len(blob) + 7) // 8, np.uint64).view(np.uint8)
    aligned[:len(blob)] = np.frombuffer(blob, np.uint8)
    out = C.c_void_p()
    assert _lib.lib.comb_pool_import(aligned.ctypes.data, len(blob), None, C.byref(out)) == comb.COMB_ERR_INVALID
    assert _lib.lib.comb_pool_import(aligned.ctypes.data, 100, None, C.byref(out)) == comb.COMB_ERR_INVALID
    bad = aligned.copy()
    bad[0] ^= 0xff
    assert _lib.lib.comb_pool_import(bad.ctypes.data, len(blob), None, C.byref(out)) == comb.COMB_ERR_INVALID
    n = C.c_size_t()
    assert _lib.lib.comb_pool_export(pool, 1, None, aligned.ctypes.data, 64, C.byref(n)) == comb.COMB_ERR_CAPACITY
    assert _lib.lib.comb_pool_export(pool, 2, None, aligned.ctypes.data, len(blob), C.byref(n)) == comb.COMB_ERR_INVALID
    assert _lib.lib.comb_pool_refresh(pool, aligned.ctypes.data, len(blob), None) == comb.COMB_ERR_INVALID  # not imported
    comb.comb_pool_destroy(pool)


def test_fp8_pool_config_sizes_and_compact_page_table():
    """(f4) fp8 pools on the host: one byte per element + fp32 scale tables; only 128/128 head dims; comb_link_plan
    writes the compact page table (entry i of page_ids as an index into the batch's distinct-page list)."""
    kb, vb, _ = comb.comb_pool_bytes(3, 8, 128, 128, 100, kv_dtype=comb.KV_E4M3)
    kb16, vb16, _ = comb.comb_pool_bytes(3, 8, 128, 128, 100)
    assert (kb, vb) == (kb16 // 2, vb16 // 2) == (3 * 100 * 8 * 16 * 128,) * 2
    assert comb.comb_pool_scale_bytes(3, 8, 128, 128, 100) == 3 * 100 * 8 * 4
    assert comb.comb_pool_scale_bytes(3, 8, 128, 128, 100, kv_dtype=comb.KV_BF16) == 0
    for bad in (dict(Dqk=64, Dv=64), dict(Dqk=192, Dv=128), dict(Dqk=128, Dv=64)):
        cfg = comb.PoolConfig(1, 2, bad["Dqk"], bad["Dv"], 16, 8, FAKE_K, FAKE_V, FAKE_S, 0, comb.KV_E4M3, 0, FAKE_S, FAKE_S)
        out = C.c_void_p()
        assert _lib.lib.comb_pool_create(C.byref(cfg), C.byref(out)) == comb.COMB_ERR_INVALID
    for cfg in (comb.PoolConfig(1, 2, 128, 128, 16, 8, FAKE_K, FAKE_V, FAKE_S, 0, comb.KV_E4M3, 0, None, None),   # no scales
                comb.PoolConfig(1, 2, 128, 128, 16, 8, FAKE_K, FAKE_V, FAKE_S, 0, 7, 0, FAKE_S, FAKE_S),           # dtype
                comb.PoolConfig(1, 2, 128, 128, 16, 8, FAKE_K, FAKE_V, FAKE_S, 0, comb.KV_E4M3, 1, FAKE_S, FAKE_S)):
        out = C.c_void_p()
        assert _lib.lib.comb_pool_create(C.byref(cfg), C.byref(out)) == comb.COMB_ERR_INVALID
    cfg = comb.PoolConfig(1, 2, 128, 128, 16, 64, FAKE_K, FAKE_V, FAKE_S, 5, comb.KV_E4M3, 0, FAKE_S, FAKE_S + 4096)
    pool = comb.comb_pool_create(cfg)
    for c, T in enumerate([40, 16, 100, 5]):
        comb.comb_chunk_alloc(pool, c, T)
    lists = [[2, 0], [], [3, 2, 2, 1]]
    link, tabs = plan(pool, lists)
    assert link.page_ids_compact
    off = link.page_ids_compact - 0x10000
    host = link._keepalive[0]
    compact = host[off:off + 4 * int(link.total_pages)].view(np.int32)
    assert np.array_equal(tabs["cas_page_ids"][compact], tabs["page_ids"])
    assert compact.min() >= 0 and compact.max() < int(link.distinct_pages)
    # a bf16 pool writes no such table
    pool16 = make_pool(num_pages=64, Hkv=2, Dqk=128, Dv=128)
    for c, T in enumerate([40, 16, 100, 5]):
        comb.comb_chunk_alloc(pool16, c, T)
    link16, _ = plan(pool16, lists)
    assert not link16.page_ids_compact
    comb.comb_pool_destroy(pool)
    comb.comb_pool_destroy(pool16)
