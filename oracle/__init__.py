"""ORACLE — test infrastructure, not the product.

A plain, slow, obviously correct CPU statement of what the COMB link-stage path computes, written from
the paper (PAPER.md = /root/reference/PAPER.md at authoring time; the GPU box never reads it):

  O1  attention output  — ``comb_oracle.c`` (fp64, explicit concatenation in link order, one joint
      softmax, no mask: §4.2 Eq. 7-8)
  O2  page image        — :func:`page_image` (numpy, bit-exact uint16)
  O3  block tables      — :class:`PoolModel` (independent re-statement of the FIFO page policy; request-major
      tables and the chunk-major inversion of the same batch)

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It shares no code with ``paper_2602_01519_b200`` and neither imports the
other; inputs come from ``comb_synth`` (data only) and are passed in as arrays.

Pins are in tests/test_oracle_pins.py (brute force, library special case, closed forms, invariants);
no function here is "parity unpinned".
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Dict, Iterable, List, Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "comb_oracle.c")
_LIB = os.path.join(_HERE, "libcomb_oracle.so")
PAGE = 16


def build(force: bool = False) -> str:
    """Compile comb_oracle.c with gcc -O2 (no fast-math) + OpenMP.  Building the checker is not using it."""
    if force or (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fPIC", "-shared", "-fopenmp", "-std=c11", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True, capture_output=True)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        P = ctypes.c_void_p
        lib.comb_oracle_attention.restype = ctypes.c_int
        lib.comb_oracle_attention.argtypes = [ctypes.c_int, P, P, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                              ctypes.c_int, P, P, P, P, P, ctypes.c_double, P, P, ctypes.c_int]
        lib.comb_oracle_attention_samples.restype = ctypes.c_int
        lib.comb_oracle_attention_samples.argtypes = [ctypes.c_int, P, P, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                                      ctypes.c_int, P, P, P, P, P, ctypes.c_double, ctypes.c_int,
                                                      P, P, P, P]
        lib.comb_oracle_max_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def max_threads() -> int:
    return int(_load().comb_oracle_max_threads())


def _ptr(a: np.ndarray):
    return ctypes.c_void_p(a.ctypes.data)


def _chunk_ptr_arrays(k_chunks: Sequence[np.ndarray], v_chunks: Sequence[np.ndarray]):
    n = len(k_chunks)
    ks = [np.ascontiguousarray(k, dtype=np.uint16) for k in k_chunks]
    vs = [np.ascontiguousarray(v, dtype=np.uint16) for v in v_chunks]
    kp = (ctypes.c_void_p * max(n, 1))(*[k.ctypes.data for k in ks])
    vp = (ctypes.c_void_p * max(n, 1))(*[v.ctypes.data for v in vs])
    lens = np.array([k.shape[0] for k in ks], dtype=np.int32) if n else np.zeros(1, dtype=np.int32)
    return ks, vs, kp, vp, lens


def attention(q: np.ndarray, q_indptr: np.ndarray, k_chunks: Sequence[np.ndarray], v_chunks: Sequence[np.ndarray],
              chunk_indptr: np.ndarray, chunk_sel: np.ndarray, scale: float,
              num_threads: int = 0) -> Tuple[np.ndarray, np.ndarray]:
    """O1.  ``q`` bf16 bits [sum lq][Hq][Dqk]; ``k_chunks[c]`` bf16 bits [T_c][Hkv][Dqk]; ``chunk_sel`` holds,
    for request r at positions chunk_indptr[r]:chunk_indptr[r+1], indices into ``k_chunks`` in LINK ORDER.
    Returns (O fp64 [sum lq][Hq][Dv], LSE fp64 [sum lq][Hq])."""
    lib = _load()
    q = np.ascontiguousarray(q, dtype=np.uint16)
    q_indptr = np.ascontiguousarray(q_indptr, dtype=np.int32)
    chunk_indptr = np.ascontiguousarray(chunk_indptr, dtype=np.int32)
    chunk_sel = np.ascontiguousarray(chunk_sel, dtype=np.int32)
    if chunk_sel.size == 0:
        chunk_sel = np.zeros(1, dtype=np.int32)
    R = q_indptr.shape[0] - 1
    Hq, Dqk = int(q.shape[1]), int(q.shape[2])
    ks, vs, kp, vp, lens = _chunk_ptr_arrays(k_chunks, v_chunks)
    if ks:
        Hkv, Dv = int(ks[0].shape[1]), int(vs[0].shape[2])
    else:  # no chunks anywhere: shapes only matter for the output
        Hkv, Dv = Hq, Dqk
    out = np.zeros((q.shape[0], Hq, Dv), dtype=np.float64)
    lse = np.zeros((q.shape[0], Hq), dtype=np.float64)
    rc = lib.comb_oracle_attention(R, _ptr(q_indptr), _ptr(q) if q.size else None, Hq, Hkv, Dqk, Dv,
                                   _ptr(chunk_indptr), _ptr(chunk_sel), kp, vp, _ptr(lens), float(scale),
                                   _ptr(out) if out.size else None, _ptr(lse) if lse.size else None,
                                   int(num_threads))
    if rc != 0:
        raise MemoryError("comb_oracle_attention failed (rc=%d)" % rc)
    return out, lse


def attention_samples(r: int, q: np.ndarray, q_indptr: np.ndarray, k_chunks, v_chunks, chunk_indptr, chunk_sel,
                      scale: float, rows: np.ndarray, heads: np.ndarray) -> Tuple[np.ndarray, np.ndarray]:
    """O1 evaluated only at (rows[n], heads[n]) of request ``r`` — for full-size configs."""
    lib = _load()
    q = np.ascontiguousarray(q, dtype=np.uint16)
    q_indptr = np.ascontiguousarray(q_indptr, dtype=np.int32)
    chunk_indptr = np.ascontiguousarray(chunk_indptr, dtype=np.int32)
    chunk_sel = np.ascontiguousarray(chunk_sel, dtype=np.int32)
    rows = np.ascontiguousarray(rows, dtype=np.int32)
    heads = np.ascontiguousarray(heads, dtype=np.int32)
    Hq, Dqk = int(q.shape[1]), int(q.shape[2])
    ks, vs, kp, vp, lens = _chunk_ptr_arrays(k_chunks, v_chunks)
    Hkv, Dv = int(ks[0].shape[1]), int(vs[0].shape[2])
    n = rows.shape[0]
    out = np.zeros((n, Dv), dtype=np.float64)
    lse = np.zeros((n,), dtype=np.float64)
    rc = lib.comb_oracle_attention_samples(int(r), _ptr(q_indptr), _ptr(q), Hq, Hkv, Dqk, Dv, _ptr(chunk_indptr),
                                           _ptr(chunk_sel), kp, vp, _ptr(lens), float(scale), n, _ptr(rows),
                                           _ptr(heads), _ptr(out), _ptr(lse))
    if rc != 0:
        raise RuntimeError("comb_oracle_attention_samples failed (rc=%d)" % rc)
    return out, lse


def attention_for(w, requests: Optional[Iterable[int]] = None, num_threads: int = 0):
    """O1 for a ``comb_synth.Workload``-like object (duck-typed: ``links``, ``chunk_kv``, ``request_q``,
    ``lq``, ``scale``).  Materialises only the chunks the selected requests link.  Returns (O, LSE) for the
    selected requests' rows, concatenated in request order."""
    reqs = list(range(len(w.links))) if requests is None else list(requests)
    used: Dict[int, int] = {}
    ks: List[np.ndarray] = []
    vs: List[np.ndarray] = []
    sel: List[int] = []
    indptr = [0]
    for r in reqs:
        for c in w.links[r]:
            c = int(c)
            if c not in used:
                used[c] = len(ks)
                k, v = w.chunk_kv(c)
                ks.append(k)
                vs.append(v)
            sel.append(used[c])
        indptr.append(len(sel))
    qs = [w.request_q(r) for r in reqs]
    q = np.concatenate(qs, axis=0) if qs else np.zeros((0, w.num_q_heads, w.head_dim_qk), np.uint16)
    q_indptr = np.zeros(len(reqs) + 1, dtype=np.int32)
    np.cumsum([x.shape[0] for x in qs], out=q_indptr[1:])
    if not ks:  # every selected request has an empty link: still need head shapes for the output
        out = np.zeros((q.shape[0], w.num_q_heads, w.head_dim_v), dtype=np.float64)
        lse = np.full((q.shape[0], w.num_q_heads), -np.inf, dtype=np.float64)
        return out, lse
    return attention(q, q_indptr, ks, vs, np.array(indptr, np.int32), np.array(sel, np.int32), w.scale,
                     num_threads)


# ------------------------------------------------------------------------------------------------
# O3 — block tables: independent re-statement of the allocation policy (include/comb.h)
# ------------------------------------------------------------------------------------------------
_M64 = (1 << 64) - 1


def _splitmix64_stream(seed: int):
    state = seed & _M64
    while True:
        state = (state + 0x9E3779B97F4A7C15) & _M64
        z = state
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _M64
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _M64
        yield z ^ (z >> 31)


def initial_free_list(num_pages: int, shuffle_seed: int) -> List[int]:
    """seed 0: ascending ids.  Otherwise Fisher-Yates (i = n-1 .. 1, j = next() mod (i+1), swap) driven by
    splitmix64(seed) — the counter-based generator both sides implement (comb.h, free_list_shuffle_seed)."""
    a = list(range(num_pages))
    if shuffle_seed:
        g = _splitmix64_stream(shuffle_seed)
        for i in range(num_pages - 1, 0, -1):
            j = next(g) % (i + 1)
            a[i], a[j] = a[j], a[i]
    return a


class PoolModel:
    """FIFO free list: a chunk of T tokens takes ceil(T/16) ids from the head, in order; freeing a chunk
    appends its ids to the tail in page-list order ("PIC allocator ... allocate free memory";
    PAPER.md:62 steps 1-4 hash table context -> PICache)."""

    def __init__(self, num_pages: int, shuffle_seed: int = 0, evict_lru: bool = False):
        self.free = initial_free_list(num_pages, shuffle_seed)
        self.head = 0
        self.dir: Dict[int, Tuple[int, List[int]]] = {}
        # lifecycle (include/comb.h "(f4) pool lifecycle"): pins, use stamps, LRU eviction
        self.evict_lru = evict_lru
        self.pins: Dict[int, int] = {}
        self.stamp: Dict[int, int] = {}    # chunk -> tick of its last alloc / store / link
        self.born: Dict[int, int] = {}     # chunk -> creation order
        self.tick = 0
        self.births = 0
        self.evicted: List[int] = []       # by the most recent store call

    def free_pages(self) -> int:
        return len(self.free) - self.head

    def _make_room(self, need: int, keep: Sequence[int]) -> bool:
        """Evict unpinned chunks outside `keep` in ascending (use stamp, creation order) until `need` pages are
        free; all or nothing."""
        if self.free_pages() >= need:
            return True
        if not self.evict_lru:
            return False
        cands = sorted((c for c in self.dir if self.pins.get(c, 0) == 0 and c not in keep),
                       key=lambda c: (self.stamp[c], self.born[c]))
        have, take = self.free_pages(), []
        for c in cands:
            if have >= need:
                break
            take.append(c)
            have += len(self.dir[c][1])
        if have < need:
            return False
        for c in take:
            self.release(c)
            self.evicted.append(c)
        return True

    def store(self, chunk_id: int, num_tokens: int) -> List[int]:
        return self.store_batch([(chunk_id, num_tokens)])[0]

    def store_batch(self, items: Sequence[Tuple[int, int]]) -> List[List[int]]:
        """One alloc/store call naming several chunks: validated as a whole, room made for the whole batch (the
        batch's own ids are never evicted), then pages taken from the head in batch order."""
        self.evicted = []
        need = 0
        for cid, T in items:
            if cid in self.dir:
                if self.dir[cid][0] != T:
                    raise KeyError("exists with different length")
            else:
                need += (T + PAGE - 1) // PAGE
        if not self._make_room(need, [c for c, _ in items]):
            raise MemoryError("no space")
        out = []
        for cid, T in items:
            self.tick += 1
            if cid not in self.dir:
                n = (T + PAGE - 1) // PAGE
                self.dir[cid] = (T, self.free[self.head:self.head + n])
                self.head += n
                self.born[cid] = self.births
                self.births += 1
            self.stamp[cid] = self.tick
            out.append(self.dir[cid][1])
        return out

    def pin(self, chunk_id: int) -> None:
        self.pins[chunk_id] = self.pins.get(chunk_id, 0) + 1

    def unpin(self, chunk_id: int) -> None:
        assert self.pins.get(chunk_id, 0) > 0
        self.pins[chunk_id] -= 1

    def touch(self, chunk_lists: Sequence[Sequence[int]]) -> None:
        """What a comb_link does to the use stamps: ONE fresh tick for all the chunks it names."""
        self.tick += 1
        for lst in chunk_lists:
            for c in lst:
                self.stamp[int(c)] = self.tick

    def release(self, chunk_id: int) -> None:
        if self.pins.get(chunk_id, 0) > 0:
            raise RuntimeError("pinned")
        _, pages = self.dir.pop(chunk_id)
        self.free.extend(pages)

    def link(self, chunk_lists: Sequence[Sequence[int]]) -> Dict[str, np.ndarray]:
        """page_ids[r] = pages(c_0) || ... || pages(c_{m-1}) in the caller's order ("in any
        order/position"); page_ntok = 16 except the last page of each chunk; kv_len = sum T."""
        indptr = [0]
        ids: List[int] = []
        ntok: List[int] = []
        kv: List[int] = []
        for lst in chunk_lists:
            tot = 0
            for c in lst:
                T, pages = self.dir[int(c)]
                ids.extend(pages)
                ntok.extend([PAGE] * (len(pages) - 1) + [T - PAGE * (len(pages) - 1)])
                tot += T
            indptr.append(len(ids))
            kv.append(tot)
        return {"page_indptr": np.array(indptr, dtype=np.int32), "page_ids": np.array(ids, dtype=np.int32),
                "page_ntok": np.array(ntok, dtype=np.int32), "kv_len": np.array(kv, dtype=np.int32)}

    def link_chunk_major(self, chunk_lists: Sequence[Sequence[int]]) -> Dict[str, np.ndarray]:
        """The same batch inverted (include/comb.h, "chunk-major view"): an entry is one (request, linked chunk)
        pair, numbered in link order; every DISTINCT chunk gets a slot, slots ordered by descending number of
        entries, ties by first appearance; a slot lists its pages once and the entries (request, entry number)
        that link it in ascending entry number.  Order-free concatenation is what makes the
        inversion legal; the tables themselves are integer bookkeeping with exactly one right answer."""
        entries = [(r, int(c)) for r, lst in enumerate(chunk_lists) for c in lst]
        first: Dict[int, int] = {}
        count: Dict[int, int] = {}
        for e, (_, c) in enumerate(entries):
            first.setdefault(c, e)
            count[c] = count.get(c, 0) + 1
        slots = sorted(count, key=lambda c: (-count[c], first[c]))
        page_indptr, page_ids, page_ntok, row_indptr, row_req, row_entry = [0], [], [], [0], [], []
        for c in slots:
            T, pages = self.dir[c]
            page_ids.extend(pages)
            page_ntok.extend([PAGE] * (len(pages) - 1) + [T - PAGE * (len(pages) - 1)])
            page_indptr.append(len(page_ids))
            for e, (r, cc) in enumerate(entries):
                if cc == c:
                    row_req.append(r)
                    row_entry.append(e)
            row_indptr.append(len(row_req))
        entry_indptr = np.zeros(len(chunk_lists) + 1, dtype=np.int32)
        np.cumsum([len(l) for l in chunk_lists], out=entry_indptr[1:])
        return {"entry_indptr": entry_indptr, "slot_chunks": np.array(slots, dtype=np.int64),
                "cas_page_indptr": np.array(page_indptr, dtype=np.int32),
                "cas_page_ids": np.array(page_ids, dtype=np.int32),
                "cas_page_ntok": np.array(page_ntok, dtype=np.int32),
                "cas_row_indptr": np.array(row_indptr, dtype=np.int32),
                "cas_row_req": np.array(row_req, dtype=np.int32),
                "cas_row_entry": np.array(row_entry, dtype=np.int32)}


# ------------------------------------------------------------------------------------------------
# O2 — page image (bit-exact)
# ------------------------------------------------------------------------------------------------
def page_image(num_pages: int, num_kv_heads: int, head_dim: int, stored: Sequence[Tuple[np.ndarray, Sequence[int]]],
               sentinel: int = 0x7FC0) -> np.ndarray:
    """Expected arena of ONE layer for K (or V): uint16 [num_pages][Hkv][16][D].
    ``stored`` = [(chunk tensor bf16 bits [T][Hkv][D], page list)] in store order.
    img[p][g][s][:] = chunk[16*i+s][g][:] for p = pages[i], 16*i+s < T; zero bits where 16*i+s >= T;
    pages owned by no chunk keep the sentinel the harness wrote before."""
    img = np.full((num_pages, num_kv_heads, PAGE, head_dim), sentinel, dtype=np.uint16)
    for x, pages in stored:
        T = x.shape[0]
        for i, p in enumerate(pages):
            n = min(PAGE, T - PAGE * i)
            img[p] = 0
            img[p, :, :n, :] = np.transpose(x[PAGE * i:PAGE * i + n], (1, 0, 2))
    return img
