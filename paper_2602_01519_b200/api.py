"""Python binding of the C ABI in include/comb.h — same names, argument marshalling only.

PyTorch is used here for device memory and streams (plumbing); every step of the path (store, link,
prefill and decode cross-attention: §3 steps 1-8, §4.2 Eq. 7-8) runs inside
libcomb.so.  ``Pool`` owns the torch allocations the library asks the caller to provide.
"""
from __future__ import annotations

import ctypes as C
from typing import Optional, Sequence, Tuple

import numpy as np
import torch

from . import _lib
from ._lib import CombError, Link, PoolConfig, check, lib

PAGE = 16


def _ptr(t) -> Optional[int]:
    if t is None:
        return None
    if isinstance(t, torch.Tensor):
        return t.data_ptr()
    if isinstance(t, np.ndarray):
        return t.ctypes.data
    return int(t)


def _stream_ptr(stream) -> Optional[int]:
    if stream is None:
        return torch.cuda.current_stream().cuda_stream if torch.cuda.is_available() else None
    if isinstance(stream, torch.cuda.Stream):
        return stream.cuda_stream
    return int(stream)


# ------------------------------------------------------------------------------------------------
# the C calls, one to one
# ------------------------------------------------------------------------------------------------
KV_BF16, KV_E4M3 = 0, 1


def comb_pool_bytes(num_layers: int, num_kv_heads: int, head_dim_qk: int, head_dim_v: int, num_pages: int,
                    page_size: int = PAGE, kv_dtype: int = KV_BF16) -> Tuple[int, int, int]:
    cfg = PoolConfig(num_layers, num_kv_heads, head_dim_qk, head_dim_v, page_size, num_pages, None, None, None, 0,
                     kv_dtype)
    k, v, s = C.c_size_t(), C.c_size_t(), C.c_size_t()
    check(lib.comb_pool_bytes(C.byref(cfg), C.byref(k), C.byref(v), C.byref(s)), "comb_pool_bytes")
    return k.value, v.value, s.value


def comb_pool_scale_bytes(num_layers: int, num_kv_heads: int, head_dim_qk: int, head_dim_v: int, num_pages: int,
                          kv_dtype: int = KV_E4M3) -> int:
    cfg = PoolConfig(num_layers, num_kv_heads, head_dim_qk, head_dim_v, PAGE, num_pages, None, None, None, 0, kv_dtype)
    return int(lib.comb_pool_scale_bytes(C.byref(cfg)))


def comb_pool_create(cfg: PoolConfig) -> int:
    out = C.c_void_p()
    check(lib.comb_pool_create(C.byref(cfg), C.byref(out)), "comb_pool_create")
    return out.value


def comb_pool_destroy(pool: int) -> None:
    check(lib.comb_pool_destroy(pool), "comb_pool_destroy")


def comb_chunk_alloc(pool: int, chunk_id: int, num_tokens: int) -> None:
    check(lib.comb_chunk_alloc(pool, chunk_id, num_tokens), "comb_chunk_alloc")


def comb_chunk_free(pool: int, chunk_id: int) -> None:
    check(lib.comb_chunk_free(pool, chunk_id), "comb_chunk_free")


def comb_chunk_pin(pool: int, chunk_id: int) -> None:
    check(lib.comb_chunk_pin(pool, chunk_id), "comb_chunk_pin")


def comb_chunk_unpin(pool: int, chunk_id: int) -> None:
    check(lib.comb_chunk_unpin(pool, chunk_id), "comb_chunk_unpin")


def comb_pool_evicted(pool: int) -> list:
    """Chunk ids evicted by the most recent alloc/store call, in eviction order."""
    n = check(lib.comb_pool_evicted(pool, None, 0), "comb_pool_evicted")
    ids = np.zeros(max(n, 1), dtype=np.uint64)
    check(lib.comb_pool_evicted(pool, ids.ctypes.data, n), "comb_pool_evicted")
    return [int(x) for x in ids[:n]]


def comb_pool_eviction_count(pool: int) -> int:
    return int(lib.comb_pool_eviction_count(pool))


EXPORT_DIRECTORY_ONLY = 1


def comb_pool_export(pool: int, directory_only: bool = False, stream=None) -> np.ndarray:
    """(f4) self-contained blob (uint8 array, 8-byte aligned) another process hands to comb_pool_import."""
    cap = int(lib.comb_pool_export_bytes(pool))
    blob = np.zeros((cap + 7) // 8, dtype=np.uint64).view(np.uint8)
    n = C.c_size_t()
    check(lib.comb_pool_export(pool, EXPORT_DIRECTORY_ONLY if directory_only else 0,
                               None if directory_only else _stream_ptr(stream), blob.ctypes.data, blob.nbytes,
                               C.byref(n)), "comb_pool_export")
    return blob[:n.value]


def _aligned_blob(blob) -> np.ndarray:
    raw = np.frombuffer(bytes(blob), dtype=np.uint8) if not isinstance(blob, np.ndarray) else blob
    out = np.zeros((raw.size + 7) // 8, dtype=np.uint64).view(np.uint8)
    out[:raw.size] = raw
    return out


def comb_pool_import(blob, stream=None) -> int:
    """Opens an exported pool read-only in this process (CUDA IPC); returns the pool handle."""
    b = _aligned_blob(blob)
    out = C.c_void_p()
    check(lib.comb_pool_import(b.ctypes.data, len(bytes(blob)) if not isinstance(blob, np.ndarray) else blob.size,
                               _stream_ptr(stream), C.byref(out)), "comb_pool_import")
    return out.value


def comb_pool_refresh(pool: int, blob, stream=None) -> None:
    b = _aligned_blob(blob)
    check(lib.comb_pool_refresh(pool, b.ctypes.data, len(bytes(blob)) if not isinstance(blob, np.ndarray) else blob.size,
                                _stream_ptr(stream)), "comb_pool_refresh")


def comb_chunk_query(pool: int, chunk_id: int) -> Tuple[int, np.ndarray]:
    """(num_tokens, page ids) of a stored chunk."""
    nt = C.c_int32()
    n = check(lib.comb_chunk_query(pool, chunk_id, C.byref(nt), None, 0), "comb_chunk_query")
    pages = np.zeros(max(n, 1), dtype=np.int32)
    check(lib.comb_chunk_query(pool, chunk_id, C.byref(nt), pages.ctypes.data, n), "comb_chunk_query")
    return nt.value, pages[:n]


def comb_store_chunk(pool: int, layer: int, chunk_id: int, num_tokens: int, k, v, stream=None) -> None:
    check(lib.comb_store_chunk(pool, layer, chunk_id, num_tokens, _ptr(k), _ptr(v), _stream_ptr(stream)),
          "comb_store_chunk")


def comb_store_chunks(pool: int, layer: int, chunk_ids: Sequence[int], tok_indptr, k_packed, v_packed,
                      stream=None) -> None:
    ids = np.ascontiguousarray(chunk_ids, dtype=np.uint64)
    ind = np.ascontiguousarray(tok_indptr, dtype=np.int32)
    check(lib.comb_store_chunks(pool, layer, int(ids.shape[0]), ids.ctypes.data, ind.ctypes.data, _ptr(k_packed),
                                _ptr(v_packed), _stream_ptr(stream)), "comb_store_chunks")


def comb_project_store_chunks(pool: int, layer: int, chunk_ids: Sequence[int], tok_indptr, h_packed, d_model: int,
                              w_kv, stream=None) -> None:
    ids = np.ascontiguousarray(chunk_ids, dtype=np.uint64)
    ind = np.ascontiguousarray(tok_indptr, dtype=np.int32)
    check(lib.comb_project_store_chunks(pool, layer, int(ids.shape[0]), ids.ctypes.data, ind.ctypes.data,
                                        _ptr(h_packed), int(d_model), _ptr(w_kv), _stream_ptr(stream)),
          "comb_project_store_chunks")


def comb_gemm_bf16(pool: int, a, w, c, M: int, N: int, K: int, residual=None, stream=None) -> None:
    check(lib.comb_gemm_bf16(pool, _ptr(a), _ptr(w), _ptr(residual), _ptr(c), int(M), int(N), int(K),
                             _stream_ptr(stream)), "comb_gemm_bf16")


def comb_layer_workspace_bytes(pool: int, link: Link, num_q_heads: int, rows: int) -> int:
    return int(lib.comb_layer_workspace_bytes(pool, C.byref(link), num_q_heads, rows))


def comb_cross_layer_forward(pool: int, layer: int, link: Link, num_requests: int, x, q_indptr, d_model: int,
                             num_q_heads: int, w_q, w_o, scale: float, x_out, workspace, workspace_bytes: int,
                             stream=None) -> None:
    ind = None if q_indptr is None else np.ascontiguousarray(q_indptr, dtype=np.int32)
    check(lib.comb_cross_layer_forward(pool, layer, C.byref(link), num_requests, _ptr(x),
                                       None if ind is None else ind.ctypes.data, int(d_model), num_q_heads, _ptr(w_q),
                                       _ptr(w_o), float(scale), _ptr(x_out), _ptr(workspace), int(workspace_bytes),
                                       _stream_ptr(stream)), "comb_cross_layer_forward")


def comb_link_bytes(num_requests: int, total_entries: int, total_pages: int) -> int:
    return int(lib.comb_link_bytes(num_requests, total_entries, total_pages))


def comb_link_host_bytes(num_requests: int, total_entries: int) -> int:
    return int(lib.comb_link_host_bytes(num_requests, total_entries))


def comb_link(pool: int, chunk_indptr, chunk_ids, link: Link, stream=None) -> Link:
    ind = np.ascontiguousarray(chunk_indptr, dtype=np.int32)
    ids = np.ascontiguousarray(chunk_ids, dtype=np.uint64)
    check(lib.comb_link(pool, int(ind.shape[0]) - 1, ind.ctypes.data, ids.ctypes.data if ids.size else None,
                        C.byref(link), _stream_ptr(stream)), "comb_link")
    return link


def comb_link_plan(pool: int, chunk_indptr, chunk_ids, link: Link, host_buf: np.ndarray) -> Link:
    """Host-only table build (no CUDA call); ``host_buf`` is the staging area, a uint8 array of link.device_bytes
    bytes, laid out as device_buf would be."""
    ind = np.ascontiguousarray(chunk_indptr, dtype=np.int32)
    ids = np.ascontiguousarray(chunk_ids, dtype=np.uint64)
    check(lib.comb_link_plan(pool, int(ind.shape[0]) - 1, ind.ctypes.data, ids.ctypes.data if ids.size else None,
                             C.byref(link), host_buf.ctypes.data), "comb_link_plan")
    return link


def comb_workspace_bytes(pool: int, num_requests: int, num_q_heads: int, total_q: int, max_pages: int) -> int:
    return int(lib.comb_workspace_bytes(pool, num_requests, num_q_heads, total_q, max_pages))


def comb_attn_workspace_bytes(pool: int, link: Link, num_q_heads: int, total_q: int) -> int:
    return int(lib.comb_attn_workspace_bytes(pool, C.byref(link), num_q_heads, total_q))


OPT_DECODE_PATH = 1
OPT_EVICT_LRU = 2
OPT_PREFILL_CLUSTERS = 3
DECODE_AUTO, DECODE_PER_REQUEST, DECODE_CHUNK_MAJOR = 0, 1, 2


def comb_pool_set_option(pool: int, option: int, value: int) -> None:
    check(lib.comb_pool_set_option(pool, option, value), "comb_pool_set_option")


def comb_cross_attn_prefill(pool: int, layer: int, link: Link, q, q_indptr, num_q_heads: int, scale: float, out,
                            lse=None, workspace=None, workspace_bytes: int = 0, stream=None) -> None:
    ind = np.ascontiguousarray(q_indptr, dtype=np.int32)
    check(lib.comb_cross_attn_prefill(pool, layer, C.byref(link), int(ind.shape[0]) - 1, _ptr(q), ind.ctypes.data,
                                      num_q_heads, float(scale), _ptr(out), _ptr(lse), _ptr(workspace),
                                      int(workspace_bytes), _stream_ptr(stream)), "comb_cross_attn_prefill")


def comb_cross_attn_decode(pool: int, layer: int, link: Link, num_requests: int, q, num_q_heads: int, scale: float,
                           out, lse=None, workspace=None, workspace_bytes: int = 0, stream=None) -> None:
    check(lib.comb_cross_attn_decode(pool, layer, C.byref(link), num_requests, _ptr(q), num_q_heads, float(scale),
                                     _ptr(out), _ptr(lse), _ptr(workspace), int(workspace_bytes),
                                     _stream_ptr(stream)), "comb_cross_attn_decode")


def comb_cross_attn_decode_noalloc(pool: int, layer: int, link: Link, num_requests: int, q, num_q_heads: int,
                                   scale: float, out, lse=None, stream=None) -> None:
    check(lib.comb_cross_attn_decode_noalloc(pool, layer, C.byref(link), num_requests, _ptr(q), num_q_heads,
                                             float(scale), _ptr(out), _ptr(lse), _stream_ptr(stream)),
          "comb_cross_attn_decode_noalloc")


def comb_noalloc_scratch_bytes() -> int:
    return int(lib.comb_noalloc_scratch_bytes())


def comb_pool_launch_count(pool: int) -> int:
    return int(lib.comb_pool_launch_count(pool))


KERNEL_STORE, KERNEL_DECODE_SPLIT, KERNEL_DECODE_MERGE, KERNEL_PREFILL = 0, 1, 2, 3
KERNEL_DECODE_CASCADE, KERNEL_CASCADE_MERGE, KERNEL_PREFILL_MERGE, KERNEL_GEMM = 4, 5, 6, 7


def comb_profile_enable(pool: int, on: bool) -> None:
    check(lib.comb_profile_enable(pool, 1 if on else 0), "comb_profile_enable")


def comb_profile_read(pool: int, kernel: int) -> Tuple[float, int]:
    """(total device ms, launches) of one kernel class since the last read; waits for those launches."""
    ms, n = C.c_double(), C.c_int64()
    check(lib.comb_profile_read(pool, kernel, C.byref(ms), C.byref(n)), "comb_profile_read")
    return ms.value, n.value


def comb_profile_read_samples(pool: int, kernel: int, cap: int = 4096) -> np.ndarray:
    """Per-launch device ms of one kernel class since the last read (oldest first); waits for those launches."""
    buf = np.zeros(cap, np.float32)
    n = C.c_int64()
    check(lib.comb_profile_read_samples(pool, kernel, buf.ctypes.data, cap, C.byref(n)), "comb_profile_read_samples")
    return buf[:min(int(n.value), cap)].copy()


def comb_util_stream_read(src: torch.Tensor, sink: torch.Tensor, stream=None) -> None:
    check(lib.comb_util_stream_read(src.data_ptr(), src.numel() * src.element_size(), sink.data_ptr(),
                                    _stream_ptr(stream)), "comb_util_stream_read")


def comb_version() -> str:
    return lib.comb_version().decode()


# ------------------------------------------------------------------------------------------------
# convenience owner of the caller-side allocations (torch = memory + streams only)
# ------------------------------------------------------------------------------------------------
class LinkedBatch:
    """A comb_link_t plus the torch buffer (device tables) and the numpy buffer (host mirror) that back it."""

    def __init__(self, link: Link, buf: torch.Tensor, host: Optional[np.ndarray] = None):
        self.link, self.buf, self.host = link, buf, host

    def _view(self, ptr: int, n: int, dtype: torch.dtype) -> torch.Tensor:
        off = ptr - self.buf.data_ptr()
        return self.buf[off:off + n * torch.empty((), dtype=dtype).element_size()].view(dtype)

    @property
    def num_requests(self) -> int:
        return self.link.num_requests

    def tables(self) -> dict:
        """Device tables copied to host numpy arrays (synchronises)."""
        L = self.link
        R, n, t = L.num_requests, int(L.total_pages), int(L.total_tiles)
        U, E, pd = int(L.num_distinct_chunks), int(L.total_entries), int(L.distinct_pages)
        i32 = lambda ptr, cnt: self._view(ptr, cnt, torch.int32).cpu().numpy()  # noqa: E731
        u8 = lambda ptr, cnt: self._view(ptr, cnt, torch.uint8).cpu().numpy()  # noqa: E731
        out = {
            "page_indptr": i32(L.page_indptr, R + 1), "page_ids": i32(L.page_ids, n),
            "page_ntok": u8(L.page_ntok, n), "kv_len": i32(L.kv_len, R),
            "tile_indptr": i32(L.tile_indptr, R + 1),
            "tile_ntok": self._view(L.tile_ntok, t, torch.int64).cpu().numpy().view(np.uint64),
            "entry_indptr": i32(L.entry_indptr, R + 1),
            "cas_page_indptr": i32(L.cas_page_indptr, U + 1), "cas_page_ids": i32(L.cas_page_ids, pd),
            "cas_tile_indptr": i32(L.cas_tile_indptr, U + 1), "cas_row_indptr": i32(L.cas_row_indptr, U + 1),
            "cas_row_req": i32(L.cas_row_req, E), "cas_row_entry": i32(L.cas_row_entry, E),
        }
        tc = int(out["cas_tile_indptr"][-1]) if U else 0
        out["cas_tile_ntok"] = self._view(L.cas_tile_ntok, tc, torch.int64).cpu().numpy().view(np.uint64)
        return out

    def host_mirror(self) -> dict:
        """The host arrays the attention planners read (None without a host buffer)."""
        L = self.link
        if not L.host_req_pages:
            return {"req_pages": None, "cas_rows": None, "cas_pages": None}
        base = self.host.ctypes.data
        o1, o2, o3 = L.host_req_pages - base, L.host_cas_rows - base, L.host_cas_pages - base
        U = int(L.num_distinct_chunks)
        return {"req_pages": self.host[o1:o1 + 4 * L.num_requests].view(np.int32),
                "cas_rows": self.host[o2:o2 + 4 * U].view(np.int32),
                "cas_pages": self.host[o3:o3 + 4 * U].view(np.int32)}


class Pool:
    """Chunk-KV pool (a1): allocates the arenas with torch and forwards every call to libcomb.so."""

    def __init__(self, num_kv_heads: int, head_dim_qk: int, head_dim_v: int, num_pages: int, num_layers: int = 1,
                 shuffle_seed: int = 0, device: str = "cuda", sentinel: Optional[int] = None, kv_dtype: int = KV_BF16):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2602_01519_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
        self.device = torch.device(device)
        self.num_layers, self.num_kv_heads = num_layers, num_kv_heads
        self.head_dim_qk, self.head_dim_v, self.num_pages = head_dim_qk, head_dim_v, num_pages
        self.kv_dtype = kv_dtype
        kb, vb, sb = comb_pool_bytes(num_layers, num_kv_heads, head_dim_qk, head_dim_v, num_pages, kv_dtype=kv_dtype)
        # arenas as int16 bit patterns [L][pages][Hkv][16][D]; optional sentinel (e.g. 0x7FC0 = bf16 NaN) for tests.
        # fp8 pools: the same layout with one byte per element (viewed as uint8 through k_codes / v_codes) plus fp32
        # scale tables [L][pages][Hkv]; their sentinel fills every byte with its low 8 bits and the scales with -7.
        self.k_arena = self._aligned_i16(kb)
        self.v_arena = self._aligned_i16(vb)
        self.k_scale = self.v_scale = None
        if kv_dtype == KV_E4M3:
            n = num_layers * num_pages * num_kv_heads
            self.k_scale = torch.full((n,), -7.0, dtype=torch.float32, device=self.device)
            self.v_scale = torch.full((n,), -7.0, dtype=torch.float32, device=self.device)
        if sentinel is not None:
            if kv_dtype == KV_E4M3:
                self.k_arena.view(torch.uint8).fill_(sentinel & 0xff)
                self.v_arena.view(torch.uint8).fill_(sentinel & 0xff)
            else:
                s = int(np.array(sentinel, dtype=np.uint16).view(np.int16))
                self.k_arena.fill_(s)
                self.v_arena.fill_(s)
        self.scratch = torch.empty(max(sb, 256), dtype=torch.uint8, device=self.device)
        self.cfg = PoolConfig(num_layers, num_kv_heads, head_dim_qk, head_dim_v, PAGE, num_pages,
                              self.k_arena.data_ptr(), self.v_arena.data_ptr(), self.scratch.data_ptr(), shuffle_seed,
                              kv_dtype, 0, None if self.k_scale is None else self.k_scale.data_ptr(),
                              None if self.v_scale is None else self.v_scale.data_ptr())
        self.handle = comb_pool_create(self.cfg)
        self._ws: Optional[torch.Tensor] = None
        self._lws: Optional[torch.Tensor] = None

    @classmethod
    def from_export(cls, blob, device: str = "cuda", stream=None) -> "Pool":
        """(f4) read-only view, in this process, of a pool another process exported (Pool.export); no arena is
        allocated here: the exporter's bytes are mapped through CUDA IPC."""
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2602_01519_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
        self = cls.__new__(cls)
        self.device = torch.device(device)
        self.handle = comb_pool_import(blob, stream)
        hdr = np.frombuffer(bytes(blob)[16:40], dtype=np.int32)  # geometry fields of the blob's header
        self.num_layers, self.num_kv_heads, self.head_dim_qk, self.head_dim_v = (int(x) for x in hdr[:4])
        self.num_pages = int(hdr[5])
        self.k_arena = self.v_arena = self.scratch = None
        self.cfg = None
        self._ws = self._lws = None
        return self

    def export(self, directory_only: bool = False, stream=None) -> bytes:
        return comb_pool_export(self.handle, directory_only, stream).tobytes()

    def refresh(self, blob, stream=None) -> None:
        comb_pool_refresh(self.handle, blob, stream)

    def _aligned_i16(self, nbytes: int, align: int = 1024) -> torch.Tensor:
        raw = torch.empty(nbytes // 2 + align // 2, dtype=torch.int16, device=self.device)
        off = (-raw.data_ptr()) % align
        return raw[off // 2: off // 2 + nbytes // 2]

    def close(self) -> None:
        if self.handle:
            torch.cuda.synchronize()
            comb_pool_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- (a2) store ----
    def store_chunk(self, chunk_id: int, k: torch.Tensor, v: torch.Tensor, layer: int = 0, stream=None) -> None:
        comb_store_chunk(self.handle, layer, chunk_id, int(k.shape[0]), k, v, stream)

    def store_chunks(self, chunk_ids, tok_indptr, k_packed: torch.Tensor, v_packed: torch.Tensor, layer: int = 0,
                     stream=None) -> None:
        comb_store_chunks(self.handle, layer, chunk_ids, tok_indptr, k_packed, v_packed, stream)

    def project_store_chunks(self, chunk_ids, tok_indptr, h_packed: torch.Tensor, w_kv: torch.Tensor, layer: int = 0,
                             stream=None) -> None:
        """(f2) K/V projection of the chunks' hidden states with the pages written by the GEMM's epilogue."""
        comb_project_store_chunks(self.handle, layer, chunk_ids, tok_indptr, h_packed, int(h_packed.shape[1]), w_kv,
                                  stream)

    # ---- (f3) cross-attention sub-layer: x + Attn(x W_Q) W_O ----
    def layer_forward(self, lb: "LinkedBatch", x: torch.Tensor, q_indptr, w_q: torch.Tensor, w_o: torch.Tensor,
                      scale: float, layer: int = 0, out: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
        """q_indptr None = decode (one row per request)."""
        rows, d_model = int(x.shape[0]), int(x.shape[1])
        Hq = int(w_q.shape[0]) // self.head_dim_qk
        if out is None:
            out = torch.empty_like(x)
        need = comb_layer_workspace_bytes(self.handle, lb.link, Hq, rows)
        if self._lws is None or self._lws.numel() < need:
            self._lws = torch.empty(max(need, 256), dtype=torch.uint8, device=self.device)
        comb_cross_layer_forward(self.handle, layer, lb.link, lb.num_requests, x, q_indptr, d_model, Hq, w_q, w_o, scale,
                                 out, self._lws, self._lws.numel(), stream)
        return out

    # ---- (a3) link ----
    def link(self, chunk_lists: Sequence[Sequence[int]], stream=None, into: Optional[LinkedBatch] = None) -> LinkedBatch:
        indptr = np.zeros(len(chunk_lists) + 1, dtype=np.int32)
        np.cumsum([len(c) for c in chunk_lists], out=indptr[1:])
        ids = (np.concatenate([np.asarray(c, dtype=np.uint64) for c in chunk_lists])
               if indptr[-1] else np.zeros(0, dtype=np.uint64))
        return self.link_flat(indptr, ids, stream, into)

    def link_flat(self, chunk_indptr: np.ndarray, chunk_ids: np.ndarray, stream=None,
                  into: Optional[LinkedBatch] = None, host_mirror: bool = True) -> LinkedBatch:
        R = int(chunk_indptr.shape[0]) - 1
        if into is None:
            total_pages = 0
            ids = np.asarray(chunk_ids).tolist()
            for c in ids:
                nt = C.c_int32()
                total_pages += check(lib.comb_chunk_query(self.handle, int(c), C.byref(nt), None, 0), "comb_link")
            nbytes = comb_link_bytes(R, len(ids), total_pages)
            buf = torch.empty(max(nbytes, 16), dtype=torch.uint8, device=self.device)
            host = np.zeros(max(comb_link_host_bytes(R, len(ids)), 16), np.uint8) if host_mirror else None
            into = LinkedBatch(Link(), buf, host)
        into.link.device_buf = into.buf.data_ptr()
        into.link.device_bytes = into.buf.numel()
        into.link.host_buf = into.host.ctypes.data if into.host is not None else None
        into.link.host_bytes = into.host.nbytes if into.host is not None else 0
        comb_link(self.handle, chunk_indptr, chunk_ids, into.link, stream)
        return into

    # ---- (a4)/(a5) attention ----
    def workspace(self, lb: LinkedBatch, num_q_heads: int, total_q: int) -> torch.Tensor:
        need = comb_attn_workspace_bytes(self.handle, lb.link, num_q_heads, total_q)
        if self._ws is None or self._ws.numel() < need:
            self._ws = torch.empty(max(need, 256), dtype=torch.uint8, device=self.device)
        return self._ws

    def prefill(self, lb: LinkedBatch, q: torch.Tensor, q_indptr, scale: float, out: Optional[torch.Tensor] = None,
                lse: Optional[torch.Tensor] = None, layer: int = 0, want_lse: bool = True, stream=None):
        total_q, Hq = int(q.shape[0]), int(q.shape[1])
        if out is None:
            out = torch.empty((total_q, Hq, self.head_dim_v), dtype=q.dtype, device=self.device)
        if lse is None and want_lse:
            lse = torch.empty((total_q, Hq), dtype=torch.float32, device=self.device)
        ws = self.workspace(lb, Hq, total_q)
        comb_cross_attn_prefill(self.handle, layer, lb.link, q, q_indptr, Hq, scale, out, lse, ws, ws.numel(), stream)
        return out, lse

    def decode(self, lb: LinkedBatch, q: torch.Tensor, scale: float, out: Optional[torch.Tensor] = None,
               lse: Optional[torch.Tensor] = None, layer: int = 0, want_lse: bool = True, stream=None):
        R, Hq = int(q.shape[0]), int(q.shape[1])
        if out is None:
            out = torch.empty((R, Hq, self.head_dim_v), dtype=q.dtype, device=self.device)
        if lse is None and want_lse:
            lse = torch.empty((R, Hq), dtype=torch.float32, device=self.device)
        ws = self.workspace(lb, Hq, R)
        comb_cross_attn_decode(self.handle, layer, lb.link, R, q, Hq, scale, out, lse, ws, ws.numel(), stream)
        return out, lse

    def decode_noalloc(self, lb: LinkedBatch, q: torch.Tensor, scale: float, out: torch.Tensor,
                       lse: Optional[torch.Tensor] = None, layer: int = 0, stream=None):
        """comb_cross_attn_decode_noalloc: the caller passes q, out (and lse); nothing is allocated, here or in the library."""
        comb_cross_attn_decode_noalloc(self.handle, layer, lb.link, int(q.shape[0]), q, int(q.shape[1]), scale, out,
                                       lse, stream)
        return out, lse

    def set_decode_path(self, path: int) -> None:
        """DECODE_AUTO / DECODE_PER_REQUEST / DECODE_CHUNK_MAJOR (comb_pool_set_option, COMB_OPT_DECODE_PATH)."""
        comb_pool_set_option(self.handle, OPT_DECODE_PATH, path)

    @property
    def launches(self) -> int:
        return comb_pool_launch_count(self.handle)

    @property
    def free_pages(self) -> int:
        return int(lib.comb_pool_free_pages(self.handle))
