"""ctypes view of libcomb.so (the C ABI of include/comb.h).  Argument marshalling only.

The library is built in-tree by ``python paper_2602_01519_b200/build.py`` (or ``__graft_entry__.build()``).
There is NO fallback: if the shared library is missing or a symbol is absent, importing raises.
"""
from __future__ import annotations

import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
# COMB_LIBRARY names another build of the same sources (prefill_timeline.py points it at libcomb_trace.so)
LIB_PATH = os.environ.get("COMB_LIBRARY") or os.path.join(HERE, "libcomb.so")

COMB_OK = 0
COMB_ERR_INVALID = -1
COMB_ERR_NO_SPACE = -2
COMB_ERR_EXISTS = -3
COMB_ERR_UNKNOWN_CHUNK = -4
COMB_ERR_CAPACITY = -5
COMB_ERR_CUDA = -6
COMB_ERR_BUSY = -7
COMB_ERR_READ_ONLY = -8


class PoolConfig(C.Structure):
    """comb_pool_config_t"""
    _fields_ = [("num_layers", C.c_int32), ("num_kv_heads", C.c_int32), ("head_dim_qk", C.c_int32),
                ("head_dim_v", C.c_int32), ("page_size", C.c_int32), ("num_pages", C.c_int32),
                ("k_arena", C.c_void_p), ("v_arena", C.c_void_p), ("scratch", C.c_void_p),
                ("free_list_shuffle_seed", C.c_uint64),
                ("kv_dtype", C.c_int32), ("reserved", C.c_int32), ("k_scale", C.c_void_p), ("v_scale", C.c_void_p)]


class Link(C.Structure):
    """comb_link_t"""
    _fields_ = [("device_buf", C.c_void_p), ("device_bytes", C.c_size_t),
                ("host_buf", C.c_void_p), ("host_bytes", C.c_size_t),
                ("page_indptr", C.c_void_p), ("page_ids", C.c_void_p), ("page_ntok", C.c_void_p),
                ("kv_len", C.c_void_p), ("tile_indptr", C.c_void_p), ("tile_ntok", C.c_void_p),
                ("entry_indptr", C.c_void_p),
                ("cas_page_indptr", C.c_void_p), ("cas_page_ids", C.c_void_p), ("cas_tile_indptr", C.c_void_p),
                ("cas_tile_ntok", C.c_void_p), ("cas_row_indptr", C.c_void_p), ("cas_row_req", C.c_void_p),
                ("cas_row_entry", C.c_void_p), ("page_ids_compact", C.c_void_p),
                ("host_req_pages", C.c_void_p), ("host_cas_rows", C.c_void_p), ("host_cas_pages", C.c_void_p),
                ("num_requests", C.c_int32), ("max_pages_per_request", C.c_int32),
                ("total_pages", C.c_int64), ("total_tiles", C.c_int64), ("total_kv_tokens", C.c_int64),
                ("total_entries", C.c_int64), ("num_distinct_chunks", C.c_int32), ("max_rows_per_chunk", C.c_int32),
                ("distinct_pages", C.c_int64), ("distinct_kv_tokens", C.c_int64),
                ("bytes_used", C.c_size_t)]


# every symbol include/comb.h declares: name -> (restype, argtypes)
_P = C.c_void_p
_SIGS = {
    "comb_pool_bytes": (C.c_int32, [C.POINTER(PoolConfig), C.POINTER(C.c_size_t), C.POINTER(C.c_size_t),
                                    C.POINTER(C.c_size_t)]),
    "comb_pool_scale_bytes": (C.c_size_t, [C.POINTER(PoolConfig)]),
    "comb_pool_create": (C.c_int32, [C.POINTER(PoolConfig), C.POINTER(_P)]),
    "comb_pool_destroy": (C.c_int32, [_P]),
    "comb_pool_free_pages": (C.c_int32, [_P]),
    "comb_chunk_alloc": (C.c_int32, [_P, C.c_uint64, C.c_int32]),
    "comb_chunk_free": (C.c_int32, [_P, C.c_uint64]),
    "comb_chunk_pin": (C.c_int32, [_P, C.c_uint64]),
    "comb_chunk_unpin": (C.c_int32, [_P, C.c_uint64]),
    "comb_pool_evicted": (C.c_int32, [_P, _P, C.c_int32]),
    "comb_pool_eviction_count": (C.c_int64, [_P]),
    "comb_pool_export_bytes": (C.c_size_t, [_P]),
    "comb_pool_export": (C.c_int32, [_P, C.c_uint32, _P, _P, C.c_size_t, C.POINTER(C.c_size_t)]),
    "comb_pool_import": (C.c_int32, [_P, C.c_size_t, _P, C.POINTER(_P)]),
    "comb_pool_refresh": (C.c_int32, [_P, _P, C.c_size_t, _P]),
    "comb_chunk_query": (C.c_int32, [_P, C.c_uint64, C.POINTER(C.c_int32), _P, C.c_int32]),
    "comb_store_chunk": (C.c_int32, [_P, C.c_int32, C.c_uint64, C.c_int32, _P, _P, _P]),
    "comb_store_chunks": (C.c_int32, [_P, C.c_int32, C.c_int32, _P, _P, _P, _P, _P]),
    "comb_project_store_chunks": (C.c_int32, [_P, C.c_int32, C.c_int32, _P, _P, _P, C.c_int32, _P, _P]),
    "comb_cross_layer_forward": (C.c_int32, [_P, C.c_int32, C.POINTER(Link), C.c_int32, _P, _P, C.c_int32, C.c_int32,
                                             _P, _P, C.c_float, _P, _P, C.c_size_t, _P]),
    "comb_layer_workspace_bytes": (C.c_size_t, [_P, C.POINTER(Link), C.c_int32, C.c_int64]),
    "comb_gemm_bf16": (C.c_int32, [_P, _P, _P, _P, _P, C.c_int64, C.c_int32, C.c_int32, _P]),
    "comb_link_bytes": (C.c_size_t, [C.c_int32, C.c_int64, C.c_int64]),
    "comb_link_host_bytes": (C.c_size_t, [C.c_int32, C.c_int64]),
    "comb_link": (C.c_int32, [_P, C.c_int32, _P, _P, C.POINTER(Link), _P]),
    "comb_link_plan": (C.c_int32, [_P, C.c_int32, _P, _P, C.POINTER(Link), _P]),
    "comb_cross_attn_prefill": (C.c_int32, [_P, C.c_int32, C.POINTER(Link), C.c_int32, _P, _P, C.c_int32, C.c_float,
                                            _P, _P, _P, C.c_size_t, _P]),
    "comb_cross_attn_decode": (C.c_int32, [_P, C.c_int32, C.POINTER(Link), C.c_int32, _P, C.c_int32, C.c_float, _P,
                                           _P, _P, C.c_size_t, _P]),
    "comb_cross_attn_decode_noalloc": (C.c_int32, [_P, C.c_int32, C.POINTER(Link), C.c_int32, _P, C.c_int32,
                                                   C.c_float, _P, _P, _P]),
    "comb_noalloc_scratch_bytes": (C.c_size_t, []),
    "comb_workspace_bytes": (C.c_size_t, [_P, C.c_int32, C.c_int32, C.c_int64, C.c_int32]),
    "comb_attn_workspace_bytes": (C.c_size_t, [_P, C.POINTER(Link), C.c_int32, C.c_int64]),
    "comb_pool_set_option": (C.c_int32, [_P, C.c_int32, C.c_int64]),
    "comb_pool_launch_count": (C.c_int64, [_P]),
    "comb_profile_enable": (C.c_int32, [_P, C.c_int32]),
    "comb_profile_read": (C.c_int32, [_P, C.c_int32, C.POINTER(C.c_double), C.POINTER(C.c_int64)]),
    "comb_profile_read_samples": (C.c_int32, [_P, C.c_int32, _P, C.c_int64, C.POINTER(C.c_int64)]),
    "comb_util_stream_read": (C.c_int32, [_P, C.c_size_t, _P, _P]),
    "comb_strerror": (C.c_char_p, [C.c_int32]),
    "comb_version": (C.c_char_p, []),
}
EXPORTS = tuple(sorted(_SIGS))


def load() -> C.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            "libcomb.so is not built (%s). Run `python paper_2602_01519_b200/build.py`; there is no CPU or "
            "PyTorch fallback for the COMB link-stage kernels." % LIB_PATH)
    lib = C.CDLL(LIB_PATH)
    for name, (res, args) in _SIGS.items():
        try:
            fn = getattr(lib, name)
        except AttributeError as e:  # stale build: fail loudly, never fall back
            raise ImportError("libcomb.so lacks %s — rebuild with `python paper_2602_01519_b200/build.py`" % name) from e
        fn.restype = res
        fn.argtypes = args
    return lib


lib = load()


class CombError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = int(status)
        super().__init__("%s: %s (%d)" % (where, lib.comb_strerror(status).decode(), status))


def check(status: int, where: str) -> int:
    if status < 0:
        raise CombError(status, where)
    return status
