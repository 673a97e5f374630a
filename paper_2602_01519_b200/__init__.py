"""comb-link-b200: B200-native (sm_100a) link-stage cross-attention of COMB (arxiv 2602.01519).

Public surface = the C ABI of include/comb.h, mirrored one to one in :mod:`paper_2602_01519_b200.api`.
Importing this package loads libcomb.so and raises if it is not built — there is no fallback path.
"""
from . import _lib  # noqa: F401  (loads libcomb.so or raises)
from ._lib import (COMB_ERR_BUSY, COMB_ERR_READ_ONLY, COMB_ERR_CAPACITY, COMB_ERR_CUDA, COMB_ERR_EXISTS, COMB_ERR_INVALID, COMB_ERR_NO_SPACE,
                   COMB_ERR_UNKNOWN_CHUNK, COMB_OK, CombError, Link, PoolConfig)
from .api import (KV_BF16, KV_E4M3, comb_pool_scale_bytes, DECODE_AUTO, DECODE_CHUNK_MAJOR, DECODE_PER_REQUEST, KERNEL_CASCADE_MERGE, KERNEL_DECODE_CASCADE,
                  KERNEL_DECODE_MERGE, KERNEL_DECODE_SPLIT, KERNEL_GEMM, KERNEL_PREFILL, KERNEL_PREFILL_MERGE, KERNEL_STORE,
                  OPT_DECODE_PATH, OPT_EVICT_LRU, OPT_PREFILL_CLUSTERS, PAGE, LinkedBatch, Pool, comb_attn_workspace_bytes, comb_chunk_alloc,
                  comb_chunk_free, comb_chunk_pin, comb_chunk_query, comb_chunk_unpin, comb_pool_evicted,
                  comb_pool_eviction_count, comb_pool_export, comb_pool_import, comb_pool_refresh, comb_cross_attn_decode, comb_cross_attn_decode_noalloc, comb_noalloc_scratch_bytes, comb_cross_layer_forward, comb_gemm_bf16,
                  comb_layer_workspace_bytes, comb_project_store_chunks, comb_cross_attn_prefill, comb_link,
                  comb_link_bytes, comb_link_host_bytes, comb_link_plan, comb_pool_bytes, comb_pool_create,
                  comb_pool_destroy, comb_pool_launch_count, comb_pool_set_option, comb_profile_enable,
                  comb_profile_read, comb_profile_read_samples, comb_store_chunk, comb_store_chunks, comb_util_stream_read, comb_version, comb_workspace_bytes)
