"""Loads a synthetic workload (any object shaped like ``comb_synth.Workload``) into a device pool through the
public binding: batched store of the chunk population in chunk-id order, link of every request, Q upload.

Used by tests/, bench.py and __graft_entry__.smoke().  It performs none of the method's arithmetic — only
host->device copies and calls of the C ABI.  Chunks no request links may be filled by a device-side random
generator (``fill="linked"``): they occupy their pages (so page placement matches a full pool) but are never
read, which keeps the multi-GB pools of BASELINE configs 2, 3 and 5 fast to build.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Dict, List, Optional

import numpy as np
import torch

from .api import LinkedBatch, Pool

PAGE = 16


def bits_to_device(a: np.ndarray, device) -> torch.Tensor:
    """uint16 bf16 bit patterns -> device torch.bfloat16 tensor (bit copy)."""
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int16)).to(device).view(torch.bfloat16)


def device_to_bits(t: torch.Tensor) -> np.ndarray:
    return t.contiguous().view(torch.int16).cpu().numpy().view(np.uint16)


@dataclass
class Loaded:
    pool: Pool
    batch: LinkedBatch
    q: torch.Tensor                 # bf16 [sum lq][Hq][Dqk]
    q_indptr: np.ndarray
    stored_host: Dict[int, tuple]   # chunk id -> (K bits, V bits) for chunks stored from host data
    store_bytes: int                # algorithmic bytes moved by the stores (read + write)
    num_store_calls: int


def load_workload(w, *, fill: str = "all", shuffle_seed: int = 0, extra_pages: int = 0, sentinel: Optional[int] = None,
                  batch_tokens: int = 1 << 16, device: str = "cuda", keep_host: bool = True, kv_dtype: int = 0) -> Loaded:
    """``fill="all"``: every chunk of the population comes from ``w.chunk_kv`` (host, seeded).
    ``fill="linked"``: only linked chunks do; the rest get device-side N(0,1) bf16 noise."""
    assert fill in ("all", "linked")
    pool = Pool(w.num_kv_heads, w.head_dim_qk, w.head_dim_v, w.pool_pages + extra_pages, shuffle_seed=shuffle_seed,
                device=device, sentinel=sentinel, kv_dtype=kv_dtype)
    linked = set(int(c) for c in w.linked_chunks())
    stored: Dict[int, tuple] = {}
    Hkv, Dqk, Dv = w.num_kv_heads, w.head_dim_qk, w.head_dim_v
    store_bytes = 0
    calls = 0
    c = 0
    n = w.num_chunks
    gen = torch.Generator(device=device)
    gen.manual_seed(1234 + int(w.seed))
    while c < n:
        ids: List[int] = []
        tok = [0]
        while c < n and (not ids or tok[-1] + int(w.chunk_len[c]) <= batch_tokens):
            ids.append(c)
            tok.append(tok[-1] + int(w.chunk_len[c]))
            c += 1
        T = tok[-1]
        if fill == "all" or all(i in linked for i in ids):
            kh = np.empty((T, Hkv, Dqk), np.uint16)
            vh = np.empty((T, Hkv, Dv), np.uint16)
            for i, cid in enumerate(ids):
                k, v = w.chunk_kv(cid)
                kh[tok[i]:tok[i + 1]] = k
                vh[tok[i]:tok[i + 1]] = v
                if keep_host:
                    stored[cid] = (k, v)
            kd, vd = bits_to_device(kh, device), bits_to_device(vh, device)
        else:
            kd = torch.randn((T, Hkv, Dqk), device=device, generator=gen, dtype=torch.float32).to(torch.bfloat16)
            vd = torch.randn((T, Hkv, Dv), device=device, generator=gen, dtype=torch.float32).to(torch.bfloat16)
            for i, cid in enumerate(ids):
                if cid in linked:
                    k, v = w.chunk_kv(cid)
                    kd[tok[i]:tok[i + 1]] = bits_to_device(k, device)
                    vd[tok[i]:tok[i + 1]] = bits_to_device(v, device)
                    if keep_host:
                        stored[cid] = (k, v)
        pool.store_chunks(ids, np.array(tok, np.int32), kd, vd)
        calls += 1
        store_bytes += 2 * T * Hkv * (Dqk + Dv) * 2
    torch.cuda.synchronize()
    batch = pool.link([list(map(int, l)) for l in w.links])
    q = bits_to_device(w.all_q(), device)
    return Loaded(pool, batch, q, w.q_indptr, stored, store_bytes, calls)
