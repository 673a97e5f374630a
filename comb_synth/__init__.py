"""Seeded synthetic inputs for the COMB link-stage path (shared by oracle-side tests and the GPU harness).

This module holds *data generation only*: chunk lengths, link lists, and bf16 bit patterns for
Q / K / V.  It contains none of the method's arithmetic (no attention, no paging, no tables) and
imports neither ``oracle`` nor ``paper_2602_01519_b200``.

Recipe (restated in DESIGN.md §5): numpy ``Generator(PCG64)``;
  * structure (lengths, link lists) ............ ``default_rng([seed, k, 0])``
  * chunk ``c``: K then V, float32 N(0,1) → bf16 .. ``default_rng([seed, k, 1, c])``
  * request ``r``: Q, float32 N(0,1) → bf16 ....... ``default_rng([seed, k, 2, r])``
where ``k`` is the index of the config in BASELINE.json ``configs`` (0..4).  bf16 rounding is
round-to-nearest-even on the float32 bit pattern.  The workloads stand in, by shape only, for the
paper's LongBench RAG / few-shot settings (§6.1) which are not in this container.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Dict, List, Optional, Tuple

import numpy as np

PAGE = 16  # tokens per page (BASELINE.json: "page 16")


# --------------------------------------------------------------------------------------------
# bf16 <-> float bit helpers (storage format conversion, not method arithmetic)
# --------------------------------------------------------------------------------------------
def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """float32 -> bf16 bit pattern (uint16), round-to-nearest-even.  Inputs must be finite."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    u = x.view(np.uint32)
    rounding = ((u >> np.uint32(16)) & np.uint32(1)) + np.uint32(0x7FFF)
    return ((u + rounding) >> np.uint32(16)).astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    b = np.ascontiguousarray(b, dtype=np.uint16)
    return (b.astype(np.uint32) << np.uint32(16)).view(np.float32)


def bf16_bits_to_f64(b: np.ndarray) -> np.ndarray:
    return bf16_bits_to_f32(b).astype(np.float64)


# --------------------------------------------------------------------------------------------
# workload description
# --------------------------------------------------------------------------------------------
@dataclass(frozen=True)
class Workload:
    name: str
    k: int                      # index into BASELINE.json configs (seeds the generators)
    seed: int
    num_q_heads: int
    num_kv_heads: int
    head_dim_qk: int
    head_dim_v: int
    chunk_len: np.ndarray       # int32 [num_chunks]  length of every chunk in the pool population
    links: Tuple[np.ndarray, ...]   # per request: int64 chunk ids in link order
    lq: np.ndarray              # int32 [R] query tokens per request
    scale: float
    q_gain: float = 1.0         # "peaked" variant multiplies Q by 4 before bf16 rounding
    note: str = ""

    # ---- derived sizes -------------------------------------------------------------------
    @property
    def num_requests(self) -> int:
        return len(self.links)

    @property
    def num_chunks(self) -> int:
        return int(self.chunk_len.shape[0])

    @property
    def group(self) -> int:
        return self.num_q_heads // self.num_kv_heads

    def pages_of_chunk(self, c: int) -> int:
        return (int(self.chunk_len[c]) + PAGE - 1) // PAGE

    @property
    def pool_pages(self) -> int:
        """Pages needed to hold every chunk of the population."""
        return int(((self.chunk_len.astype(np.int64) + PAGE - 1) // PAGE).sum())

    def kv_len(self, r: int) -> int:
        return int(self.chunk_len[self.links[r]].sum()) if len(self.links[r]) else 0

    @property
    def total_q(self) -> int:
        return int(self.lq.sum())

    @property
    def q_indptr(self) -> np.ndarray:
        out = np.zeros(self.num_requests + 1, dtype=np.int32)
        np.cumsum(self.lq, out=out[1:])
        return out

    @property
    def chunk_indptr(self) -> np.ndarray:
        out = np.zeros(self.num_requests + 1, dtype=np.int32)
        np.cumsum([len(l) for l in self.links], out=out[1:])
        return out

    @property
    def chunk_ids_flat(self) -> np.ndarray:
        if not self.links:
            return np.zeros(0, dtype=np.uint64)
        return np.concatenate([np.asarray(l, dtype=np.uint64) for l in self.links]) \
            if sum(len(l) for l in self.links) else np.zeros(0, dtype=np.uint64)

    def linked_chunks(self) -> np.ndarray:
        """Sorted distinct chunk ids named by any request."""
        if not self.links or not sum(len(l) for l in self.links):
            return np.zeros(0, dtype=np.int64)
        return np.unique(np.concatenate([np.asarray(l, dtype=np.int64) for l in self.links]))

    # ---- work counters used by bench / DESIGN (bookkeeping, valid tokens only) ---------------
    def pair_count(self) -> int:
        """sum_r lq_r * kv_r"""
        return int(sum(int(self.lq[r]) * self.kv_len(r) for r in range(self.num_requests)))

    def attention_flops(self) -> int:
        return 2 * (self.head_dim_qk + self.head_dim_v) * self.num_q_heads * self.pair_count()

    def kv_bytes_logical(self) -> int:
        tot = sum(self.kv_len(r) for r in range(self.num_requests))
        return 2 * self.num_kv_heads * (self.head_dim_qk + self.head_dim_v) * tot

    def kv_bytes_unique(self) -> int:
        """Bytes of the DISTINCT chunks the batch links: what has to cross the HBM pins at least once."""
        tot = int(self.chunk_len[self.linked_chunks()].astype(np.int64).sum())
        return 2 * self.num_kv_heads * (self.head_dim_qk + self.head_dim_v) * tot

    # ---- tensors ---------------------------------------------------------------------------
    def chunk_kv(self, c: int) -> Tuple[np.ndarray, np.ndarray]:
        """bf16 bit patterns: K [T][Hkv][Dqk], V [T][Hkv][Dv] for chunk ``c`` (K drawn first)."""
        t = int(self.chunk_len[c])
        rng = np.random.default_rng([self.seed, self.k, 1, int(c)])
        k = rng.standard_normal((t, self.num_kv_heads, self.head_dim_qk), dtype=np.float32)
        v = rng.standard_normal((t, self.num_kv_heads, self.head_dim_v), dtype=np.float32)
        return f32_to_bf16_bits(k), f32_to_bf16_bits(v)

    def request_q(self, r: int) -> np.ndarray:
        """bf16 bit patterns: Q [lq_r][Hq][Dqk] for request ``r``."""
        rng = np.random.default_rng([self.seed, self.k, 2, int(r)])
        q = rng.standard_normal((int(self.lq[r]), self.num_q_heads, self.head_dim_qk), dtype=np.float32)
        if self.q_gain != 1.0:
            q = q * np.float32(self.q_gain)
        return f32_to_bf16_bits(q)

    def all_q(self) -> np.ndarray:
        if self.total_q == 0:
            return np.zeros((0, self.num_q_heads, self.head_dim_qk), dtype=np.uint16)
        return np.concatenate([self.request_q(r) for r in range(self.num_requests)], axis=0)

    # ---- variants ----------------------------------------------------------------------------
    def peaked(self) -> "Workload":
        return replace(self, q_gain=4.0, name=self.name + "+peaked")

    def decode_phase(self) -> "Workload":
        """Same links, one query token per request (generated tokens are treated like
        query tokens).  Q is redrawn with lq=1 from the same per-request stream."""
        return replace(self, lq=np.ones(self.num_requests, dtype=np.int32), name=self.name + "+decode")


def bounded_zipf_p(n: int, a: float) -> np.ndarray:
    """p(rank) ∝ rank^-a over ranks 1..n; rank k maps to chunk id k-1."""
    p = np.arange(1, n + 1, dtype=np.float64) ** (-a)
    return p / p.sum()


def _structure_rng(seed: int, k: int) -> np.random.Generator:
    return np.random.default_rng([seed, k, 0])


# --------------------------------------------------------------------------------------------
# the five BASELINE.json configs (+ knobs to shrink them for oracle-sized parity cases)
# --------------------------------------------------------------------------------------------
def tiny_link(seed: int = 0, lq: int = 16, n_chunks: int = 4, chunk_tokens: int = 128) -> Workload:
    """configs[0]: 1 request, 8 q heads, 2 kv heads, D 64, 4 chunks x 128 in shuffled order, 16 query tokens."""
    rng = _structure_rng(seed, 0)
    order = rng.permutation(n_chunks).astype(np.int64)
    return Workload("tiny_link", 0, seed, 8, 2, 64, 64,
                    np.full(n_chunks, chunk_tokens, dtype=np.int32), (order,),
                    np.array([lq], dtype=np.int32), 1.0 / np.sqrt(64.0))


def decode_link(seed: int = 0, requests: int = 128, pool_chunks: int = 2000, chunk_tokens: int = 512,
                chunks_per_req: int = 8, no_reuse: bool = False) -> Workload:
    """configs[1]: Llama-3-8B-shaped layer, batch 128 x 1 query token, 8 chunks x 512 by Zipf(1.1) of 2000.
    ``no_reuse``: same geometry, but the batch's requests x chunks_per_req links are drawn WITHOUT replacement across
    the whole batch (1024 distinct chunks), so every linked byte has to come from HBM — the measurement case for the
    decode kernels' DRAM rate (no L2 help from shared chunks)."""
    rng = _structure_rng(seed, 1)
    if no_reuse:
        perm = rng.permutation(pool_chunks)[:requests * chunks_per_req].astype(np.int64)
        links = tuple(perm[r * chunks_per_req:(r + 1) * chunks_per_req] for r in range(requests))
        return Workload("decode_no_reuse", 1, seed, 32, 8, 128, 128,
                        np.full(pool_chunks, chunk_tokens, dtype=np.int32), links,
                        np.ones(requests, dtype=np.int32), 1.0 / np.sqrt(128.0))
    p = bounded_zipf_p(pool_chunks, 1.1)
    links = tuple(rng.choice(pool_chunks, size=chunks_per_req, replace=False, p=p).astype(np.int64)
                  for _ in range(requests))
    return Workload("decode_link", 1, seed, 32, 8, 128, 128,
                    np.full(pool_chunks, chunk_tokens, dtype=np.int32), links,
                    np.ones(requests, dtype=np.int32), 1.0 / np.sqrt(128.0))


def rag_prefill(seed: int = 0, requests: int = 32, lq: int = 256, pool_chunks: int = 1000,
                chunk_tokens: int = 512, chunks_per_req: int = 10) -> Workload:
    """configs[2]: Llama-shaped, 32 requests x 256 query tokens, 10 chunks x 512 uniform w/o replacement of 1000."""
    rng = _structure_rng(seed, 2)
    links = tuple(rng.choice(pool_chunks, size=chunks_per_req, replace=False).astype(np.int64)
                  for _ in range(requests))
    return Workload("rag_prefill", 2, seed, 32, 8, 128, 128,
                    np.full(pool_chunks, chunk_tokens, dtype=np.int32), links,
                    np.full(requests, lq, dtype=np.int32), 1.0 / np.sqrt(128.0))


def long_fewshot(seed: int = 0, requests: int = 8, lq: int = 512, n_chunks: int = 64,
                 len_lo: int = 128, len_hi: int = 1024) -> Workload:
    """configs[3]: Llama-shaped, 8 requests x 512 query tokens, all link the same 64 variable-length chunks
    (uniform 128..1024) each in its own random order (the few-shot pattern)."""
    rng = _structure_rng(seed, 3)
    lens = rng.integers(len_lo, len_hi + 1, size=n_chunks).astype(np.int32)
    links = tuple(rng.permutation(n_chunks).astype(np.int64) for _ in range(requests))
    return Workload("long_fewshot", 3, seed, 32, 8, 128, 128, lens, links,
                    np.full(requests, lq, dtype=np.int32), 1.0 / np.sqrt(128.0))


def mla_shaped(seed: int = 0, requests: int = 64, lq: int = 128, pool_chunks: int = 4000,
               chunk_tokens: int = 256, chunks_per_req: int = 16) -> Workload:
    """configs[4]: 16 heads, qk dim 192, v dim 128, no GQA, 64 requests x 128 query tokens, 16 chunks x 256 Zipf."""
    rng = _structure_rng(seed, 4)
    p = bounded_zipf_p(pool_chunks, 1.1)
    links = tuple(rng.choice(pool_chunks, size=chunks_per_req, replace=False, p=p).astype(np.int64)
                  for _ in range(requests))
    return Workload("mla_shaped", 4, seed, 16, 16, 192, 128,
                    np.full(pool_chunks, chunk_tokens, dtype=np.int32), links,
                    np.full(requests, lq, dtype=np.int32), 1.0 / np.sqrt(192.0))


CONFIGS = {
    "tiny_link": tiny_link,
    "decode_link": decode_link,
    "rag_prefill": rag_prefill,
    "long_fewshot": long_fewshot,
    "mla_shaped": mla_shaped,
}


def custom(name: str, *, k: int = 9, seed: int = 0, num_q_heads: int, num_kv_heads: int, head_dim_qk: int,
           head_dim_v: int, chunk_len, links, lq, scale: Optional[float] = None, q_gain: float = 1.0) -> Workload:
    """Free-form workload for edge-case tests (ragged lengths, empty links, duplicates ...)."""
    chunk_len = np.asarray(chunk_len, dtype=np.int32)
    links = tuple(np.asarray(l, dtype=np.int64) for l in links)
    lq = np.asarray(lq, dtype=np.int32)
    if scale is None:
        scale = 1.0 / float(np.sqrt(head_dim_qk))
    return Workload(name, k, seed, num_q_heads, num_kv_heads, head_dim_qk, head_dim_v, chunk_len, links, lq,
                    float(scale), q_gain)


# --------------------------------------------------------------------------------------------
# inputs of the steps either side of the attention: encoder hidden states, decoder rows
# and projection weights.  Data only: N(0, std) float32 -> bf16 bits, one generator per tensor.
# --------------------------------------------------------------------------------------------
def normal_bf16(seed: int, tag: int, index: int, shape, std: float = 1.0) -> np.ndarray:
    """bf16 bit patterns of N(0, std) values from ``default_rng([seed, 99, tag, index])``."""
    rng = np.random.default_rng([seed, 99, int(tag), int(index)])
    x = rng.standard_normal(tuple(int(s) for s in shape), dtype=np.float32) * np.float32(std)
    return f32_to_bf16_bits(x)


def hidden_states(seed: int, chunk: int, tokens: int, d_model: int) -> np.ndarray:
    """H^E of one chunk, bf16 bits [tokens][d_model] (unit variance, like a normalised residual stream)."""
    return normal_bf16(seed, 1, chunk, (tokens, d_model))


def decoder_rows(seed: int, request: int, rows: int, d_model: int) -> np.ndarray:
    """X^D rows of one request, bf16 bits [rows][d_model]."""
    return normal_bf16(seed, 2, request, (rows, d_model))


def projection_weight(seed: int, kind: int, layer: int, out_features: int, in_features: int,
                      gain: float = 1.0) -> np.ndarray:
    """nn.Linear-layout weight [out][in], N(0, gain / sqrt(in)) so that outputs of unit-variance inputs have
    variance gain^2.  kind: 0 = W_KV, 1 = W_Q, 2 = W_O."""
    return normal_bf16(seed, 10 + kind, layer, (out_features, in_features), gain / float(np.sqrt(in_features)))
