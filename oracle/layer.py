"""ORACLE — test infrastructure, not the product.  The steps either side of the link-stage attention, in fp64 numpy,
written from the paper (PAPER.md = /root/reference/PAPER.md at authoring time):

  project_kv    K^cross = H^E W_K,  V^cross = H^E W_V                      PAPER.md:105-109 §4.2 Eq. 5-6
  attention_f64 A = softmax(Q K^T / sqrt d) (no mask, row-wise), H = A V   PAPER.md:112-115 Eq. 7-8, on fp64 inputs,
                over the explicit concatenation of the linked chunks
  cross_layer   x_out = x + Attn(x W_Q ; K, V) W_O                          PAPER.md:102-105 Eq. 4 (W_Q is the right
                reading), Eq. 7-8, PAPER.md:117 ("passed through the standard decoder pathway via
                residual connections"); no norm, gate or bias appears in Eq. 4-8, so none is applied
  cross_stack   the L cross layers of a model applied one after the other to the same rows (8 cross
                layers in the Llama instance; the decoder's own self-attention/MLP layers between them are outside
                the path)

Nothing is rounded between the steps: the product rounds Q, the attention output and x to bf16 at each hand-over
(they feed tensor-core contractions), the oracle does not, and the tests' tolerances account for that.
Weights are given in the nn.Linear layout the C ABI takes, [out_features][in_features], i.e. the paper's W
transposed.  A matmul is a library primitive used as one step; there is no blocking, fusion or reordering.

Pins (tests/test_oracle_pins.py): explicit-loop brute force on tiny shapes, the C oracle of O1 on bf16-exact inputs
(two independently written statements of Eq. 7-8), identity / zero weights (W_O = 0 recovers the decoder row,
PAPER.md:30; W_Q = 0 gives x + mean(V) W_O), linearity in W_O.
"""
from __future__ import annotations

from typing import List, Sequence, Tuple

import numpy as np


def bf16_to_f64(bits: np.ndarray) -> np.ndarray:
    """bf16 bit patterns -> exact fp64 values."""
    b = np.ascontiguousarray(bits, dtype=np.uint16)
    return (b.astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)


def f64_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even of fp64 values to bf16 bit patterns (via the exact fp32 value when representable; the
    double rounding fp64 -> fp32 -> bf16 can differ from a direct rounding only for values within 2^-24 relative of a
    bf16 tie, which the callers' tolerances cover)."""
    f = np.ascontiguousarray(x, dtype=np.float64).astype(np.float32)
    u = f.view(np.uint32)
    rounding = ((u >> np.uint32(16)) & np.uint32(1)) + np.uint32(0x7FFF)
    return ((u + rounding) >> np.uint32(16)).astype(np.uint16)


def project_kv(h: np.ndarray, w_kv: np.ndarray, num_kv_heads: int, head_dim_qk: int,
               head_dim_v: int) -> Tuple[np.ndarray, np.ndarray]:
    """Eq. 5-6.  h fp64 [T][d_model]; w_kv fp64 [Hkv*Dqk + Hkv*Dv][d_model] (rows of W_K^T head-major, then W_V^T).
    Returns K fp64 [T][Hkv][Dqk], V fp64 [T][Hkv][Dv]."""
    nk = num_kv_heads * head_dim_qk
    k = h @ w_kv[:nk].T
    v = h @ w_kv[nk:].T
    return (k.reshape(h.shape[0], num_kv_heads, head_dim_qk), v.reshape(h.shape[0], num_kv_heads, head_dim_v))


def attention_f64(q: np.ndarray, kcat: np.ndarray, vcat: np.ndarray, scale: float) -> Tuple[np.ndarray, np.ndarray]:
    """Eq. 7-8 for one request.  q fp64 [lq][Hq][Dqk]; kcat [kv][Hkv][Dqk], vcat [kv][Hkv][Dv] = the request's chunks
    concatenated in link order.  q-head h reads kv-head h // (Hq/Hkv).  kv == 0: O = 0, LSE = -inf (reading I13)."""
    lq, Hq, _ = q.shape
    kv, Hkv, Dv = vcat.shape[0], vcat.shape[1], vcat.shape[2]
    out = np.zeros((lq, Hq, Dv))
    lse = np.full((lq, Hq), -np.inf)
    if kv == 0:
        return out, lse
    G = Hq // Hkv
    for h in range(Hq):
        g = h // G
        s = scale * (q[:, h, :] @ kcat[:, g, :].T)          # [lq][kv]
        m = s.max(axis=1, keepdims=True)
        p = np.exp(s - m)
        l = p.sum(axis=1, keepdims=True)
        out[:, h, :] = (p @ vcat[:, g, :]) / l
        lse[:, h] = (m + np.log(l))[:, 0]
    return out, lse


def cross_layer(x: np.ndarray, q_indptr: np.ndarray, w_q: np.ndarray, w_o: np.ndarray, num_q_heads: int,
                chunks_k: Sequence[np.ndarray], chunks_v: Sequence[np.ndarray], links: Sequence[Sequence[int]],
                scale: float) -> np.ndarray:
    """x fp64 [rows][d_model] (rows of request r: q_indptr[r]..q_indptr[r+1]); w_q fp64 [Hq*Dqk][d_model];
    w_o fp64 [d_model][Hq*Dv]; chunks_k[c] fp64 [T_c][Hkv][Dqk] (what the pool holds, widened exactly).
    Returns x + Attn(x W_Q) W_O."""
    rows = x.shape[0]
    Dqk = chunks_k[0].shape[2] if len(chunks_k) else w_q.shape[0] // num_q_heads
    Dv = w_o.shape[1] // num_q_heads
    q = (x @ w_q.T).reshape(rows, num_q_heads, Dqk)                                   # Eq. 4
    attn = np.zeros((rows, num_q_heads, Dv))
    for r, lst in enumerate(links):
        lo, hi = int(q_indptr[r]), int(q_indptr[r + 1])
        if hi == lo:
            continue
        if len(lst):
            kcat = np.concatenate([chunks_k[int(c)] for c in lst], axis=0)
            vcat = np.concatenate([chunks_v[int(c)] for c in lst], axis=0)
            attn[lo:hi], _ = attention_f64(q[lo:hi], kcat, vcat, scale)              # Eq. 7-8
    return x + attn.reshape(rows, num_q_heads * Dv) @ w_o.T


def cross_stack(x: np.ndarray, q_indptr: np.ndarray, w_q: List[np.ndarray], w_o: List[np.ndarray], num_q_heads: int,
                chunks_k: List[Sequence[np.ndarray]], chunks_v: List[Sequence[np.ndarray]],
                links: Sequence[Sequence[int]], scale: float) -> List[np.ndarray]:
    """Layers 0..L-1 applied in order; layer l reads its own K/V (chunks_k[l][c]) through the SAME links.
    Returns the row states after every layer."""
    states = []
    for l in range(len(w_q)):
        x = cross_layer(x, q_indptr, w_q[l], w_o[l], num_q_heads, chunks_k[l], chunks_v[l], links, scale)
        states.append(x)
    return states
