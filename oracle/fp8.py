"""ORACLE — test infrastructure, not the product.  fp8 (e4m3) pages with per-(page, kv-head) scales (SURVEY.md §8(f4):
"fp8 (e4m3) pages with per-page scales to halve decode bytes"; memory is what bounds concurrency).

The paper does not describe a quantised cache, so everything here is the reading DESIGN.md §2 states (I31-I33):

  e4m3          the OCP 8-bit float "E4M3FN": 1 sign, 4 exponent (bias 7), 3 mantissa bits; no infinities; the
                all-ones exponent with mantissa 7 is NaN; largest finite 448; subnormals m/8 * 2^-6.
  block         the 16 x D values of one (page, kv-head); slots past the chunk's length count as zeros.
  scale         a power of two, stored as fp32: 2^e with e the smallest integer such that amax <= 448 * 2^e, amax = max |x|
                over the block (e clamped to [-100, 100]); 1 if amax = 0.  Dividing by it is exact, and value * scale is
                exactly representable in bf16 (4 significant bits), so dequantisation never rounds.
  code          e4m3 of x / scale, round to nearest even (no saturation can occur: |x / scale| <= 448).
  page image    codes in the bf16 layout with one byte per element; slots past the length are byte 0; scales in a side
                table fp32 [page][kv-head].
  dequantised   x' = value(code) * scale, exact in fp64.  Attention over fp8 pages is DEFINED as Eq. 7-8 over x'.

Written with plain numpy loops / tables so that a reader can check it against the format by eye; the pins in
tests/test_oracle_pins.py check the code table against the closed form, hand-worked ties and saturation.
"""
from __future__ import annotations

from typing import Dict, List, Sequence, Tuple

import numpy as np

PAGE = 16
E4M3_MAX = 448.0


def e4m3_value_table() -> np.ndarray:
    """fp64 value of every code 0..255 (NaN for 0x7f and 0xff), straight from the format's definition."""
    t = np.zeros(256, np.float64)
    for code in range(256):
        s, e, m = code >> 7, (code >> 3) & 0xF, code & 7
        if e == 15 and m == 7:
            v = np.nan
        elif e == 0:
            v = (m / 8.0) * 2.0 ** -6
        else:
            v = (1.0 + m / 8.0) * 2.0 ** (e - 7)
        t[code] = -v if s else v
    return t


_TABLE = e4m3_value_table()
_POS = _TABLE[:127]  # codes 0x00..0x7e: the non-negative finite values, ascending


def e4m3_decode(codes: np.ndarray) -> np.ndarray:
    return _TABLE[np.asarray(codes, dtype=np.uint8)]


def e4m3_encode(x: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even onto the finite e4m3 values, saturating (|x| > 448 -> +-448).  x: fp32/fp64 array (the
    callers pass the fp32 quotient widened to fp64, so "nearest" is decided on the exact fp32 value).  Ties go to the
    code with an even mantissa, i.e. the even code (codes are consecutive integers along the ascending values)."""
    a = np.abs(np.asarray(x, dtype=np.float64))
    a = np.minimum(a, E4M3_MAX)
    hi = np.searchsorted(_POS, a, side="left")          # first code with value >= a
    hi = np.minimum(hi, 126)
    lo = np.maximum(hi - 1, 0)
    d_lo, d_hi = a - _POS[lo], _POS[hi] - a
    pick_hi = (d_hi < d_lo) | ((d_hi == d_lo) & (hi % 2 == 0))
    code = np.where(pick_hi, hi, lo).astype(np.uint8)
    code = np.where(a == _POS[hi], hi, code).astype(np.uint8)   # exact hits (also covers a == 0)
    return (code | (np.signbit(np.asarray(x, dtype=np.float64)).astype(np.uint8) << 7)).astype(np.uint8)


def bf16_bits_to_f32(bits: np.ndarray) -> np.ndarray:
    return (np.ascontiguousarray(bits, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def quantise_block(block_f32: np.ndarray) -> Tuple[np.ndarray, np.float32]:
    """block [rows][D] fp32 (bf16 values, zero rows past the length) -> (codes uint8 [rows][D], scale fp32)."""
    amax = float(np.max(np.abs(block_f32))) if block_f32.size else 0.0
    scale = np.float32(block_scale(amax))
    quot = block_f32.astype(np.float64) / float(scale)                      # exact: a power of two
    return e4m3_encode(quot), scale


def block_scale(amax: float) -> float:
    """2^e, e = the smallest integer with amax <= 448 * 2^e, clamped to [-100, 100]; 1.0 for an all-zero block.
    Found by stepping e (no logarithm): exact for every float."""
    if not amax > 0.0:
        return 1.0
    e = 0
    while amax > E4M3_MAX * 2.0 ** e and e < 100:
        e += 1
    while e > -100 and amax <= E4M3_MAX * 2.0 ** (e - 1):
        e -= 1
    return 2.0 ** e


def quantise_chunk(k_bits: np.ndarray, v_bits: np.ndarray):
    """One chunk, bf16 bit patterns [T][Hkv][D] -> per page i: codes [Hkv][16][D] (tail slots 0) and scales [Hkv], for
    K and for V.  Returns (k_codes [np][Hkv][16][Dqk], k_scale [np][Hkv], v_codes, v_scale)."""
    out = []
    for bits in (k_bits, v_bits):
        T, H, D = bits.shape
        npg = (T + PAGE - 1) // PAGE
        x = bf16_bits_to_f32(bits)
        codes = np.zeros((npg, H, PAGE, D), np.uint8)
        scales = np.ones((npg, H), np.float32)
        for i in range(npg):
            n = min(PAGE, T - PAGE * i)
            for h in range(H):
                c, s = quantise_block(x[PAGE * i:PAGE * i + n, h, :])
                codes[i, h, :n, :] = c
                scales[i, h] = s
        out += [codes, scales]
    return tuple(out)


def dequantise_chunk(codes: np.ndarray, scales: np.ndarray, T: int) -> np.ndarray:
    """codes [np][Hkv][16][D], scales [np][Hkv] -> fp64 [T][Hkv][D]: value(code) * scale, exact."""
    npg, H, _, D = codes.shape
    x = e4m3_decode(codes) * scales.astype(np.float64)[:, :, None, None]      # [np][H][16][D]
    return np.ascontiguousarray(x.transpose(0, 2, 1, 3).reshape(npg * PAGE, H, D)[:T])


def page_image(num_pages: int, dims: Tuple[int, int, int], chunks: Dict[int, Tuple[np.ndarray, np.ndarray]],
               pages: Dict[int, Sequence[int]], sentinel: int = 0xA5, scale_sentinel: float = -7.0):
    """Expected fp8 arenas after storing `chunks` (id -> (K bits, V bits)) at `pages` (id -> page list): codes
    uint8 [num_pages][Hkv][16][D] and scales fp32 [num_pages][Hkv] for K and V; pages owned by no chunk keep the
    sentinels the harness wrote before."""
    Hkv, Dqk, Dv = dims
    k = np.full((num_pages, Hkv, PAGE, Dqk), sentinel, np.uint8)
    v = np.full((num_pages, Hkv, PAGE, Dv), sentinel, np.uint8)
    ks = np.full((num_pages, Hkv), scale_sentinel, np.float32)
    vs = np.full((num_pages, Hkv), scale_sentinel, np.float32)
    for cid, (kb, vb) in chunks.items():
        kc, ksc, vc, vsc = quantise_chunk(kb, vb)
        for i, p in enumerate(pages[cid]):
            k[p], v[p], ks[p], vs[p] = kc[i], vc[i], ksc[i], vsc[i]
    return k, ks, v, vs


def attention_for(w, requests: Sequence[int] = None):
    """Eq. 7-8 over the DEQUANTISED chunks of workload `w`, per request, in fp64 numpy: explicit
    concatenation in link order, one joint softmax, GQA head h -> kv-head h // G.
    Returns (O [sum lq][Hq][Dv], LSE [sum lq][Hq]) like oracle.attention_for."""
    reqs = list(range(w.num_requests)) if requests is None else list(requests)
    G = w.num_q_heads // w.num_kv_heads
    deq: Dict[int, Tuple[np.ndarray, np.ndarray]] = {}
    outs: List[np.ndarray] = []
    lses: List[np.ndarray] = []
    for r in reqs:
        ks, vs = [], []
        for c in w.links[r]:
            c = int(c)
            if c not in deq:
                kb, vb = w.chunk_kv(c)
                kc, ksc, vc, vsc = quantise_chunk(kb, vb)
                deq[c] = (dequantise_chunk(kc, ksc, kb.shape[0]), dequantise_chunk(vc, vsc, vb.shape[0]))
            ks.append(deq[c][0])
            vs.append(deq[c][1])
        q = bf16_bits_to_f32(w.request_q(r)).astype(np.float64)             # [lq][Hq][Dqk]
        lq = q.shape[0]
        O = np.zeros((lq, w.num_q_heads, w.head_dim_v))
        L = np.full((lq, w.num_q_heads), -np.inf)
        if ks:
            K, V = np.concatenate(ks), np.concatenate(vs)                    # [kv][Hkv][D]
            for h in range(w.num_q_heads):
                s = (q[:, h, :] @ K[:, h // G, :].T) * w.scale               # [lq][kv]
                m = s.max(axis=1, keepdims=True)
                p = np.exp(s - m)
                l = p.sum(axis=1, keepdims=True)
                O[:, h, :] = (p @ V[:, h // G, :]) / l
                L[:, h] = (m + np.log(l))[:, 0]
        outs.append(O)
        lses.append(L)
    return np.concatenate(outs), np.concatenate(lses)
