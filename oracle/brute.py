"""ORACLE pin P1 — brute force on tiny inputs (test infrastructure, not the product).

A second, separately written statement of PAPER.md:112-119 §4.2 Eq. 7-8 used only to pin
``comb_oracle.c``: pure Python loops over Python floats, the softmax written literally as
exp(s_j) / sum_j exp(s_j) with NO max subtraction, keys gathered chunk by chunk in link order.
Tiny shapes only (it is O(lq * Hq * kv * D) interpreted Python).
"""
from __future__ import annotations

import math
from typing import List, Sequence

import numpy as np


def _bf16_to_float(bits: int) -> float:
    return float(np.array([int(bits) << 16], dtype=np.uint32).view(np.float32)[0])


def attention_brute(q_bits: np.ndarray, k_chunks: Sequence[np.ndarray], v_chunks: Sequence[np.ndarray],
                    link: Sequence[int], scale: float):
    """One request.  q_bits [lq][Hq][Dqk]; k_chunks[c] [T][Hkv][Dqk]; link = chunk indices in link order.
    Returns nested lists O[lq][Hq][Dv], LSE[lq][Hq]."""
    lq, Hq, Dqk = q_bits.shape
    Hkv = k_chunks[0].shape[1]
    Dv = v_chunks[0].shape[2]
    G = Hq // Hkv
    O: List = []
    L: List = []
    for i in range(lq):
        O.append([])
        L.append([])
        for h in range(Hq):
            g = h // G
            qv = [_bf16_to_float(q_bits[i, h, c]) for c in range(Dqk)]
            weights: List[float] = []
            values: List[List[float]] = []
            for c_idx in link:                      # "concatenated along l_doc" in link order
                K = k_chunks[c_idx]
                V = v_chunks[c_idx]
                for t in range(K.shape[0]):
                    s = 0.0
                    for c in range(Dqk):
                        s += qv[c] * _bf16_to_float(K[t, g, c])
                    weights.append(math.exp(scale * s))          # literal softmax numerator
                    values.append([_bf16_to_float(V[t, g, c]) for c in range(Dv)])
            if not weights:
                O[i].append([0.0] * Dv)
                L[i].append(-math.inf)
                continue
            z = math.fsum(weights)
            O[i].append([math.fsum(w * v[c] for w, v in zip(weights, values)) / z for c in range(Dv)])
            L[i].append(math.log(z))
    return O, L


def attention_request(q: np.ndarray, kcat: np.ndarray, vcat: np.ndarray, scale: float):
    """The same brute force on fp64 inputs, keys already concatenated: q [lq][Hq][Dqk], kcat [kv][Hkv][Dqk],
    vcat [kv][Hkv][Dv] -> (O [lq][Hq][Dv], LSE [lq][Hq]) as numpy arrays.  Pins oracle/layer.py::attention_f64."""
    lq, Hq, Dqk = q.shape
    kv, Hkv, Dv = vcat.shape
    G = Hq // Hkv
    O = np.zeros((lq, Hq, Dv))
    L = np.full((lq, Hq), -math.inf)
    for i in range(lq):
        for h in range(Hq):
            g = h // G
            weights = []
            for t in range(kv):
                s = 0.0
                for c in range(Dqk):
                    s += float(q[i, h, c]) * float(kcat[t, g, c])
                weights.append(math.exp(scale * s))
            if not weights:
                continue
            z = math.fsum(weights)
            for c in range(Dv):
                O[i, h, c] = math.fsum(w * float(vcat[t, g, c]) for t, w in enumerate(weights)) / z
            L[i, h] = math.log(z)
    return O, L
