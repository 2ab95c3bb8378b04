"""Eq. 1 softmax attention over the retained set, in fp64 (oracle).

TEST INFRASTRUCTURE - see ``oracle/__init__.py``.

PAPER.md:101-104, Eq. 1:   alpha_ji = exp(q_j . k_i / sqrt(d)) / sum_i' exp(q_j . k_i' / sqrt(d))
and the attention output    o_j = sum_i alpha_ji v_i   over the tokens i left in the cache.

The method computes *exact* attention over a heuristically chosen subset, so the oracle is
the textbook definition written out over that subset: stored bf16 q, k_i, v_i are upcast
to fp64 exactly, s_i = (q . k_i) * scale, m = max_i s_i, e_i = exp(s_i - m),
alpha_i = e_i / sum e, o = sum alpha_i v_i.  Grouped-query attention maps query head h to
KV head h // G with G = n_q_heads // n_kv_heads (reading G19 of DESIGN.md).  No causal mask
(the cache holds only positions <= the query's), no bias, no soft-cap, no re-indexing of
positions (G17, G18).

``merge_partials`` is the log-sum-exp merge used by any split of the retained set
(task statement: "split-K ... with a log-sum-exp merge"): for partials (m_a, l_a, o_a)
with o_a un-normalised, m = max m_a, l = sum l_a e^{m_a - m}, o = sum o_a e^{m_a - m},
result o / l.
"""
from __future__ import annotations

from typing import Iterable, Sequence, Tuple

import numpy as np


def bf16_bits_to_f64(u16: np.ndarray) -> np.ndarray:
    """Exact upcast of bfloat16 bit patterns (uint16) to float64."""
    u16 = np.ascontiguousarray(u16, dtype=np.uint16)
    return (u16.astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)


def softmax_weights(scores: np.ndarray) -> np.ndarray:
    """Eq. 1 along the last axis, max-subtracted, fp64."""
    s = np.asarray(scores, dtype=np.float64)
    m = np.max(s, axis=-1, keepdims=True)
    e = np.exp(s - m)
    return e / np.sum(e, axis=-1, keepdims=True)


def attend_retained(
    q_bits: np.ndarray,  # [n_q, d]            uint16 bf16 bits: the newest token's queries
    k_bits: np.ndarray,  # [n_pos, n_kv, d]    uint16 bf16 bits: keys by absolute position
    v_bits: np.ndarray,  # [n_pos, n_kv, d]
    retained: Sequence[int],  # A(t): absolute positions attention sees
    scale: float,
) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """Returns (o [n_q, d] fp64, lse [n_q] fp64 natural log, alpha [n_q, n_ret] fp64)."""
    n_q, d = q_bits.shape
    n_kv = k_bits.shape[1]
    if n_q % n_kv:
        raise ValueError("n_q_heads must be a multiple of n_kv_heads")
    G = n_q // n_kv
    idx = np.asarray(list(retained), dtype=np.int64)
    if idx.size == 0:
        raise ValueError("attention over an empty set is undefined (Eq. 1 denominator)")
    q = bf16_bits_to_f64(q_bits)
    k = bf16_bits_to_f64(k_bits[idx])  # [n_ret, n_kv, d]
    v = bf16_bits_to_f64(v_bits[idx])
    o = np.empty((n_q, d), dtype=np.float64)
    lse = np.empty((n_q,), dtype=np.float64)
    alpha = np.empty((n_q, idx.size), dtype=np.float64)
    for h in range(n_q):
        g = h // G
        s = (k[:, g, :] @ q[h]) * scale  # s_i = q . k_i / sqrt(d)
        m = np.max(s)
        e = np.exp(s - m)
        denom = np.sum(e)
        a = e / denom
        alpha[h] = a
        o[h] = a @ v[:, g, :]
        lse[h] = m + np.log(denom)
    return o, lse, alpha


def partial_state(
    q_bits: np.ndarray, k_bits: np.ndarray, v_bits: np.ndarray, subset: Sequence[int], scale: float
) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """Un-normalised partial (m [n_q], l [n_q], o [n_q, d]) of one part of a split."""
    n_q, d = q_bits.shape
    G = n_q // k_bits.shape[1]
    idx = np.asarray(list(subset), dtype=np.int64)
    q = bf16_bits_to_f64(q_bits)
    k = bf16_bits_to_f64(k_bits[idx])
    v = bf16_bits_to_f64(v_bits[idx])
    m = np.empty((n_q,))
    l = np.empty((n_q,))
    o = np.empty((n_q, d))
    for h in range(n_q):
        g = h // G
        s = (k[:, g, :] @ q[h]) * scale
        m[h] = np.max(s)
        e = np.exp(s - m[h])
        l[h] = np.sum(e)
        o[h] = e @ v[:, g, :]
    return m, l, o


def merge_partials(parts: Iterable[Tuple[np.ndarray, np.ndarray, np.ndarray]]) -> Tuple[np.ndarray, np.ndarray]:
    """LSE merge of partial states; returns (o [n_q, d], lse [n_q])."""
    parts = list(parts)
    m = np.max(np.stack([p[0] for p in parts]), axis=0)
    l = np.zeros_like(m)
    o = np.zeros_like(parts[0][2])
    for m_a, l_a, o_a in parts:
        w = np.exp(m_a - m)
        l = l + l_a * w
        o = o + o_a * w[:, None]
    return o / l[:, None], m + np.log(l)
