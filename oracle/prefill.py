"""Causal self-attention of a chunk's prefill tokens, in fp64 (oracle).

TEST INFRASTRUCTURE - see ``oracle/__init__.py``.

PAPER.md:95 (chunks are submitted to the engine, which first runs the prompt + speech tokens
through the model - the "prefill") and PAPER.md:77 (decoding is 95.3 % of model time; prefill is the
rest).  The model is a decoder (it "autoregressively generates text tokens conditioned
on the full speech token sequence"), so the prefill token at position x attends, by Eq. 1
(PAPER.md:101-104), to the cache positions y <= x:

    o_x = sum_{y <= x} alpha_xy v_y,   alpha_xy = softmax_y (q_x . k_y * scale)

written out per query position; GQA head map h -> h // G (reading G19).
"""
from __future__ import annotations

from typing import Tuple

import numpy as np

from .attention import bf16_bits_to_f64, softmax_weights


def causal_attention(q_bits: np.ndarray, k_bits: np.ndarray, v_bits: np.ndarray, pos_begin: int, scale: float
                     ) -> Tuple[np.ndarray, np.ndarray]:
    """q_bits [n_tok, n_q, d] uint16: queries of positions pos_begin .. pos_begin + n_tok - 1;
    k_bits, v_bits [n_pos, n_kv, d] uint16 by absolute position, n_pos >= pos_begin + n_tok.
    Returns (o [n_tok, n_q, d] fp64, lse [n_tok, n_q] fp64)."""
    n_tok, n_q, d = q_bits.shape
    n_kv = k_bits.shape[1]
    G = n_q // n_kv
    q = bf16_bits_to_f64(q_bits)
    k = bf16_bits_to_f64(k_bits)
    v = bf16_bits_to_f64(v_bits)
    o = np.zeros((n_tok, n_q, d), dtype=np.float64)
    lse = np.zeros((n_tok, n_q), dtype=np.float64)
    for i in range(n_tok):
        x = pos_begin + i
        for h in range(n_q):
            s = (k[: x + 1, h // G] @ q[i, h]) * scale
            a = softmax_weights(s)
            o[i, h] = a @ v[: x + 1, h // G]
            m = np.max(s)
            lse[i, h] = m + np.log(np.sum(np.exp(s - m)))
    return o, lse
