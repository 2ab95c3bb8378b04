"""Attention-sparsity profile of one decode step (oracle).

TEST INFRASTRUCTURE - see ``oracle/__init__.py``.

PAPER.md:77 ("at any individual decode step, fewer than 25% of speech tokens account for 99% of
attention weight") and the caption of Fig. 5: every token of the KV cache falls in
one of four groups - speech tokens "required to retain 99% of total attention weight (kept
speech)", speech tokens outside that set (evictable speech), decoded tokens inside the 99% set
(kept text) and outside it (evictable text).  System-prompt tokens are counted apart (the paper's
figure leaves them out; they are never evicted).

Definition written out (per query head):
    alpha_x = softmax over the RESIDENT positions x of (q . k_x) * scale          (Eq. 1)
    the "mass set" = the fewest tokens whose weights sum to >= frac (0.99): sort by weight
    descending (ties: ascending position), take the shortest prefix reaching frac
    k_mass = its size; k_prompt / k_speech / k_text = its members per region
    mass_<region> = sum of alpha over the region; coverage = sum of alpha over a candidate
    retained set A (what a window policy would keep): the attention mass the policy preserves.

Regions: prompt = [0, P) U [P+S, P+S+M), speech = [P, P+S), text = [P+S+M, len).
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Iterable, List, Sequence

import numpy as np

from .attention import bf16_bits_to_f64, softmax_weights


@dataclass
class HeadProfile:
    n_resident: int
    n_prompt: int
    n_speech: int
    n_text: int
    k_mass: int
    k_prompt: int
    k_speech: int
    k_text: int
    coverage: float
    mass_prompt: float
    mass_speech: float
    mass_text: float
    mass_set: List[int]  # positions of the mass set, in the order they were taken
    alpha: np.ndarray  # weights of the resident positions, in ascending position order


def region_of(x: int, P: int, S: int, M: int) -> int:
    """0 = system prompt (either one), 1 = speech, 2 = text."""
    if x < P:
        return 0
    if x < P + S:
        return 1
    if x < P + S + M:
        return 0
    return 2


def mass_set_indices(alpha: np.ndarray, frac: float) -> List[int]:
    """Indices (into alpha) of the fewest entries whose sum reaches frac: descending weight, ties by
    ascending index, cumulative sum taken in that order."""
    order = sorted(range(len(alpha)), key=lambda i: (-alpha[i], i))
    acc = 0.0
    out: List[int] = []
    for i in order:
        out.append(i)
        acc += float(alpha[i])
        if acc >= frac:
            break
    return out


def profile_head(q_bits: np.ndarray, k_bits: np.ndarray, resident: Sequence[int], P: int, S: int, M: int,
                 candidate: Iterable[int], scale: float, frac: float = 0.99) -> HeadProfile:
    """q_bits [d] uint16 (one query head), k_bits [n_pos, d] uint16 (its KV head, by absolute position)."""
    res = sorted(int(x) for x in resident)
    if not res:
        raise ValueError("empty resident set")
    q = bf16_bits_to_f64(q_bits)
    k = bf16_bits_to_f64(k_bits[np.asarray(res, dtype=np.int64)])
    alpha = softmax_weights((k @ q) * scale)
    reg = np.asarray([region_of(x, P, S, M) for x in res])
    ms = mass_set_indices(alpha, frac)
    cand = set(int(x) for x in candidate)
    in_cand = np.asarray([x in cand for x in res])
    return HeadProfile(
        n_resident=len(res), n_prompt=int(np.sum(reg == 0)), n_speech=int(np.sum(reg == 1)), n_text=int(np.sum(reg == 2)),
        k_mass=len(ms), k_prompt=int(sum(reg[i] == 0 for i in ms)), k_speech=int(sum(reg[i] == 1 for i in ms)),
        k_text=int(sum(reg[i] == 2 for i in ms)),
        coverage=float(np.sum(alpha[in_cand])), mass_prompt=float(np.sum(alpha[reg == 0])),
        mass_speech=float(np.sum(alpha[reg == 1])), mass_text=float(np.sum(alpha[reg == 2])),
        mass_set=[res[i] for i in ms], alpha=alpha)


def profile_step(q_bits: np.ndarray, k_bits: np.ndarray, resident: Sequence[int], P: int, S: int, M: int,
                 candidate: Iterable[int], scale: float, frac: float = 0.99) -> List[HeadProfile]:
    """All query heads of one (layer, sequence): q_bits [n_q, d], k_bits [n_pos, n_kv, d]; KV head of
    query head h is h // (n_q // n_kv) (reading G19)."""
    n_q = q_bits.shape[0]
    n_kv = k_bits.shape[1]
    G = n_q // n_kv
    cand = list(candidate)
    return [profile_head(q_bits[h], k_bits[:, h // G], resident, P, S, M, cand, scale, frac) for h in range(n_q)]
