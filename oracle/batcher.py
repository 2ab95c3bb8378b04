"""Batch formation: chunks -> batches of sequence slots with their cache geometry (oracle).

TEST INFRASTRUCTURE - see ``oracle/__init__.py``.

PAPER.md:95 (section 3.1): "Chunks are submitted as a batch to an inference engine ... to amortize the GPU idle
time across concurrent requests."  PAPER.md:170 (section 4.1): "a batch size of 16 chunks" and "The maximum
number of new tokens is set to 32,768 for recordings within the model's nominal context length of 60 minutes;
for shorter recordings, it is scaled as |32,768 x d / d_nominal| where d is the recording duration in seconds,
and d_nominal is 3600 seconds."  PAPER.md:99: each request is [system prompt][speech tokens][system prompt]
[text tokens].

Written out, in the paper's order (readings G24-G26 of DESIGN.md):
  1. the chunks, in time order, are cut into consecutive batches of at most `batch_size`; chunk j goes to
     batch j // batch_size, slot j % batch_size                                       (G24: no re-ordering)
  2. a chunk's duration d is its span, first segment's start to last segment's end (G23); its speech region
     holds S = ceil(rate * d) tokens, rate = 7.5 tokens per second of audio (BASELINE.json configs: 60 s -> 450,
     300 s -> 2250, 60 min -> 27000)                                                  (G25: ceil)
  3. its output budget is T = floor(32768 * d / 3600), and 32768 when d >= 3600; the "recording" of the rule
     is what is submitted as one request, i.e. the chunk; at least 1                  (G26: the garbled
     brackets of PAPER.md:170 are read as a floor)
  4. the sequence may grow to n_prefix + S + n_mid + T tokens: that bounds its logical blocks.
All arithmetic on d is IEEE double on the float32 segment times (exactly representable), in the order written.
"""
from __future__ import annotations

import math
from typing import Dict, List, Sequence, Tuple


def chunk_geometry(d: float, rate: float = 7.5, max_new_nominal: int = 32768, d_nominal: float = 3600.0) -> Tuple[int, int]:
    """(S, T) of one chunk of duration d seconds: speech tokens and the output-token budget."""
    S = int(math.ceil(rate * d))
    T = max_new_nominal if d >= d_nominal else int(math.floor(max_new_nominal * d / d_nominal))
    return S, max(1, T)


def form_batches(segments: Sequence[Tuple[float, float]], chunks: Sequence[Sequence[int]], batch_size: int = 16,
                 rate: float = 7.5, max_new_nominal: int = 32768, d_nominal: float = 3600.0) -> List[List[Dict[str, int]]]:
    """chunks: lists of segment indices (oracle.chunker.greedy_chunks).  Returns the batches; each entry is
    {"chunk": j, "slot": position in its batch, "n_speech": S, "max_new": T}."""
    batches: List[List[Dict[str, int]]] = []
    for j, ch in enumerate(chunks):
        if j % batch_size == 0:
            batches.append([])
        d = float(segments[ch[-1]][1]) - float(segments[ch[0]][0])
        S, T = chunk_geometry(d, rate, max_new_nominal, d_nominal)
        batches[-1].append({"chunk": j, "slot": len(batches[-1]), "n_speech": S, "max_new": T})
    return batches


def max_blocks(n_prefix: int, n_speech: int, n_mid: int, max_new: int, page_size: int) -> int:
    """Logical blocks a sequence of that geometry may ever span (what murmur_cache_desc_t.max_blocks_per_seq
    has to cover)."""
    return (n_prefix + n_speech + n_mid + max_new + page_size - 1) // page_size
