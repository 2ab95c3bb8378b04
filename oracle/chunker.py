"""Greedy merge of VAD segments into chunks (oracle).

TEST INFRASTRUCTURE - see ``oracle/__init__.py``.

PAPER.md:95: "Segments are greedily merged to construct chunks {C_1, ..., C_m} where each chunk
satisfies |C_i| <= c = 300 s".  Written out: walk the segments in time order, keep adding a segment
to the open chunk while the chunk's span (start of its first segment to end of the one being added)
stays <= c, otherwise close the chunk and open a new one with that segment.  A segment longer than c
is a chunk by itself (reading G23 of DESIGN.md).
"""
from __future__ import annotations

from typing import List, Sequence, Tuple


def greedy_chunks(segments: Sequence[Tuple[float, float]], c: float) -> List[List[int]]:
    chunks: List[List[int]] = []
    for i, (a, b) in enumerate(segments):
        if chunks and b - segments[chunks[-1][0]][0] <= c:
            chunks[-1].append(i)
        else:
            chunks.append([i])
    return chunks
