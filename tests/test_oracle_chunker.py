"""Pins of oracle/chunker.py (greedy VAD-segment merge) that do not load the product: by-hand
cases worked from the sentence "Segments are greedily merged to construct chunks ... where each chunk satisfies
|C_i| <= c", the defining properties of a maximal greedy partition, and a brute force over all ordered
partitions on tiny inputs (the greedy one is the partition whose chunks each take as many segments as fit)."""
import itertools

import numpy as np
import pytest

from oracle import chunker as o_chunk


def test_by_hand_cases():
    # [0,100] + [110,290]: span 290 <= 300 -> one chunk; adding [295,400] would span 400 -> new chunk;
    # [410,760] is 350 s long: a chunk by itself (reading G23); [761,800] cannot join it (span 390)
    seg = [(0, 100), (110, 290), (295, 400), (410, 760), (761, 800)]
    assert o_chunk.greedy_chunks(seg, 300.0) == [[0, 1], [2], [3], [4]]
    assert o_chunk.greedy_chunks([], 300.0) == []
    assert o_chunk.greedy_chunks([(5, 6)], 300.0) == [[0]]


def test_span_exactly_c_is_allowed():
    # |C| <= c: a span of exactly c stays in the chunk, one tick more does not
    assert o_chunk.greedy_chunks([(0, 100), (100, 300)], 300.0) == [[0, 1]]
    assert o_chunk.greedy_chunks([(0, 100), (100, 300.5)], 300.0) == [[0], [1]]


def test_touching_segments_and_gaps_count_towards_the_span():
    # the span runs from the first segment's start to the last one's end: silence in between counts
    assert o_chunk.greedy_chunks([(0, 10), (10, 20), (20, 30)], 30.0) == [[0, 1, 2]]
    assert o_chunk.greedy_chunks([(0, 10), (25, 31)], 30.0) == [[0], [1]]  # 16 s of speech, but a 31 s span
    assert o_chunk.greedy_chunks([(0, 10), (25, 30)], 30.0) == [[0, 1]]


def test_segment_longer_than_c_is_alone_and_does_not_absorb_neighbours():
    got = o_chunk.greedy_chunks([(0, 5), (6, 400), (401, 405), (406, 410)], 300.0)
    assert got == [[0], [1], [2, 3]]


def test_a_60_minute_recording_of_back_to_back_300_s_segments_gives_12_chunks():
    # BASELINE.json config 2: "one 60 min recording cut into 300 s chunks" = 12 sequences
    seg = [(300.0 * i, 300.0 * (i + 1)) for i in range(12)]
    assert o_chunk.greedy_chunks(seg, 300.0) == [[i] for i in range(12)]
    seg = [(10.0 * i, 10.0 * (i + 1)) for i in range(360)]
    got = o_chunk.greedy_chunks(seg, 300.0)
    assert len(got) == 12 and all(len(ch) == 30 for ch in got)


def _ordered_partitions(n):
    for cuts in itertools.product((0, 1), repeat=max(0, n - 1)):
        parts, cur = [], [0]
        for i, cut in enumerate(cuts, start=1):
            if cut:
                parts.append(cur)
                cur = [i]
            else:
                cur.append(i)
        if n:
            parts.append(cur)
        yield parts


@pytest.mark.parametrize("seed", range(12))
def test_brute_force_tiny(seed):
    """Among all ordered partitions whose chunks respect |C| <= c (single over-long segments excepted), the greedy
    one is the unique partition that is lexicographically largest in chunk sizes (each chunk takes all that fits)."""
    rng = np.random.default_rng(seed)
    n = int(rng.integers(1, 9))
    t, seg = 0.0, []
    for _ in range(n):
        t += float(rng.integers(0, 4))
        d = float(rng.integers(1, 14))
        seg.append((t, t + d))
        t += d
    c = float(rng.choice([10.0, 15.0, 25.0]))
    ok = [p for p in _ordered_partitions(n)
          if all(len(ch) == 1 or seg[ch[-1]][1] - seg[ch[0]][0] <= c for ch in p)]
    best = max(ok, key=lambda p: [len(ch) for ch in p])
    assert o_chunk.greedy_chunks(seg, c) == best


@pytest.mark.parametrize("seed", range(10))
def test_maximal_greedy_property(seed):
    rng = np.random.default_rng(100 + seed)
    t, seg = 0.0, []
    for _ in range(int(rng.integers(0, 150))):
        t += float(rng.uniform(0, 20))
        d = float(rng.uniform(0.2, rng.choice([30.0, 120.0, 400.0])))
        seg.append((t, t + d))
        t += d
    c = float(rng.choice([60.0, 300.0]))
    got = o_chunk.greedy_chunks(seg, c)
    assert [i for ch in got for i in ch] == list(range(len(seg)))  # a partition, in order
    for j, ch in enumerate(got):
        assert seg[ch[-1]][1] - seg[ch[0]][0] <= c or len(ch) == 1
        if j + 1 < len(got):  # the next segment did not fit
            assert seg[got[j + 1][0]][1] - seg[ch[0]][0] > c
