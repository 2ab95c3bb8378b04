"""murmur_chunk_plan (host logic) against oracle/chunker.py, plus the properties that
define a greedy merge.  No GPU needed: the function does no device work.  The oracle's own pins live in
tests/test_oracle_chunker.py, which does not load the product."""
import numpy as np
import pytest

from oracle import chunker as o_chunk
from paper_2606_01483_b200 import binding


def _segments(rng, n, max_seg=120.0, max_gap=20.0):
    t, out = 0.0, []
    for _ in range(n):
        t += float(np.float32(rng.uniform(0, max_gap)))
        d = float(np.float32(rng.uniform(0.2, max_seg)))
        out.append((float(np.float32(t)), float(np.float32(t + d))))
        t = out[-1][1]
    return out


@pytest.mark.parametrize("seed", range(20))
def test_matches_oracle_and_is_a_maximal_greedy_partition(seed):
    rng = np.random.default_rng(seed)
    seg = _segments(rng, int(rng.integers(0, 200)), max_seg=float(rng.choice([30.0, 120.0, 400.0])))
    c = float(rng.choice([60.0, 300.0]))
    got = binding.chunk_plan(seg, c)
    assert got == o_chunk.greedy_chunks(seg, c)
    assert [i for ch in got for i in ch] == list(range(len(seg)))  # a partition, in order
    for j, ch in enumerate(got):
        span = seg[ch[-1]][1] - seg[ch[0]][0]
        assert span <= c or len(ch) == 1  # |C| <= c unless one segment alone exceeds it
        if j + 1 < len(got):  # greedy: the next segment did not fit
            assert seg[got[j + 1][0]][1] - seg[ch[0]][0] > c


def test_argument_errors():
    with pytest.raises(binding.MurmurError):
        binding.chunk_plan([(0, 10), (5, 20)], 300.0)  # overlapping
    with pytest.raises(binding.MurmurError):
        binding.chunk_plan([(0, 10)], 0.0)
