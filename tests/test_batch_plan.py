"""murmur_batch_plan (host logic) against oracle/batcher.py on seeded segment lists: batch and
slot of every chunk, speech-token count, output budget and block bound - all integers, bit-exact.  No GPU needed.
The oracle's own pins are in tests/test_oracle_batcher.py."""
import numpy as np
import pytest

from oracle import batcher as o_batch
from oracle import chunker as o_chunk
from paper_2606_01483_b200 import binding


def _segments(rng, n, max_seg):
    t, out = 0.0, []
    for _ in range(n):
        t += float(np.float32(rng.uniform(0, 20.0)))
        d = float(np.float32(rng.uniform(0.2, max_seg)))
        out.append((float(np.float32(t)), float(np.float32(t + d))))
        t = out[-1][1]
    return out


@pytest.mark.parametrize("seed", range(16))
def test_matches_oracle(seed):
    rng = np.random.default_rng(seed)
    seg = _segments(rng, int(rng.integers(0, 400)), float(rng.choice([30.0, 120.0, 400.0, 5000.0])))
    chunks = o_chunk.greedy_chunks(seg, 300.0)
    B = int(rng.choice([1, 5, 16]))
    P, M, page = int(rng.integers(0, 100)), int(rng.integers(0, 8)), int(rng.choice([16, 64]))
    got = binding.batch_plan(seg, chunks, batch_size=B, n_prefix=P, n_mid=M, page_size=page)
    want = o_batch.form_batches(seg, chunks, batch_size=B)
    assert len(got) == len(want)
    for gb, wb in zip(got, want):
        assert len(gb) == len(wb)
        for g, w in zip(gb, wb):
            assert {k: g[k] for k in ("chunk", "slot", "n_speech", "max_new")} == w
            assert g["max_blocks"] == o_batch.max_blocks(P, w["n_speech"], M, w["max_new"], page)


def test_config2_shape_end_to_end_from_segments():
    # one hour of back-to-back 10 s segments -> 12 chunks of 300 s -> one batch of 12 slots, S = 2250
    seg = [(10.0 * i, 10.0 * (i + 1)) for i in range(360)]
    chunks = binding.chunk_plan(seg, 300.0)
    got = binding.batch_plan(seg, chunks, n_prefix=64, page_size=64)
    assert len(got) == 1 and [e["slot"] for e in got[0]] == list(range(12))
    assert all(e["n_speech"] == 2250 and e["max_new"] == 2730 for e in got[0])
    assert got[0][0]["max_blocks"] == (64 + 2250 + 2730 + 63) // 64


def test_other_rates_and_budgets():
    seg = [(0.0, 100.0), (200.0, 250.0)]
    got = binding.batch_plan(seg, [[0], [1]], batch_size=1, tokens_per_s=12.5, max_new_nominal=1000, d_nominal=200.0)
    want = o_batch.form_batches(seg, [[0], [1]], batch_size=1, rate=12.5, max_new_nominal=1000, d_nominal=200.0)
    assert [[{k: e[k] for k in ("chunk", "slot", "n_speech", "max_new")} for e in b] for b in got] == want
    assert got[0][0]["n_speech"] == 1250 and got[0][0]["max_new"] == 500 and got[1][0]["max_new"] == 250


def test_argument_errors():
    seg = [(0.0, 10.0), (20.0, 30.0)]
    with pytest.raises(binding.MurmurError):
        binding.batch_plan(seg, [[0], [1]], batch_size=0)
    with pytest.raises(binding.MurmurError):
        binding.batch_plan(seg, [[1], [0]])  # chunk table not ascending from 0
    with pytest.raises(binding.MurmurError):
        binding.batch_plan(seg, [[0], [1]], tokens_per_s=0.0)
    with pytest.raises(binding.MurmurError):
        binding.batch_plan(seg, [[0], [1]], tokens_per_s=1e12)  # does not fit int32
    assert binding.batch_plan(seg, []) == []
