"""Pins of oracle/batcher.py (batch formation) - values the paper and BASELINE.json fix, worked
by hand, plus the properties that define "consecutive batches of at most B".  Does not load the product."""
import numpy as np
import pytest

from oracle import batcher as o_batch
from oracle import chunker as o_chunk


def test_token_counts_of_the_baseline_configs():
    # BASELINE.json configs: 60 s -> 450 speech tokens, 300 s -> 2250, 60 min -> 27000 (7.5 tokens per second)
    assert o_batch.chunk_geometry(60.0)[0] == 450
    assert o_batch.chunk_geometry(300.0)[0] == 2250
    assert o_batch.chunk_geometry(3600.0)[0] == 27000
    assert o_batch.chunk_geometry(600.0)[0] == 4500
    # a partial token's worth of audio still needs a token (ceil): 0.1 s -> 0.75 -> 1; 60.1 s -> 450.75 -> 451
    assert o_batch.chunk_geometry(0.1)[0] == 1
    assert o_batch.chunk_geometry(60.1)[0] == 451


def test_max_new_tokens_rule_by_hand():
    # 32,768 within the nominal 60 minutes, scaled by d / 3600 below, rounded down
    assert o_batch.chunk_geometry(3600.0)[1] == 32768
    assert o_batch.chunk_geometry(5000.0)[1] == 32768
    assert o_batch.chunk_geometry(1800.0)[1] == 16384
    assert o_batch.chunk_geometry(300.0)[1] == 2730  # 32768 / 12 = 2730.67
    assert o_batch.chunk_geometry(60.0)[1] == 546    # 32768 / 60 = 546.13
    assert o_batch.chunk_geometry(450.0)[1] == 4096  # 32768 / 8, exact
    assert o_batch.chunk_geometry(0.01)[1] == 1      # never zero


def test_one_hour_in_300_s_chunks_is_one_batch_of_12():
    # BASELINE.json config 2: "12 sequences (one 60 min recording cut into 300 s chunks)", batch size 16
    seg = [(300.0 * i, 300.0 * (i + 1)) for i in range(12)]
    b = o_batch.form_batches(seg, o_chunk.greedy_chunks(seg, 300.0))
    assert len(b) == 1 and [e["slot"] for e in b[0]] == list(range(12))
    assert all(e["n_speech"] == 2250 and e["max_new"] == 2730 for e in b[0])


def test_17_chunks_give_16_plus_1():
    seg = [(100.0 * i, 100.0 * i + 90.0) for i in range(17)]
    chunks = [[i] for i in range(17)]
    b = o_batch.form_batches(seg, chunks)
    assert [len(x) for x in b] == [16, 1]
    assert b[1][0] == {"chunk": 16, "slot": 0, "n_speech": 675, "max_new": 819}  # 90 s: 675 tokens; 32768 / 40 = 819.2
    assert o_batch.form_batches(seg, []) == []


def test_duration_is_the_span_of_the_chunk():
    # G23: silence between the segments of a chunk is fed to the model: [0,10] + [50,60] is a 60 s chunk
    b = o_batch.form_batches([(0.0, 10.0), (50.0, 60.0)], [[0, 1]])
    assert b[0][0]["n_speech"] == 450 and b[0][0]["max_new"] == 546


def test_max_blocks():
    assert o_batch.max_blocks(64, 2250, 0, 1500, 64) == 60  # 3814 tokens / 64 = 59.6
    assert o_batch.max_blocks(64, 2250, 0, 1526, 64) == 60  # exactly 3840
    assert o_batch.max_blocks(64, 2250, 0, 1527, 64) == 61
    assert o_batch.max_blocks(0, 1, 0, 1, 16) == 1


@pytest.mark.parametrize("seed", range(10))
def test_partition_properties(seed):
    rng = np.random.default_rng(seed)
    n = int(rng.integers(0, 120))
    t, seg = 0.0, []
    for _ in range(n):
        t += float(rng.uniform(0, 5))
        d = float(rng.uniform(1, 400))
        seg.append((t, t + d))
        t += d
    chunks = o_chunk.greedy_chunks(seg, 300.0)
    B = int(rng.choice([1, 3, 16]))
    b = o_batch.form_batches(seg, chunks, batch_size=B)
    flat = [e["chunk"] for batch in b for e in batch]
    assert flat == list(range(len(chunks)))  # every chunk once, in time order
    assert all(len(batch) == B for batch in b[:-1]) and all(1 <= len(batch) <= B for batch in b)
    for batch in b:
        assert [e["slot"] for e in batch] == list(range(len(batch)))
        for e in batch:
            ch = chunks[e["chunk"]]
            d = seg[ch[-1]][1] - seg[ch[0]][0]
            assert 7.5 * d <= e["n_speech"] < 7.5 * d + 1  # smallest integer >= 7.5 d
            x = 32768 * d / 3600
            if d >= 3600:
                assert e["max_new"] == 32768
            elif x < 1:
                assert e["max_new"] == 1
            else:
                assert e["max_new"] <= x < e["max_new"] + 1  # largest integer <= 32768 d / 3600
