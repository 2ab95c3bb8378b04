"""Pins for oracle/paged_cache.py (no GPU): C2/C3 conventions, P4 (bulk == stepwise), P5 (worked
table through the allocator), P6 (conservation / injectivity), error behaviour."""
import random

import pytest

from oracle import policy
from oracle.paged_cache import BadState, OraclePagedCache, OutOfPages
from oracle.policy import Policy


def test_allocator_pops_ascending_and_is_lifo():
    c = OraclePagedCache(n_pages=8, page_size=4, max_seqs=4, max_blocks_per_seq=8)
    assert c.free_stack == [7, 6, 5, 4, 3, 2, 1, 0]
    c.seq_begin(0, 0, 0, 0, policy.NO_EVICTION)
    c.seq_begin(1, 0, 0, 0, policy.NO_EVICTION)
    pos = c.append([0, 1], [5, 4])  # seq 0 needs 2 blocks, seq 1 needs 1
    assert pos == [[0, 1, 2, 3, 4], [0, 1, 2, 3]]
    assert c.seqs[0].block_table == [0, 1] and c.seqs[1].block_table == [2]
    c.append([1, 0], [1, 3])  # call order matters: seq 1 first
    assert c.seqs[1].block_table == [2, 3] and c.seqs[0].block_table == [0, 1]
    c.append([0], [1])
    assert c.seqs[0].block_table == [0, 1, 4]
    c.seq_end(1)  # pushes 2 then 3 -> next pops return 3 then 2
    c.append([0], [8])
    assert c.seqs[0].block_table == [0, 1, 4, 3, 2]
    c.check_invariants()


def test_oom_is_all_or_nothing():
    c = OraclePagedCache(n_pages=3, page_size=2, max_seqs=2, max_blocks_per_seq=8)
    c.seq_begin(0, 0, 0, 0, policy.NO_EVICTION)
    c.seq_begin(1, 0, 0, 0, policy.NO_EVICTION)
    c.append([0], [3])
    before = (list(c.free_stack), list(c.seqs[0].block_table), c.seqs[0].length, c.seqs[1].length)
    with pytest.raises(OutOfPages):
        c.append([1, 0], [2, 2])  # needs 1 + 1 = 2 pages, 1 free
    assert before == (list(c.free_stack), list(c.seqs[0].block_table), c.seqs[0].length, c.seqs[1].length)
    c.append([1], [2])
    c.check_invariants()


def test_state_errors():
    c = OraclePagedCache(4, 2, 2, 2)
    with pytest.raises(BadState):
        c.append([0], [1])
    c.seq_begin(0, 0, 0, 0, policy.NO_EVICTION)
    with pytest.raises(BadState):
        c.seq_begin(0, 0, 0, 0, policy.NO_EVICTION)
    with pytest.raises(BadState):
        c.append([0, 0], [1, 1])
    with pytest.raises(BadState):
        c.append([0], [5])  # 3 blocks > max_blocks_per_seq
    with pytest.raises(BadState):
        c.seq_begin(7, 0, 0, 0, policy.NO_EVICTION)


def test_P5_worked_example_through_the_allocator(golden):
    pol = Policy(w_speech=4, delay=2, n_sink_speech=0, w_out=3, n_sink_out=1)
    c = OraclePagedCache(n_pages=6, page_size=4, max_seqs=1, max_blocks_per_seq=8)
    c.seq_begin(0, 2, 10, 0, pol)
    c.append([0], [12])
    for line in golden("worked_example_hybrid.txt"):
        t_s, _l, A_s, _ra, blocks_s = [x.strip() for x in line.split("|")]
        c.append([0], [1])
        c.evict([0])
        assert c.seqs[0].t == int(t_s)
        assert c.retained(0) == [int(x) for x in A_s.split()]
        assert c.live_blocks(0) == [int(x) for x in blocks_s.split()]
        c.check_invariants()
    # t = 8: block 1 (page 1) was freed and is on top of the stack
    assert c.free_stack[-1] == 1
    assert c.live_pages(0) == [0, 2, 3, 4]
    # runs: [0,1] in block 0 (k=0); [8..12] starts in block 2 (k=1); [17..19] in block 4 (k=3)
    assert c.runs(0) == [(0, 2, 0), (8, 5, 1), (17, 3, 3)]
    # evict is idempotent
    snap = (list(c.free_stack), list(c.seqs[0].block_table))
    c.evict([0])
    assert snap == (list(c.free_stack), list(c.seqs[0].block_table))


def _random_case(rng):
    p = rng.choice([1, 2, 4, 8])
    P, S, M = rng.randint(0, 6), rng.randint(0, 40), rng.randint(0, 3)
    pol = Policy(rng.randint(0, 20), rng.randint(0, 10), rng.randint(0, 3), rng.randint(0, 12), rng.randint(0, 3))
    return p, P, S, M, pol


def test_P4_bulk_append_then_evict_equals_stepwise_and_P6_invariants():
    rng = random.Random(1234)
    for _ in range(60):
        p, P, S, M, pol = _random_case(rng)
        T = rng.randint(1, 40)
        n_pages = -(-(P + S + M + T) // p) + 2
        a = OraclePagedCache(n_pages, p, 1, n_pages)
        b = OraclePagedCache(n_pages, p, 1, n_pages)
        a.seq_begin(0, P, S, M, pol)
        b.seq_begin(0, P, S, M, pol)
        a.append([0], [P + S + M])
        for _t in range(T):
            a.append([0], [1])
            a.evict([0])
            a.check_invariants()
            # every retained position is addressable (its block is live)
            for x in a.retained(0):
                a.slot_of(0, x)
        b.append([0], [P + S + M + T])
        b.evict([0])
        b.check_invariants()
        assert a.retained(0) == b.retained(0)
        assert a.live_blocks(0) == b.live_blocks(0)  # same live-block SET (page ids may differ)
        assert [r[:2] for r in a.runs(0)] == [r[:2] for r in b.runs(0)]
        # live blocks are exactly the blocks holding a resident position or a free slot
        st = a.seqs[0]
        R = policy.resident_positions(P, S, M, st.t, pol)
        want = sorted({x // p for x in R} | ({st.length // p} if st.length % p else set()))
        assert a.live_blocks(0) == want


def test_multi_sequence_evict_order_defines_free_stack():
    pol = Policy(2, 0, 0, 2, 0)
    c = OraclePagedCache(n_pages=16, page_size=2, max_seqs=2, max_blocks_per_seq=8)
    c.seq_begin(0, 0, 6, 0, pol)
    c.seq_begin(1, 0, 6, 0, pol)
    c.append([0, 1], [10, 10])  # seq0 pages 0..4, seq1 pages 5..9; t = 4, l = min(4, 4) = 4
    c.evict([1, 0])  # seq 1 first: frees its blocks 0,1 (speech r<4) and block 3 (out u<2)
    assert c.live_blocks(1) == [2, 4] and c.live_blocks(0) == [2, 4]
    assert c.free_stack[-6:] == [5, 6, 8, 0, 1, 3]
    c.check_invariants()
