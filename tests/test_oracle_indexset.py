"""Pins of oracle/indexset.py (general index-set eviction with dense stable compaction).

The paper defines no such policy (PAPER.md:224 names it as future work), so these are pins against the
properties the definition must have and against the parts of the oracle that ARE pinned to the paper:
identity on the full set, equality with the positional policy's attention when the set is A(t) (Eq. 1),
a brute-force physical simulation on tiny cases, idempotence, stability, page conservation.
"""
import random

import numpy as np
import pytest

from oracle import attention as o_attn
from oracle import indexset as ix
from oracle import paged_cache as pc
from oracle import policy as pol


def _positional(N=40, p=4, P=2, S=10, M=1, t=6, policy=(4, 2, 1, 3, 1), L=2, H=2, evict=True):
    c = pc.OraclePagedCache(N, p, 4, 32)
    c.seq_begin(0, P, S, M, pol.Policy(*policy))
    c.append([0], [P + S + M + t])
    if evict:
        c.evict([0])
    return c, ix.OracleIndexedCache(c, L, H)


def _all(sets_fn, L, H):
    return [[sets_fn(l, h) for h in range(H)] for l in range(L)]


def test_identity_on_the_full_set_moves_nothing_and_frees_nothing():
    W = 0x7FFFFFFF
    c, ic = _positional(policy=(W, 0, 0, W, 0))
    n = c.seqs[0].length
    pages = c.live_pages(0)
    free0 = list(c.free_stack)
    moved = ic.evict_indexed(0, _all(lambda l, h: range(n), 2, 2))
    assert moved == 0
    assert ic.seqs[0].blocks == pages and c.free_stack == free0
    assert all(ic.positions(0, l, h) == list(range(n)) for l in range(2) for h in range(2))
    assert ic.seqs[0].next_pos == n and 0 not in c.seqs
    ic.check_invariants()


def test_set_equal_to_A_t_gives_the_positional_policys_attention():
    """With sel = A(t) for every (l, h), Eq. 1 over the slabs == Eq. 1 over the retained set (1e-12)."""
    rng = np.random.default_rng(3)
    c, ic = _positional(P=3, S=20, M=2, t=9, policy=(6, 3, 1, 4, 2), p=4, N=60, L=1, H=2)
    st = c.seqs[0]
    A = c.retained(0)
    n = st.length
    k = rng.integers(0, 2**16, size=(n, 2, 8), dtype=np.uint16) & np.uint16(0xBFFF)  # finite bf16 patterns
    v = rng.integers(0, 2**16, size=(n, 2, 8), dtype=np.uint16) & np.uint16(0xBFFF)
    q = rng.integers(0, 2**16, size=(6, 8), dtype=np.uint16) & np.uint16(0xBFFF)
    k &= np.uint16(0x3FFF | 0x8000)  # keep magnitudes small (exponent < 2^0 ..)
    q &= np.uint16(0x3FFF | 0x8000)
    o_ref, lse_ref, _ = o_attn.attend_retained(q, k, v, A, 0.3)
    ic.evict_indexed(0, [[A, A]])
    o, lse = ix.attend_indexed(q, k, v, [ic.positions(0, 0, h) for h in range(2)], 0.3)
    assert np.max(np.abs(o - o_ref)) < 1e-12 and np.max(np.abs(lse - lse_ref)) < 1e-12


def _brute_force_move(mem, old_addr, blocks_new, sel, p):
    """Physical simulation: mem[(page, l, h, slot)] = position stored there.  Gathers every selected row into a
    temporary, then writes slot s of slab (l, h); returns (new mem, rows whose address changed)."""
    tmp, moved = {}, 0
    for (l, h), xs in sel.items():
        for s, x in enumerate(xs):
            tmp[(l, h, s)] = mem[old_addr(l, h, x)]
    out = {}
    for (l, h, s), val in tmp.items():
        dst = (blocks_new[s // p], l, h, s % p)
        out[dst] = val
        src = old_addr(l, h, sel[(l, h)][s])
        if (src[0], src[3]) != (dst[0], dst[3]):
            moved += 1
    return out, moved


@pytest.mark.parametrize("seed", range(12))
def test_brute_force_physical_simulation_tiny(seed):
    rng = random.Random(seed)
    p = rng.choice([1, 2, 4])
    L, H = 2, 2
    P, S, M, t = rng.randint(0, 3), rng.randint(1, 9), rng.randint(0, 2), rng.randint(1, 8)
    policy = (rng.randint(1, 6), rng.randint(0, 4), rng.randint(0, 2), rng.randint(1, 5), rng.randint(0, 2))
    c, ic = _positional(N=64, p=p, P=P, S=S, M=M, t=t, policy=policy, L=L, H=H)
    st = c.seqs[0]
    resident = sorted(x for x in pol.resident_positions(P, S, M, st.t, st.pol) if x < st.length)
    live, pages = c.live_blocks(0), c.live_pages(0)
    mem = {(pages[live.index(x // p)], l, h, x % p): x for x in resident for l in range(L) for h in range(H)}
    sel = {(l, h): sorted(rng.sample(resident, rng.randint(1, len(resident)))) for l in range(L) for h in range(H)}
    moved = ic.evict_indexed(0, _all(lambda l, h: sel[(l, h)], L, H))
    q = ic.seqs[0]
    mem2, moved_bf = _brute_force_move(mem, lambda l, h, x: (pages[live.index(x // p)], l, h, x % p), q.blocks, sel, p)
    assert moved == moved_bf
    for (l, h), xs in sel.items():  # slot s of slab (l, h) holds the s-th smallest selected position
        assert [mem2[(q.blocks[s // p], l, h, s % p)] for s in range(len(xs))] == xs == ic.positions(0, l, h)
    assert len(q.blocks) == -(-max(len(x) for x in sel.values()) // p)
    assert q.blocks == pages[: len(q.blocks)] and c.free_stack[len(c.free_stack) - (len(pages) - len(q.blocks)):] == pages[len(q.blocks):]
    ic.check_invariants()
    # second eviction, from indexed mode: subsets of the slabs
    sel2 = {key: sorted(rng.sample(xs, rng.randint(1, len(xs)))) for key, xs in sel.items()}
    blocks_before = list(q.blocks)
    slot = {key: {x: s for s, x in enumerate(xs)} for key, xs in sel.items()}
    moved2 = ic.evict_indexed(0, _all(lambda l, h: sel2[(l, h)], L, H))
    q2 = ic.seqs[0]
    mem3, moved2_bf = _brute_force_move(
        mem2, lambda l, h, x: (blocks_before[slot[(l, h)][x] // p], l, h, slot[(l, h)][x] % p), q2.blocks, sel2, p)
    assert moved2 == moved2_bf
    for (l, h), xs in sel2.items():
        assert [mem3[(q2.blocks[s // p], l, h, s % p)] for s in range(len(xs))] == xs
    ic.check_invariants()


def test_idempotent_and_stable():
    c, ic = _positional()
    res = sorted(x for x in pol.resident_positions(2, 10, 1, 6, c.seqs[0].pol) if x < c.seqs[0].length)
    sel = _all(lambda l, h: res[l + h::2], 2, 2)
    ic.evict_indexed(0, sel)
    state = ([[ic.positions(0, l, h) for h in range(2)] for l in range(2)], list(ic.seqs[0].blocks), list(c.free_stack))
    assert ic.evict_indexed(0, sel) == 0  # same sets again: nothing moves, nothing is freed
    assert state == ([[ic.positions(0, l, h) for h in range(2)] for l in range(2)], list(ic.seqs[0].blocks), list(c.free_stack))
    for l in range(2):
        for h in range(2):
            xs = ic.positions(0, l, h)
            assert xs == sorted(xs) == list(sel[l][h])  # order of the original positions is preserved


def test_rejects_positions_that_are_not_held():
    c, ic = _positional(policy=(4, 2, 0, 3, 1))
    dead = sorted(pol.dead_positions(2, 10, 1, 6, c.seqs[0].pol))
    assert dead
    with pytest.raises(pc.BadState):
        ic.evict_indexed(0, _all(lambda l, h: [0, dead[0]], 2, 2))
    with pytest.raises(ValueError):
        ic.evict_indexed(0, _all(lambda l, h: [1, 0], 2, 2))  # not ascending
    ic.evict_indexed(0, _all(lambda l, h: [0, 1], 2, 2))
    with pytest.raises(pc.BadState):
        ic.evict_indexed(0, _all(lambda l, h: [0, 5], 2, 2))  # 5 is no longer in any slab


def test_append_positions_continue_and_pages_follow_the_longest_slab():
    c, ic = _positional(p=4, policy=(0x7FFFFFFF, 0, 0, 0x7FFFFFFF, 0))
    n = c.seqs[0].length  # 19
    ic.evict_indexed(0, [[[0, 1, 2], [0]], [[0, 1, 2, 3], [5, 7]]])  # longest slab: 4 rows -> 1 block
    assert len(ic.seqs[0].blocks) == 1
    top = c.free_stack[-1]
    ic.append_indexed([0])  # longest slab 4 -> 5 rows: a second block, popped from the top of the stack
    assert ic.seqs[0].blocks[1] == top and len(ic.seqs[0].blocks) == 2
    assert ic.positions(0, 0, 1) == [0, n] and ic.positions(0, 1, 0) == [0, 1, 2, 3, n]
    for k in range(3):
        ic.append_indexed([0])
    assert len(ic.seqs[0].blocks) == 2 and ic.positions(0, 0, 1) == [0, n, n + 1, n + 2, n + 3]
    ic.append_indexed([0])  # 8 -> 9 rows
    assert len(ic.seqs[0].blocks) == 3
    ic.check_invariants()


@pytest.mark.parametrize("seed", range(6))
def test_page_conservation_under_random_operations(seed):
    rng = random.Random(100 + seed)
    p = rng.choice([2, 4])
    c = pc.OraclePagedCache(48, p, 4, 32)
    ic = ix.OracleIndexedCache(c, 2, 2)
    for s in range(3):
        c.seq_begin(s, 2, 8, 0, pol.Policy(4, 2, 0, 3, 1))
        c.append([s], [10 + rng.randint(1, 6)])
        c.evict([s])
    for s in (0, 1):
        st = c.seqs[s]
        res = sorted(x for x in pol.resident_positions(st.P, st.S, st.M, st.t, st.pol) if x < st.length)
        ic.evict_indexed(s, _all(lambda l, h: sorted(rng.sample(res, rng.randint(1, len(res)))), 2, 2))
        ic.check_invariants()
    for _ in range(40):
        op = rng.random()
        s = rng.choice(list(ic.seqs))
        if op < 0.5:
            ic.append_indexed([s] if rng.random() < 0.5 else list(ic.seqs))
        elif op < 0.85:
            ic.evict_indexed(s, _all(lambda l, h: sorted(rng.sample(ic.positions(s, l, h), rng.randint(1, len(ic.positions(s, l, h))))), 2, 2))
        else:
            c.append([2], [1])
            c.evict([2])
        ic.check_invariants()
    for s in list(ic.seqs):
        ic.seq_end(s)
    c.seq_end(2)
    assert sorted(c.free_stack) == list(range(48))


def test_attend_indexed_closed_forms():
    one = np.uint16(0x3F80)  # bf16 1.0
    k = np.full((5, 2, 4), one, dtype=np.uint16)
    v = np.zeros((5, 2, 4), dtype=np.uint16)
    v[3, 0] = np.uint16(0x4000)  # 2.0
    v[1, 1] = np.uint16(0x4040)  # 3.0
    q = np.full((4, 4), one, dtype=np.uint16)
    o, lse = ix.attend_indexed(q, k, v, [[3], [1, 2]], 1.0)
    assert np.allclose(o[0], 2.0) and np.allclose(o[1], 2.0)        # one row: o = v
    assert np.allclose(o[2], 1.5) and np.allclose(o[3], 1.5)        # identical keys: o = mean of v
    assert np.allclose(lse[:2], 4.0) and np.allclose(lse[2:], 4.0 + np.log(2.0))


def test_mass_sets_cover_the_mass_and_contain_prompts_and_recent():
    rng = np.random.default_rng(7)
    P, S, M, n = 2, 30, 1, 40
    kf = rng.standard_normal((n, 2, 16)).astype(np.float32)
    qf = rng.standard_normal((6, 16)).astype(np.float32) * 2
    tob = lambda a: (a.view(np.uint32) >> np.uint32(16)).astype(np.uint16)
    k, q = tob(kf), tob(qf)
    resident = [x for x in range(n) if x not in (5, 6, 7)]
    sel = ix.select_mass_sets(q, k, resident, P, S, M, n, 0.5, 0.9, 3)
    for h in range(2):
        assert sel[h] == sorted(sel[h]) and set(sel[h]) <= set(resident)
        assert {0, 1, 32, 37, 38, 39} <= set(sel[h])  # both prompts and the 3 newest positions
        kk = o_attn.bf16_bits_to_f64(k[np.asarray(resident), h])
        for g in range(3):
            a = o_attn.softmax_weights((kk @ o_attn.bf16_bits_to_f64(q[h * 3 + g])) * 0.5)
            inside = sum(a[i] for i, x in enumerate(resident) if x in set(sel[h]))
            assert inside >= 0.9 - 1e-12  # every query head of the group keeps >= frac of its mass
    full = ix.select_mass_sets(q, k, resident, P, S, M, n, 0.5, 1.0, 0)
    assert all(s == resident for s in full)  # frac = 1 keeps everything (all weights > 0 here)
    # a dominant key: its mass set is that key alone
    k2 = k.copy()
    k2[11] = tob((qf[0] * 8).astype(np.float32))[None, :].repeat(2, axis=0)
    q2 = np.repeat(q[:1], 6, axis=0)
    dom = ix.select_mass_sets(q2, k2, resident, P, S, M, n, 1.0, 0.99, 0)
    assert dom[0] == [0, 1, 11, 32] and dom[1] == [0, 1, 11, 32]
