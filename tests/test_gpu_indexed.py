"""Parity of the index-set eviction path (murmur_kv_evict_indexed / _append_indexed / _decode_attn_indexed /
murmur_select_mass_sets) against oracle/indexset.py on the same seeded inputs: slab position tables,
page lists and the free stack bit-exact, gathered rows bit-exact, bytes moved equal, attention within 2e-2 / 2e-3."""
import math
import random

import numpy as np
import pytest
import torch

import workloads
from oracle import attention as o_attn
from oracle import indexset as o_ix
from oracle import policy as o_policy
from workloads import Config, Geometry, seq_spec

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def dev():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return "cuda:0"


def _mk(cfg, dev, **kw):
    from harness import SideBySide

    return SideBySide(cfg, device=dev, **kw)


def _sets_to_device(sel, L, H, dev):
    cap = max(len(sel[l][h]) for l in range(L) for h in range(H))
    pos = torch.zeros(L, H, cap, dtype=torch.int32)
    cnt = torch.zeros(L, H, dtype=torch.int32)
    for l in range(L):
        for h in range(H):
            pos[l, h, : len(sel[l][h])] = torch.tensor(sel[l][h], dtype=torch.int32)
            cnt[l, h] = len(sel[l][h])
    return pos.to(dev), cnt.to(dev)


def _check_indexed(sbs, oix, i, q=None):
    """Slab tables, rows, pages and (optionally) attention of indexed sequence i against the oracle."""
    L, H = sbs.cfg.geom.n_layers, sbs.cfg.geom.n_kv_heads
    st = oix.seqs[i]
    kb, vb = sbs.kv_by_position(i)
    cap = st.max_len()
    gk, gv = sbs.gpu.gather_indexed(i, cap)
    gk, gv = workloads.to_bits(gk), workloads.to_bits(gv)
    for l in range(L):
        for h in range(H):
            want = oix.positions(i, l, h)
            assert sbs.gpu.indexed_positions(i, l, h).tolist() == want, f"positions of slab ({l}, {h})"
            assert np.array_equal(gk[l, h, : len(want)], kb[l][want, h]), f"K rows of slab ({l}, {h})"
            assert np.array_equal(gv[l, h, : len(want)], vb[l][want, h]), f"V rows of slab ({l}, {h})"
    assert sbs.gpu.free_stack().tolist() == sbs.oracle.free_stack
    assert sbs.gpu.stats()["free_pages"] == len(sbs.oracle.free_stack)
    assert sbs.gpu.last_error() == 0
    if q is not None:
        from paper_2606_01483_b200 import MURMUR_ATTN_AUTO, MURMUR_ATTN_GENERIC, MURMUR_ATTN_MMA
        from paper_2606_01483_b200.binding import MURMUR_OPT_ATTN_VARIANT

        qb = workloads.to_bits(q)
        refs = [o_ix.attend_indexed(qb[l, 0], kb[l], vb[l], [oix.positions(i, l, h) for h in range(H)], sbs.scale) for l in range(L)]
        # both kernels: tensor cores (streaming mma.sync kernel, pages of >= 16 rows) and the FFMA path
        for variant in (MURMUR_ATTN_MMA, MURMUR_ATTN_GENERIC):
            sbs.gpu.set_option(MURMUR_OPT_ATTN_VARIANT, variant)
            lse = torch.empty(L, 1, sbs.cfg.geom.n_q_heads, dtype=torch.float32, device=sbs.device)
            out = sbs.gpu.decode_attn_indexed([i], q, lse=lse, sm_scale=sbs.scale)
            got = out.float().cpu().numpy().astype(np.float64)
            errs = []
            for l in range(L):
                o_ref, lse_ref = refs[l]
                errs.append(np.abs(got[l, 0] - o_ref))
                assert np.max(np.abs(lse[l, 0].cpu().numpy() - lse_ref)) < 2e-3, variant
            e = np.stack(errs)
            assert np.isfinite(got).all() and e.max() <= 2e-2 and e.mean() <= 2e-3, (variant, e.max(), e.mean())
        sbs.gpu.set_option(MURMUR_OPT_ATTN_VARIANT, MURMUR_ATTN_AUTO)


@pytest.mark.parametrize("seed,page", [(0, 16), (1, 16), (2, 64), (3, 32)])
def test_random_index_sets_compaction_append_and_attention(dev, seed, page):
    rng = random.Random(300 + seed)
    L, H = 3, 4
    specs = [seq_spec(6, 90, 60, 40, 24, delay=8, n_sink_speech=1, n_sink_out=2), seq_spec(5, 70, 60, 32, 16, n_sink_out=1)]
    cfg = Config(f"idx{seed}", 120 + seed, Geometry(n_layers=L), page, tuple(specs))
    sbs = _mk(cfg, dev, extra_tokens=64)
    sbs.gpu.indexed_enable()
    oix = o_ix.OracleIndexedCache(sbs.oracle, L, H)
    sbs.bulk_prefill([0, 1], 30)
    sbs.check_integer_state([0, 1])
    st = sbs.oracle.seqs[0]
    resident = sorted(x for x in o_policy.resident_positions(st.P, st.S, st.M, st.t, st.pol) if x < st.length)
    # sequence 0 enters indexed mode with a random set per (layer, head); sequence 1 stays positional
    sel = [[sorted(rng.sample(resident, rng.randint(1, len(resident)))) for _ in range(H)] for _ in range(L)]
    sel[0][0] = list(resident)  # one slab keeps everything
    sel[L - 1][H - 1] = [resident[-1]]  # one slab keeps a single row
    pos_d, cnt_d = _sets_to_device(sel, L, H, dev)
    moved = sbs.gpu.kv_evict_indexed(0, pos_d, cnt_d)
    assert moved == 512 * oix.evict_indexed(0, sel)
    q = sbs.data[0].q_step(31).unsqueeze(1).contiguous()
    _check_indexed(sbs, oix, 0, q)
    from paper_2606_01483_b200 import MurmurError

    with pytest.raises(MurmurError) as e:  # positional calls are refused for an indexed sequence
        sbs.gpu.kv_evict([0])
    assert e.value.status == 2
    # appends (past a page boundary), interleaved with decode steps of the positional sequence on the same free stack
    for k in range(page + 3):
        u = 30 + k
        kn, vn = sbs.data[0].out_kv(u, u + 1)
        sbs._store(0, kn, vn)
        sbs.gpu.kv_append_indexed([0], kn.contiguous(), vn.contiguous())
        oix.append_indexed([0])
        if k % 5 == 0:
            sbs.fused_step([1])
            sbs.check_integer_state([1], check_free_stack=False)
        if k % 7 == 0 or k >= page:
            _check_indexed(sbs, oix, 0, sbs.data[0].q_step(u + 1).unsqueeze(1).contiguous())
    # a second eviction, from indexed mode: subsets of what the slabs hold now
    sel2 = [[sorted(rng.sample(oix.positions(0, l, h), rng.randint(1, len(oix.positions(0, l, h))))) for h in range(H)] for l in range(L)]
    pos_d, cnt_d = _sets_to_device(sel2, L, H, dev)
    moved = sbs.gpu.kv_evict_indexed(0, pos_d, cnt_d)
    assert moved == 512 * oix.evict_indexed(0, sel2)
    _check_indexed(sbs, oix, 0, q)
    assert sbs.gpu.kv_evict_indexed(0, pos_d, cnt_d) == 0  # idempotent: nothing moves, nothing is freed
    assert oix.evict_indexed(0, sel2) == 0
    _check_indexed(sbs, oix, 0)
    sbs.gpu.seq_end(0)
    oix.seq_end(0)
    assert sbs.gpu.free_stack().tolist() == sbs.oracle.free_stack
    sbs.check_integer_state([1])
    oix.check_invariants()
    sbs.close()


@pytest.mark.parametrize("page", [16, 64])
def test_long_ragged_slabs_attention(dev, page):
    """Slabs of very different lengths (1 row ... ~700 rows = 11 tiles of 64: the 4-stage ring of the streaming
    tensor-core kernel wraps several times, groups get odd and even tile counts, the last tile is partial), windows
    off so that everything is resident; then a few head-ragged appends across a tile boundary."""
    from workloads import WINDOW_OFF

    rng = random.Random(77 + page)
    L, H = 2, 4
    specs = [seq_spec(8, 650, 40, WINDOW_OFF, WINDOW_OFF)]
    cfg = Config(f"idxlong{page}", 140, Geometry(n_layers=L), page, tuple(specs))
    sbs = _mk(cfg, dev, extra_tokens=64)
    sbs.gpu.indexed_enable()
    oix = o_ix.OracleIndexedCache(sbs.oracle, L, H)
    sbs.bulk_prefill([0], 30)
    st = sbs.oracle.seqs[0]
    resident = sorted(x for x in o_policy.resident_positions(st.P, st.S, st.M, st.t, st.pol) if x < st.length)
    sizes = [len(resident), 1, 63, 64, 65, 191, 256, 449]
    sel = [[sorted(rng.sample(resident, sizes[(l * H + h) % len(sizes)])) for h in range(H)] for l in range(L)]
    pos_d, cnt_d = _sets_to_device(sel, L, H, dev)
    moved = sbs.gpu.kv_evict_indexed(0, pos_d, cnt_d)
    assert moved == 512 * oix.evict_indexed(0, sel)
    _check_indexed(sbs, oix, 0, sbs.data[0].q_step(31).unsqueeze(1).contiguous())
    for k in range(3):  # 63 -> 66, 64 -> 67, 191 -> 194, 256 -> 259 rows: across tile and page boundaries
        u = 30 + k
        kn, vn = sbs.data[0].out_kv(u, u + 1)
        sbs._store(0, kn, vn)
        sbs.gpu.kv_append_indexed([0], kn.contiguous(), vn.contiguous())
        oix.append_indexed([0])
        _check_indexed(sbs, oix, 0, sbs.data[0].q_step(u + 1).unsqueeze(1).contiguous())
    sbs.close()


def test_mass_sets_are_valid_and_drive_an_eviction(dev):
    """murmur_select_mass_sets: every query head keeps >= frac of its Eq. 1 mass inside its KV head's set (checked with the
    oracle's fp64 weights), prompts and the newest positions are in, the set sizes are those of the oracle up to the
    fp32-vs-fp64 boundary; the sets then drive an eviction whose attention matches Eq. 1 over exactly those sets."""
    L, H, G = 2, 4, 7
    W = workloads.WINDOW_OFF
    cfg = Config("idxmass", 130, Geometry(n_layers=L), 16, (seq_spec(8, 200, 40, W, W, M=2),), locality_rho=0.5)
    sbs = _mk(cfg, dev)
    sbs.gpu.indexed_enable()
    oix = o_ix.OracleIndexedCache(sbs.oracle, L, H)
    sbs.bulk_prefill([0], 30)
    st = sbs.oracle.seqs[0]
    n = st.length
    q = sbs.data[0].q_step(30)  # [L, n_q, d]
    frac, n_recent = 0.95, 4
    pos_d, cnt_d = sbs.gpu.select_mass_sets(0, q.contiguous(), frac, n_recent, cap=n, sm_scale=sbs.scale)
    assert sbs.gpu.last_error() == 0
    kb, _ = sbs.kv_by_position(0)
    qb = workloads.to_bits(q)
    sel = []
    for l in range(L):
        want = o_ix.select_mass_sets(qb[l], kb[l], range(n), st.P, st.S, st.M, n, sbs.scale, frac, n_recent)
        row = []
        for h in range(H):
            got = pos_d[l, h, : int(cnt_d[l, h])].cpu().tolist()
            assert got == sorted(set(got)) and 0 <= got[0] and got[-1] < n
            assert set(range(st.P)) <= set(got) and set(range(st.P + st.S, st.P + st.S + st.M)) <= set(got)
            assert set(range(n - n_recent, n)) <= set(got)
            assert abs(len(got) - len(want[h])) <= max(2, len(want[h]) // 50), (l, h, len(got), len(want[h]))
            kk = o_attn.bf16_bits_to_f64(kb[l][:, h])
            for g in range(G):
                a = o_attn.softmax_weights((kk @ o_attn.bf16_bits_to_f64(qb[l, h * G + g])) * sbs.scale)
                assert a[got].sum() >= frac - 2e-4, (l, h, g)
            row.append(got)
        sel.append(row)
    assert any(len(sel[l][h]) < n // 2 for l in range(L) for h in range(H)), "the locality-biased data should be sparse"
    sbs.evict([0])  # the live page list must be current before entering indexed mode
    moved = sbs.gpu.kv_evict_indexed(0, pos_d, cnt_d)
    assert moved == 512 * oix.evict_indexed(0, sel)
    _check_indexed(sbs, oix, 0, q.unsqueeze(1).contiguous())
    sbs.close()


def test_indexed_error_behaviour(dev):
    from paper_2606_01483_b200 import MurmurCache, MurmurError

    c = MurmurCache(2, 28, 4, 128, 16, max_seqs=2, max_blocks_per_seq=8, n_pages=10, device=dev)
    c.seq_begin(0, 4, 20, 0, (8, 4, 0, 8, 1))
    kv = torch.zeros(2, 40, 4, 128, dtype=torch.bfloat16, device=dev)
    c.kv_append([0], [40], kv, kv.clone())
    pos = torch.zeros(2, 4, 4, dtype=torch.int32, device=dev)
    pos[:, :, 1] = 1
    pos[:, :, 2] = 2
    cnt = torch.full((2, 4), 3, dtype=torch.int32, device=dev)
    with pytest.raises(MurmurError) as e:  # tables not enabled
        c.kv_evict_indexed(0, pos, cnt)
    assert e.value.status == 2
    c.indexed_enable()
    with pytest.raises(MurmurError) as e:  # appended since the last evict: the live page list is stale
        c.kv_evict_indexed(0, pos, cnt)
    assert e.value.status == 2
    c.kv_evict([0])
    bad = cnt.clone()
    bad[0, 0] = 0
    with pytest.raises(MurmurError) as e:  # an empty slab
        c.kv_evict_indexed(0, pos, bad)
    assert e.value.status == 1
    assert c.seq_state(0)["length"] == 40 and c.last_error() == 0
    c.kv_evict_indexed(0, pos, cnt)
    assert c.indexed_positions(0, 1, 3).tolist() == [0, 1, 2]
    assert len(c.free_stack()) == 10 - 1  # one block of 16 slots holds the 3 rows
    k1 = torch.zeros(2, 1, 4, 128, dtype=torch.bfloat16, device=dev)
    with pytest.raises(MurmurError) as e:
        c.kv_append([0], [1], k1, k1.clone())
    assert e.value.status == 2
    # bad sets are refused BEFORE anything moves: state, rows, pages and mode stay as they were
    before = [c.indexed_positions(0, l, h).tolist() for l in range(2) for h in range(4)]
    free_before = list(c.free_stack())
    pos2 = pos.clone()
    pos2[0, 0, 2] = 30  # position 30 is not held by slab (0, 0) any more
    pos3 = pos.clone()
    pos3[1, 2, 1], pos3[1, 2, 2] = 2, 1  # not ascending
    pos4 = pos.clone()
    pos4[1, 3, 1] = 0  # a repeated position
    for badpos in (pos2, pos3, pos4):
        with pytest.raises(MurmurError) as e:
            c.kv_evict_indexed(0, badpos, cnt)
        assert e.value.status == 1
        assert [c.indexed_positions(0, l, h).tolist() for l in range(2) for h in range(4)] == before
        assert list(c.free_stack()) == free_before and c.last_error() == 0
    two = torch.full((2, 4), 2, dtype=torch.int32, device=dev)
    c.kv_evict_indexed(0, pos, two)  # a good set still goes through afterwards
    assert c.indexed_positions(0, 0, 0).tolist() == [0, 1]
    assert c.last_error() == 0
    c.close()


def test_bad_index_set_on_a_positional_sequence_changes_nothing(dev):
    """The first murmur_kv_evict_indexed of a sequence (positional -> indexed): a set naming an evicted position or a
    position beyond the length is refused, the sequence stays positional and its rows are untouched."""
    from paper_2606_01483_b200 import MurmurCache, MurmurError

    c = MurmurCache(2, 28, 4, 128, 16, max_seqs=1, max_blocks_per_seq=8, n_pages=10, device=dev)
    c.seq_begin(0, 4, 60, 0, (16, 0, 0, 8, 1))  # speech window 16 of 60: whole blocks behind it are freed
    g = torch.Generator().manual_seed(11)
    kv = torch.randn(2, 100, 4, 128, generator=g).to(torch.bfloat16).to(dev)
    c.kv_append([0], [100], kv, kv.clone())
    c.kv_evict([0])
    retained = c.retained(0).tolist()
    pages_before, blocks_before = c.page_list(0)
    dead = next(x for x in range(100) if (x >> 4) not in set(int(b) for b in blocks_before))
    c.indexed_enable()
    good = torch.tensor(retained[:6], dtype=torch.int32)
    for badval in (dead, 100, -1):
        pos = good.repeat(2, 4, 1).contiguous()
        pos[1, 1, 5] = badval
        if badval == -1:
            pos[1, 1] = torch.tensor([-1] + retained[:5], dtype=torch.int32)
        cnt = torch.full((2, 4), 6, dtype=torch.int32, device=dev)
        with pytest.raises(MurmurError) as e:
            c.kv_evict_indexed(0, pos.to(dev), cnt)
        assert e.value.status == 1
    assert c.retained(0).tolist() == retained and c.last_error() == 0
    assert list(c.page_list(0)[0]) == list(pages_before)
    kg, vg = c.gather(0, retained, 0, 2)
    assert torch.equal(kg.cpu(), kv[:, retained].cpu())
    q = torch.randn(2, 1, 28, 128, generator=g).to(torch.bfloat16).to(dev)
    c.decode_attn([0], q)  # still a positional sequence
    c.close()
