"""Parity of the CUDA path (through the C ABI) against the oracle, on a real GPU.

Integer state (retained sets, compacted page tables, run descriptors, free stack) must be
bit-exact; attention within max-abs 2e-2 / mean-abs 2e-3 (BASELINE.json north_star).
Small and reduced-layer cases compare every element.  The full-size cases (configs 2, 3, 5 and all
15 points of config 4 at 28 layers, in the launch configuration bench.py times) compare all integer
state and, for the one-launch steps, EVERY (sequence, layer, head) of the output with the plain-C
fp64 oracle; the three-call steps before them compare sampled (sequence, layer) items.
"""
import math
import random

import numpy as np
import pytest
import torch

import workloads
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


def _variants(page_size):
    from paper_2606_01483_b200 import MURMUR_ATTN_GENERIC, MURMUR_ATTN_MMA

    return [MURMUR_ATTN_GENERIC] + ([MURMUR_ATTN_MMA] if page_size >= 16 else [])


# -------------------------------------------------------------------------------- config 1
@pytest.mark.parametrize("variant_idx", [0, 1])
def test_config1_every_step_every_head(dev, variant_idx):
    cfg = workloads.config1()
    variant = _variants(cfg.page_size)[variant_idx]
    sbs = _mk(cfg, dev, variant=variant)
    ids = [0]
    sbs.bulk_prefill(ids, 128)
    sbs.check_integer_state(ids)
    assert sbs.gpu.seq_state(0)["n_retained"] == 64 + 128 + 4 + 64
    for step in range(32):
        sbs.append_step(ids)
        sbs.evict(ids)
        sbs.check_integer_state(ids)
        q, out, lse = sbs.attend(ids, want_lse=True)
        sbs.check_attention(ids, q, out, lse)
        if step in (0, 15, 31):
            sbs.check_gather(0)
    assert sbs.t_of(0) == 160
    # evict is idempotent
    before = sbs.gpu.free_stack().tolist()
    sbs.gpu.kv_evict(ids)
    assert sbs.gpu.free_stack().tolist() == before
    sbs.check_integer_state(ids)
    sbs.close()


# -------------------------------------------------------------------------------- worked example
def test_worked_example_tiny_pages(dev, golden):
    """SURVEY 8(c) table through the GPU path with p = 4 (generic attention path)."""
    cfg = Config("worked", 9, Geometry(n_layers=2), 4,
                 (seq_spec(2, 10, 8, 4, 3, delay=2, n_sink_speech=0, n_sink_out=1),))
    sbs = _mk(cfg, dev, n_pages=6)
    sbs.bulk_prefill([0], 0, evict=False)
    for line in golden("worked_example_hybrid.txt"):
        t_s, _l, A_s, _ra, blocks_s = [x.strip() for x in line.split("|")]
        sbs.append_step([0])
        sbs.evict([0])
        assert sbs.gpu.seq_state(0)["t"] == int(t_s)
        assert sbs.gpu.retained(0).tolist() == [int(x) for x in A_s.split()]
        assert sbs.gpu.page_list(0)[1].tolist() == [int(x) for x in blocks_s.split()]
        sbs.check_integer_state([0])
        q, out, lse = sbs.attend([0], want_lse=True)
        sbs.check_attention([0], q, out, lse)
    assert sbs.gpu.free_stack().tolist()[-1] == 1
    assert sbs.gpu.runs(0) == [(0, 2, 0), (8, 5, 1), (17, 3, 3)]
    sbs.close()


# -------------------------------------------------------------------------------- random property cases
@pytest.mark.parametrize("seed", range(6))
def test_random_small_cases_stepwise(dev, seed):
    rng = random.Random(100 + seed)
    p = rng.choice([1, 2, 4, 8, 16, 32, 64])
    n_seqs = rng.randint(1, 4)
    seqs = []
    for _ in range(n_seqs):
        S = rng.randint(0, 150)
        seqs.append(seq_spec(rng.randint(0, 70), S, rng.randint(3, 40), rng.choice([0, 1, 7, 40, 64, 200]),
                             rng.choice([0, 1, 5, 33, 100]), M=rng.choice([0, 0, 3]),
                             delay=rng.choice([0, 1, 6, 20]), n_sink_speech=rng.choice([0, 0, 2, 9]),
                             n_sink_out=rng.choice([0, 1, 4])))
    cfg = Config(f"rand{seed}", 50 + seed, Geometry(n_layers=2), p, tuple(seqs))
    for variant in _variants(p):
        sbs = _mk(cfg, dev, variant=variant)
        ids = list(range(n_seqs))
        sbs.bulk_prefill(ids, 0, evict=False)
        active = list(ids)
        step = 0
        while active:
            sbs.append_step(active)
            order = active[::-1] if step % 2 else active  # call order defines the free-stack order
            sbs.evict(order)
            sbs.check_integer_state(active)
            # a sequence whose retained set is empty (P = 0, all windows 0) cannot be attended
            att = [i for i in active if len(sbs.oracle.retained(i)) > 0]
            if att:
                q, out, lse = sbs.attend(att, want_lse=True)
                sbs.check_attention(att, q, out, lse)
            for i in list(active):
                if sbs.t_of(i) >= cfg.seqs[i].T:
                    sbs.gpu.seq_end(i)
                    sbs.oracle.seq_end(i)
                    active.remove(i)
            step += 1
        assert sbs.gpu.free_stack().tolist() == sbs.oracle.free_stack
        assert len(sbs.oracle.free_stack) == sbs.oracle.N
        sbs.close()


# -------------------------------------------------------------------------------- config 2, reduced layers
def test_config2_two_layers_stepwise_around_delay_and_window_edges(dev):
    cfg = workloads.config2().with_layers(2).with_seqs(workloads.config2().seqs[:5])
    sbs = _mk(cfg, dev)
    ids = list(range(cfg.batch))
    sbs.bulk_prefill(ids, 250)
    sbs.check_integer_state(ids)
    for step in range(16):  # t = 251 .. 266 crosses d = 256 and k_o + w_o = 260
        sbs.append_step(ids)
        sbs.evict(ids)
        sbs.check_integer_state(ids)
        q, out, lse = sbs.attend(ids, want_lse=True)
        sbs.check_attention(ids, q, out, lse)
    assert sbs.gpu.seq_state(0)["n_retained"] == 836
    sbs.check_gather(2, layers=(0, 1))
    sbs.close()


def test_split_k_grid_invariance(dev):
    """Any partition of the tile list (1, 3, 37, 148, 1000 CTAs) gives the same answer within
    rounding, and each is within tolerance of the oracle (pins the cross-CTA LSE merge)."""
    from paper_2606_01483_b200 import MURMUR_ATTN_GENERIC, MURMUR_ATTN_MMA, MURMUR_OPT_ATTN_GRID, MURMUR_OPT_ATTN_VARIANT

    cfg = workloads.config2().with_layers(3).with_seqs(workloads.config2().seqs[:3])
    sbs = _mk(cfg, dev)
    ids = [0, 1, 2]
    sbs.bulk_prefill(ids, 300)
    sbs.append_step(ids)
    sbs.evict(ids)
    q = sbs.queries(ids)
    outs = []
    for grid in (1, 3, 37, 148, 1000):
        sbs.gpu.set_option(MURMUR_OPT_ATTN_GRID, grid)
        lse = torch.empty(q.shape[:3], dtype=torch.float32, device=dev)
        out = sbs.gpu.decode_attn(ids, q, lse=lse, sm_scale=sbs.scale)
        sbs.check_attention(ids, q, out, lse)
        outs.append(out.float())
    for o in outs[1:]:
        assert (o - outs[0]).abs().max().item() <= 2e-2
    sbs.gpu.set_option(MURMUR_OPT_ATTN_VARIANT, MURMUR_ATTN_GENERIC)
    out = sbs.gpu.decode_attn(ids, q, sm_scale=sbs.scale)
    assert (out.float() - outs[0]).abs().max().item() <= 2e-2
    sbs.gpu.set_option(MURMUR_OPT_ATTN_VARIANT, MURMUR_ATTN_MMA)
    sbs.close()


def test_l2_keep_fraction_does_not_change_results(dev):
    """MURMUR_OPT_L2_KEEP_PCT is a cache hint (which share of the K/V rows is read with L2::evict_last): automatic,
    0, 40 and 100 % give bit-identical outputs, for the attention call and for one-launch steps."""
    from paper_2606_01483_b200.binding import MURMUR_OPT_L2_KEEP_PCT

    cfg = workloads.config2().with_layers(3).with_seqs(workloads.config2().seqs[:3])
    ids = [0, 1, 2]
    outs = []
    for pct in (-1, 0, 40, 100):
        sbs = _mk(cfg, dev)
        sbs.gpu.set_option(MURMUR_OPT_L2_KEEP_PCT, pct)
        sbs.bulk_prefill(ids, 300)
        sbs.append_step(ids)
        sbs.evict(ids)
        q = sbs.queries(ids)
        lse = torch.empty(q.shape[:3], dtype=torch.float32, device=dev)
        out = sbs.gpu.decode_attn(ids, q, lse=lse, sm_scale=sbs.scale)
        if pct == -1:
            sbs.check_attention(ids, q, out, lse)
        steps = []
        for _ in range(3):
            qs, os_, _ = sbs.fused_step(ids, want_lse=True)
            steps.append(os_.clone())
        sbs.check_integer_state(ids)
        outs.append([out.clone()] + steps)
        sbs.close()
    for o in outs[1:]:
        for a, b in zip(o, outs[0]):
            assert torch.equal(a, b)
    from paper_2606_01483_b200 import MurmurError

    sbs = _mk(cfg, dev)
    with pytest.raises(MurmurError):
        sbs.gpu.set_option(MURMUR_OPT_L2_KEEP_PCT, 101)
    sbs.close()


def test_window_off_equals_full_attention(dev):
    """I1 on the GPU: windows >= lengths -> every position retained, nothing freed."""
    W = workloads.WINDOW_OFF
    cfg = Config("full", 7, Geometry(n_layers=2), 16, (seq_spec(64, 300, 40, W, W), seq_spec(10, 77, 40, W, W)))
    sbs = _mk(cfg, dev)
    ids = [0, 1]
    sbs.bulk_prefill(ids, 30)
    for _ in range(3):
        sbs.append_step(ids)
        sbs.evict(ids)
        sbs.check_integer_state(ids)
        for i in ids:
            assert sbs.gpu.retained(i).tolist() == list(range(sbs.oracle.seqs[i].length))
        q, out, lse = sbs.attend(ids, want_lse=True)
        sbs.check_attention(ids, q, out, lse)
    sbs.close()


def test_large_logits_sink_scale_16(dev):
    """P10: sink keys x16 (logits ~ +-60) stay finite in the fp32 softmax."""
    cfg = Config("sinks", 8, Geometry(n_layers=1), 64, (seq_spec(64, 200, 10, 64, 32),))
    sbs = _mk(cfg, dev)
    k, v = sbs.data[0].prefill_kv()
    k = k.clone()
    k[:, :4] = (k[:, :4].float() * 4.0).to(torch.bfloat16)  # x4 on top of the recipe's x4
    sbs.data[0]._prefill = (k, v)
    sbs.bulk_prefill([0], 5)
    q, out, lse = sbs.attend([0], want_lse=True)
    assert torch.isfinite(out.float()).all() and torch.isfinite(lse).all()
    sbs.check_attention([0], q, out, lse)
    sbs.close()


# -------------------------------------------------------------------------------- config 4 (sweep), reduced
@pytest.mark.parametrize("ws,wo", [(128, 64), (256, 1024), (1024, 256), (2250, 64), (2250, 1024)])
def test_config4_sweep_points_two_layers(dev, ws, wo):
    cfg = workloads.config4(ws, wo).with_layers(2).with_seqs(workloads.config4(ws, wo).seqs[:2])
    sbs = _mk(cfg, dev)
    ids = [0, 1]
    sbs.bulk_prefill(ids, 1100)
    for _ in range(2):
        sbs.append_step(ids)
        sbs.evict(ids)
        sbs.check_integer_state(ids)
        q, out, lse = sbs.attend(ids, want_lse=True)
        sbs.check_attention(ids, q, out, lse)
    want = 64 + min(ws, 2250) + 4 + min(wo, sbs.t_of(0) - 4)
    assert sbs.gpu.seq_state(0)["n_retained"] == want
    sbs.close()


# -------------------------------------------------------------------------------- config 4 (sweep), full size
_SWEEP_SHARED = {}


@pytest.mark.parametrize("ws,wo", workloads.config4_points())
def test_config4_all_sweep_points_full_size(dev, ws, wo):
    """Every point of the window sweep at 28 layers x 12 sequences: one step as three API calls and one
    one-launch step, each with bit-exact integer state and EVERY (sequence, layer, head) of the output
    compared with the fp64 oracle.  The seeded values are the same at every point (only the windows
    change), so the generators and the host copy of the bulk append are shared between the points."""
    cfg = workloads.config4(ws, wo)
    if "data" not in _SWEEP_SHARED:
        _SWEEP_SHARED["data"] = [workloads.SeqData(cfg, i, device=dev) for i in range(cfg.batch)]
        _SWEEP_SHARED["bulk"] = {}
    sbs = _mk(cfg, dev, use_c_oracle=True, data=_SWEEP_SHARED["data"], bulk_bits=_SWEEP_SHARED["bulk"])
    ids = list(range(cfg.batch))
    sbs.bulk_prefill(ids, 1100)
    sbs.check_integer_state(ids)
    sbs.append_step(ids)
    sbs.evict(ids)
    sbs.check_integer_state(ids)
    q, out, lse = sbs.attend(ids, want_lse=True)
    sbs.check_attention(ids, q, out, lse)
    n0 = sbs.gpu.stats()["kernel_launches"]
    q, out, lse = sbs.fused_step(ids, want_lse=True)
    assert sbs.gpu.stats()["kernel_launches"] == n0 + 1
    sbs.check_integer_state(ids)
    sbs.check_attention(ids, q, out, lse)
    want = 64 + min(ws, 2250) + 4 + min(wo, sbs.t_of(0) - 4)
    assert all(sbs.gpu.seq_state(i)["n_retained"] == want for i in ids)
    sbs.close()


# -------------------------------------------------------------------------------- config 5 (ragged), reduced
def test_config5_ragged_two_layers_sequences_finish_at_different_steps(dev):
    full = workloads.config5()
    cfg = full.with_layers(2)
    sbs = _mk(cfg, dev)
    ids = list(range(cfg.batch))
    # every sequence starts 1..12 tokens before its own end so that they leave the batch one by one
    rng = random.Random(5)
    left = {i: rng.randint(1, 12) for i in ids}
    for i in ids:  # per-sequence bulk prefill (different t0), evicted straight away
        sbs.bulk_prefill([i], cfg.seqs[i].T - left[i])
    sbs.check_integer_state(ids)
    active = list(ids)
    while active:
        sbs.append_step(active)
        sbs.evict(active)
        sbs.check_integer_state(active)
        q, out, lse = sbs.attend(active, want_lse=True)
        sbs.check_attention(active, q, out, lse)
        for i in list(active):
            if sbs.t_of(i) >= cfg.seqs[i].T:
                sbs.gpu.seq_end(i)
                sbs.oracle.seq_end(i)
                active.remove(i)
        assert sbs.gpu.free_stack().tolist() == sbs.oracle.free_stack
    assert len(sbs.oracle.free_stack) == sbs.oracle.N
    sbs.close()


# -------------------------------------------------------------------------------- full-size, sampled
def _full_size_steps(sbs, ids, n_steps, sample_layers, seq_subset):
    """Full-size steps in the launch configuration bench.py times: first as three API calls (sampled
    items compared), then the same number of steps through murmur_decode_step (one launch per step),
    of which EVERY (sequence, layer, head) is compared with the fp64 oracle."""
    for _ in range(n_steps):
        sbs.append_step(ids)
        sbs.evict(ids)
        sbs.check_integer_state(ids)
        q, out, lse = sbs.attend(ids, want_lse=True)
        assert torch.isfinite(out.float()).all()
        sbs.check_attention(ids, q, out, lse, layers=sample_layers, seq_subset=seq_subset)
    launches0 = sbs.gpu.stats()["kernel_launches"]
    for k in range(n_steps):
        q, out, lse = sbs.fused_step(ids, want_lse=True)
        if k == 0:
            assert sbs.gpu.stats()["kernel_launches"] == launches0 + 1, "murmur_decode_step must be ONE launch"
        sbs.check_integer_state(ids)
        assert torch.isfinite(out.float()).all()
        sbs.check_attention(ids, q, out, lse)  # full tensor: all sequences, layers and heads


def test_config2_full_size_28_layers_full_tensor(dev):
    cfg = workloads.config2()
    sbs = _mk(cfg, dev, use_c_oracle=True)
    ids = list(range(12))
    sbs.bulk_prefill(ids, 300)
    sbs.check_integer_state(ids)
    _full_size_steps(sbs, ids, 3, sample_layers=[0, 13, 27], seq_subset=[0, 5, 11])
    assert sbs.gpu.stats()["attn_grid"] == sbs.gpu.stats()["sm_count"]
    sbs.close()


@pytest.mark.parametrize("evicted", [False, True])
def test_config3_full_size_28_layers_full_tensor(dev, evicted):
    cfg = workloads.config3(evicted)
    sbs = _mk(cfg, dev, use_c_oracle=True)
    sbs.bulk_prefill([0], 1030)  # past d = 1024 and k_o + w_o = 516
    sbs.check_integer_state([0])
    _full_size_steps(sbs, [0], 3, sample_layers=[0, 27], seq_subset=[0])
    want = (64 + 27000 + sbs.t_of(0)) if not evicted else (64 + 2048 + 4 + 512)
    assert sbs.gpu.seq_state(0)["n_retained"] == want
    sbs.close()


def test_config5_full_size_28_layers_full_tensor(dev):
    cfg = workloads.config5()
    sbs = _mk(cfg, dev, use_c_oracle=True, extra_tokens=8)
    ids = list(range(32))
    for i in ids:
        sbs.bulk_prefill([i], min(cfg.seqs[i].T - 2, 1200))
    sbs.check_integer_state(ids)
    _full_size_steps(sbs, ids, 3, sample_layers=[5, 27], seq_subset=[0, 9, 31])
    sbs.close()


# -------------------------------------------------------------------------------- host-buffer entry
@pytest.mark.parametrize("mode", ["pinned_zero_copy", "pinned_packed_staged", "pinned_staged", "pageable"])
def test_decode_step_host_matches_device_calls(dev, mode):
    """murmur_decode_step_host from page-locked buffers in place (zero-copy: the kernel reads q / k_new / v_new and
    writes out through the buffers' device-mapped addresses), from page-locked buffers with zero-copy switched
    off (staged; packed back to back = one copy), and from pageable buffers (always staged)."""
    from paper_2606_01483_b200 import binding

    cfg = workloads.config1().with_layers(3)
    a = _mk(cfg, dev)
    if mode in ("pinned_packed_staged", "pinned_staged"):
        a.gpu.set_option(binding.MURMUR_OPT_HOST_ZERO_COPY, 0)
    a.bulk_prefill([0], 100)
    for _ in range(4):
        u = a.t_of(0)
        k, v = a.data[0].out_kv(u, u + 1)
        q = a.data[0].q_step(u + 1).unsqueeze(1).contiguous()
        if mode == "pinned_packed_staged":  # packed back to back in one pinned block: a single host-to-device copy
            hb = torch.empty(2 * k.numel() + q.numel(), dtype=torch.bfloat16).pin_memory()
            hb[: k.numel()] = k.reshape(-1).cpu()
            hb[k.numel(): 2 * k.numel()] = v.reshape(-1).cpu()
            hb[2 * k.numel():] = q.reshape(-1).cpu()
            kh, vh, qh = hb[: k.numel()].view(k.shape), hb[k.numel(): 2 * k.numel()].view(v.shape), hb[2 * k.numel():].view(q.shape)
            oh = torch.empty(q.shape, dtype=torch.bfloat16).pin_memory()
        elif mode == "pageable":
            kh, vh, qh = k.cpu(), v.cpu(), q.cpu()
            oh = torch.empty(q.shape, dtype=torch.bfloat16)
        else:
            kh, vh, qh = k.cpu().pin_memory(), v.cpu().pin_memory(), q.cpu().pin_memory()
            oh = torch.empty(q.shape, dtype=torch.bfloat16).pin_memory()
        n0 = a.gpu.stats()["host_zero_copy_steps"]
        a.gpu.decode_step_host([0], kh, vh, qh, oh)
        torch.cuda.synchronize()
        assert a.gpu.stats()["host_zero_copy_steps"] - n0 == (1 if mode == "pinned_zero_copy" else 0)
        a._store(0, k, v)
        a.oracle.append([0], [1])
        a.oracle.evict([0])
        a.check_integer_state([0])
        a.check_attention([0], q, oh.to(dev))
        a.check_gather(0, layers=None)  # the rows the kernel scattered from the host buffer
    a.close()


# -------------------------------------------------------------------------------- fused step / PDL
@pytest.mark.parametrize("pdl,fuse", [(1, 2), (0, 2), (1, 1), (0, 1), (1, 0), (0, 0)])
def test_decode_step_fused_prologue_ragged_every_step(dev, pdl, fuse):
    """murmur_decode_step (fuse 2: the whole step in one launch; 1: append+evict in one launch, then
    attention; 0: three launches; each with / without programmatic dependent launch) on a
    ragged page-16 batch whose windows start sliding and whose sequences finish at different steps:
    integer state bit-exact after every step, attention within tolerance, for every option mix."""
    from paper_2606_01483_b200 import MURMUR_OPT_FUSE_STEP, MURMUR_OPT_PDL

    base = workloads.config5()
    specs = [workloads.seq_spec(8, 70 + 9 * i, 40 + 7 * i, 32 if i % 2 else 48, 16 if i % 3 else 32, n_sink_out=2 + i % 3)
             for i in range(5)]
    cfg = base.with_seqs(specs).with_layers(2)
    a = _mk(cfg, dev)
    a.gpu.set_option(MURMUR_OPT_PDL, pdl)
    a.gpu.set_option(MURMUR_OPT_FUSE_STEP, fuse)
    active = list(range(cfg.batch))
    a.bulk_prefill(active, 1)
    a.check_integer_state(active)
    step = 0
    while active:
        q, out, lse = a.fused_step(active, want_lse=True)
        a.check_integer_state(active)
        a.check_attention(active, q, out, lse)
        done = [i for i in active if a.t_of(i) >= cfg.seqs[i].T]
        for i in done:
            a.gpu.seq_end(i)
            a.oracle.seq_end(i)
        active = [i for i in active if i not in done]
        step += 1
    assert step == max(s.T for s in specs) - 1
    assert list(a.gpu.free_stack()) == a.oracle.free_stack
    a.close()


@pytest.mark.parametrize("seed", range(8))
def test_decode_step_one_launch_random_policies(dev, seed):
    """The one-launch step on random small cases: page 16/32/64, windows 0 / tiny / larger than the
    sequence, speech sinks, a second prompt, output window 0 (the new token is appended but not
    attended), sequences that start without an evict (tile table missing -> generated in the kernel),
    new pages popped in the same step in which others are freed, reversed call order."""
    rng = random.Random(900 + seed)
    p = rng.choice([16, 32, 64])
    n_seqs = rng.randint(1, 5)
    seqs = []
    for _ in range(n_seqs):
        seqs.append(seq_spec(rng.randint(1, 70), rng.randint(0, 200), rng.randint(3, 70), rng.choice([0, 1, 7, 40, 64, 300]),
                             rng.choice([0, 1, 5, 33, 100]), M=rng.choice([0, 0, 3]),
                             delay=rng.choice([0, 1, 6, 20]), n_sink_speech=rng.choice([0, 0, 2, 9]),
                             n_sink_out=rng.choice([0, 1, 4])))
    cfg = Config(f"randstep{seed}", 70 + seed, Geometry(n_layers=2), p, tuple(seqs))
    sbs = _mk(cfg, dev)
    ids = list(range(n_seqs))
    sbs.bulk_prefill(ids, 0, evict=bool(seed % 2))
    active = list(ids)
    step = 0
    while active:
        order = active[::-1] if step % 2 else list(active)
        q, out, lse = sbs.fused_step(order, want_lse=True)
        sbs.check_integer_state(active)
        sbs.check_attention(order, q, out, lse)
        for i in list(active):
            if sbs.t_of(i) >= cfg.seqs[i].T:
                sbs.gpu.seq_end(i)
                sbs.oracle.seq_end(i)
                active.remove(i)
        step += 1
    assert sbs.gpu.free_stack().tolist() == sbs.oracle.free_stack
    assert len(sbs.oracle.free_stack) == sbs.oracle.N
    sbs.close()


@pytest.mark.parametrize("n_seqs,one_launch", [(33, True), (64, True), (70, False)])
def test_decode_step_many_sequences(dev, n_seqs, one_launch):
    """Up to 64 sequences the whole step is ONE launch (the step kernel's per-sequence tables hold 64); beyond that
    murmur_decode_step takes the two-launch form and the attention call is split in chunks; results are the same.
    Ragged windows, so that the new-block prefix sums and the free stack see work in both halves of the list."""
    specs = [seq_spec(4, 20 + (i % 7), 8, 16, 8 + (i % 3), n_sink_out=1 + (i % 2)) for i in range(n_seqs)]
    cfg = Config("many", 90, Geometry(n_layers=2), 16, tuple(specs))
    sbs = _mk(cfg, dev)
    ids = list(range(n_seqs))
    sbs.bulk_prefill(ids, 1)
    for k in range(6):
        order = ids[::-1] if k % 2 else ids
        n0 = sbs.gpu.stats()["kernel_launches"]
        q, out, lse = sbs.fused_step(order, want_lse=True)
        assert (sbs.gpu.stats()["kernel_launches"] - n0 == 1) == one_launch
        sbs.check_integer_state(ids)
        sbs.check_attention(order, q, out, lse)
    sbs.close()


def test_decode_step_back_to_back_without_host_sync(dev):
    """200 fused steps enqueued back to back (PDL chain: each launch's set-up overlaps its predecessor)
    with no host synchronisation in between.  Afterwards the final integer state is checked, and the
    outputs of eight sampled steps (first, around the window edges t = 256 / 260, middle, last) are
    compared with the oracle over the retained sets recorded at those steps (a missing
    griddepcontrol.wait would corrupt tables or outputs)."""
    cfg = workloads.config2().with_layers(2)
    a = _mk(cfg, dev)
    ids = list(range(cfg.batch))
    a.bulk_prefill(ids, 250)
    sampled = {0, 1, 5, 6, 9, 10, 100, 199}  # steps 5 / 9 are t = 256 (= d) and t = 260 (= k_o + w_o)
    outs, rets = {}, {}
    for k in range(200):
        q, out, lse = a.fused_step(ids, want_lse=True)
        if k in sampled:
            outs[k] = (q, out, lse)
            rets[k] = {i: list(a.oracle.retained(i)) for i in ids}
    torch.cuda.synchronize()
    a.check_integer_state(ids)
    for k in sorted(sampled):
        q, out, lse = outs[k]
        a.check_attention(ids, q, out, lse, retained=rets[k])
    a.close()


def test_chained_steps_with_more_ctas_than_sms(dev):
    """Chained step launches whose grid exceeds one wave (MURMUR_OPT_ATTN_GRID = 1000): a second-wave CTA starts
    after first-wave keepers of its OWN launch have already added to the go-ahead counter, so it must accept
    "counter >= expected", not only equality - otherwise it spins out the whole time-out (0.3 - 3 ms) on every step
    with the step's commit stalled behind it.  Results must match the oracle, and the chained steps may not be
    slower than a small multiple of the same steps launched without programmatic dependent launch (no chain)."""
    from paper_2606_01483_b200 import MURMUR_OPT_ATTN_GRID, MURMUR_OPT_PDL

    cfg = workloads.config2().with_layers(2)
    a = _mk(cfg, dev)
    ids = list(range(cfg.batch))
    a.bulk_prefill(ids, 250)
    a.gpu.set_option(MURMUR_OPT_ATTN_GRID, 1000)
    keep = []
    for k in range(12):  # back to back, no host sync: steps 1.. are chained
        keep.append(a.fused_step(ids, want_lse=True) + ({i: list(a.oracle.retained(i)) for i in ids},))
    torch.cuda.synchronize()
    a.check_integer_state(ids)
    for q, out, lse, ret in keep[-3:]:
        a.check_attention(ids, q, out, lse, retained=ret)
    # timing: the same device inputs every step, GPU side only (the oracle is not advanced from here on)
    q, out, _lse, _ = keep[-1]
    k_new = torch.randn(2, len(ids), 4, 128, device=dev).to(torch.bfloat16)
    v_new = torch.randn(2, len(ids), 4, 128, device=dev).to(torch.bfloat16)
    times = {}
    for pdl in (1, 0, 1, 0):
        a.gpu.set_option(MURMUR_OPT_PDL, pdl)
        for _ in range(3):
            a.gpu.decode_step(ids, k_new, v_new, q, out, None, a.scale)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(30):
            a.gpu.decode_step(ids, k_new, v_new, q, out, None, a.scale)
        e1.record()
        torch.cuda.synchronize()
        times[pdl] = min(times.get(pdl, 1e9), e0.elapsed_time(e1) / 30)
    assert a.gpu.last_error() == 0
    assert times[1] < 3.0 * times[0] + 0.02, f"chained {times[1] * 1e3:.1f} us/step vs unchained {times[0] * 1e3:.1f} us/step"
    a.close()


def test_decode_step_soak_small_pages_many_allocations(dev):
    """600 one-launch steps enqueued without host synchronisation on a page-16 cache with small
    windows: every sequence allocates a page every 16 steps while others are freed in the same launch
    (the free stack is reused continuously).  Integer state and outputs are checked at three points."""
    specs = [seq_spec(5 + i, 90 + 11 * i, 700, 64, 48, delay=10 + i, n_sink_speech=i % 2, n_sink_out=3) for i in range(6)]
    cfg = Config("soak", 97, Geometry(n_layers=3), 16, tuple(specs))
    sbs = _mk(cfg, dev, n_pages=6 * 16 + 40)  # far fewer pages than an un-evicted run needs: reuse is mandatory
    ids = list(range(6))
    sbs.bulk_prefill(ids, 1)
    for k in range(600):
        order = ids[::-1] if k % 3 == 0 else ids
        q, out, lse = sbs.fused_step(order, want_lse=True)
        if k in (199, 399, 599):
            sbs.check_integer_state(ids)
            sbs.check_attention(order, q, out, lse)
    assert sbs.gpu.last_error() == 0
    sbs.close()



# -------------------------------------------------------------------------------- per-layer engine mode
def _ragged16_specs_with_w_out_0():
    """Ragged page-16 batch; the last sequence has w_out = 0: its newest token is dead as soon as it is
    appended, so the step that completes a block frees the very block the token was written to."""
    specs = [seq_spec(8, 70 + 9 * i, 40 + 7 * i, 32 if i % 2 else 48, 16 if i % 3 else 32, n_sink_out=2 + i % 3)
             for i in range(4)]
    specs.append(seq_spec(5, 60, 45, 32, 0, n_sink_out=1))
    return specs


def test_per_layer_mode_append_write_only_layers(dev):
    """The reserve-once / write-per-layer append (murmur_kv_append with layer_begin > 0) as an engine
    issues it - append(0), evict, attn(0), then append(l), attn(l) for every further layer - on a ragged
    page-16 batch over more than two pages of tokens: integer state bit-exact after every step, the rows
    of ALL layers gathered back bit-exact (a row written to the wrong page shows up here), attention of
    every layer within tolerance.  Includes a w_out = 0 sequence (the evict after layer 0 frees the block
    the newest token lives in; the later layers' rows for it are dropped, not an error)."""
    specs = _ragged16_specs_with_w_out_0()
    cfg = workloads.config5().with_seqs(specs).with_layers(3)
    a = _mk(cfg, dev)
    active = list(range(cfg.batch))
    a.bulk_prefill(active, 1)
    a.check_integer_state(active)
    step = 0
    while active:
        order = active[::-1] if step % 2 else list(active)
        q, out, lse = a.per_layer_step(order, want_lse=True)
        a.check_integer_state(active)
        a.check_attention(order, q, out, lse)
        if step % 5 == 0 or any((a.oracle.seqs[i].length % 16) in (0, 1) for i in active):
            for i in active:
                a.check_gather(i, layers=None)
        done = [i for i in active if a.t_of(i) >= cfg.seqs[i].T]
        for i in done:
            a.gpu.seq_end(i)
            a.oracle.seq_end(i)
        active = [i for i in active if i not in done]
        step += 1
    assert step == max(s.T for s in specs) - 1 and step > 2 * 16
    assert list(a.gpu.free_stack()) == a.oracle.free_stack
    assert a.gpu.last_error() == 0
    a.close()


def test_decode_step_layers_one_launch_per_layer_range(dev):
    """murmur_decode_step_layers: the step issued in layer ranges, ONE launch per call - the opening call
    (layers [0, 1)) reserves, commits and evicts, the others (issued out of order here) only write their
    rows and attend.  Ragged page-16 batch with a w_out = 0 sequence, run past two pages of tokens; integer
    state bit-exact, rows of all layers gathered back bit-exact, attention of every layer in tolerance."""
    specs = _ragged16_specs_with_w_out_0()
    cfg = workloads.config5().with_seqs(specs).with_layers(4)
    a = _mk(cfg, dev)
    active = list(range(cfg.batch))
    a.bulk_prefill(active, 1)
    step = 0
    while active:
        order = active[::-1] if step % 2 else list(active)
        n0 = a.gpu.stats()["kernel_launches"]
        ranges = [(0, 1), (2, 4), (1, 2)] if step % 2 else [(0, 2), (2, 3), (3, 4)]
        q, out, lse = a.layer_range_step(order, ranges, want_lse=True)
        assert a.gpu.stats()["kernel_launches"] == n0 + 3, "one launch per layer range"
        a.check_integer_state(active)
        a.check_attention(order, q, out, lse)
        if step % 5 == 0 or any((a.oracle.seqs[i].length % 16) in (0, 1) for i in active):
            for i in active:
                a.check_gather(i, layers=None)
        done = [i for i in active if a.t_of(i) >= cfg.seqs[i].T]
        for i in done:
            a.gpu.seq_end(i)
            a.oracle.seq_end(i)
        active = [i for i in active if i not in done]
        step += 1
    assert step > 2 * 16
    assert list(a.gpu.free_stack()) == a.oracle.free_stack
    assert a.gpu.last_error() == 0
    a.close()


def test_decode_step_layers_rejects_a_range_of_an_unopened_step(dev):
    from paper_2606_01483_b200 import MurmurCache, MurmurError

    c = MurmurCache(3, 28, 4, 128, 16, max_seqs=2, max_blocks_per_seq=8, n_pages=8, device=dev)
    c.seq_begin(0, 4, 20, 0, (8, 4, 0, 8, 1))
    kv = torch.zeros(3, 30, 4, 128, dtype=torch.bfloat16, device=dev)
    c.kv_append([0], [30], kv, kv.clone())  # appended, not evicted: no step is open
    k1 = torch.zeros(1, 1, 4, 128, dtype=torch.bfloat16, device=dev)
    q1 = torch.zeros(1, 1, 28, 128, dtype=torch.bfloat16, device=dev)
    with pytest.raises(MurmurError) as e:
        c.decode_step_layers([0], k1, k1.clone(), q1, torch.empty_like(q1), 1, 2)
    assert e.value.status == 2
    assert c.seq_state(0)["length"] == 30
    c.decode_step_layers([0], k1, k1.clone(), q1, torch.empty_like(q1), 0, 1)  # opens the step
    assert c.seq_state(0)["length"] == 31
    c.decode_step_layers([0], k1, k1.clone(), q1, torch.empty_like(q1), 2, 3)
    assert c.seq_state(0)["length"] == 31 and c.last_error() == 0

    def refused(lb, le):
        n = le - lb
        k, q = k1.expand(n, 1, 4, 128).contiguous(), q1.expand(n, 1, 28, 128).contiguous()
        with pytest.raises(MurmurError) as e:
            c.decode_step_layers([0], k, k.clone(), q, torch.empty_like(q), lb, le)
        assert e.value.status == 2
        assert c.seq_state(0)["length"] == 31

    refused(2, 3)  # layer 2 was already issued in this step: a second write would overwrite the token's rows
    refused(1, 3)  # ... also as part of a larger range
    c.decode_step_layers([0], k1, k1.clone(), q1, torch.empty_like(q1), 1, 2)  # the last open layer: the step closes
    refused(1, 2)  # every layer issued: no step is open any more
    # a plain append + evict leaves evict_len == len as an opening call would, but opens no step
    c.kv_append([0], [1], kv[:, :1].contiguous(), kv[:, :1].contiguous())
    c.kv_evict([0])
    with pytest.raises(MurmurError) as e:
        c.decode_step_layers([0], k1, k1.clone(), q1, torch.empty_like(q1), 1, 2)
    assert e.value.status == 2 and c.seq_state(0)["length"] == 32 and c.last_error() == 0
    c.close()


@pytest.mark.parametrize("mode", ["one_launch", "two_launches", "three_calls", "per_layer", "layer_calls"])
def test_evict_unmaps_the_block_of_the_newest_token(dev, mode):
    """w_out = 0 with page 16: at every step whose token completes a block of dead outputs, the same
    step's eviction frees the block that token was just written to.  Every form of the step must leave
    identical integer state (the page goes back on the stack in the same step) and attend without it."""
    from paper_2606_01483_b200 import MURMUR_OPT_FUSE_STEP

    specs = [seq_spec(5, 60, 50, 32, 0, n_sink_out=1), seq_spec(3, 29, 50, 16, 0, n_sink_out=0, delay=4),
             seq_spec(16, 48, 50, 64, 8, n_sink_out=2)]
    cfg = Config("unmap", 91, Geometry(n_layers=2), 16, tuple(specs))
    a = _mk(cfg, dev)
    if mode == "two_launches":
        a.gpu.set_option(MURMUR_OPT_FUSE_STEP, 1)
    ids = [0, 1, 2]
    a.bulk_prefill(ids, 1)
    freed_same_step = 0
    for step in range(48):
        n_free0 = len(a.oracle.free_stack)
        if mode in ("one_launch", "two_launches"):
            q, out, lse = a.fused_step(ids, want_lse=True)
        elif mode == "per_layer":
            q, out, lse = a.per_layer_step(ids, want_lse=True)
        elif mode == "layer_calls":
            q, out, lse = a.layer_range_step(ids, [(0, 1), (1, 2)], want_lse=True)
        else:
            a.append_step(ids)
            a.evict(ids)
            q, out, lse = a.attend(ids, want_lse=True)
        a.check_integer_state(ids)
        a.check_attention(ids, q, out, lse)
        for i in (0, 1):  # the block of the newest token is gone whenever it was completed by this step
            st = a.oracle.seqs[i]
            if st.length % 16 == 0 and (st.length - 1) // 16 not in a.oracle.live_blocks(i):
                freed_same_step += 1
        if step % 7 == 0:
            for i in ids:
                a.check_gather(i, layers=None)
        assert len(a.oracle.free_stack) >= n_free0 - 3
    assert freed_same_step >= 4, "the case this test is named for never happened"
    assert a.gpu.last_error() == 0
    a.close()


def test_bulk_append_130_sequences_two_layers(dev):
    """More sequences than one append launch takes (128): the call is split, and with several layers
    every chunk is issued layer by layer - only the first layer's launch reserves, the others write
    through the block table.  Rows of both layers gathered back bit-exact; then three decode steps."""
    specs = [seq_spec(3, 10 + (i % 5), 8, 8, 4, n_sink_out=1) for i in range(130)]
    cfg = Config("many130", 92, Geometry(n_layers=2), 16, tuple(specs))
    sbs = _mk(cfg, dev)
    ids = list(range(130))
    sbs.bulk_prefill(ids, 2, evict=False)  # ONE call, 130 sequences x (prefill + 2) tokens
    for i in (0, 1, 63, 127, 128, 129):
        sbs.check_gather(i, layers=None)
    sbs.evict(ids)
    sbs.check_integer_state(ids)
    for _ in range(3):
        sbs.append_step(ids)
        sbs.evict(ids)
        sbs.check_integer_state(ids)
        q, out, lse = sbs.attend(ids, want_lse=True)
        sbs.check_attention(ids, q, out, lse, seq_subset=[0, 31, 32, 127, 128, 129])
    for i in (0, 64, 128, 129):
        sbs.check_gather(i, layers=None)
    assert sbs.gpu.last_error() == 0
    sbs.close()

# -------------------------------------------------------------------------------- CUDA graph replay
@pytest.mark.parametrize("layered", [False, True])
def test_decode_step_cuda_graph_replay(dev, layered):
    """One captured decode step (one launch, or the per-layer-range launches of a step) replayed 40 times with
    refilled input buffers on a ragged page-16 batch (windows slide, pages are allocated and freed inside the
    replays), then murmur_mirror_sync: integer state bit-exact, every replay's output within tolerance, and the
    handle usable through the normal calls afterwards."""
    specs = [seq_spec(8, 70 + 9 * i, 80, 32 if i % 2 else 48, 16 if i % 3 else 32, n_sink_out=2 + i % 3) for i in range(4)]
    cfg = workloads.config5().with_seqs(specs).with_layers(3)
    a = _mk(cfg, dev)
    ids = list(range(cfg.batch))
    a.bulk_prefill(ids, 1)
    a.fused_step(ids)  # un-captured step first: one-time kernel attributes are set outside the capture
    if layered:
        a.layer_range_step(ids, [(0, 1), (1, 3)])
    L = cfg.geom.n_layers
    k_buf = torch.empty(L, len(ids), 4, 128, dtype=torch.bfloat16, device=dev)
    v_buf = torch.empty_like(k_buf)
    q_buf = torch.empty(L, len(ids), 28, 128, dtype=torch.bfloat16, device=dev)
    out_buf = torch.empty_like(q_buf)

    def fill():
        ks, vs = [], []
        for i in ids:
            u = a.t_of(i)
            k, v = a.data[i].out_kv(u, u + 1)
            ks.append(k)
            vs.append(v)
            a._store(i, k, v)
        k_buf.copy_(torch.cat(ks, dim=1))
        v_buf.copy_(torch.cat(vs, dim=1))
        a.oracle.append(ids, [1] * len(ids))
        a.oracle.evict(ids)
        q_buf.copy_(a.queries(ids))

    fill()
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        if layered:
            a.gpu.decode_step_layers(ids, k_buf[0:1], v_buf[0:1], q_buf[0:1], out_buf[0:1], 0, 1, None, a.scale)
            a.gpu.decode_step_layers(ids, k_buf[1:3], v_buf[1:3], q_buf[1:3], out_buf[1:3], 1, 3, None, a.scale)
        else:
            a.gpu.decode_step(ids, k_buf, v_buf, q_buf, out_buf, None, a.scale)
    for step in range(40):
        if step:
            fill()
        g.replay()
        torch.cuda.synchronize()
        if step % 4 == 0 or step >= 36:
            a.check_attention(ids, q_buf, out_buf)
    # the host mirror has not seen the replays: ordinary calls are refused until murmur_mirror_sync has run
    from paper_2606_01483_b200 import MurmurError
    for call in (lambda: a.gpu.kv_evict(ids), lambda: a.gpu.decode_step(ids, k_buf, v_buf, q_buf, out_buf, None, a.scale)):
        with pytest.raises(MurmurError) as e:
            call()
        assert e.value.status == 2
    a.gpu.mirror_sync()
    a.check_integer_state(ids)
    # and on through the ordinary calls
    q, out, lse = a.fused_step(ids, want_lse=True)
    a.check_integer_state(ids)
    a.check_attention(ids, q, out, lse)
    a.close()


# -------------------------------------------------------------------------------- per-layer windows
def test_decode_attn_windowed_per_layer_groups(dev):
    """murmur_decode_attn_windowed: layers 0-1 attend a tighter window than layers 2-3 while residency
    follows the sequences' own (loosest) policy; each group is checked against Eq. 1 over the A(t) of
    ITS window, and a window equal to the base policy reproduces murmur_decode_attn bit for bit."""
    from oracle import attention as o_attn
    from oracle import policy as o_policy
    from paper_2606_01483_b200 import MurmurError

    specs = [seq_spec(9 + i, 150 + 20 * i, 80, 64, 40, delay=32, n_sink_speech=2, n_sink_out=4) for i in range(3)]
    cfg = Config("winlayers", 95, Geometry(n_layers=4), 16, tuple(specs))
    sbs = _mk(cfg, dev)
    ids = [0, 1, 2]
    sbs.bulk_prefill(ids, 50)
    tight = (32, 16, 0, 16, 2)
    base = specs[0].policy_tuple
    for _ in range(4):
        sbs.append_step(ids)
        sbs.evict(ids)
        sbs.check_integer_state(ids)
        q = sbs.queries(ids)
        lse = torch.empty(q.shape[:3], dtype=torch.float32, device=dev)
        out = torch.empty_like(q)
        sbs.gpu.decode_attn(ids, q[0:2].contiguous(), out=out[0:2], lse=lse[0:2], sm_scale=sbs.scale, layer_begin=0, layer_end=2, window=tight)
        sbs.gpu.decode_attn(ids, q[2:4].contiguous(), out=out[2:4], lse=lse[2:4], sm_scale=sbs.scale, layer_begin=2, layer_end=4, window=base)
        plain = sbs.gpu.decode_attn(ids, q[2:4].contiguous(), sm_scale=sbs.scale, layer_begin=2, layer_end=4)
        assert torch.equal(plain, out[2:4]), "a window equal to the base policy must reproduce murmur_decode_attn (same split)"
        got = out.float().cpu().numpy().astype(np.float64)
        q_bits = workloads.to_bits(q)
        errs = []
        for j, i in enumerate(ids):
            st = sbs.oracle.seqs[i]
            kb, vb = sbs.kv_by_position(i)
            for layer in range(4):
                pol = o_policy.Policy(*(tight if layer < 2 else base))
                ret = [x for x in o_policy.retained_positions(st.P, st.S, st.M, st.t, pol) if x < st.length]
                assert set(ret) <= set(sbs.oracle.retained(i)) | set(o_policy.resident_positions(st.P, st.S, st.M, st.t, st.pol))
                o_ref, lse_ref, _ = o_attn.attend_retained(q_bits[layer, j], kb[layer], vb[layer], ret, sbs.scale)
                errs.append(np.abs(got[layer, j] - o_ref))
                assert np.max(np.abs(lse[layer, j].cpu().numpy() - lse_ref)) < 2e-3
        e = np.stack(errs)
        assert e.max() <= 2e-2 and e.mean() <= 2e-3
    # a window that reaches further back than the base policy could touch evicted positions: rejected
    for bad in ((65, 32, 2, 40, 4), (64, 33, 2, 40, 4), (64, 32, 3, 40, 4), (64, 32, 2, 41, 4), (64, 32, 2, 40, 5)):
        with pytest.raises(MurmurError):
            sbs.gpu.decode_attn(ids, q, sm_scale=sbs.scale, window=bad)
    assert sbs.gpu.last_error() == 0
    sbs.close()


# -------------------------------------------------------------------------------- errors
def test_error_behaviour_leaves_state_unchanged(dev):
    from paper_2606_01483_b200 import MurmurCache, MurmurError

    c = MurmurCache(2, 28, 4, 128, 16, max_seqs=3, max_blocks_per_seq=8, n_pages=5, device=dev)
    pol = (8, 4, 0, 8, 1)
    c.seq_begin(0, 4, 20, 0, pol)
    c.seq_begin(1, 4, 20, 0, pol)

    def kv(n):
        return torch.zeros(2, n, 4, 128, dtype=torch.bfloat16, device=dev)

    with pytest.raises(MurmurError) as e:
        c.seq_begin(0, 1, 1, 1, pol)
    assert e.value.status == 2
    with pytest.raises(MurmurError) as e:
        c.kv_append([2], [1], kv(1), kv(1))  # inactive
    assert e.value.status == 2
    with pytest.raises(MurmurError) as e:
        c.kv_append([0, 0], [1, 1], kv(2), kv(2))  # duplicate
    assert e.value.status == 1
    with pytest.raises(MurmurError) as e:
        c.kv_append([7], [1], kv(1), kv(1))  # out of range
    assert e.value.status == 1
    c.kv_append([0], [40], kv(40), kv(40))  # 3 pages
    with pytest.raises(MurmurError) as e:
        c.kv_append([1, 0], [20, 20], kv(40), kv(40))  # needs 2 + 1 pages, 2 free: all-or-nothing
    assert e.value.status == 3
    assert c.seq_state(0)["length"] == 40 and c.seq_state(1)["length"] == 0
    assert c.free_stack().tolist() == [4, 3]
    with pytest.raises(MurmurError) as e:
        c.kv_append([0], [200], kv(200), kv(200))  # > max_blocks_per_seq
    assert e.value.status == 2
    q = torch.zeros(2, 1, 28, 128, dtype=torch.bfloat16, device=dev)
    with pytest.raises(MurmurError) as e:
        c.decode_attn([0], q)  # not evicted since the last append
    assert e.value.status == 2
    c.kv_evict([0])
    c.decode_attn([0], q)
    with pytest.raises(MurmurError) as e:
        c.decode_attn([1], q)  # empty sequence
    assert e.value.status == 2
    assert c.last_error() == 0
    c.seq_end(0)
    assert sorted(c.free_stack().tolist()) == [0, 1, 2, 3, 4]
    c.close()
