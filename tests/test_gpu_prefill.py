"""Parity of murmur_prefill_attn (causal attention of the prefill tokens over the paged cache)
against oracle/prefill.py on the same seeded inputs; tolerance as for decode (2e-2 / 2e-3)."""
import math

import numpy as np
import pytest
import torch

import workloads
from oracle import attention as o_attn
from oracle import prefill as o_pre

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def dev():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return "cuda:0"


def _cache(dev, n_layers, n_tok, page, policy=None, P=8, M=0):
    from paper_2606_01483_b200 import MURMUR_WINDOW_OFF, MurmurCache

    nb = (n_tok + page - 1) // page + 2
    c = MurmurCache(n_layers, 28, 4, 128, page, 1, nb, nb + 2, device=dev)
    c.seq_begin(0, P, n_tok - P - M, M, policy or (MURMUR_WINDOW_OFF, 0, 0, MURMUR_WINDOW_OFF, 0))
    return c


def _rand(shape, seed, dev):
    g = torch.Generator().manual_seed(seed)
    return torch.randn(*shape, generator=g).to(torch.bfloat16).to(dev)


def _check(out, lse, q, k, v, pos_begin, rows, scale):
    got = out.float().cpu().numpy().astype(np.float64)
    qb, kb, vb = workloads.to_bits(q), workloads.to_bits(k), workloads.to_bits(v)
    errs = []
    for layer in range(q.shape[0]):
        if rows is None:
            o_ref, lse_ref = o_pre.causal_attention(qb[layer], kb[layer], vb[layer], pos_begin, scale)
            errs.append(np.abs(got[layer] - o_ref))
            if lse is not None:
                assert np.max(np.abs(lse[layer].cpu().numpy() - lse_ref)) < 2e-3
        else:
            for i in rows:
                o_ref, lse_ref, _ = o_attn.attend_retained(qb[layer, i], kb[layer], vb[layer], range(pos_begin + i + 1), scale)
                errs.append(np.abs(got[layer, i] - o_ref))
                if lse is not None:
                    assert np.max(np.abs(lse[layer, i].cpu().numpy() - lse_ref)) < 2e-3
    e = np.concatenate([x.ravel() for x in errs])
    assert np.isfinite(got).all()
    assert e.max() <= 2e-2 and e.mean() <= 2e-3, (e.max(), e.mean())


def _check_every_row_c(out, lse, q, k, v, layers, q_heads, scale):
    """EVERY row of the given layers and query heads against the plain-C fp64 twin of oracle/prefill.py
    (oracle/c: murmur_oracle_prefill); q_heads must cover whole GQA groups.  Returns (max, mean) abs error."""
    from oracle import c as oracle_c

    co = oracle_c.load()
    layers, q_heads = list(layers), list(q_heads)
    G = q.shape[2] // k.shape[2]
    kv_heads = sorted(set(h // G for h in q_heads))
    assert q_heads == [g * G + j for g in kv_heads for j in range(G)]
    li = torch.tensor(layers, device=q.device)
    hi = torch.tensor(q_heads, device=q.device)
    gi = torch.tensor(kv_heads, device=q.device)
    qb = workloads.to_bits(q[li][:, :, hi])
    kb, vb = workloads.to_bits(k[li][:, :, gi]), workloads.to_bits(v[li][:, :, gi])
    o_ref, lse_ref, _ = co.prefill(qb, kb, vb, 0, scale)
    got = out[li][:, :, hi].float().cpu().numpy().astype(np.float64)
    assert np.isfinite(got).all()
    e = np.abs(got - o_ref)
    assert e.max() <= 2e-2 and e.mean() <= 2e-3, (e.max(), e.mean())
    if lse is not None:
        assert np.max(np.abs(lse[li][:, :, hi].cpu().numpy() - lse_ref)) < 2e-3
    return float(e.max()), float(e.mean())


@pytest.mark.parametrize("page,n_tok", [(16, 200), (32, 130), (64, 257), (64, 64), (16, 1)])
def test_prefill_every_row_small(dev, page, n_tok):
    L = 2
    c = _cache(dev, L, n_tok, page, P=min(8, n_tok))
    k, v = _rand((L, n_tok, 4, 128), 1, dev), _rand((L, n_tok, 4, 128), 2, dev)
    k[:, :4] *= 4  # sink keys
    q = _rand((L, n_tok, 28, 128), 3, dev)
    c.kv_append([0], [n_tok], k, v)
    lse = torch.empty(L, n_tok, 28, dtype=torch.float32, device=dev)
    out = c.prefill_attn(0, 0, n_tok, q, lse=lse)
    _check(out, lse, q, k, v, 0, None, 1 / math.sqrt(128))
    assert c.last_error() == 0
    c.close()


def test_prefill_chunked_unaligned_ranges_and_layer_range(dev):
    # the chunk is prefilled in two pieces that do not start on a tile boundary; second layer only
    L, n_tok = 3, 300
    c = _cache(dev, L, n_tok, 16)
    k, v = _rand((L, n_tok, 4, 128), 4, dev), _rand((L, n_tok, 4, 128), 5, dev)
    q = _rand((L, n_tok, 28, 128), 6, dev)
    c.kv_append([0], [n_tok], k, v)
    scale = 1 / math.sqrt(128)
    for a, b in ((0, 37), (37, 300), (101, 102)):
        out = c.prefill_attn(0, a, b, q[1:2, a:b].contiguous(), layer_begin=1, layer_end=2)
        _check(out, None, q[1:2, a:b], k[1:2], v[1:2], a, None, scale)
    c.close()


@pytest.mark.parametrize("page", [16, 64])
def test_prefill_moving_row_maximum(dev, page):
    """Scores that keep growing along the key axis: every row's reference maximum moves by far more than 2^8
    again and again, in first and in second halves of the 128-key tiles (the kernel's lazy-maximum rescale of
    O and l, incl. the case where the first half of the same tile's PV is already in flight)."""
    L, n_tok = 1, 700
    c = _cache(dev, L, n_tok, page)
    k, v = _rand((L, n_tok, 4, 128), 21, dev), _rand((L, n_tok, 4, 128), 22, dev)
    q = _rand((L, n_tok, 28, 128), 23, dev)
    # a common direction u in q and k; its weight in k jumps at positions spread over both tile halves
    u = torch.zeros(128, device=dev)
    u[:8] = 1.0
    q = (q.float() + 6.0 * u).to(torch.bfloat16)
    step = torch.zeros(n_tok, device=dev)
    for pos, amp in ((40, 2.0), (100, 4.0), (130, 6.0), (200, 8.0), (330, 10.0), (447, 12.0), (448, 14.0), (600, 16.0), (699, 18.0)):
        step[pos:] = amp
    k = (k.float() + step[None, :, None, None] * u).to(torch.bfloat16)
    c.kv_append([0], [n_tok], k, v)
    lse = torch.empty(L, n_tok, 28, dtype=torch.float32, device=dev)
    out = c.prefill_attn(0, 0, n_tok, q, lse=lse)
    _check(out, lse, q, k, v, 0, None, 1 / math.sqrt(128))
    assert c.last_error() == 0
    c.close()


def test_prefill_many_single_tile_items_per_cta(dev):
    """100 positions x 28 layers: 448 work items of ONE 128-key tile each, three per persistent CTA back to back, every
    one with rows past the sequence length in its last (only) tile - the hand-overs between softmax, epilogue, producer
    and issuer that a multi-tile item spaces out all fall on top of each other.  The first run is compared with the oracle
    on every row of every layer and head; then repeated, bit-identical every time."""
    L, n_tok = 28, 100
    c = _cache(dev, L, n_tok, 16)
    k, v = _rand((L, n_tok, 4, 128), 31, dev), _rand((L, n_tok, 4, 128), 32, dev)
    q = _rand((L, n_tok, 28, 128), 33, dev)
    c.kv_append([0], [n_tok], k, v)
    lse = torch.empty(L, n_tok, 28, dtype=torch.float32, device=dev)
    out = c.prefill_attn(0, 0, n_tok, q, lse=lse)
    _check_every_row_c(out, lse, q, k, v, range(L), range(28), 1 / math.sqrt(128))  # every row, layer and head
    for _ in range(50):
        again = c.prefill_attn(0, 0, n_tok, q)
        assert torch.equal(again, out)
    assert c.last_error() == 0
    c.close()


def test_prefill_config2_size_sampled_rows(dev):
    # one 300 s chunk: 64 prefix + 2250 speech tokens, 2 layers; rows around tile / page boundaries and the end
    cfg = workloads.config2().with_layers(2)
    d = workloads.SeqData(cfg, 0, device=dev)
    k, v = d.prefill_kv()
    n_tok = k.shape[1]
    c = _cache(dev, 2, n_tok, 64, P=64)
    c.kv_append([0], [n_tok], k.contiguous(), v.contiguous())
    q = _rand((2, n_tok, 28, 128), 7, dev)
    lse = torch.empty(2, n_tok, 28, dtype=torch.float32, device=dev)
    out = c.prefill_attn(0, 0, n_tok, q, lse=lse)
    torch.cuda.synchronize()
    _check(out, lse, q, k, v, 0, [0, 1, 15, 16, 63, 64, 65, 127, 128, 1000, 2047, 2048, n_tok - 2, n_tok - 1], 1 / math.sqrt(128))
    c.close()


def test_prefill_config2_size_every_row(dev):
    """The launch bench.py times - one 300 s chunk (64 prefix + 2250 speech tokens), all 28 layers in ONE launch whose
    148 persistent CTAs walk ~7 500 work items - compared with the fp64 oracle on EVERY row: all 28 query heads of
    layers 0, 9, 18 and 27 (early, middle and late items of the persistent schedule), and all 28 layers on the two
    middle KV heads (query heads 7 .. 20).  Output and log-sum-exp, tolerance as everywhere (2e-2 / 2e-3)."""
    cfg = workloads.config2()
    d = workloads.SeqData(cfg, 0, device=dev)
    k, v = d.prefill_kv()
    k, v = k.contiguous(), v.contiguous()
    L, n_tok = k.shape[0], k.shape[1]
    assert (L, n_tok) == (28, 2314)
    c = _cache(dev, L, n_tok, 64, P=64)
    c.kv_append([0], [n_tok], k, v)
    q = _rand((L, n_tok, 28, 128), 17, dev)
    lse = torch.empty(L, n_tok, 28, dtype=torch.float32, device=dev)
    out = c.prefill_attn(0, 0, n_tok, q, lse=lse)
    torch.cuda.synchronize()
    scale = 1 / math.sqrt(128)
    _check_every_row_c(out, lse, q, k, v, [0, 9, 18, 27], range(28), scale)
    for half in (range(0, 14), range(14, 28)):
        _check_every_row_c(out, lse, q, k, v, half, range(7, 21), scale)
    assert c.last_error() == 0
    c.close()


def test_prefill_rejects_evicted_cache_and_bad_ranges(dev):
    from paper_2606_01483_b200 import MurmurError

    c = _cache(dev, 1, 200, 16, policy=(16, 0, 0, 16, 0), P=8)
    k = _rand((1, 200, 4, 128), 8, dev)
    c.kv_append([0], [200], k, k.clone())
    q = _rand((1, 200, 28, 128), 9, dev)
    c.prefill_attn(0, 0, 200, q)  # fine before any evict
    with pytest.raises(MurmurError):
        c.prefill_attn(0, 0, 201, _rand((1, 201, 28, 128), 9, dev))
    with pytest.raises(MurmurError):
        c.prefill_attn(0, 5, 5, q[:, :0].contiguous())
    kk = _rand((1, 40, 4, 128), 10, dev)
    c.kv_append([0], [40], kk, kk.clone())  # 40 output tokens: the speech window slides, blocks are freed
    c.kv_evict([0])
    with pytest.raises(MurmurError):
        c.prefill_attn(0, 0, 200, q)
    c.close()
