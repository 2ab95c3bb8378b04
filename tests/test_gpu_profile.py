"""Parity of murmur_attn_profile (attention-sparsity profile, PAPER.md:77 / Fig. 5) against
oracle/sparsity.py on the same seeded inputs.

Integer fields that floating point decides (k_mass and its region split) are checked for VALIDITY
against the oracle's fp64 weights: the GPU's set size k must reach the mass fraction and k - 1 must
not, within eps of rounding (both sides would agree exactly in infinite precision); where the
boundary is not within eps the values must be equal.  Region totals are exact."""
import math

import numpy as np
import pytest
import torch

import workloads
from oracle import policy as o_policy
from oracle import sparsity as o_sp
from workloads import Config, Geometry, seq_spec

pytestmark = pytest.mark.gpu
EPS = 2e-4


@pytest.fixture(scope="module")
def dev():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return "cuda:0"


def _check_head(got, hp: o_sp.HeadProfile, frac):
    assert (got["n_resident"], got["n_prompt"], got["n_speech"], got["n_text"]) == (hp.n_resident, hp.n_prompt, hp.n_speech, hp.n_text)
    for f, want in (("coverage", hp.coverage), ("mass_prompt", hp.mass_prompt), ("mass_speech", hp.mass_speech), ("mass_text", hp.mass_text)):
        assert abs(float(got[f]) - want) < 1e-4, (f, float(got[f]), want)
    k = int(got["k_mass"])
    assert k == got["k_prompt"] + got["k_speech"] + got["k_text"]
    srt = np.sort(hp.alpha)[::-1]
    cum = np.cumsum(srt)
    assert 1 <= k <= hp.n_resident
    assert cum[k - 1] >= frac - EPS, "the reported set does not reach the mass fraction"
    assert k == 1 or cum[k - 2] < frac + EPS, "a smaller set already reaches the mass fraction"
    clear = abs(cum[hp.k_mass - 1] - frac) > EPS and (hp.k_mass == 1 or abs(cum[hp.k_mass - 2] - frac) > EPS)
    if clear:
        assert k == hp.k_mass
        # region split is unique unless the k-th and (k+1)-th weights are (nearly) tied
        gap = srt[k - 1] - srt[k] if k < len(srt) else 1.0
        if gap > 1e-6:
            assert (got["k_prompt"], got["k_speech"], got["k_text"]) == (hp.k_prompt, hp.k_speech, hp.k_text)
    return k == hp.k_mass


@pytest.mark.parametrize("page,evicted", [(64, False), (16, False), (32, True)])
def test_profile_random_small(dev, page, evicted):
    from harness import SideBySide

    pol = dict(w_speech=40, w_out=24) if evicted else dict(w_speech=workloads.WINDOW_OFF, w_out=workloads.WINDOW_OFF)
    specs = [seq_spec(9, 150, 80, pol["w_speech"], pol["w_out"], M=3 if i else 0, n_sink_speech=2 * i, n_sink_out=4)
             for i in range(2)]
    cfg = Config("prof", 60, Geometry(n_layers=2), page, tuple(specs), locality_rho=0.5)
    sbs = SideBySide(cfg, device=dev)
    ids = [0, 1]
    sbs.bulk_prefill(ids, 70)
    cand = (32, 16, 1, 20, 2)
    q = sbs.queries(ids)
    for frac in (0.99, 0.9):
        got = sbs.gpu.attn_profile(ids, q, candidate=cand, mass_frac=frac)
        q_bits = workloads.to_bits(q)
        exact = total = 0
        for j, i in enumerate(ids):
            s = sbs.oracle.seqs[i]
            resident = [x for x in o_policy.resident_positions(s.P, s.S, s.M, s.t, s.pol) if x < s.length]
            cset = [x for x in o_policy.retained_positions(s.P, s.S, s.M, s.t, o_policy.Policy(*cand)) if x < s.length]
            kb, _ = sbs.kv_by_position(i)
            for layer in range(2):
                hps = o_sp.profile_step(q_bits[layer, j], kb[layer], resident, s.P, s.S, s.M, cset, sbs.scale, frac)
                for h, hp in enumerate(hps):
                    exact += _check_head(got[layer, j, h], hp, frac)
                    total += 1
        assert exact >= 0.95 * total
    # candidate None = the sequence's own policy: coverage over its own A(t)
    own = sbs.gpu.attn_profile(ids, q)
    if not evicted:
        assert np.allclose(own["coverage"], 1.0, atol=1e-5)
    assert sbs.gpu.last_error() == 0
    sbs.close()


def _direct_cache(dev, n_tok, P, S, M, page=16):
    from paper_2606_01483_b200 import MURMUR_WINDOW_OFF, MurmurCache

    c = MurmurCache(1, 28, 4, 128, page, 1, (n_tok + page - 1) // page + 1, (n_tok + page - 1) // page + 2, device=dev)
    c.seq_begin(0, P, S, M, (MURMUR_WINDOW_OFF, 0, 0, MURMUR_WINDOW_OFF, 0))
    return c


def test_profile_identical_keys_ties_by_position(dev):
    # uniform weights: the mass set is the first ceil(frac * n) positions; region split follows positions
    n, P, S, M = 150, 10, 100, 5
    c = _direct_cache(dev, n, P, S, M)
    row = torch.linspace(-1, 1, 128).to(torch.bfloat16)
    k = row.expand(1, n, 4, 128).contiguous().to(dev)
    c.kv_append([0], [n], k, k.clone())
    q = torch.randn(1, 1, 28, 128, generator=torch.Generator().manual_seed(3)).to(torch.bfloat16).to(dev)
    for frac, want in ((0.5, 75), (0.901, 136), (0.997, 150)):
        got = c.attn_profile([0], q, candidate=(20, 0, 0, 10, 0), mass_frac=frac)[0, 0]
        assert (got["k_mass"] == want).all(), (frac, got["k_mass"])
        take = list(range(want))
        reg = [o_sp.region_of(x, P, S, M) for x in take]
        assert (got["k_prompt"] == reg.count(0)).all() and (got["k_speech"] == reg.count(1)).all() and (got["k_text"] == reg.count(2)).all()
        assert (got["n_prompt"] == 15).all() and (got["n_speech"] == 100).all() and (got["n_text"] == 35).all()
        # candidate at t = 35, w_s 20, d 0 -> l = min(35, 80) = 35: speech [45, 65), prompts, last 10 outputs
        assert np.allclose(got["coverage"], (15 + 20 + 10) / n, atol=1e-5)
    c.close()


def test_profile_one_dominant_key(dev):
    n, P, S, M = 90, 6, 60, 0
    c = _direct_cache(dev, n, P, S, M, page=64)
    g = torch.Generator().manual_seed(5)
    k = (torch.randn(1, n, 4, 128, generator=g) * 0.05)
    q = torch.zeros(1, 1, 28, 128)
    q[..., 0] = 8.0
    k[0, 40, :, 0] = 60.0  # logit (8 * 60) / sqrt(128) = 42 above the rest
    kb = k.to(torch.bfloat16).to(dev)
    c.kv_append([0], [n], kb, kb.clone())
    got = c.attn_profile([0], q.to(torch.bfloat16).to(dev), mass_frac=0.99)[0, 0]
    assert (got["k_mass"] == 1).all() and (got["k_speech"] == 1).all()
    assert np.allclose(got["mass_speech"], 1.0, atol=1e-6)
    c.close()


def test_profile_argument_errors(dev):
    from paper_2606_01483_b200 import MurmurError

    c = _direct_cache(dev, 20, 2, 10, 0)
    q = torch.zeros(1, 1, 28, 128, dtype=torch.bfloat16, device=dev)
    with pytest.raises(MurmurError):  # empty sequence
        c.attn_profile([0], q)
    k = torch.zeros(1, 5, 4, 128, dtype=torch.bfloat16, device=dev)
    c.kv_append([0], [5], k, k.clone())
    with pytest.raises(MurmurError):
        c.attn_profile([0], q, mass_frac=0.0)
    with pytest.raises(MurmurError):
        c.attn_profile([0], q, candidate=(-1, 0, 0, 0, 0))
    assert (c.attn_profile([0], q)["k_mass"] == 5).all()  # zero keys: uniform, ceil(0.99 * 5) = 5
    c.close()
