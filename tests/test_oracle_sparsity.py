"""Pins of oracle/sparsity.py (the 99 %-mass set of PAPER.md:77 / Fig. 5) against
closed forms, brute force and invariants - nothing here calls the CUDA path."""
import itertools
import math

import numpy as np
import pytest
import torch

from oracle import sparsity as sp


def _bits(x: np.ndarray) -> np.ndarray:
    return torch.tensor(np.asarray(x, dtype=np.float32)).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)


def test_identical_keys_give_uniform_weights_and_ceil_frac_n():
    # closed form: uniform alpha = 1/n -> the mass set is the first ceil(frac * n) positions (ties by position)
    n, d, P, S, M = 50, 16, 5, 30, 2
    k = np.tile(np.linspace(-1, 1, d, dtype=np.float32), (n, 1))
    q = np.ones(d, dtype=np.float32)
    hp = sp.profile_head(_bits(q), _bits(k), range(n), P, S, M, range(n), 0.25, 0.99)
    assert np.allclose(hp.alpha, 1.0 / n)
    assert hp.k_mass == math.ceil(0.99 * n) == 50
    hp = sp.profile_head(_bits(q), _bits(k), range(n), P, S, M, range(10), 0.25, 0.5)
    assert hp.k_mass == 25 and hp.mass_set == list(range(25))
    # regions of positions 0..24: prompt [0,5), speech [5,35)
    assert (hp.k_prompt, hp.k_speech, hp.k_text) == (5, 20, 0)
    assert (hp.n_prompt, hp.n_speech, hp.n_text) == (7, 30, 13)
    assert hp.coverage == pytest.approx(10 / n)


def test_one_dominant_key():
    n, d = 40, 8
    rng = np.random.default_rng(1)
    k = rng.standard_normal((n, d)).astype(np.float32) * 0.1
    q = np.zeros(d, dtype=np.float32)
    q[0] = 1.0
    k[17, 0] = 60.0  # logit 60 above the rest: alpha_17 = 1 - O(e^-59)
    hp = sp.profile_head(_bits(q), _bits(k), range(n), 4, 20, 0, [17], 1.0)
    assert hp.k_mass == 1 and hp.mass_set == [17] and hp.k_speech == 1
    assert hp.coverage == pytest.approx(1.0, abs=1e-12)


def test_geometric_weights_closed_form():
    # scores s_i = -i * ln 2 -> alpha_i = 2^-i / (2 - 2^-(n-1)): smallest k with 1 - 2^-k >= frac * (1 - 2^-n)
    n, d = 24, 4
    k = np.zeros((n, d), dtype=np.float32)
    k[:, 0] = -np.arange(n)  # exactly representable in bf16 (small integers)
    q = np.array([1.0, 0, 0, 0], dtype=np.float32)
    for frac in (0.5, 0.9, 0.99, 0.999):
        hp = sp.profile_head(_bits(q), _bits(k), range(n), 0, n, 0, [], math.log(2.0), frac)
        want = next(kk for kk in range(1, n + 1) if 1 - 2.0 ** -kk >= frac * (1 - 2.0 ** -n))
        assert hp.k_mass == want and hp.mass_set == list(range(want))


@pytest.mark.parametrize("seed", range(5))
def test_mass_set_is_a_minimum_cardinality_set_brute_force(seed):
    rng = np.random.default_rng(10 + seed)
    n, d = 9, 8
    k = rng.standard_normal((n, d)).astype(np.float32)
    q = rng.standard_normal(d).astype(np.float32) * 2
    frac = [0.5, 0.8, 0.9, 0.95, 0.99][seed]
    hp = sp.profile_head(_bits(q), _bits(k), range(n), 2, 4, 1, [], 0.5, frac)
    a = hp.alpha
    best = min(r for r in range(1, n + 1) for c in itertools.combinations(range(n), r) if sum(a[list(c)]) >= frac)
    assert hp.k_mass == best
    assert sum(a[hp.mass_set]) >= frac
    assert hp.k_mass == 1 or sum(a[hp.mass_set[:-1]]) < frac


def test_invariants_on_random_input():
    rng = np.random.default_rng(7)
    n, d, P, S, M = 120, 32, 10, 70, 5
    k = rng.standard_normal((n, 2, d)).astype(np.float32)
    q = rng.standard_normal((4, d)).astype(np.float32)
    resident = [x for x in range(n) if not (30 <= x < 50)]  # an evicted hole
    cand = [x for x in resident if x < 20 or x >= 100]
    hps = sp.profile_step(_bits(q), _bits(k), resident, P, S, M, cand, 1 / math.sqrt(d))
    for h, hp in enumerate(hps):
        assert hp.n_resident == len(resident) == hp.n_prompt + hp.n_speech + hp.n_text
        assert hp.mass_prompt + hp.mass_speech + hp.mass_text == pytest.approx(1.0, abs=1e-12)
        assert hp.k_mass == hp.k_prompt + hp.k_speech + hp.k_text <= hp.n_resident
        assert 0.0 <= hp.coverage <= 1.0
        comp = sp.profile_head(_bits(q[h]), _bits(k[:, h // 2]), resident, P, S, M, set(resident) - set(cand), 1 / math.sqrt(d))
        assert hp.coverage + comp.coverage == pytest.approx(1.0, abs=1e-12)
        # the weights are those of oracle.attention (library softmax over the same scores)
        kk = torch.tensor(k[resident][:, h // 2]).to(torch.bfloat16).double()
        qq = torch.tensor(q[h]).to(torch.bfloat16).double()
        assert np.allclose(hp.alpha, torch.softmax(kk @ qq / math.sqrt(d), dim=0).numpy(), atol=1e-14)
    # GQA: heads 0,1 share KV head 0 - different queries, same keys
    assert hps[0].n_resident == hps[1].n_resident


def test_region_map():
    P, S, M = 3, 4, 2
    assert [sp.region_of(x, P, S, M) for x in range(12)] == [0, 0, 0, 1, 1, 1, 1, 0, 0, 2, 2, 2]
