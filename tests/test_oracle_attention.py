"""Pins for oracle/attention.py and its plain-C twin (no GPU).

I1, I3, P8, P9, P10, P11, P12 of SURVEY.md section 8(c), plus a pure-Python brute force and a
GQA head-map check.  The library routine used as the independent definition of Eq. 1 is
torch.nn.functional.scaled_dot_product_attention on CPU in fp64.
"""
import math

import numpy as np
import pytest
import torch

from oracle import attention, policy
from oracle.policy import Policy
from workloads import from_bits, to_bits


def _rand_bits(rng, *shape, scale=1.0):
    x = torch.from_numpy(rng.standard_normal(shape).astype(np.float32) * scale).to(torch.bfloat16)
    return to_bits(x)


def _sdpa_f64(q_bits, k_bits, v_bits, idx, scale):
    """Independent definition: library SDPA, fp64, GQA expanded by repeat_interleave."""
    q = from_bits(q_bits).double()  # [n_q, d]
    k = from_bits(k_bits[idx]).double()  # [n, n_kv, d]
    v = from_bits(v_bits[idx]).double()
    G = q.shape[0] // k.shape[1]
    kk = k.permute(1, 0, 2).repeat_interleave(G, dim=0)  # [n_q, n, d]
    vv = v.permute(1, 0, 2).repeat_interleave(G, dim=0)
    o = torch.nn.functional.scaled_dot_product_attention(q[:, None, :], kk, vv, scale=scale)
    return o[:, 0, :].numpy()


# ---------------------------------------------------------------------------- I1
def test_I1_windows_off_equals_full_attention_library_routine():
    rng = np.random.default_rng(1)
    P, S, M, t = 5, 40, 2, 9
    n = P + S + M + t
    q, k, v = _rand_bits(rng, 28, 128), _rand_bits(rng, n, 4, 128), _rand_bits(rng, n, 4, 128)
    scale = 1.0 / math.sqrt(128)
    A = policy.retained_positions(P, S, M, t, Policy(10**6, 0, 0, 10**6, 0))
    assert A == list(range(n))
    o, lse, alpha = attention.attend_retained(q, k, v, A, scale)
    ref = _sdpa_f64(q, k, v, np.arange(n), scale)
    assert np.max(np.abs(o - ref)) < 1e-12


def test_subset_equals_library_routine_on_gathered_rows():
    rng = np.random.default_rng(2)
    pol = Policy(8, 4, 1, 6, 2)
    P, S, M, t = 3, 30, 1, 20
    n = P + S + M + t
    q, k, v = _rand_bits(rng, 14, 64), _rand_bits(rng, n, 2, 64), _rand_bits(rng, n, 2, 64)
    A = policy.retained_positions(P, S, M, t, pol)
    assert 0 < len(A) < n
    o, _, _ = attention.attend_retained(q, k, v, A, 0.125)
    assert np.max(np.abs(o - _sdpa_f64(q, k, v, np.asarray(A), 0.125))) < 1e-12


# ---------------------------------------------------------------------------- I3
def test_I3_weights_sum_to_one_and_nonnegative():
    rng = np.random.default_rng(3)
    q, k, v = _rand_bits(rng, 28, 128), _rand_bits(rng, 300, 4, 128, scale=3.0), _rand_bits(rng, 300, 4, 128)
    _, _, alpha = attention.attend_retained(q, k, v, range(0, 300, 2), 1 / math.sqrt(128))
    assert np.all(alpha >= 0)
    assert np.max(np.abs(alpha.sum(axis=1) - 1.0)) < 1e-12


# ---------------------------------------------------------------------------- brute force
def test_brute_force_pure_python_tiny():
    """Eq. 1 with math.exp and nested loops on a tiny case; catches transposed operands, a wrong
    head map or a dropped scale."""
    rng = np.random.default_rng(4)
    n_q, n_kv, d, n = 6, 3, 4, 7
    q, k, v = _rand_bits(rng, n_q, d), _rand_bits(rng, n, n_kv, d), _rand_bits(rng, n, n_kv, d)
    qf, kf, vf = (attention.bf16_bits_to_f64(a) for a in (q, k, v))
    subset = [0, 2, 3, 6]
    scale = 0.37
    o, lse, _ = attention.attend_retained(q, k, v, subset, scale)
    for h in range(n_q):
        g = h // 2
        s = [sum(qf[h][c] * kf[i][g][c] for c in range(d)) * scale for i in subset]
        den = sum(math.exp(x) for x in s)
        for c in range(d):
            ref = sum(math.exp(s[a]) / den * vf[i][g][c] for a, i in enumerate(subset))
            assert abs(o[h][c] - ref) < 1e-12
        assert abs(lse[h] - math.log(den)) < 1e-12


def test_gqa_head_map_consecutive_heads_share_kv_head():
    """G19: kv = h // G.  Make KV head 1 the only one with a non-trivial V."""
    n_q, n_kv, d, n = 8, 4, 16, 5
    rng = np.random.default_rng(5)
    q, k = _rand_bits(rng, n_q, d), _rand_bits(rng, n, n_kv, d)
    vz = np.zeros((n, n_kv, d), dtype=np.float32)
    vz[:, 1, :] = 1.0
    v = to_bits(torch.from_numpy(vz).to(torch.bfloat16))
    o, _, _ = attention.attend_retained(q, k, v, range(n), 0.25)
    nonzero_heads = [h for h in range(n_q) if np.any(o[h] != 0)]
    assert nonzero_heads == [2, 3]


# ---------------------------------------------------------------------------- P8
def test_P8_special_cases():
    rng = np.random.default_rng(6)
    q, k, v = _rand_bits(rng, 28, 128), _rand_bits(rng, 50, 4, 128), _rand_bits(rng, 50, 4, 128)
    vf = attention.bf16_bits_to_f64(v)
    # one retained key: o = v exactly
    o, _, alpha = attention.attend_retained(q, k, v, [17], 0.1)
    assert np.all(alpha == 1.0)
    for h in range(28):
        assert np.array_equal(o[h], vf[17, h // 7])
    # identical keys: o = mean of v
    k_same = np.repeat(k[:1], 50, axis=0)
    o, _, _ = attention.attend_retained(q, k_same, v, range(50), 0.1)
    for h in range(28):
        assert np.max(np.abs(o[h] - vf[:, h // 7].mean(axis=0))) < 1e-12
    # order of the retained set does not matter
    idx = list(range(0, 50, 3))
    o1, l1, _ = attention.attend_retained(q, k, v, idx, 0.1)
    o2, l2, _ = attention.attend_retained(q, k, v, idx[::-1], 0.1)
    assert np.max(np.abs(o1 - o2)) < 1e-12 and np.max(np.abs(l1 - l2)) < 1e-12


# ---------------------------------------------------------------------------- P9
def test_P9_lse_merge_of_any_partition_equals_unsplit():
    rng = np.random.default_rng(7)
    q, k, v = _rand_bits(rng, 28, 128), _rand_bits(rng, 97, 4, 128, scale=2.0), _rand_bits(rng, 97, 4, 128)
    scale = 1 / math.sqrt(128)
    idx = list(range(97))
    o_ref, lse_ref, _ = attention.attend_retained(q, k, v, idx, scale)
    for cuts in ([50], [1, 2, 96], [10, 20, 30, 40, 50, 60, 70, 80, 90], [96]):
        parts, lo = [], 0
        for c in cuts + [97]:
            parts.append(attention.partial_state(q, k, v, idx[lo:c], scale))
            lo = c
        o, lse = attention.merge_partials(parts)
        assert np.max(np.abs(o - o_ref)) < 1e-12
        assert np.max(np.abs(lse - lse_ref)) < 1e-12
    # merge is order independent
    o_rev, _ = attention.merge_partials(parts[::-1])
    assert np.max(np.abs(o_rev - o_ref)) < 1e-12


# ---------------------------------------------------------------------------- P10
@pytest.mark.parametrize("sink_scale", [4.0, 16.0])
def test_P10_large_logits_stay_finite(sink_scale):
    rng = np.random.default_rng(8)
    q, v = _rand_bits(rng, 28, 128), _rand_bits(rng, 64, 4, 128)
    kf = rng.standard_normal((64, 4, 128)).astype(np.float32)
    kf[:4] *= sink_scale
    k = to_bits(torch.from_numpy(kf).to(torch.bfloat16))
    o, lse, alpha = attention.attend_retained(q, k, v, range(64), 1 / math.sqrt(128))
    assert np.all(np.isfinite(o)) and np.all(np.isfinite(lse))
    assert np.max(np.abs(alpha.sum(axis=1) - 1)) < 1e-12


# ---------------------------------------------------------------------------- P11 / P12
def _bf16_round_f64(x):
    return attention.bf16_bits_to_f64(to_bits(torch.from_numpy(np.asarray(x, dtype=np.float32)).to(torch.bfloat16)))


def test_P11_tolerance_attainable_but_not_vacuous():
    """Rounding alpha and o to bf16 (what a bf16-P, bf16-out kernel does) stays inside the
    2e-2 / 2e-3 bars on unit-scale data, while dropping one heavy in-window key does not."""
    rng = np.random.default_rng(9)
    n = 836
    q, k, v = _rand_bits(rng, 28, 128), _rand_bits(rng, n, 4, 128), _rand_bits(rng, n, 4, 128)
    # make the newest key strongly aligned with the queries of KV group 0 (heavy weight)
    qf = attention.bf16_bits_to_f64(q)
    kf = attention.bf16_bits_to_f64(k)
    kf[n - 1, 0] = 2.0 * qf[0:7].mean(axis=0) * math.sqrt(7)
    k = to_bits(torch.from_numpy(kf.astype(np.float32)).to(torch.bfloat16))
    scale = 1 / math.sqrt(128)
    o, _, alpha = attention.attend_retained(q, k, v, range(n), scale)
    vf = attention.bf16_bits_to_f64(v)
    o_lowp = np.stack([_bf16_round_f64(alpha[h]) @ vf[:, h // 7] / _bf16_round_f64(alpha[h]).sum() for h in range(28)])
    o_lowp = _bf16_round_f64(o_lowp)
    assert np.max(np.abs(o_lowp - o)) <= 2e-2 and np.mean(np.abs(o_lowp - o)) <= 2e-3
    # P12: a wrong set is visible - drop the heavy key
    assert alpha[0, n - 1] > 0.2
    o_wrong, _, _ = attention.attend_retained(q, k, v, range(n - 1), scale)
    assert np.max(np.abs(o_wrong - o)) > 2e-2


# ---------------------------------------------------------------------------- C twin
def test_c_twin_matches_numpy_oracle():
    from oracle import c as oc

    lib = oc.load()
    rng = np.random.default_rng(10)
    L, n_q, n_kv, d = 3, 28, 4, 128
    pol = Policy(16, 5, 2, 9, 3)
    P, S, M, t = 4, 70, 3, 31
    n = P + S + M + t
    q = _rand_bits(rng, L, n_q, d)
    k, v = _rand_bits(rng, L, n, n_kv, d), _rand_bits(rng, L, n, n_kv, d)
    A = policy.retained_positions(P, S, M, t, pol)
    assert list(lib.retained(P, S, M, t, pol)) == A
    for tt in (0, 1, 5, 6, 7, 30, 200):
        assert list(lib.retained(P, S, M, tt, pol)) == policy.retained_positions(P, S, M, tt, pol)
    out, lse, used = lib.attend(q, k, v, A, 0.0883883, n_threads=2)
    assert used >= 1
    for layer in range(L):
        o_ref, lse_ref, _ = attention.attend_retained(q[layer], k[layer], v[layer], A, 0.0883883)
        assert np.max(np.abs(out[layer] - o_ref)) < 1e-12
        assert np.max(np.abs(lse[layer] - lse_ref)) < 1e-12
