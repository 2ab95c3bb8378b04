"""Pins of oracle/prefill.py: library SDPA (causal, fp64), the decode oracle (Eq. 1 over [0, x]),
closed forms and a pure-Python brute force."""
import math

import numpy as np
import torch

from oracle import attention as o_attn
from oracle import prefill as o_pre


def _bits(x):
    return torch.tensor(np.asarray(x, dtype=np.float32)).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)


def _rand(seed, n_pos, n_tok, n_q=4, n_kv=2, d=16):
    rng = np.random.default_rng(seed)
    return (_bits(rng.standard_normal((n_tok, n_q, d))), _bits(rng.standard_normal((n_pos, n_kv, d))),
            _bits(rng.standard_normal((n_pos, n_kv, d))))


def test_matches_library_causal_sdpa_fp64():
    n = 37
    q, k, v = _rand(0, n, n)
    o, _ = o_pre.causal_attention(q, k, v, 0, 0.25)
    qt = torch.tensor(o_attn.bf16_bits_to_f64(q)).permute(1, 0, 2)  # [n_q, n, d]
    kt = torch.tensor(o_attn.bf16_bits_to_f64(k)).permute(1, 0, 2).repeat_interleave(2, dim=0)
    vt = torch.tensor(o_attn.bf16_bits_to_f64(v)).permute(1, 0, 2).repeat_interleave(2, dim=0)
    ref = torch.nn.functional.scaled_dot_product_attention(qt, kt, vt, is_causal=True, scale=0.25)
    assert np.allclose(o, ref.permute(1, 0, 2).numpy(), atol=1e-12)


def test_each_row_is_the_decode_oracle_over_its_prefix():
    q, k, v = _rand(1, 50, 20)
    o, lse = o_pre.causal_attention(q, k, v, 30, 0.3)  # positions 30..49
    for i in (0, 7, 19):
        o_ref, lse_ref, _ = o_attn.attend_retained(q[i], k, v, range(30 + i + 1), 0.3)
        assert np.allclose(o[i], o_ref, atol=1e-13) and np.allclose(lse[i], lse_ref, atol=1e-12)


def test_first_position_returns_v0_and_identical_keys_return_the_running_mean():
    q, k, v = _rand(2, 9, 9)
    o, lse = o_pre.causal_attention(q, k, v, 0, 1.0)
    assert np.allclose(o[0, 0], o_attn.bf16_bits_to_f64(v)[0, 0]) and np.allclose(o[0, 3], o_attn.bf16_bits_to_f64(v)[0, 1])
    k_same = np.broadcast_to(k[:1], k.shape).copy()
    o2, _ = o_pre.causal_attention(q, k_same, v, 0, 1.0)
    vf = o_attn.bf16_bits_to_f64(v)
    for x in range(9):
        assert np.allclose(o2[x, 2], vf[: x + 1, 1].mean(axis=0), atol=1e-13)


def test_brute_force_pure_python():
    q, k, v = _rand(3, 6, 3, n_q=2, n_kv=1, d=4)
    o, _ = o_pre.causal_attention(q, k, v, 3, 0.5)
    qf, kf, vf = (o_attn.bf16_bits_to_f64(a).tolist() for a in (q, k, v))
    for i in range(3):
        for h in range(2):
            x = 3 + i
            s = [sum(qf[i][h][e] * kf[y][0][e] for e in range(4)) * 0.5 for y in range(x + 1)]
            z = sum(math.exp(t) for t in s)
            want = [sum(math.exp(s[y]) / z * vf[y][0][e] for y in range(x + 1)) for e in range(4)]
            assert np.allclose(o[i, h], want, atol=1e-12)


# ---- the plain-C twin (oracle/c: murmur_oracle_prefill), used for the full-size every-row comparisons --------
def _rand_layers(seed, L, n_pos, n_tok, n_q=28, n_kv=4, d=128):
    rng = np.random.default_rng(seed)
    return (_bits(rng.standard_normal((L, n_tok, n_q, d))), _bits(rng.standard_normal((L, n_pos, n_kv, d))),
            _bits(rng.standard_normal((L, n_pos, n_kv, d))))


def test_c_twin_matches_the_numpy_oracle_to_1e_12():
    from oracle import c as oracle_c

    co = oracle_c.load()
    for seed, (L, n_pos, n_tok, pos_begin) in enumerate([(2, 90, 90, 0), (1, 150, 40, 110), (3, 33, 1, 32)]):
        q, k, v = _rand_layers(10 + seed, L, n_pos, n_tok)
        o_c, lse_c, used = co.prefill(q, k, v, pos_begin, 1.0 / math.sqrt(128), n_threads=1 + seed)
        assert used >= 1
        for layer in range(L):
            o, lse = o_pre.causal_attention(q[layer], k[layer], v[layer], pos_begin, 1.0 / math.sqrt(128))
            assert np.max(np.abs(o_c[layer] - o)) < 1e-12 and np.max(np.abs(lse_c[layer] - lse)) < 1e-12


def test_c_twin_matches_library_causal_sdpa_fp64_and_the_decode_twin():
    from oracle import c as oracle_c

    co = oracle_c.load()
    n = 70
    q, k, v = _rand_layers(20, 1, n, n, n_q=4, n_kv=2, d=16)
    o_c, lse_c, _ = co.prefill(q, k, v, 0, 0.25)
    qt = torch.tensor(o_attn.bf16_bits_to_f64(q[0])).permute(1, 0, 2)
    kt = torch.tensor(o_attn.bf16_bits_to_f64(k[0])).permute(1, 0, 2).repeat_interleave(2, dim=0)
    vt = torch.tensor(o_attn.bf16_bits_to_f64(v[0])).permute(1, 0, 2).repeat_interleave(2, dim=0)
    ref = torch.nn.functional.scaled_dot_product_attention(qt, kt, vt, is_causal=True, scale=0.25)
    assert np.allclose(o_c[0], ref.permute(1, 0, 2).numpy(), atol=1e-12)
    # row i is the decode twin (murmur_oracle_attend) over the retained set [0, i]
    for i in (0, 13, 69):
        o_d, lse_d, _ = co.attend(q[:, i], k, v, list(range(i + 1)), 0.25)
        assert np.allclose(o_c[:, i], o_d, atol=1e-13) and np.allclose(lse_c[:, i], lse_d, atol=1e-12)
    # a wrong causal boundary (y < x instead of y <= x) would make row 0 empty / change every row: row 0 must return v_0
    assert np.allclose(o_c[0, 0, 0], o_attn.bf16_bits_to_f64(v)[0, 0, 0])


def test_c_twin_rejects_bad_sizes():
    from oracle import c as oracle_c

    co = oracle_c.load()
    q, k, v = _rand_layers(30, 1, 10, 5, n_q=4, n_kv=2, d=16)
    try:
        co.prefill(q, k, v, 6, 0.25)  # positions 6..10 need 11 cache rows
    except RuntimeError:
        pass
    else:
        raise AssertionError("pos_begin + n_tok > n_pos must be refused")
