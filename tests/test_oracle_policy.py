"""Pins for oracle/policy.py, oracle/literal_sim.py and oracle/cost_model.py (no GPU).

Pins follow SURVEY.md section 8(c): I2, P1, P2, P3, P4, P5, P7 and special cases.  Each pin is
chosen so that a plausible mistake (off-by-one in l, window of w+1, wrong region for the
sinks, missing clamp) fails at least one of them.
"""
import itertools

import pytest

from oracle import cost_model, literal_sim, policy
from oracle.policy import Policy, WINDOW_OFF


# ---------------------------------------------------------------------------- I2
def _tiny_grid():
    for S, w_s, d, k_s in itertools.product((0, 1, 5, 9), (0, 1, 3, 6, 12), (0, 1, 4), (0, 2)):
        for w_o, k_o in itertools.product((0, 1, 3, 6), (0, 1, 2)):
            yield S, w_s, d, k_s, w_o, k_o


def test_I2_closed_form_equals_literal_simulation_exhaustive_tiny():
    """Closed-form predicate == Alg. 1 / Alg. 2 transcribed as set simulations, every step."""
    n_cases = 0
    for S, w_s, d, k_s, w_o, k_o in _tiny_grid():
        for P, M in ((0, 0), (2, 0), (1, 2)):
            pol = Policy(w_s, d, k_s, w_o, k_o)
            T = 12
            for t, A_sim, R_sim in literal_sim.simulate_hybrid(P, S, M, T, w_s, d, k_s, w_o, k_o):
                assert policy.retained_positions(P, S, M, t, pol) == A_sim, (P, S, M, t, pol)
                assert policy.resident_positions(P, S, M, t, pol) == R_sim, (P, S, M, t, pol)
                n_cases += 1
    assert n_cases > 10000


def test_I2_literal_alg1_matches_paper_line2_by_hand():
    """Alg. 1 line 2 evaluated by hand for n_sink=2, w=3, 1-based."""
    got = {j: c for j, c in literal_sim.simulate_output_eviction(2, 3, 7)}
    assert got[1] == {1}
    assert got[3] == {1, 2, 3}
    assert got[5] == {1, 2, 3, 4, 5}  # {1,2} U {3,4,5}
    assert got[6] == {1, 2, 4, 5, 6}  # token 3 is the first one evicted
    assert got[7] == {1, 2, 5, 6, 7}


def test_literal_alg2_window_by_hand():
    """Alg. 2 by hand: S=8, d=2, w=3: l = 0,0,1,2,3,4,5,5 (clamped at S-w)."""
    ls = [l for _t, l, _a, _r in literal_sim.simulate_speech_eviction(8, 2, 3, 0, 8)]
    assert ls == [0, 0, 1, 2, 3, 4, 5, 5]
    steps = list(literal_sim.simulate_speech_eviction(8, 2, 3, 0, 8))
    assert steps[0][2] == {0, 1, 2} and steps[0][3] == set(range(8))
    assert steps[3][2] == {2, 3, 4} and steps[3][3] == {2, 3, 4, 5, 6, 7}  # t=4: l=2


# ---------------------------------------------------------------------------- P1
@pytest.mark.parametrize("k_o,w_o", [(4, 64), (0, 5), (3, 0), (8, 256)])
def test_P1_output_region_counts_and_first_eviction(k_o, w_o):
    pol = Policy(WINDOW_OFF, 0, 0, w_o, k_o)
    P, S, M = 3, 7, 2
    base = P + S + M
    prev = None
    for t in range(1, k_o + w_o + 6):
        A = policy.retained_positions(P, S, M, t, pol)
        outs = [x - base for x in A if x >= base]
        assert len(outs) == min(t, k_o + w_o)
        if t == k_o + w_o + 1:
            # first eviction happens exactly now and removes u = k_o
            assert set(prev + [t - 1]) - set(outs) == {k_o}
        elif t <= k_o + w_o:
            assert outs == list(range(t))
        prev = outs


# ---------------------------------------------------------------------------- P2
@pytest.mark.parametrize("S,w_s,d", [(2250, 512, 256), (20, 6, 3), (10, 4, 0), (5, 9, 2)])
def test_P2_window_start_delay_then_plus_one_then_clamp(S, w_s, d):
    pol = Policy(w_s, d, 0, WINDOW_OFF, 0)
    l_prev = 0
    for t in range(1, S + d + 10):
        l = policy.window_start(S, t, pol)
        if t <= d:
            assert l == 0  # "l_j = 0 for j < d", 0-based step counter j0 = t-1
        if l_prev < max(0, S - w_s) and t > d:
            assert l == l_prev + 1  # "advances by one each step thereafter"
        assert l <= max(0, S - w_s)  # G10 clamp
        n_sp = sum(1 for x in policy.retained_positions(0, S, 0, t, pol) if x < S)
        assert n_sp == min(w_s, S)
        l_prev = l
    assert policy.window_start(S, d + 1, pol) == min(1, max(0, S - w_s))  # G7: l = 1 at t = d+1


# ---------------------------------------------------------------------------- P3
def test_P3_eq3_values_printed_in_paper(golden):
    for line in golden("eq3_ratio.txt"):
        L_s, T, n_sink, w, printed = line.split()
        L_s, T, n_sink, w = int(L_s), int(T), int(n_sink), int(w)
        a = cost_model.eq3_ratio_sum(L_s, T, n_sink, w)
        b = cost_model.eq3_ratio_closed(L_s, T, n_sink, w)
        assert abs(a - b) < 1e-12  # the two forms of Eq. 3 agree
        assert f"{a:.2f}" == printed  # 1.51 and 1.06


def test_P3_exact_attended_total_is_consistent_with_closed_form_count():
    pol = Policy(16, 8, 0, 12, 2)
    P, S, M, T = 4, 60, 0, 50
    total = cost_model.exact_attended_total(P, S, M, T, pol)
    assert total == sum(policy.retained_count_closed_form(P, S, M, t, pol) for t in range(1, T + 1))
    # full-cache cost / evicted cost > 1 and bounded by Eq. 3 style reasoning
    full = sum(P + S + M + t for t in range(1, T + 1))
    assert full > total


# ---------------------------------------------------------------------------- P4
def test_P4_monotone_sets():
    for S, w_s, d, k_s, w_o, k_o in [(30, 8, 4, 2, 6, 2), (12, 4, 0, 0, 3, 1), (9, 20, 3, 1, 40, 0)]:
        pol = Policy(w_s, d, k_s, w_o, k_o)
        P, M = 3, 1
        R_prev = set(policy.resident_positions(P, S, M, 0, pol))
        assert R_prev == set(range(P + S + M))
        for t in range(1, 40):
            newest = P + S + M + t - 1
            A = set(policy.retained_positions(P, S, M, t, pol))
            R = set(policy.resident_positions(P, S, M, t, pol))
            D = set(policy.dead_positions(P, S, M, t, pol))
            assert A <= R
            assert A <= R_prev | {newest}
            assert R <= R_prev | {newest}
            assert R | D == set(range(P + S + M + t)) and not (R & D)
            # R \ A is exactly the speech ahead of the window (G9)
            l = policy.window_start(S, t, pol)
            assert R - A == {P + r for r in range(S) if r >= l + w_s and r >= k_s}
            R_prev = R


# ---------------------------------------------------------------------------- P5
def test_P5_worked_example_table(golden):
    pol = Policy(w_speech=4, delay=2, n_sink_speech=0, w_out=3, n_sink_out=1)
    P, S, M, p = 2, 10, 0, 4
    rows = golden("worked_example_hybrid.txt")
    assert len(rows) == 8
    for line in rows:
        t_s, l_s, A_s, RA_s, blocks_s = [c.strip() for c in line.split("|")]
        t = int(t_s)
        A = policy.retained_positions(P, S, M, t, pol)
        R = policy.resident_positions(P, S, M, t, pol)
        assert policy.window_start(S, t, pol) == int(l_s)
        assert A == [int(x) for x in A_s.split()]
        assert sorted(set(R) - set(A)) == [int(x) for x in RA_s.split()]
        dead = set(policy.dead_positions(P, S, M, t, pol))
        length = P + S + M + t
        n_blocks = -(-length // p)
        live = [b for b in range(n_blocks)
                if not ((b + 1) * p <= length and all(x in dead for x in range(b * p, (b + 1) * p)))]
        assert live == [int(x) for x in blocks_s.split()]


# ---------------------------------------------------------------------------- P7 (soft)
def test_P7_table3_kept_percent(golden):
    """kept % ~ (S + n_sink + w) / (S + T) at the final state, S = 2250, T = 2770: within 0.5 pt of
    every printed row.  A whole-sequence reading of Alg. 1 (window evicting
    speech) would give 100*(4+256)/(2250+2770) = 5.2 %, far off the printed 50.0."""
    S, T = 2250, 2770
    for line in golden("table3_kept_pct.txt"):
        n_sink, w, printed = line.split()
        pol = Policy(WINDOW_OFF, 0, 0, int(w), int(n_sink))
        kept = len(policy.retained_positions(0, S, 0, T, pol))
        pct = 100.0 * kept / (S + T)
        assert abs(pct - float(printed)) < 0.5, (n_sink, w, pct, printed)


# ---------------------------------------------------------------------------- special cases
def test_G11_windows_off_keeps_everything():
    for P, S, M, t in [(0, 0, 0, 1), (4, 9, 2, 7), (64, 450, 0, 160)]:
        assert policy.retained_positions(P, S, M, t, policy.NO_EVICTION) == list(range(P + S + M + t))
        assert policy.dead_positions(P, S, M, t, policy.NO_EVICTION) == []
    pol = Policy(9, 0, 0, 7, 0)  # windows exactly the region sizes
    assert policy.retained_positions(2, 9, 0, 7, pol) == list(range(2 + 9 + 7))


def test_closed_form_count_matches_enumeration():
    for S, w_s, d, k_s, w_o, k_o in _tiny_grid():
        pol = Policy(w_s, d, k_s, w_o, k_o)
        for t in (0, 1, 2, 5, 11):
            assert policy.retained_count_closed_form(2, S, 1, t, pol) == len(
                policy.retained_positions(2, S, 1, t, pol))


def test_config2_steady_state_count():
    """64 + 512 + 4 + 256 = 836 retained tokens per sequence from t >= 260."""
    pol = Policy(512, 256, 0, 256, 4)
    assert len(policy.retained_positions(64, 2250, 0, 260, pol)) == 836
    assert len(policy.retained_positions(64, 2250, 0, 1500, pol)) == 836
    assert len(policy.retained_positions(64, 2250, 0, 259, pol)) == 835


def test_policy_rejects_negative():
    with pytest.raises(ValueError):
        Policy(-1, 0, 0, 0, 0)
