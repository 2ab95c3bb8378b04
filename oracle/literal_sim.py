"""Alg. 1 and Alg. 2 of the paper transcribed line by line (oracle, second implementation).

TEST INFRASTRUCTURE - see ``oracle/__init__.py``.

These simulators loop over decode steps and keep explicit Python sets, in the paper's own
index conventions, so they can be checked against PAPER.md:110-117 and 130-146 by eye.
They share nothing with ``oracle/policy.py`` (which evaluates a closed form per position);
the two must agree for every step (invariant I2 of the task statement).

Alg. 1, output region, 1-based token index i, decode step j:
    1: for each decode step j do
    2:   K <- {1..n_sink} U {max(1, j-w+1)..j}
    3:   Evict {k_i, v_i | i not in K} from C
    4: end for

Alg. 2, speech region, 0-based l:
    1: l <- 0
    2: for each decode step j do
    3:   if j >= d then l <- l + 1
    5:   K <- {l..l+w-1}
    6:   Evict {k_i, v_i | i not in K} from C
    7: end for
Readings applied to Alg. 2: the step counter is 0-based (j0 = t-1, G7); Eq. 2's
sinks {0..k_s-1} are kept as well (G6); tokens AHEAD of the window are masked, not removed
(G9); l is clamped to max(0, S-w) so the window parks at the end of the speech (G10).
"""
from __future__ import annotations

from typing import Iterator, List, Set, Tuple


def simulate_output_eviction(n_sink: int, w: int, n_steps: int) -> Iterator[Tuple[int, Set[int]]]:
    """Alg. 1 verbatim.  Yields (j, C_j): the 1-based output-token indices left in the cache
    after the eviction of decode step j (token j has just been appended)."""
    cache: Set[int] = set()
    for j in range(1, n_steps + 1):  # 1: for each decode step j
        cache.add(j)  # the j-th generation token enters the cache
        keep = set(range(1, n_sink + 1)) | set(range(max(1, j - w + 1), j + 1))  # 2
        cache = {i for i in cache if i in keep}  # 3: evict i not in K (permanent)
        yield j, set(cache)


def simulate_speech_eviction(
    S: int, d: int, w: int, n_sink: int, n_steps: int
) -> Iterator[Tuple[int, int, Set[int], Set[int]]]:
    """Alg. 2 with the readings in the module docstring.

    Yields (t, l, attended, resident) with 0-based speech indices, t = j0 + 1."""
    resident: Set[int] = set(range(S))  # speech tokens are prefilled
    l = 0  # 1: l <- 0
    for j0 in range(n_steps):  # 2: for each decode step j (0-based counter)
        if j0 >= d:  # 3: if j >= d then l <- l + 1
            l = l + 1
        l = min(l, max(0, S - w))  # G10: park at the end of the speech region
        window = set(range(l, l + w))  # 5: K <- {l..l+w-1}
        sinks = set(range(min(n_sink, S)))  # Eq. 2: {1..n_sink} kept
        # 6: evict what is not in K -- permanently only behind the trailing edge (G9)
        resident = {r for r in resident if r in sinks or r >= l}
        attended = {r for r in resident if r in sinks or r in window}
        yield j0 + 1, l, attended, set(resident)


def simulate_hybrid(
    P: int, S: int, M: int, n_steps: int, w_speech: int, delay: int, n_sink_speech: int,
    w_out: int, n_sink_out: int,
) -> Iterator[Tuple[int, List[int], List[int]]]:
    """Both policies on their disjoint regions ("a hybrid that combines both").

    Yields (t, A(t), R(t)) as sorted absolute positions."""
    out_iter = simulate_output_eviction(n_sink_out, w_out, n_steps)
    sp_iter = simulate_speech_eviction(S, delay, w_speech, n_sink_speech, n_steps)
    base = P + S + M
    fixed = list(range(P)) + list(range(P + S, P + S + M))  # system prompts: never evicted
    for (j, out_cache), (t, _l, sp_att, sp_res) in zip(out_iter, sp_iter):
        assert j == t
        out_abs = [base + (i - 1) for i in out_cache]  # 1-based i -> 0-based u
        attended = sorted(fixed + [P + r for r in sp_att] + out_abs)
        resident = sorted(fixed + [P + r for r in sp_res] + out_abs)
        yield t, attended, resident
