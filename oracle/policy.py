"""Retained set A(t) and resident set R(t) of MURMUR's hybrid eviction policy (oracle).

TEST INFRASTRUCTURE - see ``oracle/__init__.py``.

Sequence layout ("[system prompt] [speech tokens] [system prompt] [text
tokens]"), 0-based absolute positions:

    PRE    = [0, P)
    SPEECH = [P, P+S)            region-relative index r
    MID    = [P+S, P+S+M)
    OUT    = [P+S+M, P+S+M+t)    region-relative index u; t counts the output tokens in the
                                 cache INCLUDING the one just appended (PAPER.md:101, 115:
                                 "j-th generation token", K contains j)

Rules followed (every reading is listed in DESIGN.md section "Readings"):

* Output tokens, Alg. 1: keep {1..n_sink} U {max(1, j-w+1)..j}, 1-based
  in the output region, j = t.  0-based: keep u < k_o or u >= t - w_o.
* Speech tokens, Eq. 2 + Alg. 2: a window of w speech tokens starting at
  l; l = 0 during a delay of d steps, then +1 per step ("if j >= d then l <- l+1" with the
  0-based step counter j0 = t-1, hence l = max(0, t - d)); sinks {0..k_s-1} of Eq. 2 kept.
  The window parks at the end of the speech region: l <= max(0, S - w_s)   (reading G10).
* System prompts are never evicted (policies exist only for speech and
  output tokens).
* Hybrid = both rules on their disjoint regions.

A(t) is what attention sees at step t.  A token is *dead* (permanently removable) once it
is behind the trailing edge of its window and is not a sink; speech tokens ahead of the
window are resident but not attended (reading G9), so R(t) = A(t) U {speech ahead}.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import List

WINDOW_OFF = 0x7FFFFFFF  # window >= any length: nothing is ever evicted (reading G11)


@dataclass(frozen=True)
class Policy:
    """Per-sequence policy parameters (paper names in brackets)."""

    w_speech: int  # speech window      [w of Alg. 2]
    delay: int  # delay steps        [d of Alg. 2]
    n_sink_speech: int  # speech sinks       [n_sink of Eq. 2]; Alg. 2 has none -> 0
    w_out: int  # output window      [w of Alg. 1]
    n_sink_out: int  # output sinks       [n_sink of Alg. 1]

    def __post_init__(self):
        for name in ("w_speech", "delay", "n_sink_speech", "w_out", "n_sink_out"):
            v = getattr(self, name)
            if not isinstance(v, int) or v < 0:
                raise ValueError(f"{name} must be a non-negative int, got {v!r}")


NO_EVICTION = Policy(WINDOW_OFF, 0, 0, WINDOW_OFF, 0)


def window_start(S: int, t: int, pol: Policy) -> int:
    """l(t): first speech index of the window at step t (Alg. 2 lines 1-4 + end clamp)."""
    return min(max(0, t - pol.delay), max(0, S - pol.w_speech))


def keep_speech(r: int, S: int, t: int, pol: Policy) -> bool:
    """Eq. 2 sinks U Alg. 2 window {l..l+w-1}."""
    l = window_start(S, t, pol)
    return r < pol.n_sink_speech or (l <= r < l + pol.w_speech)


def keep_out(u: int, t: int, pol: Policy) -> bool:
    """Alg. 1 line 2 translated to 0-based u = i - 1."""
    return u < pol.n_sink_out or u >= t - pol.w_out


def dead_speech(r: int, S: int, t: int, pol: Policy) -> bool:
    """Behind the trailing edge and not a sink: can never be attended again."""
    return r >= pol.n_sink_speech and r < window_start(S, t, pol)


def dead_out(u: int, t: int, pol: Policy) -> bool:
    return u >= pol.n_sink_out and u < t - pol.w_out


def retained_positions(P: int, S: int, M: int, t: int, pol: Policy) -> List[int]:
    """A(t): sorted absolute positions attention sees at step t (per-position predicate)."""
    out: List[int] = []
    for x in range(P):
        out.append(x)  # prefix system prompt: always kept
    for r in range(S):
        if keep_speech(r, S, t, pol):
            out.append(P + r)
    for x in range(P + S, P + S + M):
        out.append(x)  # second system prompt: always kept
    base = P + S + M
    for u in range(t):
        if keep_out(u, t, pol):
            out.append(base + u)
    return out


def resident_positions(P: int, S: int, M: int, t: int, pol: Policy) -> List[int]:
    """R(t): sorted absolute positions still in memory at step t (everything not dead)."""
    out: List[int] = list(range(P))
    for r in range(S):
        if not dead_speech(r, S, t, pol):
            out.append(P + r)
    out.extend(range(P + S, P + S + M))
    base = P + S + M
    for u in range(t):
        if not dead_out(u, t, pol):
            out.append(base + u)
    return out


def dead_positions(P: int, S: int, M: int, t: int, pol: Policy) -> List[int]:
    """Complement of R(t) inside [0, P+S+M+t)."""
    out: List[int] = []
    for r in range(S):
        if dead_speech(r, S, t, pol):
            out.append(P + r)
    base = P + S + M
    for u in range(t):
        if dead_out(u, t, pol):
            out.append(base + u)
    return out


def retained_count_closed_form(P: int, S: int, M: int, t: int, pol: Policy) -> int:
    """|A(t)| = P + M + |([0,k_s) U [l,l+w_s)) n [0,S)| + min(t, k_o + w_o)."""
    l = window_start(S, t, pol)
    sinks = min(pol.n_sink_speech, S)
    win_lo = min(l, S)
    win_hi = min(l + pol.w_speech, S)
    window_outside_sinks = max(0, win_hi - max(win_lo, sinks))
    return P + M + sinks + window_outside_sinks + min(t, pol.n_sink_out + pol.w_out)
