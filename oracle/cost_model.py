"""Eq. 3 theoretical attention-cost ratio (oracle helper, used as a pin).

TEST INFRASTRUCTURE - see ``oracle/__init__.py``.

PAPER.md:148-152, Eq. 3:
    rho = sum_{j=1..T} (L_s + j) / sum_{j=1..T} (n_sink + w + j)
        = (L_s T + T(T+1)/2) / ((n_sink + w) T + T(T+1)/2)
The paper prints rho ~ 1.51 for (n_sink=4, w=1024) and ~ 1.06 for (n_sink=512, w=1536) at
L_s ~ 2250, T ~ 2700.  Note the model charges n_sink + w + j per step for
*either* policy (it swaps L_s for n_sink + w even for output eviction); the exact count of
attended tokens under the hybrid rule is ``exact_attended_total`` below and differs - that
is a property of the paper's simplified model, not a bug (pin P3).
"""
from __future__ import annotations

from . import policy as _pol


def eq3_ratio_sum(L_s: int, T: int, n_sink: int, w: int) -> float:
    """Left form of Eq. 3: the two sums written out."""
    num = sum(L_s + j for j in range(1, T + 1))
    den = sum(n_sink + w + j for j in range(1, T + 1))
    return num / den


def eq3_ratio_closed(L_s: int, T: int, n_sink: int, w: int) -> float:
    """Right form of Eq. 3."""
    tri = T * (T + 1) / 2
    return (L_s * T + tri) / ((n_sink + w) * T + tri)


def exact_attended_total(P: int, S: int, M: int, T: int, pol: _pol.Policy) -> int:
    """sum_{t=1..T} |A(t)| under the hybrid rule of ``oracle.policy``."""
    return sum(len(_pol.retained_positions(P, S, M, t, pol)) for t in range(1, T + 1))
