"""Reliable-update schedule of SURVEY 8(c) O8, written out as a rule on a residual history (test helper).

Given h[k] = |r_{k+1}| / |b| after CGLS pass k (k = 0, 1, ...), the norm rmax0 = |r_0| / |b| the recurrence starts
from, delta and tol, a reliable update fires after pass k (1-based iteration k + 1) when

    h[k] < delta * max(rmax, h[k])  with  rmax = max of |r| / |b| since the last update (initially rmax0),   or
    h[k] <= tol,

and rmax restarts from the recomputed fp64 residual, which equals h[k] up to the drift of the inner recurrence.
The rule needs nothing but the history, so applying it to the fp64 history of oracle.cgnr predicts when
oracle.cgnr_mixed (and the CUDA solver) must fire: their inner recurrences follow the fp64 one to ~1e-6 relative.
`margin` reports how close any decision came to its threshold (relative), so that a test can tell a wrong schedule
from a coin flip on a threshold.
"""
from __future__ import annotations


def reliable_update_schedule(history, rmax0: float, delta: float, tol: float):
    """Returns (firing iterations, 1-based; smallest relative distance of any delta decision to its threshold)."""
    fired, rmax, margin = [], float(rmax0), float("inf")
    for k, h in enumerate(history):
        h = float(h)
        rmax = max(rmax, h)
        margin = min(margin, abs(h / (delta * rmax) - 1.0))
        if h < delta * rmax or h <= tol:
            fired.append(k + 1)
            rmax = h
            if h <= tol:
                break
    return fired, margin
