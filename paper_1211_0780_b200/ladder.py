"""Temperature ladders with temperature-independent swap acceptance.

The paper chose its 34 (13) temperatures "such that the acceptance rate of swaps is independent of the temperatures"
and does not print them.  This module holds the host-side arithmetic of that choice -- none of the Monte Carlo step:
the acceptance counts come from the library (xy_get_accept_counts), the new ladder goes back through xy_set_betas.

respace() is one step of the classic feedback: for neighbouring temperatures the rejection rate 1 - a_k of pair k grows
(to first order linearly) with its spacing, so spacings are rescaled by (target rejection / measured rejection)^gamma
and renormalised to keep both end temperatures fixed.
"""
import numpy as np


def respace(betas, acceptance, gamma=0.5, floor=1e-3):
    """New ladder with the same end points.  betas [R] increasing; acceptance [R-1] measured per pair (k, k+1)."""
    b = np.asarray(betas, dtype=np.float64)
    a = np.clip(np.asarray(acceptance, dtype=np.float64), 0.0, 1.0)
    if b.size < 3:
        return b.copy()
    rej = np.maximum(1.0 - a, floor)
    d = np.diff(b) * (rej.mean() / rej) ** gamma
    d *= (b[-1] - b[0]) / d.sum()
    out = np.concatenate([[b[0]], b[0] + np.cumsum(d)])
    out[-1] = b[-1]
    return out


def measure_swap_acceptance(xy, n_mcs):
    """Per-pair acceptance over the next n_mcs steps of `xy` (pair k is attempted on every other step)."""
    _, pt0 = xy.get_accept_counts()
    t0 = int(xy.get_counters()[2])
    xy.mcs(n_mcs)
    _, pt1 = xy.get_accept_counts()
    R = xy.R
    k = np.arange(R - 1)
    steps = t0 + np.arange(n_mcs)
    attempts = np.array([np.count_nonzero((steps & 1) == (kk & 1)) for kk in k], dtype=np.float64)
    return (pt1 - pt0).astype(np.float64) / np.maximum(attempts, 1.0)


def equalise_swap_acceptance(xy, betas, rounds=6, n_mcs=400, burn=100, gamma=0.5):
    """Iterates respace() on a running system.  Returns (betas, list of per-round acceptance arrays)."""
    b = np.asarray(betas, dtype=np.float64).copy()
    history = []
    for _ in range(rounds):
        xy.set_betas(b)
        xy.mcs(burn)
        a = measure_swap_acceptance(xy, n_mcs)
        history.append(a)
        b = respace(b, a, gamma=gamma)
    xy.set_betas(b)
    xy.mcs(burn)
    history.append(measure_swap_acceptance(xy, n_mcs))
    return b, history
