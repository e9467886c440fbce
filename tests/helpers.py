"""Test-side helpers that belong to neither the oracle nor the CUDA path.

* an independent, from-the-definition numpy Philox4x32-10 (used to PREDICT what the oracle and
  the GPU must draw; it is itself pinned by the known-answer vectors in tests/golden/),
* angle comparison modulo 2 pi, replica-scatter error bars, and
* brute-force definitions on tiny lattices (explicit bond loops, L=2 quadrature).
"""
import numpy as np

TWO_PI_F = np.float32(6.2831855)
STREAM_INIT, STREAM_MET_BLACK, STREAM_MET_WHITE, STREAM_PT = 0, 1, 2, 3


def philox4x32_10_np(c0, c1, c2, c3, k0, k1):
    """Vectorised Philox4x32-10; every argument broadcastable integer arrays < 2**32."""
    M0, M1 = np.uint64(0xD2511F53), np.uint64(0xCD9E8D57)
    W0, W1 = np.uint64(0x9E3779B9), np.uint64(0xBB67AE85)
    mask = np.uint64(0xFFFFFFFF)
    c0, c1, c2, c3, k0, k1 = np.broadcast_arrays(*[np.asarray(a, dtype=np.uint64) for a in (c0, c1, c2, c3, k0, k1)])
    c0, c1, c2, c3, k0, k1 = [a.copy() for a in (c0, c1, c2, c3, k0, k1)]
    for rnd in range(10):
        if rnd > 0:
            k0 = (k0 + W0) & mask
            k1 = (k1 + W1) & mask
        p0 = M0 * c0
        p1 = M1 * c2
        n0 = (p1 >> np.uint64(32)) ^ c1 ^ k0
        n1 = p1 & mask
        n2 = (p0 >> np.uint64(32)) ^ c3 ^ k1
        n3 = p0 & mask
        c0, c1, c2, c3 = n0, n1, n2, n3
    return [a.astype(np.uint32) for a in (c0, c1, c2, c3)]


def u24(w):
    return (np.asarray(w, dtype=np.uint32) >> np.uint32(8)).astype(np.float32) * np.float32(2.0 ** -24)


def site_words(L, slot, c2, stream, seed):
    """Philox words [4, L,L,L] of counter (i>>2, slot, c2, stream) for every natural site index i."""
    i = np.arange(L ** 3, dtype=np.uint64).reshape(L, L, L)
    W = philox4x32_10_np(i >> np.uint64(2), slot, c2, stream, seed & 0xFFFFFFFF, seed >> 32)
    return np.stack(W), i


def predicted_init(L, R, seed):
    out = np.empty((R, L, L, L), dtype=np.float32)
    for r in range(R):
        W, i = site_words(L, r, 0, STREAM_INIT, seed)
        w = np.take_along_axis(W, (i & np.uint64(3)).astype(np.int64)[None], axis=0)[0]
        out[r] = TWO_PI_F * u24(w)
    return out


def predicted_proposals(L, R, n_met, seed, slots=None):
    """(theta_new, u) every site would draw in Metropolis sweep number n_met (only `slots` filled if given)."""
    z, y, x = np.meshgrid(np.arange(L), np.arange(L), np.arange(L), indexing="ij")
    colour = (x + y + z) & 1
    prop = np.empty((R, L, L, L), dtype=np.float32)
    uacc = np.empty((R, L, L, L), dtype=np.float32)
    for r in (range(R) if slots is None else slots):
        Wb, i = site_words(L, r, n_met, STREAM_MET_BLACK, seed)
        Ww, _ = site_words(L, r, n_met, STREAM_MET_WHITE, seed)
        W = np.where(colour[None] == 0, Wb, Ww)
        p = ((i >> np.uint64(1)) & np.uint64(1)).astype(np.int64)
        w_prop = np.take_along_axis(W, (2 * p)[None], axis=0)[0]
        w_acc = np.take_along_axis(W, (2 * p + 1)[None], axis=0)[0]
        prop[r] = TWO_PI_F * u24(w_prop)
        uacc[r] = u24(w_acc)
    return prop, uacc


def colour_mask(L):
    z, y, x = np.meshgrid(np.arange(L), np.arange(L), np.arange(L), indexing="ij")
    return (x + y + z) & 1


def angle_diff(a, b):
    d = np.abs(np.asarray(a, dtype=np.float64) - np.asarray(b, dtype=np.float64)) % (2 * np.pi)
    return np.minimum(d, 2 * np.pi - d)


def mean_and_err_over_replicas(series):
    """series[t, r]: independent replicas r.  Mean of per-replica means, error from their scatter."""
    per = np.asarray(series, dtype=np.float64).mean(axis=0)
    return per.mean(), per.std(ddof=1) / np.sqrt(per.size)


def brute_force_observables(theta):
    """E, Mx, My, M2, M4 of ONE configuration [L,L,L] by explicit python loops over bonds."""
    import math
    L = theta.shape[0]
    t = theta.astype(np.float64)
    E = 0.0
    for z in range(L):
        for y in range(L):
            for x in range(L):
                a = t[z, y, x]
                E -= math.cos(a - t[z, y, (x + 1) % L])
                E -= math.cos(a - t[z, (y + 1) % L, x])
                E -= math.cos(a - t[(z + 1) % L, y, x])
    Mx = float(np.sum(np.cos(t)))
    My = float(np.sum(np.sin(t)))
    M2 = Mx * Mx + My * My
    return np.array([E, Mx, My, M2, M2 * M2])


def exact_mean_energy_L2(beta, M=10):
    """<E> of the 2x2x2 periodic XY model by a direct 7-D periodic-trapezoid quadrature.

    With L=2 the +mu and -mu neighbours coincide, so H = -2 sum_{12 cube edges} cos(ti - tj).
    Global rotation invariance fixes spin 0 at angle 0; the other seven angles run over an
    M-point uniform grid each (spectrally accurate for a periodic analytic integrand)."""
    g = 2 * np.pi * np.arange(M) / M
    ang = [np.zeros(1)] + [g] * 7
    shape = lambda v: [M if (k == v and v > 0) else 1 for k in range(1, 8)]
    th = [ang[v].reshape(shape(v)) for v in range(8)]
    S = 0.0
    for v in range(8):
        for bit in (1, 2, 4):
            if not v & bit:
                S = S + np.cos(th[v] - th[v | bit])
    E = -2.0 * S
    w = np.exp(-beta * (E - E.min()))
    return float((E * w).sum() / w.sum())
