"""Lock-step parity criteria P1..P5 of SURVEY.md section 8(c) / DESIGN.md section 7.

The MCS map is chaotic (rounding differences grow x3-5 per MCS), so the GPU is compared with the
oracle one call at a time from a SHARED state; these helpers hold the pass criteria.  They use
numpy only and call neither the oracle nor the CUDA path themselves.
"""
import numpy as np

from .helpers import angle_diff

# Stated device-math errors (measured by test_gpu_parity.py::test_device_math_errors):
EPS_SINCOS = 7.5e-7      # abs error of one fast sin/cos on [0, 2pi] (MUFU.SIN/COS after one FMUL by 1/2pi)
ETA_FIELD = 6 * EPS_SINCOS   # abs error of one component of the six-neighbour field h
TOL_ANGLE = 1.0e-4       # north_star: "per-site angles must agree within 1e-4 rad (mod 2pi)"
TOL_DECISION = 1.0e-6    # north_star: decisions may differ only within 1e-6 of the threshold
FRAC_DECISION = 1.0e-6   # ... and for at most 1e-6 of the decisions


def check_metropolis(start, gpu, ora, proposals, met_p, met_u, sel):
    """P1 for the sites selected by the boolean mask `sel` (one colour pass, run by the oracle from
    exactly the neighbourhood the GPU saw).  start/gpu/ora/proposals: [R,L,L,L] fp32; met_p
    (fp64), met_u (fp32): the oracle's trace of that pass.

    Every GPU site must equal, BITWISE, its old value (reject) or the proposal (accept).  The
    decisions read off the two states must agree except where |u - p_oracle| <= 1e-6, for at
    most 1e-6 of the decisions.  Returns a dict of counts."""
    sb, gb, ob, pb = (a.view(np.uint32)[sel] for a in (start, gpu, ora, proposals))
    g_acc, g_rej = gb == pb, gb == sb
    assert np.all(g_acc | g_rej), "GPU produced an angle that is neither the old value nor the proposal"
    o_acc = ob == pb
    assert np.all(o_acc | (ob == sb))
    ambiguous = pb == sb                      # proposal bit-equal to the old angle: decision unreadable
    mism = (g_acc != o_acc) & ~ambiguous
    n = int(sb.size)
    n_mism = int(mism.sum())
    if n_mism:
        d = np.abs(met_u[sel][mism].astype(np.float64) - np.minimum(met_p[sel][mism], 2.0))
        assert np.all(d <= TOL_DECISION), f"{n_mism} decision mismatches, worst {d.max():.3e} away from the threshold"
    assert n_mism <= max(1, int(np.ceil(FRAC_DECISION * n))), f"{n_mism} mismatching decisions in {n}"
    return {"decisions": n, "mismatch": n_mism, "accept_frac": float(g_acc.mean())}


def check_overrelax(gpu, ora, or_h, sel, eta=ETA_FIELD):
    """P2 for the sites selected by `sel` (one colour pass).  A site passes if |dtheta| <= 1e-4
    (mod 2pi) or |dtheta| <= 4 eta / |h_i| + 2e-6, with |h_i| from the oracle: the reflection
    theta' = 2 arg(h) - theta has condition number 2/|h|, so where the field nearly vanishes no
    fp32 implementation can meet an absolute 1e-4 (SURVEY.md finding 4).  Returns the statistics."""
    d = angle_diff(gpu[sel], ora[sel])
    h = or_h[sel]
    ok1 = d <= TOL_ANGLE
    ok2 = d <= 4.0 * eta / np.maximum(h, 1e-300) + 2e-6
    bad = ~(ok1 | ok2)
    assert not bad.any(), (f"{int(bad.sum())} sites violate both clauses; worst dtheta={d[bad].max():.3e} "
                           f"at |h|={h[bad][np.argmax(d[bad])]:.3e}")
    return {"sites": int(d.size), "max": float(d.max()), "rms": float(np.sqrt((d ** 2).mean())),
            "frac_gt_1e-4": float((~ok1).mean()), "frac_gt_1e-5": float((d > 1e-5).mean())}


def check_observables(gpu_obs, ora_obs, N):
    """P3.  |dE| <= 1e-6 * 3N, |dMx|, |dMy| <= 1e-6 * N; M2, M4 follow from Mx, My."""
    g, o = np.asarray(gpu_obs), np.asarray(ora_obs)
    dE = np.abs(g[:, 0] - o[:, 0]).max()
    dM = np.abs(g[:, 1:3] - o[:, 1:3]).max()
    assert dE <= 1e-6 * 3 * N, f"|dE| = {dE:.3e} > {1e-6 * 3 * N:.3e}"
    assert dM <= 1e-6 * N, f"|dM| = {dM:.3e} > {1e-6 * N:.3e}"
    m2 = g[:, 1] ** 2 + g[:, 2] ** 2
    assert np.allclose(g[:, 3], m2, rtol=1e-14, atol=0)
    assert np.allclose(g[:, 4], m2 * m2, rtol=1e-14, atol=0)
    return {"dE_over_3N": float(dE / (3 * N)), "dM_over_N": float(dM / N)}


def check_pt(gpu_perm, ora_perm, pt_p, pt_u):
    """P4.  Identical slot_at_rank except pairs whose |u - p| <= 1e-6."""
    gpu_perm, ora_perm = np.asarray(gpu_perm), np.asarray(ora_perm)
    diff = np.nonzero(gpu_perm != ora_perm)[0]
    for k in diff:
        pair = k if (k < len(pt_p) and not np.isnan(pt_p[k])) else k - 1
        assert abs(pt_u[pair] - min(pt_p[pair], 2.0)) <= TOL_DECISION, f"PT pair {pair} decided differently"
    return {"pairs_differing": int(len(diff) // 2)}
