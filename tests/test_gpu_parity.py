"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element.

Protocol: the MCS map is chaotic, so every comparison is
LOCK-STEP -- both sides start one call from the same state and counters.  A sweep is two colour
passes; the oracle is run pass by pass from exactly the neighbourhood the GPU saw (the white
pass from the GPU's own black result), so each decision / reflection is compared like for like.
"""
import os

import numpy as np
import pytest

from paper_1211_0780_b200 import inputs
from . import helpers as H
from . import parity as P

pytestmark = pytest.mark.gpu
SEED = inputs.SEED
NCPU = max(1, min(32, os.cpu_count() or 1))

# (L, R): several tiles in y and z, ragged row lengths (L/8 = 1, 3, 5 float4 per row), R = 1
SHAPES = [(8, 8), (16, 3), (24, 5), (32, 16), (40, 2), (48, 1), (64, 4)]


def make(xy_mod, oracle_mod, L, R, betas=None, seed=SEED):
    betas = inputs.beta_ladder(0.44, 0.47, R) if betas is None else np.asarray(betas, dtype=np.float64)
    xy = xy_mod.XY(L, R, betas, seed)
    ora = oracle_mod.XYOracle(L, R, betas, seed, threads=NCPU)
    return xy, ora


def states_for(L, R):
    yield "uniform", inputs.uniform_state(L, R, 11)
    yield "smooth", inputs.smooth_state(L, R, 12)


def metropolis_lockstep(xy, ora, S, t, slots=None):
    """One GPU Metropolis sweep from state S with n_met = t, checked pass by pass (P1)."""
    L, R = xy.L, xy.R
    col = H.colour_mask(L)
    xy.set_state(S); xy.set_counters([t, 0, 0])
    perm = xy.get_perm()
    xy.metropolis_sweep()
    G = xy.get_state()
    prop, _ = H.predicted_proposals(L, R, t, SEED, slots)
    ora.set_perm(perm); ora.set_counters([t, 0, 0]); ora.set_active_slots(slots)
    out = []
    start = S
    for c in (0, 1):
        sel = np.zeros((R, L, L, L), dtype=bool)
        sel[list(range(R)) if slots is None else list(slots)] = (col == c)
        ora.set_state(start)
        tr = ora.enable_trace(met=True)
        ora.metropolis_pass(c)
        out.append(P.check_metropolis(start, G, ora.get_state(), prop, tr["met_p"], tr["met_u"], sel))
        start = np.where(col[None] == 0, G, S)          # the GPU's black result + the untouched white sites
    ora.enable_trace()
    # untouched sites of other slots / nothing else changed
    assert np.array_equal(xy.get_counters(), [t + 1, 0, 0])
    return out


def overrelax_lockstep(xy, ora, S, slots=None):
    L, R = xy.L, xy.R
    col = H.colour_mask(L)
    xy.set_state(S)
    xy.overrelax_sweep()
    G = xy.get_state()
    ora.set_active_slots(slots)
    out = []
    start = S
    for c in (0, 1):
        sel = np.zeros((R, L, L, L), dtype=bool)
        sel[list(range(R)) if slots is None else list(slots)] = (col == c)
        ora.set_state(start)
        tr = ora.enable_trace(overrelax=True)
        ora.overrelax_pass(c)
        out.append(P.check_overrelax(G, ora.get_state(), tr["or_h"], sel))
        start = np.where(col[None] == 0, G, S)
    ora.enable_trace()
    return out, G


# ---- a1 / device math -------------------------------------------------------------------------
def test_device_philox_known_answers_and_random_counters(xy_mod):
    kat = []
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")):
        line = line.split("#")[0].split()
        if len(line) == 10:
            kat.append([int(v, 16) for v in line])
    assert len(kat) >= 3
    for row in kat:
        out = xy_mod.debug_philox(np.array([row[0:4]], dtype=np.uint32), row[4], row[5])
        assert [int(v) for v in out[0]] == row[6:10]
    rng = np.random.default_rng(5)
    ctr = rng.integers(0, 2 ** 32, size=(4096, 4), dtype=np.uint64).astype(np.uint32)
    k0, k1 = 0x12110780, 0xDEADBEEF
    out = xy_mod.debug_philox(ctr, k0, k1)
    ref = np.stack(H.philox4x32_10_np(ctr[:, 0], ctr[:, 1], ctr[:, 2], ctr[:, 3], k0, k1), axis=1)
    assert np.array_equal(out, ref)


def test_device_math_errors(xy_mod):
    """The stated errors of the kernels' fast math (parity.EPS_SINCOS and DESIGN.md section 6)."""
    rng = np.random.default_rng(6)
    x = np.concatenate([rng.random(1 << 20) * 2 * np.pi, [0.0, np.pi / 2, np.pi, 3 * np.pi / 2, 6.2831855],
                        (np.arange(1 << 16) * (2 * np.pi / (1 << 16)))]).astype(np.float32)
    c, s = xy_mod.debug_sincos(x)
    ec = c.astype(np.float64) - np.cos(x.astype(np.float64))
    es = s.astype(np.float64) - np.sin(x.astype(np.float64))
    print(f"sincos: max|err| cos {np.abs(ec).max():.3e} sin {np.abs(es).max():.3e}; bias cos {ec.mean():.2e} sin {es.mean():.2e};"
          f" rms {np.sqrt((ec ** 2).mean()):.2e}")
    assert np.abs(ec).max() <= P.EPS_SINCOS and np.abs(es).max() <= P.EPS_SINCOS
    assert abs(ec.mean()) < 1e-7 and abs(es.mean()) < 2e-8      # MUFU.COS carries a -7e-8 mean error
    # the fp64 sin / cos of the settlement of close decisions (sincos_0_2pi): libm-grade on [0, 2 pi]
    xd = np.concatenate([rng.random(1 << 20) * 2 * np.pi, x[-70000:].astype(np.float64), np.arange(9) * (np.pi / 4),
                         np.nextafter(np.arange(1, 9) * (np.pi / 4), 0), np.nextafter(np.arange(1, 9) * (np.pi / 4), 7), [6.2831854820251465]])
    cd, sd = xy_mod.debug_sincos64(xd)
    ref_c, ref_s = np.cos(xd.astype(np.longdouble)), np.sin(xd.astype(np.longdouble))
    e64 = max(float(np.abs(cd - ref_c).max()), float(np.abs(sd - ref_s).max()))
    print(f"sincos64: max|err| {e64:.3e}")
    assert e64 <= 2.5e-16
    phi = rng.random(1 << 20) * 2 * np.pi
    r = np.exp(rng.uniform(np.log(1e-6), np.log(6.0), size=phi.size))
    hx, hy = (r * np.cos(phi)).astype(np.float32), (r * np.sin(phi)).astype(np.float32)
    a = xy_mod.debug_atan2(hy, hx)
    ref = np.arctan2(hy.astype(np.float64), hx.astype(np.float64)) % (2 * np.pi)
    ea = H.angle_diff(a, ref)
    print(f"atan2: max|err| {ea.max():.3e}")
    assert ea.max() <= 8e-7          # half an ulp at 2 pi is 2.4e-7; polynomial 2.5e-7; rcp + octant folding the rest
    assert a.min() >= 0.0 and a.max() <= 6.2831855
    for yy, xx, want in ((0.0, 1.0, 0.0), (1.0, 0.0, np.pi / 2), (0.0, -1.0, np.pi), (-1.0, 0.0, 3 * np.pi / 2),
                         (1.0, 1.0, np.pi / 4), (-1.0, -1.0, 5 * np.pi / 4)):
        got = xy_mod.debug_atan2(np.array([yy]), np.array([xx]))[0]
        assert abs(got - want) <= 6e-7


@pytest.mark.parametrize("L,R,beta_hi", [(32, 4, 0.47), (16, 3, 1.5)])
def test_fast_path_window(xy_mod, oracle_mod, L, R, beta_hi):
    """The fp32 fast path of the Metropolis decision may only be trusted outside the window
    |u - p_fast| >= |beta| * 4e-5 + 1.5e-6 (xy_device.cuh): measure |p_fast - p_oracle| on every site
    (XY_OPT_TRACE records p_fast) and require it to stay inside that window, with its u-rounding of
    2^-24, wherever p <= 1 could decide anything."""
    betas = inputs.beta_ladder(0.44, beta_hi, R)
    xy, ora = make(xy_mod, oracle_mod, L, R, betas=betas)
    xy.set_option(xy_mod.XY_OPT_TRACE, 1)
    col = H.colour_mask(L)
    for name, S in states_for(L, R):
        xy.set_state(S); xy.set_counters([5, 0, 0])
        ora.set_counters([5, 0, 0])
        xy.metropolis_sweep()
        pf = xy.debug_get_trace().astype(np.float64)
        G = xy.get_state()
        start = S
        worst = 0.0
        for c in (0, 1):
            ora.set_state(start)
            tr = ora.enable_trace(met=True)
            ora.metropolis_pass(c)
            sel = np.broadcast_to(col == c, S.shape)
            p = tr["met_p"][sel]
            d = np.abs(np.minimum(pf[sel], 1.0) - np.minimum(p, 1.0))           # only p <= 1 can change a decision
            window = (np.abs(betas.astype(np.float32)).astype(np.float64) * 4e-5 + 1.5e-6)[:, None]
            ratio = (d.reshape(R, -1) + 2.0 ** -24) / window
            worst = max(worst, float(ratio.max()))
            start = np.where(col[None] == 0, G, S)
        ora.enable_trace()
        print(L, R, name, "max (|p_fast - p| + 2^-24) / window =", worst)
        assert worst < 0.5, "the fast path's error must stay well inside the re-evaluation window"


# ---- a0 -------------------------------------------------------------------------------------
@pytest.mark.parametrize("L,R", [(8, 8), (24, 3), (32, 4)])
def test_init_random_is_bit_exact(xy_mod, oracle_mod, L, R):
    xy, ora = make(xy_mod, oracle_mod, L, R)
    xy.init_random(); ora.init_random()
    G = xy.get_state()
    assert np.array_equal(G.view(np.uint32), H.predicted_init(L, R, SEED).view(np.uint32))
    assert np.array_equal(G.view(np.uint32), ora.get_state().view(np.uint32))
    xy.init_ordered(0.25)
    assert np.all(xy.get_state() == np.float32(0.25))


@pytest.mark.parametrize("L,R", [(8, 2), (40, 3)])
def test_state_roundtrip_host_and_device(xy_mod, L, R):
    import torch
    xy = xy_mod.XY(L, R, inputs.beta_ladder(0.4, 0.5, R), SEED)
    S = inputs.uniform_state(L, R, 3)
    xy.set_state(S)
    assert np.array_equal(xy.get_state().view(np.uint32), S.view(np.uint32))
    d = torch.from_numpy(S).cuda()
    xy.init_ordered(0.0)
    xy.set_state(d)
    out = torch.empty_like(d)
    xy.get_state(out)
    assert torch.equal(out, d)


# ---- a2 -------------------------------------------------------------------------------------
@pytest.mark.parametrize("L,R", SHAPES)
def test_metropolis_lockstep(xy_mod, oracle_mod, L, R):
    xy, ora = make(xy_mod, oracle_mod, L, R)
    for name, S in states_for(L, R):
        for t in (0, 7):
            stats = metropolis_lockstep(xy, ora, S, t)
            print(L, R, name, t, stats)
            assert 0.2 < stats[0]["accept_frac"] < 0.95
    met, _ = xy.get_accept_counts()
    assert met.sum() > 0


def test_metropolis_other_tilings_give_identical_states(xy_mod):
    """The tiling is an implementation detail: any valid (TILE_Y, TILE_Z) gives the same bits."""
    L, R = 32, 3
    S = inputs.uniform_state(L, R, 21)
    ref = None
    for ty, tz in ((32, 32), (8, 8), (16, 4), (4, 2), (2, 16)):
        xy = xy_mod.XY(L, R, inputs.beta_ladder(0.45, 0.46, R), SEED)
        xy.set_option(xy_mod.XY_OPT_TILE_Z, tz); xy.set_option(xy_mod.XY_OPT_TILE_Y, ty)
        xy.set_state(S); xy.metropolis_sweep(); xy.overrelax_sweep()
        G = xy.get_state()
        obs = xy.measure()
        if ref is None:
            ref, ref_obs = G, obs
        assert np.array_equal(G.view(np.uint32), ref.view(np.uint32)), (ty, tz)
        # the fp32 site terms are grouped per thread and plane before the fp64 accumulation, so the
        # grouping (not the result beyond fp32 rounding) depends on the tiling: P3's bound applies
        assert np.abs(obs[:, 0] - ref_obs[:, 0]).max() <= 1e-6 * 3 * L ** 3
        assert np.abs(obs[:, 1:3] - ref_obs[:, 1:3]).max() <= 1e-6 * L ** 3


def test_metropolis_extreme_betas(xy_mod, oracle_mod):
    """beta = 0 accepts everything (state predictable from Philox alone, O1); beta huge and an
    ordered start accepts nothing (O3); negative beta is legal (antiferromagnet)."""
    L, R = 16, 4
    xy, ora = make(xy_mod, oracle_mod, L, R, betas=[0.0, 1e30, -0.3, 0.0])
    S = inputs.ordered_state(L, R)
    xy.set_state(S); xy.set_counters([3, 0, 0]); xy.metropolis_sweep()
    G = xy.get_state()
    prop, _ = H.predicted_proposals(L, R, 3, SEED)
    for r in (0, 3):
        assert np.array_equal(G[r].view(np.uint32), prop[r].view(np.uint32))
    assert np.all(G[1] == 0.0)
    metropolis_lockstep(xy, ora, inputs.uniform_state(L, R, 4), 1)


# ---- a3 -------------------------------------------------------------------------------------
@pytest.mark.parametrize("L,R", SHAPES)
def test_overrelax_lockstep(xy_mod, oracle_mod, L, R):
    xy, ora = make(xy_mod, oracle_mod, L, R)
    for name, S in states_for(L, R):
        xy.set_state(S)
        E0 = xy.measure()[:, 0]
        stats, G = overrelax_lockstep(xy, ora, S)
        print(L, R, name, stats)
        assert np.all((G >= 0.0) & (G <= np.float32(6.2831855)))
        E1 = xy.measure()[:, 0]
        assert np.all(np.abs(E1 - E0) <= 1e-5 * np.abs(E0) + 1e-3), "over-relaxation must conserve E (P:43)"
    assert np.array_equal(xy.get_counters(), [0, 2, 0])


def test_overrelax_fixed_points_and_vanishing_field(xy_mod, oracle_mod):
    """Helical states are fixed points (h_i parallel to S_i, O7).  Where the field (nearly)
    vanishes the reflection is ill-conditioned: the result must stay a finite angle in range and
    pass the conditioned clause of P2 (R6: h = 0 exactly leaves the spin alone)."""
    L, R = 16, 2
    xy, ora = make(xy_mod, oracle_mod, L, R, betas=[0.45, 0.46])
    for k in ((1, 0, 0), (0, 2, 0), (0, 0, 3), (1, 1, 1)):
        S = inputs.helical_state(L, R, k, phase=0.3)
        xy.set_state(S); xy.overrelax_sweep()
        assert H.angle_diff(xy.get_state(), S).max() < 5e-6
    # 2x2x2 blocks of 0 / pi: every site sees three neighbours at 0 and three at pi -> |h| ~ 1e-7
    z, y, x = np.meshgrid(np.arange(L), np.arange(L), np.arange(L), indexing="ij")
    S = np.where((x // 2 + y // 2 + z // 2) % 2 == 0, 0.0, np.pi).astype(np.float32)
    S = np.broadcast_to(S, (R, L, L, L)).copy()
    stats, G = overrelax_lockstep(xy, ora, S)
    assert np.isfinite(G).all() and G.min() >= 0.0 and G.max() <= np.float32(6.2831855)


# ---- a4 -------------------------------------------------------------------------------------
@pytest.mark.parametrize("L,R", SHAPES)
def test_measure_against_oracle(xy_mod, oracle_mod, L, R):
    xy, ora = make(xy_mod, oracle_mod, L, R)
    for name, S in states_for(L, R):
        xy.set_state(S); ora.set_state(S)
        stats = P.check_observables(xy.measure(), ora.measure(), L ** 3)
        print(L, R, name, stats)
    # by RANK: after a permutation the rows move with the labels
    if R >= 3:
        perm = np.roll(np.arange(R, dtype=np.int32), 1)
        xy.set_perm(perm); ora.set_perm(perm)
        g = xy.measure()
        P.check_observables(g, ora.measure(), L ** 3)
        assert np.array_equal(xy.get_perm(), perm)
        assert np.allclose(xy.get_beta_of_slot()[perm], inputs.beta_ladder(0.44, 0.47, R))


@pytest.mark.parametrize("L,R", SHAPES)
def test_measure_fused_into_overrelax(xy_mod, oracle_mod, L, R):
    """The white over-relaxation pass carries the reduction (default): its observables must equal the
    oracle's on the state the sweep leaves behind, and the standalone reduction's on that same state."""
    xy, ora = make(xy_mod, oracle_mod, L, R)
    assert xy.get_option(xy_mod.XY_OPT_FUSED_MEASURE) == 1
    for name, S in states_for(L, R):
        xy.set_state(S)
        xy.overrelax_sweep()
        n0 = xy.get_launch_count()
        fused = xy.measure()
        assert xy.get_launch_count() - n0 <= 1, "only the finalize kernel may run: no second pass over the spins"
        G = xy.get_state()
        ora.set_state(G)
        print(L, R, name, P.check_observables(fused, ora.measure(), L ** 3))
        xy.set_state(G)                                  # invalidates the cache -> standalone reduction
        P.check_observables(fused, xy.measure(), L ** 3)
    xy.set_option(xy_mod.XY_OPT_FUSED_MEASURE, 0)
    xy.overrelax_sweep()
    n0 = xy.get_launch_count()
    unfused = xy.measure()
    assert xy.get_launch_count() - n0 == 2
    ora.set_state(xy.get_state())
    P.check_observables(unfused, ora.measure(), L ** 3)


@pytest.mark.parametrize("L,R", SHAPES + [(160, 1)])
def test_stiffness_sums_against_oracle(xy_mod, oracle_mod, L, R):
    """f1 (Eq. 6): the six per-direction bond sums, GPU vs oracle, by rank; fp32 bond terms
    with the stated 7.5e-7 sin/cos error -> |delta| <= 4e-6 * N per sum; E = -(Cx+Cy+Cz)."""
    xy, ora = make(xy_mod, oracle_mod, L, R)
    N = L ** 3
    if R >= 3:
        perm = np.roll(np.arange(R, dtype=np.int32), 1)
        xy.set_perm(perm); ora.set_perm(perm)
    for name, S in states_for(L, R):
        xy.set_state(S); ora.set_state(S)
        g, o = xy.measure_stiffness(), ora.measure_stiffness()
        assert np.all(np.abs(g - o) <= 4e-6 * N), (name, np.abs(g - o).max() / N)
        assert np.all(np.abs(g[:, :3].sum(axis=1) + xy.measure()[:, 0]) <= 4e-6 * 3 * N)
    # closed forms on the GPU: ordered (rho_s = 1 at T = 0) and helical, each axis separately
    xy.set_state(inputs.ordered_state(L, R, 0.7))
    assert np.all(np.abs(xy.measure_stiffness() - np.array([N, N, N, 0, 0, 0.0])) <= 4e-6 * N)
    for k in ((1, 0, 0), (0, 2, 0), (0, 0, 3)):
        xy.set_state(inputs.helical_state(L, R, k, phase=0.3))
        want = np.array([N * np.cos(2 * np.pi * kk / L) for kk in k] + [-N * np.sin(2 * np.pi * kk / L) for kk in k])
        assert np.all(np.abs(xy.measure_stiffness() - want) <= 4e-6 * N), k
    # the call must leave the state and the cached observables alone
    xy.set_state(S)
    a = xy.measure(); xy.measure_stiffness()
    assert np.array_equal(a, xy.measure()) and np.array_equal(xy.get_state().view(np.uint32), S.view(np.uint32))


def test_measure_closed_forms(xy_mod):
    """O3 / O7 / O8 on the GPU reduction: ordered, helical (each axis separately) and staggered."""
    L, R = 16, 2
    N = L ** 3
    xy = xy_mod.XY(L, R, [0.45, 0.46], SEED)
    xy.set_state(inputs.ordered_state(L, R, 0.0))
    o = xy.measure()
    assert np.allclose(o, [[-3.0 * N, N, 0.0, float(N) ** 2, float(N) ** 4]] * R, rtol=1e-7, atol=1e-3)
    for k in ((1, 0, 0), (0, 2, 0), (0, 0, 3), (2, 1, 3)):
        xy.set_state(inputs.helical_state(L, R, k))
        o = xy.measure()
        E = -N * sum(np.cos(2 * np.pi * kk / L) for kk in k)
        assert np.all(np.abs(o[:, 0] - E) <= 1e-6 * 3 * N), (k, o[:, 0], E)
        assert np.all(np.abs(o[:, 1:3]) <= 1e-6 * N)
    xy.set_state(inputs.staggered_state(L, R))
    o = xy.measure()
    assert np.all(np.abs(o[:, 0] - 3.0 * N) <= 1e-6 * 3 * N) and np.all(np.abs(o[:, 1:3]) <= 1e-6 * N)
    # global rotation leaves E and |M|^2 unchanged (O6)
    S = inputs.smooth_state(L, R, 9)
    xy.set_state(S); a = xy.measure()
    xy.set_state(((S.astype(np.float64) + 1.2345) % (2 * np.pi)).astype(np.float32)); b = xy.measure()
    assert np.all(np.abs(a[:, 0] - b[:, 0]) <= 2e-6 * 3 * N)
    assert np.allclose(a[:, 3], b[:, 3], rtol=1e-5)


def test_measure_is_deterministic_and_cached(xy_mod):
    L, R = 32, 4
    xy = xy_mod.XY(L, R, inputs.beta_ladder(0.45, 0.46, R), SEED)
    xy.init_random()
    a = xy.measure()
    n0 = xy.get_launch_count()
    b = xy.measure()
    assert xy.get_launch_count() == n0, "an unchanged state must not be reduced again"
    assert np.array_equal(a, b)
    xy.set_state(xy.get_state())
    assert np.array_equal(xy.measure(), a), "fixed-order reduction: bit-identical run to run"


# ---- a5 -------------------------------------------------------------------------------------
def test_pt_forced_swaps_at_equal_beta(xy_mod):
    """O10: all beta equal -> every attempted pair swaps; the permutation after t exchanges is known."""
    for R in (1, 2, 5, 8):
        xy = xy_mod.XY(8, R, [0.45] * R, SEED)
        xy.init_random()
        want = list(range(R))
        for t in range(6):
            xy.pt_exchange()
            for k in range(t & 1, R - 1, 2):
                want[k], want[k + 1] = want[k + 1], want[k]
            assert list(xy.get_perm()) == want
        assert np.array_equal(xy.get_counters(), [0, 0, 6])
        _, pt = xy.get_accept_counts()
        assert pt.sum() == sum(len(range(t & 1, R - 1, 2)) for t in range(6))


@pytest.mark.parametrize("L,R,lo,hi", [(8, 8, 0.44, 0.47), (16, 16, 0.40, 0.50), (32, 16, 0.450, 0.458)])
def test_pt_lockstep(xy_mod, oracle_mod, L, R, lo, hi):
    """P4: both sides compute E from the shared state; decisions and label bookkeeping agree."""
    betas = inputs.beta_ladder(lo, hi, R)
    xy, ora = make(xy_mod, oracle_mod, L, R, betas=betas)
    # replicas thermalised a little so that energies are ordered like the betas
    xy.init_random()
    xy.mcs(30)
    n_swapped = 0
    for t in range(30, 50):
        S, perm = xy.get_state(), xy.get_perm()
        ora.set_state(S); ora.set_perm(perm); ora.set_counters([0, 0, t])
        xy.set_counters([0, 0, t])
        tr = ora.enable_trace(pt=True)
        xy.pt_exchange(); ora.pt_exchange()
        g = xy.get_perm()
        P.check_pt(g, ora.get_perm(), tr["pt_p"], tr["pt_u"])
        n_swapped += int((g != perm).sum()) // 2
        bos = xy.get_beta_of_slot()
        assert np.array_equal(bos[g], betas), "beta labels must follow slot_at_rank"
        assert np.array_equal(bos, ora.get_beta_of_slot()) or not np.array_equal(g, ora.get_perm())
        xy.metropolis_sweep(); xy.overrelax_sweep()
    assert n_swapped > 0


# ---- one full MCS (P5) and free run (P6) --------------------------------------------------------
def mcs_lockstep(xy, ora, t):
    """Advance the GPU one MCS from its current state with counters (t,t,t); check every stage."""
    L, R = xy.L, xy.R
    S, perm = xy.get_state(), xy.get_perm()
    metropolis_lockstep(xy, ora, S, t)
    S1 = xy.get_state()
    _, S2 = overrelax_lockstep(xy, ora, S1)
    ora.set_state(S2); ora.set_perm(perm); ora.set_counters([t + 1, t + 1, t])
    xy.set_counters([t + 1, t + 1, t])
    obs = xy.measure()
    P.check_observables(obs, ora.measure(), L ** 3)
    tr = ora.enable_trace(pt=True)
    xy.pt_exchange(); ora.pt_exchange()
    P.check_pt(xy.get_perm(), ora.get_perm(), tr["pt_p"], tr["pt_u"])
    ora.enable_trace()
    return obs


@pytest.mark.parametrize("idx", [0, 1, 2])
def test_full_mcs_lockstep_on_configs(xy_mod, oracle_mod, idx):
    """P5 on BASELINE.json configs 1-3 at their STATED lengths (200 / 2000 / 1000 MCS): a free-running GPU
    trajectory; the MCS t in {0..9, T/4, T/2, T-1} are re-done by the oracle from the GPU's state with the
    GPU's counters, every stage against its own criterion (P1-P4)."""
    cfg = inputs.CONFIGS[idx]
    n_mcs = cfg.mcs
    xy, ora = make(xy_mod, oracle_mod, cfg.L, cfg.R, betas=inputs.betas_of(cfg))
    xy.init_random()
    sampled = sorted(set(list(range(10)) + [n_mcs // 4, n_mcs // 2, n_mcs - 1]))
    t = 0
    for s in sampled:
        if s > t:
            xy.mcs(s - t)
            t = s
        assert np.array_equal(xy.get_counters(), [t, t, t])
        obs = mcs_lockstep(xy, ora, t)
        print(cfg.name, "MCS", t, "ok; E/N rank 0", obs[0, 0] / cfg.L ** 3)
        t += 1
    assert t == n_mcs


@pytest.mark.parametrize("L,R", [(80, 3), (96, 2)])
def test_paper_other_sizes_and_nonuniform_ladder(xy_mod, oracle_mod, L, R):
    """the paper's L = 80 and 96 have no compile-time kernel variant (their rows do
    not split into whole warps per parity class) and its temperature ladders are not uniform: the
    run-time-geometry kernel on a non-uniformly spaced, unsorted beta set, lock-step against the oracle."""
    betas = np.array([1.0 / 2.2019, 1.0 / 2.25, 1.0 / 2.19][:R])          # T_c of P:76 and two neighbours, unsorted
    xy, ora = make(xy_mod, oracle_mod, L, R, betas=betas)
    xy.init_random()
    t = 0
    for s in (0, 1, 5):
        if s > t:
            xy.mcs(s - t)
            t = s
        mcs_lockstep(xy, ora, t)
        t += 1
    g, o = xy.measure_stiffness(), None
    ora.set_state(xy.get_state()); ora.set_perm(xy.get_perm())
    o = ora.measure_stiffness()
    assert np.all(np.abs(g - o) <= 4e-6 * L ** 3)


def test_free_run_divergence_report(xy_mod, oracle_mod):
    """P6: GPU and oracle run freely from the same start.  Only k = 1 is asserted (chaos: the
    difference grows x3-5 per MCS, SURVEY.md finding 3); the curve is printed."""
    L, R = 16, 4
    xy, ora = make(xy_mod, oracle_mod, L, R, betas=inputs.beta_ladder(0.45, 0.458, R))
    xy.init_random(); ora.init_random()
    curve = []
    for k in range(1, 13):
        xy.mcs(1); ora.mcs()
        d = H.angle_diff(xy.get_state(), ora.get_state())
        curve.append((k, float(np.sqrt((d ** 2).mean())), float(d.max())))
    print("free-run rms/max difference per MCS:", curve)
    assert curve[0][2] <= 1e-3 and curve[0][1] <= 1e-5


def test_mcs_series_matches_stepwise_calls(xy_mod):
    """xy_mcs(n) with a device series == n x (sweep, sweep, measure, exchange) called one by one."""
    import torch
    L, R, n = 16, 6, 9
    betas = inputs.beta_ladder(0.44, 0.47, R)
    a = xy_mod.XY(L, R, betas, SEED); b = xy_mod.XY(L, R, betas, SEED)
    a.set_option(xy_mod.XY_OPT_RESIDENT, 0)                  # the per-pass kernels (the resident path: test_resident_*)
    a.init_random(); b.init_random()
    series = torch.zeros(n, R, 5, dtype=torch.float64, device="cuda")
    a.mcs(n, series)
    rows = []
    for _ in range(n):
        b.metropolis_sweep(); b.overrelax_sweep(); rows.append(b.measure()); b.pt_exchange()
    assert np.array_equal(series.cpu().numpy(), np.stack(rows))
    assert np.array_equal(a.get_state().view(np.uint32), b.get_state().view(np.uint32))
    assert np.array_equal(a.get_perm(), b.get_perm())


# ---- full-size configs, sampled (the launch configuration bench.py times) -----------------------
def sampled_slots_lockstep(xy, ora, name, slots, times):
    """A free-running GPU trajectory; at every MCS in `times` the oracle re-does Metropolis and over-relaxation for the
    sampled slots (every site of those slots), and the reduction + exchange for all slots."""
    L = xy.L
    t = 0
    for s_t in times:
        xy.mcs(s_t - t)
        t = s_t
        assert np.array_equal(xy.get_counters(), [t, t, t])
        S, perm = xy.get_state(), xy.get_perm()
        stats = metropolis_lockstep(xy, ora, S, t, slots=slots)
        print(name, "MCS", t, "metropolis", stats)
        S1 = xy.get_state()
        del S
        stats, S2 = overrelax_lockstep(xy, ora, S1, slots=slots)
        print(name, "MCS", t, "overrelax", stats)
        del S1
        ora.set_active_slots(None)
        ora.set_state(S2); ora.set_perm(perm); ora.set_counters([t + 1, t + 1, t]); xy.set_counters([t + 1, t + 1, t])
        del S2
        print(name, "MCS", t, "measure", P.check_observables(xy.measure(), ora.measure(), L ** 3))
        tr = ora.enable_trace(pt=True)
        xy.pt_exchange(); ora.pt_exchange()
        print(name, "MCS", t, "pt", P.check_pt(xy.get_perm(), ora.get_perm(), tr["pt_p"], tr["pt_u"]))
        ora.enable_trace()
        t += 1


@pytest.mark.parametrize("idx,slots", [(3, (0, 17, 31)), (4, (0, 37, 63))])
def test_full_size_configs_sampled_slots(xy_mod, oracle_mod, idx, slots):
    """BASELINE.json configs 4 and 5 at full size and full length on the GPU with the default tiling (the
    launch configuration bench.py times); at three sampled MCS the oracle re-does Metropolis and
    over-relaxation for three sampled slots (every site of those slots), and the reduction + exchange for
    all slots."""
    cfg = inputs.CONFIGS[idx]
    L, R = cfg.L, cfg.R
    xy, ora = make(xy_mod, oracle_mod, L, R, betas=inputs.betas_of(cfg))
    if cfg.start == "random":
        xy.init_random()
        G = xy.get_state()
        for r in slots:
            W, i = H.site_words(L, r, 0, H.STREAM_INIT, SEED)
            w = np.take_along_axis(W, (i & np.uint64(3)).astype(np.int64)[None], axis=0)[0]
            assert np.array_equal(G[r].view(np.uint32), (H.TWO_PI_F * H.u24(w)).view(np.uint32))
        del G
    else:
        xy.init_ordered(0.0)
    # MCS 3 (just after the start), T/2 and T-1 of the stated 500: the late samples compare an equilibrated
    # state (small-|h| sites, acceptance ~0.55), not only the easy regime right after an ordered start
    sampled_slots_lockstep(xy, ora, cfg.name, slots, (3, cfg.mcs // 2, cfg.mcs - 1))


# ---- f3: the paper's own workload families and ladders ----------------------------------------------------
@pytest.mark.parametrize("name,slots", [("paper_L64_R34", None), ("paper_L80_R34", (0, 16, 33)), ("paper_L96_R34", (5, 33)),
                                        ("paper_L160_R13", (0, 6, 12))])
def test_paper_families_lockstep(xy_mod, oracle_mod, name, slots):
    """L = 64 ... 160 with R = 34 temperatures in T = [2.1, 2.3] (R = 13 in [2.19, 2.21] at
    L = 160) on a NON-uniform (geometric) ladder: a free-running GPU trajectory, re-done by the oracle at MCS 0, 1 and 6
    (whole system at L = 64, sampled slots above) -- Metropolis, over-relaxation, reduction and exchange."""
    fam = inputs.paper_family(name)
    betas = inputs.betas_of_family(fam)
    xy, ora = make(xy_mod, oracle_mod, fam.L, fam.R, betas=betas)
    xy.init_random()
    if slots is None:
        t = 0
        for s_t in (0, 1, 6):
            xy.mcs(s_t - t)
            t = s_t
            mcs_lockstep(xy, ora, t)
            t += 1
    else:
        sampled_slots_lockstep(xy, ora, name, slots, (0, 1, 6))
    assert np.array_equal(xy.get_beta_of_slot()[xy.get_perm()], betas)


def test_ladder_equalises_the_swap_acceptance(xy_mod):
    """P:62 "chosen such that the acceptance rate of swaps is independent of the temperatures": starting from the
    geometric ladder over a range that straddles T_c, ladder.equalise_swap_acceptance (host arithmetic on
    xy_get_accept_counts, new ladder through xy_set_betas) must flatten the measured per-pair acceptance while keeping
    both end temperatures; xy_set_betas must leave the permutation and the spins alone."""
    from paper_1211_0780_b200 import ladder
    L, R = 16, 12
    b0 = inputs.geometric_beta_ladder(1.9, 2.6, R)
    xy = xy_mod.XY(L, R, b0, SEED)
    xy.init_random()
    xy.mcs(300)
    perm, S = xy.get_perm(), xy.get_state()
    xy.set_betas(b0 * 1.0)
    assert np.array_equal(xy.get_perm(), perm) and np.array_equal(xy.get_state().view(np.uint32), S.view(np.uint32))
    assert np.array_equal(xy.get_beta_of_slot()[perm], b0)
    b, hist = ladder.equalise_swap_acceptance(xy, b0, rounds=8, n_mcs=1500, burn=200)
    first, last = hist[0], hist[-1]
    print("acceptance per pair, geometric ladder:", np.round(first, 3).tolist())
    print("acceptance per pair, tuned ladder:    ", np.round(last, 3).tolist())
    print("tuned betas:", np.round(b, 5).tolist())
    assert b[0] == b0[0] and b[-1] == b0[-1] and np.all(np.diff(b) > 0)
    assert np.array_equal(xy.get_beta_of_slot()[xy.get_perm()], b)
    assert (last.max() - last.min()) < 0.5 * (first.max() - first.min())
    assert last.min() > first.min()


@pytest.mark.parametrize("L,R", [(200, 2), (256, 1), (8, 64), (16, 200)])
def test_large_lattices_and_many_replicas(xy_mod, oracle_mod, L, R):
    """Sizes beyond the BASELINE configs: L = 200 and 256 (run-time-geometry kernel, rows of 25 and 32 float4)
    and replica counts far above the tile count (R = 64 at L = 8, R = 200 at L = 16): one Metropolis sweep,
    one over-relaxation sweep, the reduction and the stiffness sums after two free MCS, lock-step."""
    xy, ora = make(xy_mod, oracle_mod, L, R)
    xy.init_random(); xy.mcs(2)
    S = xy.get_state()
    print(L, R, "metropolis", metropolis_lockstep(xy, ora, S, 2))
    S1 = xy.get_state()
    stats, S2 = overrelax_lockstep(xy, ora, S1)
    print(L, R, "overrelax", stats)
    ora.set_active_slots(None)
    ora.set_state(S2); ora.set_perm(xy.get_perm())
    print(L, R, "measure", P.check_observables(xy.measure(), ora.measure(), L ** 3))
    assert np.all(np.abs(xy.measure_stiffness() - ora.measure_stiffness()) <= 4e-6 * L ** 3)


def test_set_state_reduces_out_of_range_angles(xy_mod, oracle_mod):
    """include/xy.h: the stated errors hold for angles in [0, 2 pi]; xy_set_state reduces anything else modulo
    2 pi (in-range angles pass bit for bit, NaN / inf become 0).  A sweep from such input must then equal the
    sweep from the reduced input, and the reduced angles must be the same directions."""
    L, R = 16, 2
    rng = np.random.default_rng(17)
    S = ((rng.random((R, L, L, L)) - 0.5) * 200.0).astype(np.float32)          # angles in [-100, 100)
    S[0, 0, 0, :4] = [np.nan, np.inf, -np.inf, 6.2831855]
    xy, ora = make(xy_mod, oracle_mod, L, R)
    xy.set_state(S)
    G = xy.get_state()
    assert np.isfinite(G).all() and G.min() >= 0.0 and G.max() <= np.float32(6.2831855)
    assert list(G[0, 0, 0, :4]) == [0.0, 0.0, 0.0, np.float32(6.2831855)]
    fin = np.isfinite(S)
    assert H.angle_diff(G[fin], S[fin]).max() <= 4e-6 + 100 * 6e-8            # fl32 of the double reduction
    inr = (S >= 0) & (S <= np.float32(6.2831855))
    assert np.array_equal(G[inr].view(np.uint32), S[inr].view(np.uint32))
    metropolis_lockstep(xy, ora, G, 0)
    a = xy.get_state()
    xy.set_state(S); xy.set_counters([0, 0, 0]); xy.metropolis_sweep()
    assert np.array_equal(xy.get_state().view(np.uint32), a.view(np.uint32))



# ---- f2 stage A: the resident kernel (whole steps of a small lattice in one persistent launch) ------------------
@pytest.mark.parametrize("L,R,n_or", [(8, 8, 1), (8, 3, 1), (8, 20, 2), (8, 64, 1), (16, 4, 1), (16, 5, 0), (24, 2, 1), (32, 3, 1),
                                      (32, 16, 1), (40, 2, 1), (48, 2, 2),
                                      # several slots per thread block (R > 132 blocks' worth): the slot split of the
                                      # threads, a partially filled last block (R = 133: 66 full blocks + one slot),
                                      # the tag exchange between many one-block "clusters"
                                      (8, 133, 1), (8, 200, 1), (8, 512, 1), (16, 200, 1)])
def test_resident_kernel_equals_per_pass_kernels(xy_mod, L, R, n_or):
    """XY_OPT_RESIDENT: n whole steps in one launch with the spins resident in shared
    memory must leave BITWISE the states, labels, counters and Metropolis / exchange acceptance counts of the
    per-pass kernels (same site arithmetic, same Philox keying, decisions settled in fp64 on both paths), over
    several calls; the observables (series rows and xy_measure afterwards) agree within the P3 bound, their fp32
    terms being grouped differently before the fp64 accumulation."""
    import torch
    betas = inputs.beta_ladder(0.445, 0.46, R)
    N = L ** 3
    runs = []
    for resident in (1, 0):
        xy = xy_mod.XY(L, R, betas, SEED)
        xy.set_option(xy_mod.XY_OPT_RESIDENT, resident)
        xy.set_option(xy_mod.XY_OPT_OR_PER_MCS, n_or)
        if resident:
            plan = xy.get_resident_plan()
            assert plan["resident"] == 1, plan
            assert (plan["slots_per_block"] > 1) == (R > 132), plan
        xy.init_random()
        s1 = torch.zeros(6, R, 5, dtype=torch.float64, device="cuda")
        s2 = torch.zeros(5, R, 5, dtype=torch.float64, device="cuda")
        n0 = xy.get_launch_count()
        xy.mcs(6, s1); xy.mcs(5, s2); xy.mcs(1); xy.mcs(3)
        launches = xy.get_launch_count() - n0
        obs = xy.measure()
        runs.append((xy.get_state(), xy.get_perm(), xy.get_counters(), xy.get_accept_counts(), xy.get_beta_of_slot(),
                     s1.cpu().numpy(), s2.cpu().numpy(), obs, launches))
        # a sweep by the per-pass kernels continues seamlessly from what the resident kernel wrote back
        xy.metropolis_sweep(); xy.overrelax_sweep(); xy.pt_exchange()
        runs[-1] += (xy.get_state(), xy.get_perm())
    a, b = runs
    assert a[8] == 4, "one launch per xy_mcs call"
    assert np.array_equal(a[0].view(np.uint32), b[0].view(np.uint32)), "states differ"
    assert np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2]) and np.array_equal(a[2], [15, 15 * n_or, 15])
    assert np.array_equal(a[3][0], b[3][0]) and np.array_equal(a[3][1], b[3][1])
    assert np.array_equal(a[4], b[4])
    for x, y in ((a[5], b[5]), (a[6], b[6]), (a[7], b[7])):
        assert np.abs(x[..., 0] - y[..., 0]).max() <= 1e-6 * 3 * N and np.abs(x[..., 1:3] - y[..., 1:3]).max() <= 1e-6 * N
        assert np.allclose(x[..., 3], x[..., 1] ** 2 + x[..., 2] ** 2, rtol=1e-13) and np.allclose(x[..., 4], x[..., 3] ** 2, rtol=1e-13)
    assert np.all(a[5][..., 3] > 0)
    assert np.array_equal(a[9].view(np.uint32), b[9].view(np.uint32)) and np.array_equal(a[10], b[10])


def xy_mcs_lockstep(xy_mod, xy, ora, S, perm, t):
    """ONE xy_mcs(1) call against the oracle, stage by stage (P1-P4 directly, for the paths that run a whole step
    without handing the intermediate states back: the resident kernel, the slot-chunk schedule).

    (a) P1.  With XY_OPT_OR_PER_MCS = 0 the call is Metropolis sweep + reduction + exchange, so the state it leaves is
        the Metropolis result M: every site bitwise old-or-proposal, decisions against the oracle's trace, pass by
        pass (the oracle's white pass starts from the GPU's own black result), exactly like metropolis_lockstep.
    (b) P2.  The same call from the same state and counters with one over-relaxation sweep leaves G; the Metropolis
        part is deterministic, so the over-relaxation went from M to G: the oracle's two passes from M with its |h|
        trace, under the conditioning clause of check_overrelax.
    (c) P3 / P4.  The series row of that call (by rank, before the exchange) against the oracle's observables of G,
        and the exchange replayed in the oracle from the same energies."""
    import torch
    L, R = xy.L, xy.R
    col = H.colour_mask(L)
    prop, _ = H.predicted_proposals(L, R, t, SEED)
    stats = {}
    xy.set_option(xy_mod.XY_OPT_OR_PER_MCS, 0)
    xy.set_state(S); xy.set_perm(perm); xy.set_counters([t, t, t])
    xy.mcs(1)
    M = xy.get_state()
    assert np.array_equal(xy.get_counters(), [t + 1, t, t + 1])
    ora.set_active_slots(None); ora.set_perm(perm); ora.set_counters([t, t, t])
    start = S
    for c in (0, 1):
        sel = np.broadcast_to(col == c, S.shape)
        ora.set_state(start)
        tr = ora.enable_trace(met=True)
        ora.metropolis_pass(c)
        stats[f"met{c}"] = P.check_metropolis(start, M, ora.get_state(), prop, tr["met_p"], tr["met_u"], sel)
        start = np.where(col[None] == 0, M, S)
    ora.enable_trace()
    xy.set_option(xy_mod.XY_OPT_OR_PER_MCS, 1)
    xy.set_state(S); xy.set_perm(perm); xy.set_counters([t, t, t])
    row = torch.zeros(1, R, 5, dtype=torch.float64, device="cuda")
    xy.mcs(1, row)
    G = xy.get_state()
    assert np.array_equal(xy.get_counters(), [t + 1, t + 1, t + 1])
    start = M
    for c in (0, 1):
        sel = np.broadcast_to(col == c, S.shape)
        ora.set_state(start)
        tr = ora.enable_trace(overrelax=True)
        ora.overrelax_pass(c)
        stats[f"or{c}"] = P.check_overrelax(G, ora.get_state(), tr["or_h"], sel)
        start = np.where(col[None] == 0, G, M)
    ora.enable_trace()
    stats["obs"] = P.check_observables(row.cpu().numpy()[0], ora_obs_of(G, ora, perm), L ** 3)
    tr = ora.enable_trace(pt=True)
    ora.set_state(G); ora.set_perm(perm); ora.set_counters([t + 1, t + 1, t])
    ora.pt_exchange()
    P.check_pt(xy.get_perm(), ora.get_perm(), tr["pt_p"], tr["pt_u"])
    ora.enable_trace()
    P.check_observables(xy.measure(), ora_obs_of(G, ora, xy.get_perm()), L ** 3)      # by rank AFTER the exchange
    return stats, G


# (L, R, warm-up MCS, config index or None).  Every code path of the resident kernel: configs 1 and 2 as they are
# benchmarked; several slots per block (R > 132), with a partially filled last block (R = 133); one block per slot and
# clusters of 2, 4, 8 blocks per slot (the planner takes the largest co-resident cluster, so R decides); every lattice
# size that has a kernel; a random start (warm = 0) and an equilibrated state (50 steps).
RESIDENT_LOCKSTEP = [(8, 8, 0, 0), (8, 8, 50, 0), (8, 133, 0, None), (8, 200, 50, None),          # one block per slot; two slots per block
                     (16, 3, 50, None), (16, 100, 0, None), (16, 140, 50, None),             # 8 blocks per slot; 1; two slots per block
                     (24, 5, 0, None), (24, 30, 50, None), (24, 60, 0, None), (24, 100, 0, None),   # 8, 4, 2, 1 blocks per slot
                     (32, 16, 50, 1), (32, 16, 0, 1), (32, 3, 0, None), (32, 36, 0, None),  # 4 (config 2), 8, 2 blocks per slot
                     (40, 2, 0, None), (48, 2, 50, None)]


@pytest.mark.parametrize("L,R,warm,cfg", RESIDENT_LOCKSTEP)
def test_resident_kernel_lockstep_P1_P2_against_oracle(xy_mod, oracle_mod, L, R, warm, cfg):
    """The default xy_mcs path of configs 1-2 (L <= 48: resident_mcs_kernel) against the ORACLE with the same bars as
    the per-pass kernels: P1 decision by decision, P2 with the conditioning clause, P3, P4 (xy_mcs_lockstep)."""
    betas = inputs.betas_of(inputs.CONFIGS[cfg]) if cfg is not None else inputs.beta_ladder(0.45, 0.458, R)
    xy, ora = make(xy_mod, oracle_mod, L, R, betas=betas)
    plan = xy.get_resident_plan()
    assert xy.get_option(xy_mod.XY_OPT_RESIDENT) == 1 and plan["resident"] == 1, plan
    assert (plan["slots_per_block"] > 1) == (R > 132), plan
    xy.init_random()
    if warm:
        xy.mcs(warm)
    S, perm = xy.get_state(), xy.get_perm()
    for t in (warm, warm + 1):
        stats, S = xy_mcs_lockstep(xy_mod, xy, ora, S, perm, t)
        perm = xy.get_perm()
        print(L, R, "t", t, "plan", plan, stats)
    # two resident launches per lock-step (plus the layout conversions, the standalone rank gather of xy_measure ...):
    # no Metropolis / over-relaxation colour-pass kernel ran
    xy.set_option(xy_mod.XY_OPT_PROFILE, 1); xy.get_kernel_times()
    xy.mcs(1)
    kt = xy.get_kernel_times()
    assert kt["resident"][1] == 1 and kt["metropolis"][1] == 0 and kt["overrelax"][1] == 0, kt


def test_resident_plan_reports_the_path_xy_mcs_takes(xy_mod):
    """xy_get_resident_plan()[0] is 1 exactly when xy_mcs will run the resident kernel: a plan exists, the option is
    on and the Metropolis trace hook (which needs the per-pass kernels) is off; the kernel classes that actually ran
    say the same."""
    def classes_of_one_step(xy):
        xy.set_option(xy_mod.XY_OPT_PROFILE, 1); xy.get_kernel_times()
        xy.mcs(1)
        kt = xy.get_kernel_times()
        xy.set_option(xy_mod.XY_OPT_PROFILE, 0)
        return kt["resident"][1], kt["metropolis"][1]
    xy = xy_mod.XY(8, 8, inputs.beta_ladder(0.44, 0.47, 8), SEED)
    xy.init_random()
    assert xy.get_resident_plan()["resident"] == 1 and classes_of_one_step(xy) == (1, 0)
    xy.set_option(xy_mod.XY_OPT_TRACE, 1)
    assert xy.get_resident_plan()["resident"] == 0 and classes_of_one_step(xy) == (0, 2)
    xy.set_option(xy_mod.XY_OPT_TRACE, 0)
    assert xy.get_resident_plan()["resident"] == 1
    xy.set_option(xy_mod.XY_OPT_RESIDENT, 0)
    assert xy.get_resident_plan()["resident"] == 0 and classes_of_one_step(xy) == (0, 2)
    big = xy_mod.XY(64, 2, inputs.beta_ladder(0.45, 0.46, 2), SEED)
    big.init_random()
    assert big.get_resident_plan()["resident"] == 0 and classes_of_one_step(big) == (0, 2)


def test_slot_chunk_step_lockstep_against_oracle(xy_mod, oracle_mod):
    """XY_OPT_SLOT_CHUNK against the ORACLE (not only against the default schedule): one xy_mcs(1) at L = 64 with the
    passes of 2 of 3 slots back to back (a ragged last chunk), P1-P4 stage by stage, from an equilibrated state."""
    L, R = 64, 3
    xy, ora = make(xy_mod, oracle_mod, L, R, betas=inputs.beta_ladder(0.4530, 0.4555, R))
    xy.set_option(xy_mod.XY_OPT_SLOT_CHUNK, 2)
    xy.init_random(); xy.mcs(20)
    S, perm = xy.get_state(), xy.get_perm()
    for t in (20, 21):
        stats, S = xy_mcs_lockstep(xy_mod, xy, ora, S, perm, t)
        perm = xy.get_perm()
        print(L, R, "chunk 2, t", t, stats)


def ora_obs_of(state, ora, perm):
    """Oracle observables (by rank under `perm`) of a given state; leaves the oracle's state set to it."""
    ora.set_state(state); ora.set_perm(perm)
    return ora.measure()


# ---- pipeline hazards --------------------------------------------------------------------------
@pytest.mark.parametrize("L,R", [(32, 3), (64, 2), (128, 1), (160, 1)])
def test_free_run_is_reproducible_across_kernel_variants(xy_mod, L, R):
    """compute-sanitizer is closed on this pool, so races in the TMA / mbarrier pipeline are hunted
    this way: a hazard between the bulk copies, the staging and the updates would make a free run
    differ from run to run or from tiling to tiling.  The site arithmetic does not depend on the tile
    shape, and the compile-time-geometry kernel does the same operations in the same order as the
    run-time-geometry one, so 6 MCS from the same seed must end in BITWISE identical states."""
    betas = inputs.beta_ladder(0.4535, 0.4550, R)
    ref = None
    variants = [dict(), dict(), dict(generic=1), dict(tz=8), dict(generic=1, tz=L), dict(ty=8, tz=16), dict(resident=1)]
    for v in variants:
        xy = xy_mod.XY(L, R, betas, SEED)
        xy.set_option(xy_mod.XY_OPT_RESIDENT, v.get("resident", 0))       # L = 32: the resident kernel is one more variant
        if "generic" in v:
            xy.set_option(xy_mod.XY_OPT_GENERIC_KERNEL, 1)
        if "ty" in v:
            xy.set_option(xy_mod.XY_OPT_TILE_Y, v["ty"])
        if "tz" in v:
            xy.set_option(xy_mod.XY_OPT_TILE_Z, v["tz"])
        xy.init_random()
        xy.mcs(6)
        S, perm, obs = xy.get_state(), xy.get_perm(), xy.measure()
        if ref is None:
            ref = (S, perm, obs)
            continue
        assert np.array_equal(S.view(np.uint32), ref[0].view(np.uint32)), v
        assert np.array_equal(perm, ref[1]), v
        assert np.allclose(obs[:, :3], ref[2][:, :3], rtol=0, atol=1e-6 * 3 * L ** 3), v


@pytest.mark.parametrize("L,R", [(64, 3), (96, 2), (160, 1)])
def test_chained_launches_equal_serialised_launches(xy_mod, L, R):
    """Programmatic dependent launch (the kernels of a step may become resident during their predecessor's tail and
    wait there for its completion) must not change a single bit.  XY_OPT_PROFILE = 1 puts an event record between any
    two launches, which is plain stream order without overlap, and disables graph replay: 8 steps that way against 8
    steps the default way (first step eager, then the captured graph with programmatic edges), and against 8 single
    sweep-by-sweep calls."""
    betas = inputs.beta_ladder(0.4535, 0.4550, R)
    runs = []
    for mode in ("default", "profiled", "stepwise"):
        xy = xy_mod.XY(L, R, betas, SEED)
        xy.set_option(xy_mod.XY_OPT_RESIDENT, 0)
        xy.set_option(xy_mod.XY_OPT_PROFILE, 1 if mode == "profiled" else 0)
        xy.init_random()
        if mode == "stepwise":
            for _ in range(8):
                xy.metropolis_sweep(); xy.overrelax_sweep(); xy.measure(to_host=False); xy.pt_exchange()
        else:
            xy.mcs(8)
        runs.append((xy.get_state(), xy.get_perm(), xy.get_accept_counts(), xy.measure()))
        if mode == "profiled":
            kt = xy.get_kernel_times()
            assert kt["metropolis"][1] == 16 and kt["overrelax"][1] == 16 and kt["fixup"][1] == 16, kt
    for other in runs[1:]:
        assert np.array_equal(runs[0][0].view(np.uint32), other[0].view(np.uint32))
        assert np.array_equal(runs[0][1], other[1])
        assert np.array_equal(runs[0][2][0], other[2][0]) and np.array_equal(runs[0][2][1], other[2][1])
        assert np.array_equal(runs[0][3], other[3])


@pytest.mark.parametrize("L,R,chunk,n_or", [(32, 5, 2, 1), (64, 3, 1, 2), (160, 3, 2, 1)])
def test_slot_chunk_schedule_equals_default(xy_mod, L, R, chunk, n_or):
    """XY_OPT_SLOT_CHUNK (SURVEY 8(f) f2 for large lattices: the four colour passes of K slots back to back, so that
    they stay in L2) reorders launches over independent slots only: states, labels, counters and acceptance counts
    must be bitwise those of the default schedule, the observables equal (same kernels, same tiles), under graph
    replay and with eager launches."""
    import torch
    betas = inputs.beta_ladder(0.45, 0.458, R)
    out = []
    for k, graph in ((0, 1), (chunk, 1), (chunk, 0)):
        xy = xy_mod.XY(L, R, betas, SEED)
        xy.set_option(xy_mod.XY_OPT_RESIDENT, 0)
        xy.set_option(xy_mod.XY_OPT_OR_PER_MCS, n_or)
        xy.set_option(xy_mod.XY_OPT_SLOT_CHUNK, k)
        xy.set_option(xy_mod.XY_OPT_CUDA_GRAPH, graph)
        xy.init_random()
        series = torch.zeros(5, R, 5, dtype=torch.float64, device="cuda")
        xy.mcs(5, series)
        out.append((xy.get_state(), xy.get_perm(), xy.get_counters(), xy.get_accept_counts(), series.cpu().numpy(), xy.measure()))
    ref = out[0]
    for o in out[1:]:
        assert np.array_equal(o[0].view(np.uint32), ref[0].view(np.uint32))
        assert np.array_equal(o[1], ref[1]) and list(o[2]) == list(ref[2])
        assert np.array_equal(o[3][0], ref[3][0]) and np.array_equal(o[3][1], ref[3][1])
        assert np.array_equal(o[4], ref[4]) and np.array_equal(o[5], ref[5])


@pytest.mark.parametrize("L,R", [(16, 6), (64, 3)])
def test_checkpoint_resume_is_bitwise(xy_mod, L, R):
    """SURVEY section 5 (checkpoint / resume): state, permutation and counters read through the C ABI and restored into a
    NEW context continue the trajectory bit for bit -- the chain is a deterministic function of (seed, betas, state,
    labels, counters).  L = 16 runs the resident kernel, L = 64 the per-pass kernels under graph replay."""
    betas = inputs.beta_ladder(0.45, 0.46, R)
    ref = xy_mod.XY(L, R, betas, SEED)
    ref.init_random()
    ref.mcs(20)
    a = xy_mod.XY(L, R, betas, SEED)
    a.init_random()
    a.mcs(9)
    state, perm, counters = a.get_state(), a.get_perm(), a.get_counters()
    a.close()
    b = xy_mod.XY(L, R, betas, SEED)
    b.set_state(state); b.set_perm(perm); b.set_counters(counters)
    b.mcs(11)
    assert list(b.get_counters()) == list(ref.get_counters())
    assert np.array_equal(b.get_perm(), ref.get_perm())
    assert np.array_equal(b.get_state().view(np.uint32), ref.get_state().view(np.uint32))
    assert np.array_equal(b.get_beta_of_slot(), ref.get_beta_of_slot())
    assert np.array_equal(b.measure(), ref.measure())


def test_mcs_with_several_overrelaxation_sweeps(xy_mod):
    """XY_OPT_OR_PER_MCS: xy_mcs must equal the same calls made one by one, bit for bit, and its
    series rows must be the observables of the state the last over-relaxation sweep left behind."""
    import torch
    L, R, n = 32, 4, 3
    betas = inputs.beta_ladder(0.45, 0.46, R)
    a, b = xy_mod.XY(L, R, betas, SEED), xy_mod.XY(L, R, betas, SEED)
    a.init_random(); b.init_random()
    a.set_option(xy_mod.XY_OPT_RESIDENT, 0)
    a.set_option(xy_mod.XY_OPT_OR_PER_MCS, 3)
    series = torch.zeros(n, R, 5, dtype=torch.float64, device="cuda")
    a.mcs(n, series)
    rows = []
    for _ in range(n):
        b.metropolis_sweep()
        for _ in range(3):
            b.overrelax_sweep()
        rows.append(b.measure())
        b.pt_exchange()
    assert np.array_equal(a.get_state().view(np.uint32), b.get_state().view(np.uint32))
    assert np.array_equal(a.get_perm(), b.get_perm())
    assert np.array_equal(a.get_counters(), [n, 3 * n, n])
    assert np.array_equal(series.cpu().numpy(), np.stack(rows))


@pytest.mark.parametrize("L,R,fused,n_or", [(8, 8, 1, 1), (32, 5, 1, 2), (32, 3, 0, 1), (64, 2, 1, 1)])
def test_mcs_graph_replay_equals_eager_launches(xy_mod, L, R, fused, n_or):
    """XY_OPT_CUDA_GRAPH: xy_mcs replays one captured graph per step with the counters on the device.
    States, permutations, counters, acceptance counts and the observable series must equal, bit for
    bit, those of eagerly launched steps -- over two calls, so the graph is re-used with new counters."""
    import torch
    betas = inputs.beta_ladder(0.45, 0.46, R)
    runs = []
    for graph in (1, 0):
        xy = xy_mod.XY(L, R, betas, SEED)
        xy.set_option(xy_mod.XY_OPT_RESIDENT, 0)
        xy.set_option(xy_mod.XY_OPT_CUDA_GRAPH, graph)
        xy.set_option(xy_mod.XY_OPT_FUSED_MEASURE, fused)
        xy.set_option(xy_mod.XY_OPT_OR_PER_MCS, n_or)
        xy.init_random()
        s1 = torch.zeros(7, R, 5, dtype=torch.float64, device="cuda")
        s2 = torch.zeros(5, R, 5, dtype=torch.float64, device="cuda")
        n0 = xy.get_launch_count()
        xy.mcs(7, s1)
        xy.mcs(5, s2)
        xy.mcs(4)                                             # no series
        runs.append((xy.get_state(), xy.get_perm(), xy.get_counters(), xy.get_accept_counts(), s1.cpu().numpy(),
                     s2.cpu().numpy(), xy.measure(), xy.get_launch_count() - n0))
    a, b = runs
    assert np.array_equal(a[0].view(np.uint32), b[0].view(np.uint32))
    assert np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2]) and np.array_equal(a[2], [16, 16 * n_or, 16])
    assert np.array_equal(a[3][0], b[3][0]) and np.array_equal(a[3][1], b[3][1])
    assert np.array_equal(a[4], b[4]) and np.array_equal(a[5], b[5]) and np.array_equal(a[6], b[6])
    assert np.all(a[4][:, :, 3] > 0)                          # every row was written
    assert a[7] == b[7] + 3, "same kernels per step, plus one counter upload per call"


def test_user_stream_and_context_lifetime(xy_mod):
    """A caller-owned (non-blocking) torch stream: same results as the library's own stream, graph replay
    included; and contexts can be created and destroyed repeatedly without leaking device memory."""
    import torch
    L, R = 32, 4
    betas = inputs.beta_ladder(0.45, 0.46, R)
    ref = xy_mod.XY(L, R, betas, SEED)
    ref.init_random(); ref.mcs(6)
    want = ref.get_state()
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        xy = xy_mod.XY(L, R, betas, SEED, stream=st)
        xy.init_random(); xy.mcs(6)
        got = xy.get_state()
    assert np.array_equal(got.view(np.uint32), want.view(np.uint32))
    xy.close(); ref.close()
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(40):
        t = xy_mod.XY(L, R, betas, SEED)
        t.init_random(); t.mcs(3); t.measure()
        t.close()
    torch.cuda.synchronize()
    assert free0 - torch.cuda.mem_get_info()[0] < 64 << 20


def test_gpu_sampler_against_closed_forms(xy_mod):
    """The GPU chain pinned to mathematics instead of to the oracle:
    high-temperature series <cos> per bond = t + 8 t^3 t' (t = I1/I0) at beta = 0.1, with the exchanges on
    (all beta equal: every attempted pair swaps, which must not change anything); beta = 0 gives <E> = 0;
    and the ordered state at huge beta is a fixed point of the whole step with E/N = -3."""
    import torch
    from scipy.special import i0, i1
    L, R, T, burn = 16, 32, 400, 20
    N = L ** 3
    for beta in (0.1, 0.0):
        xy = xy_mod.XY(L, R, np.full(R, beta), SEED + 7)
        xy.init_random()
        series = torch.zeros(burn + T, R, 5, dtype=torch.float64, device="cuda")
        xy.mcs(burn + T, series)
        e = series.cpu().numpy()[burn:, :, 0] / N
        mean, err = H.mean_and_err_over_replicas(e)
        if beta > 0:
            t = i1(beta) / i0(beta)
            want = -3 * (t + 8 * t ** 3 * (1 - t / beta - t * t))
        else:
            want = 0.0
        print("beta", beta, "E/N", mean, "+-", err, "want", want)
        assert err < 3e-4 and abs(mean - want) < 4 * err + 2e-4, (beta, mean, want, err)
    xy = xy_mod.XY(L, 4, np.full(4, 1e30), SEED)
    xy.init_ordered(0.0)
    xy.mcs(5)
    assert np.array_equal(xy.get_state(), np.zeros((4, L, L, L), dtype=np.float32))
    o = xy.measure()
    assert np.allclose(o[:, 0], -3.0 * N) and np.allclose(o[:, 1], N) and np.allclose(o[:, 2], 0.0)


# ---- P7: long-run statistics ---------------------------------------------------------------------
def _run_means(series, N):
    """series [T,R,5] (after the discarded head) -> time averages E/N [R], <M2> [R], <M4> [R]."""
    return series[..., 0].mean(axis=0) / N, series[..., 3].mean(axis=0), series[..., 4].mean(axis=0)


def _stored_oracle_runs(cfg):
    """tests/golden/p7_oracle_<cfg>.txt (written by tests/golden/make_p7_oracle.py, which calls only the oracle)
    -> arrays [n_runs, R] of <E>/N, <M2>, <M4> and the acceptance fractions [n_runs, 2]."""
    path = os.path.join(os.path.dirname(__file__), "golden", f"p7_oracle_{cfg.name}.txt")
    rows, acc = {}, {}
    for line in open(path):
        w = line.split("#")[0].split()
        if not w:
            continue
        if w[0] == "acc":
            acc[int(w[1])] = (float(w[2]), float(w[3]))
        else:
            rows.setdefault(int(w[0]), {})[int(w[1])] = [float(v) for v in w[2:5]]
    ks = sorted(k for k in rows if len(rows[k]) == cfg.R and k in acc)
    a = np.array([[rows[k][r] for r in range(cfg.R)] for k in ks])            # [n_runs, R, 3]
    return a[..., 0], a[..., 1], a[..., 2], np.array([acc[k] for k in ks])


def _welch(a, b):
    """Welch's t and its Welch-Satterthwaite degrees of freedom for two samples along axis 0."""
    va, vb = a.var(axis=0, ddof=1) / a.shape[0], b.var(axis=0, ddof=1) / b.shape[0]
    t = (a.mean(axis=0) - b.mean(axis=0)) / np.sqrt(va + vb)
    dof = (va + vb) ** 2 / (va ** 2 / (a.shape[0] - 1) + vb ** 2 / (b.shape[0] - 1))
    return t, dof


@pytest.mark.parametrize("idx,n_gpu_runs,n_live_oracle_runs", [(0, 48, 48), (1, 16, 0), (2, 16, 0)])
def test_long_run_statistics(xy_mod, oracle_mod, idx, n_gpu_runs, n_live_oracle_runs):
    """P7 (north_star: "Long-run <E> and Binder ratio must agree within 3 sigma") on BASELINE.json configs 1-3
    at their stated lengths (200 / 2000 / 1000 MCS, first quarter discarded).

    The time series of one run is autocorrelated and its replicas are coupled by the exchanges, so sigma comes
    from the scatter over INDEPENDENT runs (all seeds different): Welch's t of GPU runs against oracle runs,
    per rank and for the average over ranks, for <E>/N and for Q2 = <M4>/<M2>^2 (from the runs' pooled moments
    via leave-one-out jackknife values, because Q2 is a ratio of time averages).  Config 1's oracle runs are
    made here; for configs 2-3 (35 s and 5 min of 16 cores per run) they are the stored
    tests/golden/p7_oracle_*.txt, written by a committed script that calls only the oracle.

    Bars: |t| < 3 on the rank average; the 2R per-rank values (two observables) are tested simultaneously, so
    each gets the two-sided Student-t quantile at the 3-sigma level divided by 2R (Bonferroni), with Welch's
    degrees of freedom."""
    import torch
    from scipy import stats
    cfg = inputs.CONFIGS[idx]
    L, R, N, n_mcs = cfg.L, cfg.R, cfg.L ** 3, cfg.mcs
    betas = inputs.betas_of(cfg)
    head = n_mcs // 4
    G = []
    for k in range(n_gpu_runs):
        xy = xy_mod.XY(L, R, betas, SEED + 1000 + k)
        xy.init_random()
        series = torch.zeros(n_mcs, R, 5, dtype=torch.float64, device="cuda")
        xy.mcs(n_mcs, series)
        G.append(_run_means(series.cpu().numpy()[head:], N))
    gm, gpt = xy.get_accept_counts()
    g_acc = (gm.sum() / (n_mcs * R * N), gpt.sum() / max(1, n_mcs * (R - 1) / 2))
    ge, g2, g4 = (np.stack([g[j] for g in G]) for j in range(3))                 # [n_runs, R]
    if n_live_oracle_runs:
        O = []
        for k in range(n_live_oracle_runs):
            ora = oracle_mod.XYOracle(L, R, betas, SEED + 2000 + k, threads=NCPU)
            ora.init_random()
            O.append(_run_means(np.stack([ora.mcs() for _ in range(n_mcs)])[head:], N))
        oe, o2, o4 = (np.stack([o[j] for o in O]) for j in range(3))
        om, opt = ora.get_accept_counts()
        o_acc = (om.sum() / (n_mcs * R * N), opt.sum() / max(1, n_mcs * (R - 1) / 2))
    else:
        oe, o2, o4, acc = _stored_oracle_runs(cfg)
        assert oe.shape[0] >= 4, "too few stored oracle runs"
        o_acc = tuple(acc[-1])

    def q2_jackknife(m2, m4):
        """Per run pseudo-values of Q2 = mean(M4)/mean(M2)^2 (pooled over runs): their mean and scatter give the
        estimate and its error without the bias of averaging per-run ratios."""
        n = m2.shape[0]
        full = m4.mean(axis=0) / m2.mean(axis=0) ** 2
        loo = (m4.sum(axis=0) - m4) / (n - 1) / ((m2.sum(axis=0) - m2) / (n - 1)) ** 2
        return n * full - (n - 1) * loo

    p3 = 2.0 * stats.norm.sf(3.0)                                              # two-sided 3-sigma level
    report = []
    for name, a, b in (("E/N", ge, oe), ("Q2", q2_jackknife(g2, g4), q2_jackknife(o2, o4))):
        t, dof = _welch(a, b)
        bound = stats.t.isf(p3 / (2 * 2 * R), dof)                              # Bonferroni over the 2R per-rank tests
        t_all, dof_all = _welch(a.mean(axis=1), b.mean(axis=1))
        report.append((name, float(np.abs(t).max()), float(bound.min()), float(t_all), float(dof_all)))
        print(f"P7 {cfg.name} {name}: gpu runs {a.shape[0]}, oracle runs {b.shape[0]}; rank 0/{R - 1} gpu {a.mean(axis=0)[[0, -1]]} "
              f"oracle {b.mean(axis=0)[[0, -1]]}; per-rank t {np.round(t, 2).tolist()}; max|t| {np.abs(t).max():.2f} "
              f"(Bonferroni bound {bound.min():.2f}, dof {dof.min():.1f}); t(rank average) {t_all:.2f} (dof {dof_all:.1f})")
        assert np.all(np.abs(t) < bound), (name, t, bound)
        assert abs(t_all) < 3.0, (name, t_all)
    print(f"P7 {cfg.name} acceptance: gpu metropolis {g_acc[0]:.4f} exchange {g_acc[1]:.4f}; oracle {o_acc[0]:.4f} {o_acc[1]:.4f}")
    assert abs(g_acc[0] / o_acc[0] - 1) < 0.01 and g_acc[1] > 0 and abs(g_acc[1] / max(o_acc[1], 1e-9) - 1) < 0.2
