"""Seeded synthetic inputs shared by the tests, bench.py and smoke().

This module holds NONE of the method's arithmetic (no Hamiltonian, no update rule, no RNG of
the method): only the workload table of BASELINE.json, the beta ladders, and generators of
spin configurations used as test inputs.  It is the one module both the CUDA path's callers
and the oracle's callers may import.

The paper's workloads are lattices produced by the simulation itself, not a
data set, so the five BASELINE.json configs ARE the stand-ins: cubic periodic L^3, R replicas,
beta linearly spaced around beta_c ~ 0.4542 (the paper's own non-uniform ladder, PAPER.md:62,
is not printed).
"""
from collections import namedtuple

import numpy as np

SEED = 0x12110780          # BASELINE.json gives none; DESIGN.md fixes this one for every config

Config = namedtuple("Config", "name L R beta_lo beta_hi start mcs measure_every")

# BASELINE.json "configs", in order.  CONFIGS[0] is the small case the oracle finishes in
# seconds; CONFIGS[4] (L=160, R=64) is the one the metric is quoted on.
CONFIGS = (
    Config("cfg1_L8_R8", 8, 8, 0.44, 0.47, "random", 200, 1),
    Config("cfg2_L32_R16", 32, 16, 0.450, 0.458, "random", 2000, 1),
    Config("cfg3_L64_R32", 64, 32, 0.4530, 0.4555, "random", 1000, 1),
    Config("cfg4_L128_R32", 128, 32, 0.4537, 0.4547, "ordered", 500, 5),
    Config("cfg5_L160_R64", 160, 64, 0.4538, 0.4546, "random", 500, 1),
)
HEADLINE = CONFIGS[4]


def config(name_or_index):
    if isinstance(name_or_index, int):
        return CONFIGS[name_or_index]
    for c in CONFIGS:
        if c.name == name_or_index:
            return c
    raise KeyError(name_or_index)


# The paper's own workload families: 34 temperatures in T = [2.1, 2.3] for L = 64, 80, 96, 128 and 13 in
# T = [2.19, 2.21] for L = 160, "chosen such that the acceptance rate of swaps is independent of the temperatures".  The
# ladder itself is not printed: the stand-in starts geometric in beta (non-uniform) and ladder.equalise_swap_acceptance
# moves the inner temperatures until the measured per-pair acceptance is flat.
PaperFamily = namedtuple("PaperFamily", "name L R T_lo T_hi start mcs")
PAPER_FAMILIES = (
    PaperFamily("paper_L64_R34", 64, 34, 2.1, 2.3, "random", 200),
    PaperFamily("paper_L80_R34", 80, 34, 2.1, 2.3, "random", 200),
    PaperFamily("paper_L96_R34", 96, 34, 2.1, 2.3, "random", 200),
    PaperFamily("paper_L128_R34", 128, 34, 2.1, 2.3, "random", 200),
    PaperFamily("paper_L160_R13", 160, 13, 2.19, 2.21, "random", 200),
)


def paper_family(name):
    for f in PAPER_FAMILIES:
        if f.name == name:
            return f
    raise KeyError(name)


def geometric_beta_ladder(T_lo, T_hi, R):
    """R inverse temperatures from 1/T_hi up to 1/T_lo, constant RATIO between neighbours (so non-uniform in beta and in T)."""
    lo, hi = 1.0 / T_hi, 1.0 / T_lo
    if R == 1:
        return np.array([lo], dtype=np.float64)
    k = np.arange(R, dtype=np.float64)
    b = lo * (hi / lo) ** (k / (R - 1))
    b[0], b[-1] = lo, hi
    return b


def betas_of_family(fam):
    return geometric_beta_ladder(fam.T_lo, fam.T_hi, fam.R)


def beta_ladder(beta_lo, beta_hi, R):
    """beta_k = lo + k (hi - lo)/(R-1), k = 0..R-1, in double, inclusive ends."""
    if R == 1:
        return np.array([beta_lo], dtype=np.float64)
    k = np.arange(R, dtype=np.float64)
    return beta_lo + k * ((beta_hi - beta_lo) / (R - 1))


def betas_of(cfg):
    return beta_ladder(cfg.beta_lo, cfg.beta_hi, cfg.R)


# ----------------------------------------------------------------------------------------
# Spin configurations used as test inputs, natural layout [R, z, y, x], fp32 angles.
# ----------------------------------------------------------------------------------------
def uniform_state(L, R, seed):
    """i.i.d. angles uniform on [0, 2pi) -- the value distribution of a random start."""
    rng = np.random.default_rng(seed)
    s = rng.random((R, L, L, L), dtype=np.float32) * np.float32(2 * np.pi)
    return np.minimum(s, np.float32(6.2831850)).astype(np.float32)


def ordered_state(L, R, theta0=0.0):
    return np.full((R, L, L, L), theta0, dtype=np.float32)


def helical_state(L, R, k=(1, 0, 0), phase=0.0):
    """theta = 2pi (kx x + ky y + kz z)/L + phase, reduced to [0, 2pi): a spin wave."""
    z, y, x = np.meshgrid(np.arange(L), np.arange(L), np.arange(L), indexing="ij")
    t = (2.0 * np.pi * ((k[0] * x + k[1] * y + k[2] * z) % L) / L + phase) % (2.0 * np.pi)
    return np.broadcast_to(t.astype(np.float32), (R, L, L, L)).copy()


def staggered_state(L, R):
    """theta = 0 on even (x+y+z), pi on odd."""
    z, y, x = np.meshgrid(np.arange(L), np.arange(L), np.arange(L), indexing="ij")
    t = np.where(((x + y + z) & 1) == 0, 0.0, np.pi).astype(np.float32)
    return np.broadcast_to(t, (R, L, L, L)).copy()


def smooth_state(L, R, seed, width=0.6):
    """Angles clustered around a per-replica mean direction (a partially ordered state, like
    the equilibrium configurations at beta >= beta_c that the big lattices spend their time in)."""
    rng = np.random.default_rng(seed)
    mean = rng.random((R, 1, 1, 1)) * 2 * np.pi
    t = (mean + width * rng.standard_normal((R, L, L, L))) % (2 * np.pi)
    return np.minimum(t, 6.2831850).astype(np.float32)
