#!/usr/bin/env python
"""Writes tests/golden/p7_oracle_<config>.txt: the ORACLE's long-run statistics of a BASELINE.json config at its
full stated length, for the P7 parity test (north_star "Long-run <E> and Binder ratio must
agree within 3 sigma").

Calls only oracle/ and the seeded input recipe (paper_1211_0780_b200.inputs holds no arithmetic of the method).
One oracle run of config 3 (L=64, R=32, 1000 MCS) costs about 5 core-hours / #cores, far too slow to repeat
inside the GPU test run, and the oracle is a deterministic function of (seed, betas, L, R) (its result does
not depend on the thread count: tests/test_oracle_pins.py), so its per-run time averages are stored once.

    python tests/golden/make_p7_oracle.py --config 1 --runs 8      # cfg2_L32_R16, 2000 MCS
    python tests/golden/make_p7_oracle.py --config 2 --runs 6      # cfg3_L64_R32, 1000 MCS

Run k uses seed SEED + 2000 + k, a random start, the config's linear beta ladder and every MCS of the stated
length; the first quarter is discarded; per rank the time averages of E/N, |M|^2 and |M|^4 are written with
17 significant digits.  Existing runs in the output file are kept (runs are appended), so the work can be
split over several invocations (--first K).
"""
import argparse
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import xy_oracle  # noqa: E402
from paper_1211_0780_b200 import inputs  # noqa: E402

SEED_OFFSET = 2000


def run_one(cfg, k, threads):
    betas = inputs.betas_of(cfg)
    ora = xy_oracle.XYOracle(cfg.L, cfg.R, betas, inputs.SEED + SEED_OFFSET + k, threads=threads)
    if cfg.start == "random":
        ora.init_random()
    else:
        ora.init_ordered(0.0)
    series = np.stack([ora.mcs() for _ in range(cfg.mcs)])           # [T, R, 5] by rank
    tail = series[cfg.mcs // 4:]
    N = cfg.L ** 3
    met, pt = ora.get_accept_counts()
    return (tail[..., 0].mean(axis=0) / N, tail[..., 3].mean(axis=0), tail[..., 4].mean(axis=0),
            met.sum() / (cfg.mcs * cfg.R * N), pt.sum() / max(1, cfg.mcs * (cfg.R - 1) / 2))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, required=True)
    ap.add_argument("--runs", type=int, default=8)
    ap.add_argument("--first", type=int, default=0)
    ap.add_argument("--threads", type=int, default=os.cpu_count() or 1)
    ap.add_argument("--out", default=None)
    a = ap.parse_args()
    cfg = inputs.CONFIGS[a.config]
    out = a.out or os.path.join(os.path.dirname(os.path.abspath(__file__)), f"p7_oracle_{cfg.name}.txt")
    if not os.path.exists(out):
        with open(out, "w") as f:
            f.write(f"# Oracle long-run statistics of BASELINE.json config {cfg.name}: L={cfg.L} R={cfg.R} "
                    f"beta {cfg.beta_lo}..{cfg.beta_hi} linear, {cfg.start} start, {cfg.mcs} MCS, first {cfg.mcs // 4} discarded.\n"
                    "# Written by tests/golden/make_p7_oracle.py, which calls only oracle/ (PAPER.md:30 MCS; :45-50 Eq. 3; :52-56 Eqs. 4-5).\n"
                    f"# Run k uses seed 0x{inputs.SEED:x} + {SEED_OFFSET} + k.  Columns: run rank <E>/N <|M|^2> <|M|^4>; lines 'acc run "
                    "metropolis_accept_fraction pt_accept_fraction'.\n")
    for k in range(a.first, a.first + a.runs):
        t0 = time.time()
        e, m2, m4, amet, apt = run_one(cfg, k, a.threads)
        with open(out, "a") as f:
            for r in range(cfg.R):
                f.write(f"{k} {r} {e[r]:.17g} {m2[r]:.17g} {m4[r]:.17g}\n")
            f.write(f"acc {k} {amet:.6f} {apt:.6f}\n")
        print(f"{cfg.name} run {k}: {time.time() - t0:.1f} s, <E>/N rank0 {e[0]:.6f}, met acc {amet:.4f}, pt acc {apt:.4f}", flush=True)


if __name__ == "__main__":
    main()
