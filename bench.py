#!/usr/bin/env python
"""bench.py -- spin-updates/ns of one Monte Carlo step (MCS) of the 3-D XY model at L=160 x 64 replicas.

A "step" is one pass of the whole hot path over all R replicas: checkerboard Metropolis sweep,
checkerboard over-relaxation sweep, observable reduction, replica exchange.  One
spin-update = one Metropolis attempt or one over-relaxation reflection of one site, so a step
performs 2 * L^3 * R spin-updates.  Prints ONE JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 0..4]

N > 1 (under torchrun): the path does not shard (north_star: one GPU) -- every rank runs an
independent replica set of the same size ("replicas only", weak scaling), no data-path collective.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1211_0780_b200 import inputs  # noqa: E402  (no CUDA needed to import)

METRIC = "spin-updates/ns per MCS at L=160x64 replicas"
UNIT = "spin-updates/ns"
BYTES_PER_UPDATE = 12          # colour-split layout: read own + other colour, write own
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel from the committed
# `ncu --set full` capture (profiles/), keyed by config name; None until captured.
NCU_TRAFFIC_BYTES = {}
try:
    with open(os.path.join(ROOT, "profiles", "traffic.json.txt")) as _f:
        NCU_TRAFFIC_BYTES = json.load(_f)
except Exception:
    pass


def measured_peak_gbs():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons every 50 ms DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, device_index):
        self.rows, self.proc, self.thread = [], None, None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "50", "-i", str(device_index)],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [c.strip() for c in line.split(",")]))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()          # exactly the process started above
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        rows = [r for t, r in self.rows if t0 <= t <= t1 + 0.2 and len(r) >= 7] or [r for _, r in self.rows if len(r) >= 7]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm = sorted(float(r[0]) for r in rows)
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        reasons = [n for i, n in enumerate(names) if any(r[3 + i].lower().startswith("active") for r in rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(rows[0][1]), "power_w_max": max(float(r[2]) for r in rows),
                "samples": len(rows), "reasons": reasons}


def combine_ranks(ms_local, units_local, dist=None, device="cpu"):
    """max over ranks of the elapsed time, sum over ranks of the units processed (spin-updates)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(ms_local), float(units_local)
    import torch
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units_local)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


NCU_PEAK_GBS = 8184.0          # ncu's own denominator for dram % of peak: 3996 MHz x 8192 bit x 2


def config_keys(cfg):
    """The workload description both arms print (the reference arm adds what it sampled)."""
    return {"workload": cfg.name, "L": cfg.L, "R": cfg.R, "beta": [cfg.beta_lo, cfg.beta_hi], "start": cfg.start,
            "ladder": "geometric in beta (PAPER.md:62 family)" if cfg.name.startswith("paper_") else "linear in beta",
            "state_bytes": 4 * cfg.L ** 3 * cfg.R}


def oracle_sample_rate(cfg, n_slots, steps, warmup, threads):
    """The CPU oracle, as it stands, on a bounded sample: full MCS of the first n_slots temperatures of cfg.
    XYOracle.mcs() reduces the observables once per step and hands the energies to the exchange."""
    from oracle import xy_oracle
    betas = inputs.betas_of(cfg)[:n_slots]
    ora = xy_oracle.XYOracle(cfg.L, n_slots, betas, inputs.SEED, threads=threads)
    if cfg.start == "random":
        ora.init_random()
    else:
        ora.init_ordered(0.0)
    for _ in range(warmup):
        ora.mcs()
    t0 = time.perf_counter()
    for _ in range(steps):
        ora.mcs()
    dt = time.perf_counter() - t0
    updates = 2.0 * cfg.L ** 3 * n_slots * steps
    return updates / dt * 1e-9, dt / steps * 1e3


def run_reference(args, cfg):
    """--impl reference: the oracle on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    cores = os.cpu_count() or 1
    n_slots = max(1, min(cfg.R, cores))
    value, ms = oracle_sample_rate(cfg, n_slots, args.steps, args.warmup, threads=n_slots)
    sample = f"full MCS (Metropolis+OR+measure+PT) of the first {n_slots} of {cfg.R} temperatures at L={cfg.L}, one thread per replica"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": dict(config_keys(cfg), sampled_replicas=n_slots),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": n_slots, "kind": "oracle", "sample": sample,
                         "ns_per_update_per_core": n_slots / value},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def time_other_workloads(binding, torch, skip_name, steps=20, warmup=5):
    """Driver-timed numbers for the workloads the headline is NOT quoted on: BASELINE.json configs 1-4 and the paper's
    own five families, `steps` steps of xy_mcs each after `warmup` (CUDA events, device-resident state,
    the library's default path: the resident kernel for L <= 48, graph-replayed per-pass kernels above).  Configs 1-3
    and the L = 64 family fit in the 126 MB L2 and are not flushed between steps (stated per entry): their numbers are
    updates/ns, not an HBM roofline."""
    work = [(c.name, c.L, c.R, inputs.betas_of(c), c.start, "linear in beta") for c in inputs.CONFIGS]
    work += [(f.name, f.L, f.R, inputs.betas_of_family(f), f.start, "geometric in beta (PAPER.md:62 family)") for f in inputs.PAPER_FAMILIES]
    out = []
    for name, L, R, betas, start, ladder in work:
        if name == skip_name:
            continue
        xy = binding.XY(L, R, betas, inputs.SEED)
        xy.init_random() if start == "random" else xy.init_ordered(0.0)
        xy.mcs(warmup)
        torch.cuda.synchronize()
        n0 = xy.get_launch_count()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        xy.mcs(steps)
        b.record()
        torch.cuda.synchronize()
        xy.synchronize()                               # raises if a close-decision queue overflowed or a launch aborted
        ms = a.elapsed_time(b) / steps
        plan = xy.get_resident_plan()
        state = 4 * L ** 3 * R
        out.append({"workload": name, "L": L, "R": R, "ladder": ladder, "start": start, "steps": steps, "warmup": warmup,
                    "ms_per_step": ms, "updates_per_ns": 2.0 * L ** 3 * R / (ms * 1e-3) * 1e-9,
                    "path": ("resident kernel: %d block(s) per slot, %d slot(s) per block, %d blocks" % (plan["blocks_per_slot"], plan["slots_per_block"], plan["blocks"]))
                            if plan["resident"] else "per-pass kernels, tiles %d x %d, graph replay" % (xy.get_option(binding.XY_OPT_TILE_Y), xy.get_option(binding.XY_OPT_TILE_Z)),
                    "gpu_launches": xy.get_launch_count() - n0,
                    "memory": "state %.1f MB: %s" % (state / 1e6, "L2-resident, no flush between steps" if state < 120e6 else "larger than L2 (HBM)"),
                    "hbm_roofline_frac": (2.0 * L ** 3 * R * BYTES_PER_UPDATE / (ms * 1e-3) * 1e-9 / measured_peak_gbs()[0]) if state >= 120e6 else None})
        xy.close()
    return out


def run_ours(args, cfg):
    import torch
    import torch.distributed as dist
    from paper_1211_0780_b200 import binding
    from paper_1211_0780_b200.build import build_library

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback for the product path)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        build_library()
    if world > 1:
        dist.barrier()
    binding.load_library()

    L, R, N = cfg.L, cfg.R, cfg.L ** 3
    updates_per_step = 2.0 * N * R
    xy = binding.XY(L, R, inputs.betas_of(cfg), inputs.SEED + rank)      # independent replica set per rank
    if cfg.start == "random":
        xy.init_random()
    else:
        xy.init_ordered(0.0)
    if args.tile_y:
        xy.set_option(binding.XY_OPT_TILE_Y, args.tile_y)
    if args.tile_z:
        xy.set_option(binding.XY_OPT_TILE_Z, args.tile_z)
    if args.generic_kernel:
        xy.set_option(binding.XY_OPT_GENERIC_KERNEL, 1)
    if args.slot_chunk:
        xy.set_option(binding.XY_OPT_SLOT_CHUNK, args.slot_chunk)
    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident throughput ("value"): K steps, nothing but the library's own kernels on the stream ----
    xy.mcs(args.warmup)
    barrier()
    n0 = xy.get_launch_count()
    sampler = ClockSampler(local) if rank == 0 else None
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.time()
    e0.record()
    xy.mcs(args.steps)
    e1.record()
    barrier()
    ms_local = e0.elapsed_time(e1)
    launches = xy.get_launch_count() - n0
    # ---- the same K steps again with a CUDA-event pair around every launch (XY_OPT_PROFILE): per-kernel
    #      durations for the roofline; the event records cost ~2 % of a step, so this pass is not the headline
    xy.set_option(binding.XY_OPT_PROFILE, 1)
    xy.mcs(1)
    xy.get_kernel_times()
    barrier()
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record()
    xy.mcs(args.steps)
    p1.record()
    barrier()
    t1 = time.time()
    ms_profiled = p0.elapsed_time(p1)
    ktimes = xy.get_kernel_times()
    clocks = sampler.stop(t0, t1) if sampler else None
    ms, units = combine_ranks(ms_local, updates_per_step * args.steps, dist if world > 1 else None, "cuda")
    obs = xy.measure()

    # ---- end to end through the C ABI with HOST buffers ---------------------------------------------
    # step = xy_set_state(pinned host natural-layout state) -> MCS -> xy_measure(host out) + xy_get_perm(host out)
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    xy.set_option(binding.XY_OPT_PROFILE, 0)
    host = torch.empty(R * N, dtype=torch.float32, pin_memory=True)
    xy.get_state(host)
    for _ in range(2):
        xy.set_state(host); xy.mcs(1); xy.measure(); xy.get_perm()
    barrier()
    e0.record()
    for _ in range(e2e_steps):
        xy.set_state(host); xy.mcs(1); xy.measure(); xy.get_perm()
    e1.record()
    barrier()
    e2e_ms, e2e_units = combine_ranks(e0.elapsed_time(e1), updates_per_step * e2e_steps, dist if world > 1 else None, "cuda")

    if world > 1:
        dist.destroy_process_group()
    if rank != 0:
        return
    peak, peak_src = measured_peak_gbs()
    # dominant kernel = the class with the largest device time in the timed region
    dom = max(("metropolis", "overrelax", "measure", "resident"), key=lambda k: ktimes[k][0])
    # the resident kernel (small lattices) runs all K steps in ONE launch: its algorithmic bytes are those of K whole steps
    per_launch_bytes = {"metropolis": BYTES_PER_UPDATE * N * R / 2, "overrelax": BYTES_PER_UPDATE * N * R / 2,
                        "measure": 4.0 * N * R, "resident": BYTES_PER_UPDATE * updates_per_step * args.steps}
    kern = {}
    for k, (tot, n) in ktimes.items():
        if n:
            kern[k] = {"launches": n, "avg_ms": tot / n, "share": tot / (ms_profiled + 1e-30)}
            if k in per_launch_bytes:
                kern[k]["algorithmic_GBps"] = per_launch_bytes[k] / (tot / n * 1e-3) * 1e-9
    ach = kern[dom]["algorithmic_GBps"]
    traffic = NCU_TRAFFIC_BYTES.get(cfg.name, {}).get(dom)
    out = {
        "metric": METRIC, "value": units / (ms * 1e-3) * 1e-9, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": dict(config_keys(cfg), l2=f"inputs larger than L2 (state {4 * N * R / 1e9:.2f} GB >> 126 MB)" if 4 * N * R > 4e8
                   else "state fits in L2; no flush", parallelism="replicas only" if world > 1 else "1 GPU",
                   tile_y=xy.get_option(binding.XY_OPT_TILE_Y), tile_z=xy.get_option(binding.XY_OPT_TILE_Z),
                   slot_chunk=xy.get_option(binding.XY_OPT_SLOT_CHUNK)),
        "site_mcs_per_ns": units / 2 / (ms * 1e-3) * 1e-9,
        "hbm_roofline_frac_whole_mcs": units * BYTES_PER_UPDATE / (ms * 1e-3) * 1e-9 / peak,
        "roofline": {"bound": "hbm", "kernel": dom, "achieved": ach, "peak": peak, "peak_source": peak_src, "unit": "GB/s",
                     "frac": ach / peak, "traffic": traffic, "traffic_build": NCU_TRAFFIC_BYTES.get(cfg.name, {}).get("build"),
                     "bytes_per_update": BYTES_PER_UPDATE,
                     "algorithmic_bytes_per_launch": per_launch_bytes[dom],
                     # the second denominator SURVEY.md 8(d) asks for, labelled: ncu's theoretical DRAM peak, and the
                     # dram throughput % ncu itself reported for this kernel in the committed capture (profiles/)
                     "note": ("spins resident in shared memory for the whole call (XY_OPT_RESIDENT): no HBM traffic inside the timed region; "
                              "achieved is the 12 B/update model over time, for comparison with the per-pass kernels") if dom == "resident" else None,
                     "frac_of_ncu_peak": ach / NCU_PEAK_GBS, "ncu_peak": NCU_PEAK_GBS,
                     "ncu_dram_pct_of_peak_sustained_elapsed": NCU_TRAFFIC_BYTES.get(cfg.name, {}).get(dom + "_dram_pct")},
        "hbm_roofline_frac_whole_mcs_of_ncu_peak": units * BYTES_PER_UPDATE / (ms * 1e-3) * 1e-9 / NCU_PEAK_GBS,
        "kernels": kern,
        "path": xy.get_resident_plan(),
        "kernels_measured": f"second pass of {args.steps} steps with a CUDA-event pair around every launch: {ms_profiled / args.steps:.4f} ms per step",
        "e2e": {"value": e2e_units / (e2e_ms * 1e-3) * 1e-9, "unit": UNIT, "h2d_bytes_per_step": 4 * N * R,
                "d2h_bytes_per_step": R * 5 * 8 + R * 4, "steps": e2e_steps, "ms_per_step": e2e_ms / e2e_steps,
                "call": "xy_set_state(pinned host) -> xy_mcs(1) -> xy_measure(host) + xy_get_perm(host)"},
        "gpu_launches": launches,
        "clocks": clocks,
        "observables_rank0": {"E_per_site": obs[0, 0] / N, "m": float(np.sqrt(obs[0, 3])) / N},
    }
    if world == 1 and not args.no_other_workloads and not any((args.tile_y, args.tile_z, args.generic_kernel, args.slot_chunk)):
        xy.close()
        out["other_workloads"] = time_other_workloads(binding, torch, cfg.name)
    if not args.no_cpu_baseline and world == 1:
        cores = os.cpu_count() or 1
        n_slots = max(1, min(R, cores))
        v, _ = oracle_sample_rate(cfg, n_slots, 2, 1, threads=n_slots)
        out["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": n_slots, "kind": "oracle",
                               "sample": f"2 timed MCS (after 1 warm-up) of the first {n_slots} of {R} temperatures at L={L}, "
                                         "one thread per replica; one reduction per step",
                               "ns_per_update_per_core": n_slots / v, "gpu_over_cpu": out["value"] / v}
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="index into BASELINE.json configs (default 4: L=160, R=64)")
    ap.add_argument("--family", default=None, help="one of the paper's own workload families instead (PAPER.md:62), e.g. paper_L80_R34: "
                                                  "non-uniform (geometric) ladder; see inputs.PAPER_FAMILIES")
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-workloads", action="store_true", help="skip the short timings of the other configs / paper families")
    ap.add_argument("--tile-z", type=int, default=0, help="override the march length (tuning; 0 = library default)")
    ap.add_argument("--tile-y", type=int, default=0, help="override the tile rows (tuning; 0 = library default)")
    ap.add_argument("--generic-kernel", action="store_true", help="force the run-time-geometry colour-pass kernel (tuning)")
    ap.add_argument("--slot-chunk", type=int, default=0, help="XY_OPT_SLOT_CHUNK: run the colour passes of K slots at a time back to back "
                                                          "(L2-resident schedule, SURVEY 8(f) f2; 0 = library default: all slots per pass)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    cfg = inputs.CONFIGS[args.config]
    if args.family:                                 # same fields as a Config; the ladder is geometric in beta, not linear
        fam = inputs.paper_family(args.family)
        b = inputs.betas_of_family(fam)
        cfg = inputs.Config(fam.name, fam.L, fam.R, float(b[0]), float(b[-1]), fam.start, fam.mcs, 1)
        inputs.betas_of = lambda c, _b=b: _b      # every arm of this run uses the family's ladder
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
