#!/usr/bin/env python
"""bench.py -- atom-steps/s of the FP64 Tersoff/SW force + NVE hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config I] [--impl ours|reference]

A "step" is one velocity-Verlet NVE step of the whole hot path (kick+drift, neighbour rebuild every
10th step, pair kernel, gather, kick) on BASELINE.json config I (default 1 = configs[1]: Tersoff,
512 000 atoms).  Prints ONE JSON line.  N > 1 runs independent replicas
(the path is single-GPU by north_star: "replicas only"), one process per GPU under torchrun.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import md_inputs as mi  # noqa: E402

METRIC = "atom-steps/s (FP64 Tersoff/SW force+integrate)"
UNIT = "atom-steps/s"
# Algorithmic work of the dominant kernel (pair kernel): flop-equivalents per atom
# with add = mul = 1, fma = 2, div = 16, sqrt = 20, exp = 35, log = 50.
PAIR_FLOP_PER_ATOM = {"tersoff": 1370.0 + 340.0 + 300.0, "sw": 2300.0}
FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12      # 148 SMs x 64 DFMA/clk x 1.965 GHz = 37.2


def measured_peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return {}


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.05)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for t, line in self.rows:
            if not (t0 - 0.03 <= t <= t1 + 0.03):
                continue
            p = [c.strip() for c in line.split(",")]
            try:
                sm.append(float(p[0])); mx.append(float(p[1]))
            except Exception:
                continue
            for nm, v in zip(names, p[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no sample inside the timed region"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons),
                "samples": len(sm)}


def reference_sample_ncell(full_ncell, steps, warmup):
    """Bounded sample for the oracle: same recipe and seed, fewer cells, sized for <= ~100 s of CPU."""
    budget_atom_steps = 100.0 / 8e-6                         # oracle ~8 us per atom-step (1 core)
    n_max = budget_atom_steps / max(1, steps + warmup)
    nc = int((n_max / 8.0) ** (1.0 / 3.0))
    return max(3, min(full_ncell, nc))


def run_oracle(cfg_index, steps, warmup, ncell):
    import oracle                                            # the one CPU leg allowed to use oracle/
    c = mi.make_config(cfg_index, ncell=ncell)
    K = c["max_neighbors"] if c["potential"] == "tersoff" else 40
    st = {k: c[k] for k in ("x", "y", "z", "vx", "vy", "vz", "box", "mass")}
    r = oracle.nve_run(c["potential"], c["params"], st, warmup, c["dt"], c["rebuild_every"], c["r_list"], K)
    t0 = time.perf_counter()
    oracle.nve_run(c["potential"], c["params"], st, steps, c["dt"], c["rebuild_every"], c["r_list"], K, f=r["f"])
    dt = time.perf_counter() - t0
    return c["n"], dt


def main_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    full = mi.CONFIGS[args.config]
    ncell = reference_sample_ncell(full["ncell"], args.steps, args.warmup)
    n, dt = run_oracle(args.config, args.steps, args.warmup, ncell)
    value = n * args.steps / dt
    sample = (f"{ncell}^3 cells = {n} atoms of the same recipe and seed (of {full['ncell']}^3), "
              f"{args.steps} steps, 1 thread")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": full["name"], "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def traffic_from_profiles(kernel):
    """dram bytes per launch of `kernel` from the committed ncu summary (data file, not code)."""
    try:
        t = json.load(open(os.path.join(ROOT, "profiles", "traffic.json")))
        return t.get(kernel)
    except Exception:
        return None


def max_over_ranks(values, device, world):
    """Times of the slowest rank (the contract's max over ranks); identity for one rank."""
    import torch
    import torch.distributed as dist
    tv = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(tv, op=dist.ReduceOp.MAX)
    return [float(v) for v in tv.cpu()]


def aggregate_value(n_per_rank, steps, world, ms_max):
    """Whole-job atom-steps/s of `world` replicas of n_per_rank atoms each, timed by the slowest rank."""
    return world * n_per_rank * steps / (ms_max * 1e-3)


def main_ours(args):
    import torch
    import torch.distributed as dist

    import paper_1610_03343_b200 as md

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    c = mi.make_config(args.config)
    pot, n, K = c["potential"], c["n"], c["max_neighbors"]
    box, mass, dt, rebuild, r_list = list(c["box"]), c["mass"], c["dt"], c["rebuild_every"], c["r_list"]
    host0 = {k: torch.from_numpy(c[k].copy()) for k in ("x", "y", "z", "vx", "vy", "vz")}
    d = {k: v.to(dev) for k, v in host0.items()}
    f = torch.zeros((3, n), dtype=torch.float64, device=dev)
    pe = torch.zeros(n, dtype=torch.float64, device=dev)
    nl = md.md_neighbors_create(n, K)
    prec = md.MD_FP32 if args.fp32 else md.MD_FP64

    def run(first, nsteps, f_valid=True):
        md.md_nve_run(nl, pot, c["params"], n, d["x"], d["y"], d["z"], d["vx"], d["vy"], d["vz"], f, f_valid, pe,
                      box, mass, dt, nsteps, rebuild, r_list, precision=prec, first_step=first)

    run(0, 0, f_valid=False)                       # forces of the initial state
    run(0, args.warmup)
    step0 = args.warmup
    max_row = md.md_neighbors_status(nl)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2

    chunk = rebuild                                # one timed call = one rebuild cycle of md_nve_run

    def timed_pass(profile):
        """K steps as ceil(K/chunk) md_nve_run calls of `chunk` steps (the last one shorter), each bracketed
        by its own CUDA-event pair; L2 flushed (256 MiB written, then read back so that no dirty foreign
        lines are left to evict) before every call, outside the event pairs."""
        nonlocal step0
        md.md_profile_enable(nl, profile)
        md.md_profile_read(nl)
        sizes = [min(chunk, args.steps - k) for k in range(0, args.steps, chunk)]
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in sizes]
        barrier()
        t0 = time.perf_counter()
        done = 0
        for k, sz in enumerate(sizes):
            flush.zero_()                          # L2 flush between timed iterations (not timed)
            flush.sum()
            ev[k][0].record()
            run(step0 + done, sz)
            ev[k][1].record()
            done += sz
        torch.cuda.synchronize()
        t1 = time.perf_counter()
        barrier()
        step0 += args.steps
        ms = sum(a.elapsed_time(b) for a, b in ev)
        kinds_ms, launches = md.md_profile_read(nl)
        md.md_profile_enable(nl, False)
        return ms, kinds_ms, launches, t0, t1

    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.1)
    ms_total, _, launches, t0, t1 = timed_pass(False)
    clocks = sampler.stop(t0, t1)
    # same loop with per-kernel-kind events (roofline of the dominant kernel)
    ms_prof, kinds_ms, launches_prof, _, _ = timed_pass(True)
    # back-to-back steps, one C call, no flush (what a production MD loop does)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(); run(step0, args.steps); e1.record()
    torch.cuda.synchronize()
    ms_b2b = e0.elapsed_time(e1)
    step0 += args.steps
    md.md_neighbors_status(nl)
    e_final = float(pe.sum())

    # end to end through the C ABI with HOST (pinned) buffers: H2D + K steps + D2H inside the timed region
    hp = {k: v.clone().pin_memory() for k, v in host0.items()}
    hf = torch.zeros((3, n), dtype=torch.float64).pin_memory()
    hpe = torch.zeros(n, dtype=torch.float64).pin_memory()
    nl2 = md.md_neighbors_create(n, K)

    def e2e_call(nsteps):
        for k, v in host0.items():
            hp[k].copy_(v)
        barrier()
        t = time.perf_counter()
        md.md_nve_run_host(nl2, pot, c["params"], n, hp["x"], hp["y"], hp["z"], hp["vx"], hp["vy"], hp["vz"],
                           hf, hpe, box, mass, dt, nsteps, rebuild, r_list, precision=prec)
        return time.perf_counter() - t
    e2e_call(max(3, args.warmup))
    e2e_s = e2e_call(args.steps)
    md.md_neighbors_status(nl2)

    ms_total, ms_prof, ms_b2b, e2e_ms = max_over_ranks([ms_total, ms_prof, ms_b2b, e2e_s * 1e3], dev, world)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    peaks = measured_peaks()
    fp64_peak = md.md_probe_fp64_peak(20000)
    n_pair = max(1, launches_prof["pair"])
    pair_ms = kinds_ms["pair"] / n_pair
    achieved = PAIR_FLOP_PER_ATOM[pot] * n / (pair_ms * 1e-3) / 1e12
    _, long_rows = md.md_neighbors_row_stats(nl)
    kern = "k_sw_pairs_cta" if pot == "sw" else ("k_tersoff_pairs_cta" if long_rows * 256 > n else "k_tersoff_atom")
    value = aggregate_value(n, args.steps, world, ms_total)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_total / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32" if args.fp32 else "f64", "data": "synthetic",
        "config": {"workload": c["name"], "potential": pot, "atoms_per_gpu": n, "dt_fs": dt,
                   "rebuild_every": rebuild, "r_list": r_list, "max_neighbors": K, "max_row_seen": max_row,
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "steps_per_timed_call": chunk,
                   "l2": f"flushed (256 MiB written then read) before every timed md_nve_run call of {chunk} steps, "
                         "outside the CUDA-event pairs"},
        "clocks": clocks,
        "e2e": {"value": world * n * args.steps / (e2e_ms * 1e-3), "unit": UNIT,
                "h2d_bytes_per_step": 6 * 8 * n / args.steps, "d2h_bytes_per_step": 10 * 8 * n / args.steps,
                "what": f"md_nve_run_host: pinned host x,v -> device, {args.steps} steps, x,v,f,pe -> host"},
        "gpu_launches": int(sum(launches.values())),
        "roofline": {"bound": "alu", "kernel": kern, "achieved": achieved, "peak": fp64_peak, "unit": "TFLOP/s",
                     "frac": achieved / fp64_peak, "traffic": traffic_from_profiles(kern),
                     "peak_source": "md_probe_fp64_peak (measured DFMA rate, this run); nominal "
                                    f"{FP64_NOMINAL_TFLOPS:.1f}",
                     "flop_equiv_per_atom": PAIR_FLOP_PER_ATOM[pot], "kernel_ms": pair_ms,
                     "kernel_share_of_step": kinds_ms["pair"] / max(1e-9, sum(kinds_ms.values()))},
        "kernels_ms_per_step": {k: v / args.steps for k, v in kinds_ms.items()},
        "ms_per_step_profiled": ms_prof / args.steps,
        "back_to_back": {"value": world * n * args.steps / (ms_b2b * 1e-3), "unit": UNIT,
                         "ms_per_step": ms_b2b / args.steps, "l2": "not flushed; one md_nve_run call"},
        "hbm": {"hbm_gbs_peak": peaks.get("hbm_gbs"), "peak_source": "MEASURED_PEAKS.json" if peaks else "absent"},
        "final_pe_per_atom": e_final / n,
        "paper_context": "K40 FP64 Tersoff, 512000 atoms ~ 100 X5670 cores ~ 2.7e7 atom-steps/s (PAPER.md:365-373)",
    }
    if world == 1 and not args.no_cpu_baseline:
        ncell = 40 if c["ncell"] >= 40 else c["ncell"]
        cb_steps = 3
        n_cb, dt_cb = run_oracle(args.config if c["ncell"] <= 40 else 1, cb_steps, 0, ncell)
        line["cpu_baseline"] = {"value": n_cb * cb_steps / dt_cb, "unit": UNIT, "cores": 1, "kind": "oracle",
                                "sample": f"{n_cb} atoms of the same recipe, {cb_steps} NVE steps incl. one "
                                          f"list build, given initial forces, 1 thread, {dt_cb:.1f} s"}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--config", type=int, default=1, help="0-based index into BASELINE.json configs")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--fp32", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    return main_reference(args) if args.impl == "reference" else main_ours(args)


if __name__ == "__main__":
    sys.exit(main())
