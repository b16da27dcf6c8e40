#!/usr/bin/env python
"""bench.py -- atom-steps/s of the FP64 Tersoff/SW force + NVE hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config I] [--impl ours|reference] [--only-headline]

A "step" is one velocity-Verlet NVE step of the whole hot path (kick+drift, neighbour rebuild every
10th step, pair kernel, gather, kick) on BASELINE.json config I (default 1 = configs[1]: Tersoff,
512 000 atoms).  Prints ONE JSON line: the headline config in the contract's
keys, and under `configs` a bounded run of every other BASELINE config (3, 4, 5, 5 in FP32 as NVE runs;
config 1 and the 512 000-atom crystal as full-output evaluations in atom-evals/s), each with its exact
pair / triplet counts, the pair phase's fraction of the measured FP64 peak and the whole step's fraction of
the measured HBM bandwidth.  `--config 0` alone prints config 1's evaluation line.  N > 1 runs independent
replicas (the path is single-GPU by north_star: "replicas only"), one process per GPU under torchrun.
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
FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12      # 148 SMs x 64 DFMA/clk x 1.965 GHz = 37.2


def pair_flop_equiv(pot, listed, in_range, triplets):
    """Algorithmic work of one pair phase in flop-equivalents (SURVEY.md section 8(d):
    add = mul = 1, fma = 2, div = 16, sqrt = 20, exp = 35, log = 50), from EXACT integer counts of listed
    directed pairs, in-range directed pairs and ordered in-range triplets (md_pair_counts).
    Tersoff: 342 per in-range pair + (28 zeta pass + 25 force pass) per ordered triplet (M = 4: 2004 per atom).
    SW: 20 per listed pair (screen) + 178 per in-range pair + 30 per ordered triplet -- the definition's
    count; the kernel evaluates the triplet sum through moments and executes fewer."""
    if pot == "tersoff":
        return 342.0 * in_range + 53.0 * triplets
    return 20.0 * listed + 178.0 * in_range + 30.0 * triplets


def step_bytes(listed, in_range, n, rebuild_every, fp32):
    """Algorithmic HBM bytes of one md_nve_run step, from the same counts.
    pair phase : x,y,z 24 + NN 4 + MASK 8 + own-half f 24 per atom; list entry 4 per listed pair; reverse
                 slot 1 + record 32 (16 in FP32 mode) per in-range pair   (neighbour coordinates: L2-served)
    gather+VV  : MASK 8 + own-half f 24 + v 24 + x 24 read, v 24 + x 24 written per atom; record per in-range pair
    build      : x,y,z read twice 48 + cell-ordered copies written and read 96 + NN 4 per atom; list entry
                 written and read 8 + reverse slot 1 per listed pair -- every `rebuild_every` steps"""
    rec = 16.0 if fp32 else 32.0
    pair = 60.0 * n + 4.0 * listed + (1.0 + rec) * in_range
    gather = 128.0 * n + rec * in_range
    build = (148.0 * n + 9.0 * listed) / rebuild_every
    return pair + gather + build


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


def run_oracle(cfg_index, steps, warmup, ncell, threads=1):
    """Oracle NVE on `ncell`^3 cells of config `cfg_index`: `warmup` untimed steps (they also provide the
    forces), then `steps` timed ones.  threads > 1: the force evaluation on that many threads."""
    import oracle                                            # the one CPU leg allowed to use oracle/
    c = mi.make_config(cfg_index, ncell=ncell)
    K = c["max_neighbors"] if c["potential"] == "tersoff" else 40
    st = {k: c[k] for k in ("x", "y", "z", "vx", "vy", "vz", "box", "mass")}
    r = oracle.nve_run(c["potential"], c["params"], st, warmup, c["dt"], c["rebuild_every"], c["r_list"], K)
    t0 = time.perf_counter()
    if threads > 1:
        oracle.nve_run_threads(c["potential"], c["params"], st, steps, c["dt"], c["rebuild_every"], c["r_list"], K,
                               threads, r["f"])
    else:
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
    """dram bytes per launch of `kernel` from the committed ncu summary (data file, not code); measured at
    512 000 atoms, so None for any other size."""
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


class Gpu:
    """Device, rank and barrier shared by the measurements of one bench.py process."""

    def __init__(self):
        import torch
        import torch.distributed as dist
        self.torch, self.dist = torch, dist
        self.rank = int(os.environ.get("RANK", "0"))
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.local = int(os.environ.get("LOCAL_RANK", "0"))
        if not torch.cuda.is_available():
            raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
        torch.cuda.set_device(self.local)
        self.dev = f"cuda:{self.local}"
        if self.world > 1:
            dist.init_process_group("nccl", device_id=torch.device(self.dev))
        self.flush = torch.empty(256 << 20, dtype=torch.uint8, device=self.dev)   # > 126 MB L2

    def barrier(self):
        if self.world > 1:
            self.dist.barrier()
        self.torch.cuda.synchronize()

    def flush_l2(self):
        """256 MiB written, then read back so that no dirty foreign lines are left to evict."""
        self.flush.zero_()
        self.flush.sum()

    def close(self):
        if self.world > 1:
            self.dist.destroy_process_group()


def kernel_name(md, nl, pot, n):
    if pot == "sw":
        return "k_screen+k_sw_sorted"
    _, long_rows = md.md_neighbors_row_stats(nl)
    # md_nve_run asks for no virial: the register path is the 128-register lean kernel (tersoff.cu, launch())
    return "k_screen+k_tersoff_sorted|k_tersoff_binned" if long_rows * 256 > n else "k_tersoff_lean"


def measure_nve(gpu, md, cfg_index, steps, warmup, fp32, peaks, fp64_peak, with_e2e, sampler=None):
    """K NVE steps of BASELINE config `cfg_index` as ceil(K/chunk) md_nve_run calls of one rebuild cycle each,
    every call bracketed by its own CUDA-event pair, L2 flushed before every call outside the pairs; a second
    pass with the library's per-kernel-kind events; one back-to-back call; optionally the host-buffer call."""
    torch = gpu.torch
    c = mi.make_config(cfg_index)
    pot, n, K = c["potential"], c["n"], c["max_neighbors"]
    box, mass, dt, rebuild, r_list = list(c["box"]), c["mass"], c["dt"], c["rebuild_every"], c["r_list"]
    host0 = {k: torch.from_numpy(c[k].copy()) for k in ("x", "y", "z", "vx", "vy", "vz")}
    d = {k: v.to(gpu.dev) for k, v in host0.items()}
    f = torch.zeros((3, n), dtype=torch.float64, device=gpu.dev)
    pe = torch.zeros(n, dtype=torch.float64, device=gpu.dev)
    nl = md.md_neighbors_create(n, K)
    prec = md.MD_FP32 if fp32 else md.MD_FP64

    def run(first, nsteps, f_valid=True):
        md.md_nve_run(nl, pot, c["params"], n, d["x"], d["y"], d["z"], d["vx"], d["vy"], d["vz"], f, f_valid, pe,
                      box, mass, dt, nsteps, rebuild, r_list, precision=prec, first_step=first)

    run(0, 0, f_valid=False)                       # forces of the initial state
    run(0, warmup)
    step0 = warmup
    max_row = md.md_neighbors_status(nl)
    chunk = rebuild                                # one timed call = one rebuild cycle of md_nve_run

    def timed_pass(profile):
        nonlocal step0
        md.md_profile_enable(nl, profile)
        md.md_profile_read(nl)
        sizes = [min(chunk, steps - k) for k in range(0, steps, chunk)]
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in sizes]
        gpu.barrier()
        t0 = time.perf_counter()
        done = 0
        for k, sz in enumerate(sizes):
            gpu.flush_l2()                         # L2 flush between timed iterations (not timed)
            ev[k][0].record()
            run(step0 + done, sz)
            ev[k][1].record()
            done += sz
        torch.cuda.synchronize()
        t1 = time.perf_counter()
        gpu.barrier()
        step0 += steps
        ms = sum(a.elapsed_time(b) for a, b in ev)
        kinds_ms, launches = md.md_profile_read(nl)
        md.md_profile_enable(nl, False)
        return ms, kinds_ms, launches, t0, t1

    if sampler is not None:
        sampler.start()
        time.sleep(0.1)
    ms_total, _, launches, t0, t1 = timed_pass(False)
    clocks = sampler.stop(t0, t1) if sampler is not None else None
    ms_prof, kinds_ms, _, _, _ = timed_pass(True)  # same loop with per-kernel-kind events
    gpu.barrier()                                  # back-to-back steps, one C call, no flush
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(); run(step0, steps); e1.record()
    torch.cuda.synchronize()
    ms_b2b = e0.elapsed_time(e1)
    step0 += steps
    md.md_neighbors_status(nl)
    listed, in_range, triplets = md.md_pair_counts(nl)
    kern = kernel_name(md, nl, pot, n)
    e_final = float(pe.sum())

    e2e_ms = None
    if with_e2e:                                   # C ABI with HOST (pinned) buffers: H2D + K steps + D2H timed
        hp = {k: v.clone().pin_memory() for k, v in host0.items()}
        hf = torch.zeros((3, n), dtype=torch.float64).pin_memory()
        hpe = torch.zeros(n, dtype=torch.float64).pin_memory()
        nl2 = md.md_neighbors_create(n, K)

        def e2e_call(nsteps):
            for k, v in host0.items():
                hp[k].copy_(v)
            gpu.barrier()
            t = time.perf_counter()
            md.md_nve_run_host(nl2, pot, c["params"], n, hp["x"], hp["y"], hp["z"], hp["vx"], hp["vy"], hp["vz"],
                               hf, hpe, box, mass, dt, nsteps, rebuild, r_list, precision=prec)
            return time.perf_counter() - t
        e2e_call(max(3, warmup))
        e2e_ms = e2e_call(steps) * 1e3
        md.md_neighbors_destroy(nl2)
    md.md_neighbors_destroy(nl)

    vals = gpu_max([ms_total, ms_prof, ms_b2b, e2e_ms if e2e_ms is not None else 0.0], gpu)
    ms_total, ms_prof, ms_b2b = vals[:3]
    e2e_ms = vals[3] if e2e_ms is not None else None
    world = gpu.world
    pair_ms = kinds_ms["pair"] / steps             # one pair phase per step
    flops = pair_flop_equiv(pot, listed, in_range, triplets)
    achieved = flops / (pair_ms * 1e-3) / 1e12
    nbytes = step_bytes(listed, in_range, n, rebuild, fp32)
    hbm_peak = peaks.get("hbm_gbs")
    hbm_gbs = nbytes / (ms_total / steps * 1e-3) / 1e9
    return {
        "c": c, "value": aggregate_value(n, steps, world, ms_total), "ms_per_step": ms_total / steps,
        "ms_per_step_profiled": ms_prof / steps, "ms_b2b": ms_b2b, "e2e_ms": e2e_ms, "clocks": clocks,
        "launches": launches, "kinds_ms": kinds_ms, "max_row": max_row, "kernel": kern, "pair_ms": pair_ms,
        "counts": {"listed_pairs": listed, "in_range_pairs": in_range, "ordered_triplets": triplets,
                   "listed_per_atom": listed / n, "in_range_per_atom": in_range / n,
                   "ordered_triplets_per_atom": triplets / n},
        "alu": {"achieved": achieved, "peak": fp64_peak, "unit": "TFLOP/s", "frac": achieved / fp64_peak,
                "flop_equiv_per_atom": flops / n, "kernel": kern, "kernel_ms": pair_ms},
        "hbm": {"achieved": hbm_gbs, "peak": hbm_peak, "unit": "GB/s",
                "frac": hbm_gbs / hbm_peak if hbm_peak else None, "bytes_per_atom_step": nbytes / n,
                "what": "algorithmic bytes of a whole md_nve_run step / ms_per_step",
                "peak_source": "MEASURED_PEAKS.json" if hbm_peak else "absent"},
        "final_pe_per_atom": e_final / n,
    }


def gpu_max(values, gpu):
    return max_over_ranks(values, gpu.dev, gpu.world)


def measure_eval(gpu, md, cfg_index, calls, warmup, fp64_peak, peaks):
    """Config 1's mode: ONE evaluation of energy, forces, virial and heat current per "step" (atom-evals/s).
    Each call is bracketed by its own event pair; L2 is flushed before every call."""
    torch = gpu.torch
    c = mi.make_config(cfg_index)
    pot, n, K = c["potential"], c["n"], c["max_neighbors"]
    box = list(c["box"])
    d = {k: torch.from_numpy(c[k]).to(gpu.dev) for k in ("x", "y", "z", "vx", "vy", "vz")}
    pe = torch.zeros(n, dtype=torch.float64, device=gpu.dev)
    f = torch.zeros((3, n), dtype=torch.float64, device=gpu.dev)
    W = torch.zeros((9, n), dtype=torch.float64, device=gpu.dev)
    J = torch.zeros((3, n), dtype=torch.float64, device=gpu.dev)
    nl = md.md_neighbors_create(n, K)
    md.md_build_neighbors(nl, n, d["x"], d["y"], d["z"], box, c["r_list"])
    fn = md.md_tersoff_force if pot == "tersoff" else md.md_sw_force

    def call():
        fn(nl, n, d["x"], d["y"], d["z"], d["vx"], d["vy"], d["vz"], box, c["params"], md.MD_FP64,
           pe=pe, f=f, virial=W, heat=J)
    for _ in range(max(3, warmup)):
        call()
    md.md_neighbors_status(nl)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(calls)]
    gpu.barrier()
    for a, b in ev:
        gpu.flush_l2()
        a.record(); call(); b.record()
    torch.cuda.synchronize()
    ms = sum(a.elapsed_time(b) for a, b in ev)
    ms, = gpu_max([ms], gpu)
    listed, in_range, triplets = md.md_pair_counts(nl)
    md.md_neighbors_destroy(nl)
    rec = 32.0
    # pair kernel + k_gather with all outputs: adds list entry 4 + neighbour coordinates (L2) per in-range pair,
    # W 72 read + 72 written, J 24, v 24, x 24, U 8 per atom
    nbytes = (60.0 + 8.0) * n + 4.0 * listed + (1.0 + rec) * in_range + (8 + 24 + 24 + 24 + 144 + 24 + 24) * n \
        + (rec + 4.0) * in_range
    hbm_peak = peaks.get("hbm_gbs")
    return {"workload": c["name"], "atoms": n, "outputs": "pe, f, virial(9), heat", "calls": calls,
            "value": gpu.world * n * calls / (ms * 1e-3), "unit": "atom-evals/s", "us_per_eval": 1e3 * ms / calls,
            "hbm_frac": (nbytes / (ms / calls * 1e-3) / 1e9 / hbm_peak) if hbm_peak else None,
            "bytes_per_atom_eval": nbytes / n, "in_range_per_atom": in_range / n}


def measure_multi_eval(gpu, md, calls, warmup, peaks):
    """Multi-element Tersoff: full-output evaluations of a 512 000-atom 3C-SiC crystal
    (zinc-blende, a = 4.32 A, sigma 0.05 A, 300 K), list cut-off 3.0 + 0.5 A, in atom-evals/s."""
    torch = gpu.torch
    s = mi.zincblende_crystal(40, mi.SIC_LATTICE_A, 0.05, 300.0, mi.BASE_SEED + 7)
    n, K, box = s["n"], 32, list(s["box"])
    d = {k: torch.from_numpy(s[k]).to(gpu.dev) for k in ("x", "y", "z", "vx", "vy", "vz")}
    types = torch.from_numpy(s["types"]).to(gpu.dev)
    pe = torch.zeros(n, dtype=torch.float64, device=gpu.dev)
    f = torch.zeros((3, n), dtype=torch.float64, device=gpu.dev)
    W = torch.zeros((9, n), dtype=torch.float64, device=gpu.dev)
    J = torch.zeros((3, n), dtype=torch.float64, device=gpu.dev)
    nl = md.md_neighbors_create(n, K)
    md.md_build_neighbors(nl, n, d["x"], d["y"], d["z"], box, 3.5)

    def call():
        md.md_tersoff_multi_force(nl, n, d["x"], d["y"], d["z"], d["vx"], d["vy"], d["vz"], box, types,
                                  mi.TERSOFF_SIC_ELEMENTS, mi.TERSOFF_SIC_CHI, md.MD_FP64, pe=pe, f=f, virial=W, heat=J)
    for _ in range(max(3, warmup)):
        call()
    md.md_neighbors_status(nl)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(calls)]
    gpu.barrier()
    for a, b in ev:
        gpu.flush_l2()
        a.record(); call(); b.record()
    torch.cuda.synchronize()
    ms, = gpu_max([sum(a.elapsed_time(b) for a, b in ev)], gpu)
    listed, in_range, triplets = md.md_pair_counts(nl)
    md.md_neighbors_destroy(nl)
    return {"workload": "3C-SiC 512000 atoms, multi-element Tersoff (Tersoff 1989 parameters)", "atoms": n,
            "outputs": "pe, f, virial(9), heat", "calls": calls, "value": gpu.world * n * calls / (ms * 1e-3),
            "unit": "atom-evals/s", "us_per_eval": 1e3 * ms / calls, "listed_per_atom": listed / n,
            "in_range_per_atom": in_range / n, "ordered_triplets_per_atom": triplets / n}


def measure_literal_ab(gpu, md, cfg_index, calls, warmup):
    """the paper's literal Algorithm 3 + 2 (md_tersoff_force_literal) beside the stored-P design
    (md_tersoff_force), forces only, same list, per-call event pairs, L2 flushed before every call."""
    torch = gpu.torch
    c = mi.make_config(cfg_index)
    n, K, box = c["n"], c["max_neighbors"], list(c["box"])
    d = {k: torch.from_numpy(c[k]).to(gpu.dev) for k in ("x", "y", "z", "vx", "vy", "vz")}
    f = torch.zeros((3, n), dtype=torch.float64, device=gpu.dev)
    nl = md.md_neighbors_create(n, K)
    md.md_build_neighbors(nl, n, d["x"], d["y"], d["z"], box, c["r_list"])
    out = {"workload": c["name"], "atoms": n, "outputs": "f"}
    for name, fn in (("stored_P", md.md_tersoff_force), ("literal_alg3_alg2", md.md_tersoff_force_literal)):
        def call():
            fn(nl, n, d["x"], d["y"], d["z"], d["vx"], d["vy"], d["vz"], box, c["params"], md.MD_FP64, f=f)
        for _ in range(max(3, warmup)):
            call()
        md.md_neighbors_status(nl)
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(calls)]
        gpu.barrier()
        for a, b in ev:
            gpu.flush_l2()
            a.record(); call(); b.record()
        torch.cuda.synchronize()
        ms, = gpu_max([sum(a.elapsed_time(b) for a, b in ev)], gpu)
        out[name] = {"us_per_eval": 1e3 * ms / calls, "atom_evals_per_s": gpu.world * n * calls / (ms * 1e-3)}
    md.md_neighbors_destroy(nl)
    out["literal_over_stored"] = out["literal_alg3_alg2"]["us_per_eval"] / out["stored_P"]["us_per_eval"]
    return out


def measure_ensembles(gpu, md, cfg_index, steps, warmup):
    """md_npt_run (Berendsen NPT, the paper's benchmark ensemble: velocity-Verlet + per-atom
    virial + two scalars read back per step) and md_nve_heat_run (Green-Kubo sampling every 10th step) on the
    headline workload, in atom-steps/s, one call of `steps` steps each, CUDA events around the call."""
    torch = gpu.torch
    c = mi.make_config(cfg_index)
    pot, n, K = c["potential"], c["n"], c["max_neighbors"]
    out = {"workload": c["name"], "atoms": n, "steps": steps}
    ber = dict(T0=300.0, tau_T=100.0, P0=0.0, tau_P=1000.0, beta=1.0 / 0.6104)
    for name in ("npt_berendsen", "nve_green_kubo_every_10"):
        d = {k: torch.from_numpy(c[k].copy()).to(gpu.dev) for k in ("x", "y", "z", "vx", "vy", "vz")}
        f = torch.zeros((3, n), dtype=torch.float64, device=gpu.dev)
        nl = md.md_neighbors_create(n, K)
        box = list(c["box"])

        def run(first, nsteps, f_valid):
            if name == "npt_berendsen":
                md.md_npt_run(nl, pot, c["params"], n, d["x"], d["y"], d["z"], d["vx"], d["vy"], d["vz"], f, f_valid, box,
                              c["mass"], c["dt"], nsteps, c["rebuild_every"], c["r_list"], ber, first_step=first)
            else:
                md.md_nve_heat_run(nl, pot, c["params"], n, d["x"], d["y"], d["z"], d["vx"], d["vy"], d["vz"], f, f_valid,
                                   box, c["mass"], c["dt"], nsteps, c["rebuild_every"], c["r_list"], 10, first_step=first)
        run(0, warmup, False)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        gpu.barrier()
        gpu.flush_l2()
        e0.record(); run(warmup, steps, True); e1.record()
        torch.cuda.synchronize()
        ms, = gpu_max([e0.elapsed_time(e1)], gpu)
        md.md_neighbors_status(nl)
        md.md_neighbors_destroy(nl)
        out[name] = {"value": gpu.world * n * steps / (ms * 1e-3), "unit": UNIT, "ms_per_step": ms / steps}
    return out


def summary(r):
    """The per-config entry of the line's `configs` object."""
    c = r["c"]
    return {"workload": c["name"], "potential": c["potential"], "atoms": c["n"], "dt_fs": c["dt"],
            "value": r["value"], "unit": UNIT, "ms_per_step": r["ms_per_step"],
            "kernels_ms_per_step": {k: v / max(1, r["steps"]) for k, v in r["kinds_ms"].items()},
            "pair_kernel": r["kernel"], "pair_ms": r["pair_ms"], "alu_frac": r["alu"]["frac"],
            "alu_tflops": r["alu"]["achieved"], "flop_equiv_per_atom": r["alu"]["flop_equiv_per_atom"],
            "hbm_frac": r["hbm"]["frac"], "hbm_gbs": r["hbm"]["achieved"],
            "bytes_per_atom_step": r["hbm"]["bytes_per_atom_step"], "counts_per_atom": {
                k: r["counts"][k] for k in ("listed_per_atom", "in_range_per_atom", "ordered_triplets_per_atom")},
            "steps": r["steps"], "max_row_seen": r["max_row"]}


def main_ours(args):
    import paper_1610_03343_b200 as md

    gpu = Gpu()
    peaks = measured_peaks()
    fp64_peak = md.md_probe_fp64_peak(20000)
    if mi.CONFIGS[args.config]["steps"] == 0:                # config 1: evaluation mode
        r = measure_eval(gpu, md, args.config, args.steps, args.warmup, fp64_peak, peaks)
        if gpu.rank == 0:
            print(json.dumps({"metric": "atom-evals/s (FP64 Tersoff: energy, forces, virial, heat current)",
                              "n_gpus": gpu.world, "steps": args.steps, "warmup": args.warmup,
                              "higher_is_better": True, "dtype": "f64", "data": "synthetic", **r}))
        gpu.close()
        return 0

    sampler = ClockSampler(gpu.local)
    r = measure_nve(gpu, md, args.config, args.steps, args.warmup, args.fp32, peaks, fp64_peak, True, sampler)
    r["steps"] = args.steps
    c, n, world = r["c"], r["c"]["n"], gpu.world
    extra = {}
    if not args.only_headline:
        # the other BASELINE configs, bounded (their own length or --steps, whichever is shorter)
        for idx, fp32 in ((2, False), (4, False), (4, True), (3, False)):
            if idx == args.config and fp32 == args.fp32:
                continue
            k = min(args.steps, mi.CONFIGS[idx]["steps"])
            q = measure_nve(gpu, md, idx, k, args.warmup, fp32, peaks, fp64_peak, False)
            q["steps"] = k
            extra[mi.CONFIGS[idx]["name"] + ("_fp32" if fp32 else "")] = summary(q)
        extra["cfg1_tersoff_512_eval"] = measure_eval(gpu, md, 0, 200, args.warmup, fp64_peak, peaks)
        extra["cfg2_size_full_output_eval"] = measure_eval(gpu, md, 1, 20, args.warmup, fp64_peak, peaks)
        extra["multi_element_sic_512k_eval"] = measure_multi_eval(gpu, md, 20, args.warmup, peaks)
        extra["ensembles_cfg2"] = measure_ensembles(gpu, md, 1, 100, 20)
        extra["literal_vs_stored_P_cfg2"] = measure_literal_ab(gpu, md, 1, 20, args.warmup)
        extra["literal_vs_stored_P_cfg4"] = measure_literal_ab(gpu, md, 3, 5, args.warmup)
    if gpu.rank != 0:
        gpu.close()
        return 0

    kinds_ms, steps = r["kinds_ms"], args.steps
    line = {
        "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": world, "steps": steps,
        "warmup": args.warmup, "ms_per_step": r["ms_per_step"], "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32" if args.fp32 else "f64", "data": "synthetic",
        "config": {"workload": c["name"], "potential": c["potential"], "atoms_per_gpu": n, "dt_fs": c["dt"],
                   "rebuild_every": c["rebuild_every"], "r_list": c["r_list"], "max_neighbors": c["max_neighbors"],
                   "max_row_seen": r["max_row"],
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "steps_per_timed_call": c["rebuild_every"],
                   "l2": f"flushed (256 MiB written then read) before every timed md_nve_run call of "
                         f"{c['rebuild_every']} steps, outside the CUDA-event pairs"},
        "clocks": r["clocks"],
        "e2e": {"value": world * n * steps / (r["e2e_ms"] * 1e-3), "unit": UNIT,
                "h2d_bytes_per_step": 6 * 8 * n / steps, "d2h_bytes_per_step": 10 * 8 * n / steps,
                "what": f"md_nve_run_host: pinned host x,v -> device, {steps} steps, x,v,f,pe -> host"},
        "gpu_launches": int(sum(r["launches"].values())),
        "roofline": {"bound": "alu", "kernel": r["kernel"], "achieved": r["alu"]["achieved"], "peak": fp64_peak,
                     "unit": "TFLOP/s", "frac": r["alu"]["frac"], "traffic": traffic_from_profiles(r["kernel"]) if n == 512000 else None,
                     "peak_source": "md_probe_fp64_peak (measured DFMA rate, this run); nominal "
                                    f"{FP64_NOMINAL_TFLOPS:.1f}",
                     "flop_equiv_per_atom": r["alu"]["flop_equiv_per_atom"], "kernel_ms": r["pair_ms"],
                     "counts_per_atom": {k: r["counts"][k] for k in ("listed_per_atom", "in_range_per_atom",
                                                                     "ordered_triplets_per_atom")},
                     "kernel_share_of_step": kinds_ms["pair"] / max(1e-9, sum(kinds_ms.values()))},
        "hbm": r["hbm"],
        "kernels_ms_per_step": {k: v / steps for k, v in kinds_ms.items()},
        "ms_per_step_profiled": r["ms_per_step_profiled"],
        "back_to_back": {"value": world * n * steps / (r["ms_b2b"] * 1e-3), "unit": UNIT,
                         "ms_per_step": r["ms_b2b"] / steps, "l2": "not flushed; one md_nve_run call"},
        "final_pe_per_atom": r["final_pe_per_atom"],
        "paper_context": "K40 FP64 Tersoff, 512000 atoms ~ 100 X5670 cores ~ 2.7e7 atom-steps/s (PAPER.md:365-373)",
    }
    if extra:
        line["configs"] = extra
    if world == 1 and not args.no_cpu_baseline:
        # the oracle as it stands on this box's host cores: one full rebuild cycle (the GPU's cadence)
        src = args.config if c["ncell"] <= 40 else 1
        ncell = min(40, c["ncell"])
        cb_steps = c["rebuild_every"]
        n_cb, dt_cb = run_oracle(src, cb_steps, 0, ncell)
        line["cpu_baseline"] = {"value": n_cb * cb_steps / dt_cb, "unit": UNIT, "cores": 1, "kind": "oracle",
                                "sample": f"{n_cb} atoms of the same recipe, {cb_steps} NVE steps = one rebuild "
                                          f"cycle incl. its list build, given initial forces, 1 thread, {dt_cb:.1f} s"}
        cores = len(os.sched_getaffinity(0))
        if cores > 1:
            n_ca, dt_ca = run_oracle(src, cb_steps, 0, ncell, threads=cores)
            line["cpu_baseline_all_cores"] = {
                "value": n_ca * cb_steps / dt_ca, "unit": UNIT, "cores": cores, "kind": "oracle",
                "sample": f"same sample; force evaluation on {cores} threads over atom ranges with per-thread "
                          f"force buffers, list build and integrator on one; {dt_ca:.1f} s"}
    print(json.dumps(line))
    gpu.close()
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
    ap.add_argument("--only-headline", action="store_true", help="skip the `configs` summary of the other configs")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    return main_reference(args) if args.impl == "reference" else main_ours(args)


if __name__ == "__main__":
    sys.exit(main())
