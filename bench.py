#!/usr/bin/env python
"""bench.py -- Sutton-Chen MD hot path on B200: pair interactions/s and MD steps/s.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

One "step" = one pass of the whole hot path over the synthetic cluster: a velocity-Verlet MD step
(half kick + drift, [cutoff variant: skin check / cell sort / neighbour rows], density sweep, force +
energy sweep, half kick + kinetic-energy reduction) through libscmd's sc_step.  Default workload:
BASELINE.json configs[3], the Ni65536 fcc cluster, all pairs, FP64 -- the configuration the metric's
roofline target (N >= 65,536) is quoted on.  Other workloads (same JSON line):
    Ni<N>-<fcc|liquid|mackay>-<allpairs|cutoff10>-<fp64|mixed>
Prints ONE JSON line.  N > 1 GPUs = N independent replicas
(the paper's own use: up to 15 independent trajectories per temperature); the
only collective is the timing reduction.  `--gpus N` with N > 1 and no torchrun environment
starts the N ranks itself (re-executes under `python -m torch.distributed.run`); under torchrun
(the driver's launch) it is one of the ranks.  The default run also times, 20 steps each, the
mixed all-pairs and the cutoff-list variants of the same cluster and reports them in `also`.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

from paper_1210_3559_b200 import workloads as W  # noqa: E402

METRIC = "pair_interactions_per_s"
UNIT = "ordered pairs/s (both sweeps)"

# ALU instructions per ordered pair in the shipped (9,6) kernels (SASS-counted):
# thread-level FP64-pipe instructions (FP64 path) / FMA-pipe lane operations (mixed path)
I_DENSITY = {"fp64": 11, "mixed": 16}
I_FORCE_ENERGY = {"fp64": 22, "mixed": 27}
# Newton's-third-law sweeps (all pairs, default from N = 2961 up to 262144: csrc/sc_allpairs_n3.cuh): 13 / 25 FP64 instructions
# per UNORDERED pair = 6.5 / 12.5 per ordered pair
I_DENSITY_N3 = {"fp64": 6.5, "mixed": 10.0}      # mixed: 20 / 30 FMA-pipe lane operations per unordered pair
I_FORCE_ENERGY_N3 = {"fp64": 12.5, "mixed": 15.0}
# nominal B200 ALU peaks: 148 SMs x lanes x 2 FLOP x 1.965 GHz
SM_COUNT, SM_MAX_GHZ = 148, 1.965
LANES = {"fp64": 64, "mixed": 128}
PEAK_TFLOPS = {k: SM_COUNT * v * 2 * SM_MAX_GHZ / 1e3 for k, v in LANES.items()}
DEFAULT_WORKLOAD = "Ni65536-fcc-allpairs-fp64"


class Spec:
    """Parsed workload name."""

    def __init__(self, name: str):
        parts = name.split("-")
        if len(parts) != 4 or not parts[0].startswith("Ni"):
            raise SystemExit(f"unknown workload {name}: want Ni<N>-<fcc|liquid|mackay>-<allpairs|cutoff<r>>-<fp64|mixed>")
        self.name = name
        self.n_atoms = int(parts[0][2:])
        self.kind, self.pairs, self.prec = parts[1], parts[2], parts[3]
        if self.kind not in ("fcc", "liquid", "mackay") or self.prec not in ("fp64", "mixed"):
            raise SystemExit(f"unknown workload {name}")
        self.r_cut = 0.0 if self.pairs == "allpairs" else float(self.pairs.replace("cutoff", ""))
        self.skin = 1.0 if self.r_cut > 0 else 0.0                      # BASELINE.json config 4: skin 1 A

    def generate(self, rank: int = 0) -> W.Workload:
        n = self.n_atoms
        if self.kind == "mackay":
            if n == 147:
                return W.config_c1(seed=1001 + rank)
            shells = {309: 4, 561: 5, 923: 6, 1415: 7, 2057: 8}[n]          # 8 shells: the paper's Ni2057
            return W.mackay_cluster(shells, 1000.0, 1001 + rank)
        if self.kind == "liquid":
            return W.config_c3(seed=3001 + rank, n_atoms=n)
        if n == 1415:
            return W.config_c2(seed=2001 + rank)
        if n == 65536:
            return W.config_c4(seed=4001 + rank)
        k = int(round(np.log2(n) / 2))
        return W.fcc_cluster(n, 1500.0, 5000 + k + rank)                # C5 sweep member


def make_workload(name: str, rank: int = 0) -> W.Workload:
    return Spec(name).generate(rank)


# ------------------------------------------------------------------------------------------- #
# clocks
# ------------------------------------------------------------------------------------------- #
class ClockSampler:
    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.QUERY}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append((time.time(), line.strip()))

    def mark(self):
        """Samples taken before this call are dropped (warm-up)."""
        self.t_mark = time.time()

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        t_mark = getattr(self, "t_mark", 0.0)
        for stamp, line in self.lines:
            if stamp < t_mark:
                continue
            parts = [p.strip() for p in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1])); pw.append(float(parts[2]))
            except ValueError:
                continue
            for nm, val in zip(names, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------- #
# distributed plumbing (replicas only; the timing reduction is the one collective)
# ------------------------------------------------------------------------------------------- #
def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def aggregate(local_ms: float, local_units: float, world: int, backend_device="cuda"):
    """-> (max over ranks of the timed milliseconds, sum over ranks of the units processed)."""
    if world == 1:
        return local_ms, local_units
    import torch
    import torch.distributed as dist
    t = torch.tensor([local_ms], dtype=torch.float64, device=backend_device)
    u = torch.tensor([local_units], dtype=torch.float64, device=backend_device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


# ------------------------------------------------------------------------------------------- #
# reference arm / cpu baseline: the oracle as it stands, on host cores, bounded sample
# ------------------------------------------------------------------------------------------- #
def oracle_sample_rows(n_atoms: int, target_pair_passes: float = 2.5e9) -> np.ndarray:
    """Rows of the workload the CPU baseline evaluates: evenly spaced, sized for ~10-30 s."""
    nrows = int(max(1, min(n_atoms, target_pair_passes / (2.0 * n_atoms))))
    return np.unique(np.linspace(0, n_atoms - 1, nrows).astype(np.int64))


def oracle_time_sample(w: W.Workload, rows: np.ndarray, r_cut: float = 0.0, pair_fraction: float = 1.0):
    """Both sweeps of the binary64 oracle build for `rows` (all j; with a cutoff the oracle still visits
    every j and filters): seconds, ordered pair interactions credited (in-range ones for a cutoff)."""
    from oracle.sc_oracle import Oracle
    o = Oracle("plain")
    P = o.params(r_cut=r_cut)
    rho_all = np.full(w.n_atoms, 100.0)          # timing only: any positive density works as s_j input
    t0 = time.perf_counter()
    rho_rows = o.density_rows(w.pos, P, rows)
    rho_all[rows] = rho_rows
    o.forces_rows(w.pos, P, rho_all, rows)
    dt = time.perf_counter() - t0
    return dt, float(rows.size) * (w.n_atoms - 1) * pair_fraction


def in_range_fraction(w: W.Workload, r_cut: float) -> float:
    """Share of the N(N-1) ordered pairs with r < r_cut (1 for all pairs), from a row sample."""
    if r_cut <= 0:
        return 1.0
    rows = np.unique(np.linspace(0, w.n_atoms - 1, 256).astype(np.int64))
    hits = 0
    for i in rows:
        d2 = ((w.pos - w.pos[i]) ** 2).sum(axis=1)
        hits += int((d2 < r_cut * r_cut).sum()) - 1
    return hits / (rows.size * (w.n_atoms - 1.0))


ORACLE_BUILD = "binary64 oracle build (gcc -O3 -march=native -fopenmp, no fast-math, no FMA contraction)"


def cpu_baseline(w: W.Workload, r_cut: float = 0.0, pair_fraction: float = 1.0, budget_s: float = 10.0) -> dict:
    """The oracle as it stands on the host cores: (i) on all cores (OpenMP over rows) -- whole
    evaluations of the workload or, when one would exceed the budget, an evenly spaced row sample of it,
    repeated for ~budget_s; (ii) on ONE thread (the paper compared its GPU with a single CPU core,
    PAPER.md:129), a smaller row sample of the same workload."""
    from oracle import sc_oracle
    cores = os.cpu_count() or 1
    filt = ", filtered at r_c" if r_cut > 0 else ""
    sc_oracle.set_threads(cores)
    rows = oracle_sample_rows(w.n_atoms, target_pair_passes=2.0e10)
    total_s, total_pairs, reps = 0.0, 0.0, 0
    while reps < 8 and (reps == 0 or total_s < budget_s):
        dt, pairs = oracle_time_sample(w, rows, r_cut, pair_fraction)
        total_s += dt; total_pairs += pairs; reps += 1
    what = "all rows" if rows.size == w.n_atoms else f"{rows.size} evenly spaced rows i"
    # single thread: ~1/cores of the pair visits, so that it takes about as long
    sc_oracle.set_threads(1)
    rows1 = oracle_sample_rows(w.n_atoms, target_pair_passes=2.0e10 / cores)
    s1, p1, reps1 = 0.0, 0.0, 0
    while reps1 < 4 and (reps1 == 0 or s1 < 0.6 * budget_s):
        dt, pairs = oracle_time_sample(w, rows1, r_cut, pair_fraction)
        s1 += dt; p1 += pairs; reps1 += 1
    sc_oracle.set_threads(cores)
    what1 = "all rows" if rows1.size == w.n_atoms else f"{rows1.size} evenly spaced rows i"
    return {"value": total_pairs / total_s, "unit": UNIT, "cores": cores, "kind": "oracle",
            "seconds": total_s,
            "sample": f"{reps} x ({what} of {w.name}, all j, both sweeps{filt}), {ORACLE_BUILD}, OpenMP on all {cores} host cores",
            "single_thread": {"value": p1 / s1, "unit": UNIT, "cores": 1, "seconds": s1,
                              "sample": f"{reps1} x ({what1} of {w.name}, all j, both sweeps{filt}), same build, 1 thread"}}


def config_dict(spec: Spec, n_atoms: int, pairs_per_step: float, world: int, md_per_call: int) -> dict:
    """The `config` object of the JSON line: the same keys from both arms."""
    return {"workload": spec.name, "n_atoms": n_atoms, "pairs_per_step": pairs_per_step,
            "r_cut": spec.r_cut, "skin": spec.skin,
            "parallelism": "replicas only" if world > 1 else "1 GPU",
            "l2": "flushed between timed steps (256 MiB memset outside the per-step events)",
            "md_steps_per_bench_step": md_per_call,
            "step": f"sc_step(dt=1 fs, nsteps={md_per_call}): kick+drift, [skin check / rebuild,] density sweep, "
                    "force+energy sweep, kick+KE"}


def run_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return
    from oracle import sc_oracle
    sc_oracle.set_threads(os.cpu_count() or 1)
    spec = Spec(args.workload)
    w = spec.generate()
    frac = in_range_fraction(w, spec.r_cut)
    rows = oracle_sample_rows(w.n_atoms, target_pair_passes=6e8)
    for _ in range(args.warmup):
        oracle_time_sample(w, rows, spec.r_cut, frac)
    total_s, total_pairs = 0.0, 0.0
    for _ in range(args.steps):
        dt, pairs = oracle_time_sample(w, rows, spec.r_cut, frac)
        total_s += dt; total_pairs += pairs
    value = total_pairs / total_s
    sample = (f"each step = {rows.size} evenly spaced rows i of {w.name} (all j, both sweeps), "
              f"{ORACLE_BUILD}, OpenMP on {os.cpu_count()} host cores")
    n = w.n_atoms
    pairs_per_step = float(n) * (n - 1) * frac       # in-range ordered pairs of one whole evaluation (estimate for a cutoff)
    md_per_call = 1
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total_s / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(spec, n, pairs_per_step, 1, md_per_call),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------- #
# our arm
# ------------------------------------------------------------------------------------------- #
PATH_NAMES = {0: "one-sided", 1: "newton3", 2: "one-launch", 3: "lists"}


def measure(scmd, spec: Spec, steps: int, warmup: int, rank: int, world: int, dev, one_sided: bool,
            with_e2e: bool, sampler: "ClockSampler | None"):
    """Time `steps` bench steps of one workload on this rank.  -> dict of local results (no collectives)."""
    import torch
    w = spec.generate(rank)
    N = w.n_atoms
    prec = scmd.SC_PREC_MIXED if spec.prec == "mixed" else scmd.SC_PREC_FP64
    sc = scmd.SuttonChen(N, r_cut=spec.r_cut, skin=spec.skin, precision=prec)
    d_pos = torch.as_tensor(w.pos, device=dev)
    d_vel = torch.as_tensor(w.vel, device=dev)
    if one_sided:
        sc.sc_set_option(scmd.SC_OPT_NEWTON3, 2)
    sc.sc_set_state(d_pos, d_vel)
    sc.sc_energy()                                                     # first evaluation (builds the rows)
    stats0 = sc.sc_stats()
    pairs_per_step = float(stats0["n_pairs_in_cut"])                   # N(N-1) for all pairs
    # which kernels the library runs for this context is the library's choice: ask it (SC_INFO_STEP_PATH).
    # In the one-launch loop (small all-pairs clusters, csrc/sc_small.cuh) a bench step is one sc_step call of
    # MD_PER_CALL MD steps and the roofline kernel is the loop itself.
    # Where the library runs all steps of a call in one launch (SC_INFO_ONE_LAUNCH: the one-sided loop for small
    # clusters, the Newton's-third-law loop up to 16384 atoms) a bench step is one sc_step call of 100 MD steps and the
    # roofline kernel is the loop itself: the WHOLE step (both sweeps, finalize phases, integrator, grid barriers) is
    # set against the sweeps' instruction counts.
    step_path = sc.sc_get_option(scmd.SC_INFO_STEP_PATH)
    one_launch = sc.sc_get_option(scmd.SC_INFO_ONE_LAUNCH) == 1
    md_per_call = 100 if one_launch else 1
    if not one_launch:
        sc.sc_profile(True)
        sweep_path = sc.sc_get_option(scmd.SC_INFO_STEP_PATH)          # profiling forbids the loops: the path that is timed
    else:
        sweep_path = step_path
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > 126 MB L2
    stream = torch.cuda.current_stream()

    def one_step():
        sc.sc_step(1.0, md_per_call)

    for _ in range(max(warmup, 3)):
        one_step()
    torch.cuda.synchronize()
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    if sampler is not None:
        sampler.mark()                                                 # samples before this are dropped (warm-up)
    launches0 = sc.sc_launch_count()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    ms_force, ms_density = [], []
    torch.cuda.synchronize()
    for k in range(steps):
        flush.zero_()                                                  # L2 flush, outside the timed events
        ev[k][0].record(stream)
        one_step()
        ev[k][1].record(stream)
        if one_launch:
            continue
        prof = sc.sc_profile_read()                                    # synchronises
        ms_force.append(prof["ms_force"]); ms_density.append(prof["ms_density"])
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    launches = sc.sc_launch_count() - launches0
    if one_launch:
        # the loop itself; on the Newton's-third-law path also the call's first half kick + drift and three scalar reductions
        per_call = 1 if step_path == 2 else 5
        assert launches == per_call * steps, f"one-launch loop expected, {launches} launches in {steps} calls"
    stats1 = sc.sc_stats()
    local_ms = sum(a.elapsed_time(b) for a, b in ev)
    out = dict(w=w, N=N, pairs_per_step=pairs_per_step, md_per_call=md_per_call, one_launch=one_launch,
               sweep_path=sweep_path, local_ms=local_ms, launches=launches, stats0=stats0, stats1=stats1,
               ms_force=ms_force, ms_density=ms_density)

    if with_e2e:
        # end to end through the host-buffer entry point: upload positions, both sweeps (cutoff: plus the
        # cell sort and row build, since new positions invalidate the rows), download forces + energy
        # (pinned host memory), every step
        h_pos = torch.as_tensor(w.pos).pin_memory()
        h_force = torch.empty(N, 3, dtype=torch.float64).pin_memory()
        for _ in range(2):
            sc.sc_eval_host(h_pos, h_force)
        torch.cuda.synchronize()
        e2e_steps = max(3, min(steps, 10))
        t_e2e = 0.0
        for _ in range(e2e_steps):
            flush.zero_()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            sc.sc_eval_host(h_pos, h_force)                            # returns after the D2H copy
            t_e2e += time.perf_counter() - t0
        out.update(e2e_ms=t_e2e * 1e3, e2e_steps=e2e_steps)
    sc.close()
    del flush
    return out


def roofline_block(scmd, spec: Spec, m: dict, steps: int) -> dict:
    N, pairs_per_step, path = m["N"], m["pairs_per_step"], m["sweep_path"]
    i_f, i_d, peak = I_FORCE_ENERGY[spec.prec], I_DENSITY[spec.prec], PEAK_TFLOPS[spec.prec]
    newton3 = path == 1
    if newton3:
        i_f, i_d = I_FORCE_ENERGY_N3[spec.prec], I_DENSITY_N3[spec.prec]
    if m["one_launch"]:
        # one kernel holds both sweeps: split its time in proportion to the instruction counts
        t_both = m["local_ms"] * 1e-3 / (steps * m["md_per_call"])
        t_force, t_density = t_both * i_f / (i_f + i_d), t_both * i_d / (i_f + i_d)
    else:
        t_force = statistics.mean(m["ms_force"]) * 1e-3
        t_density = statistics.mean(m["ms_density"]) * 1e-3
    achieved = i_f * 2.0 * pairs_per_step / t_force / 1e12
    probe_kind = 0 if spec.prec == "fp64" else 2
    try:
        rate, _ = scmd.probe_throughput(probe_kind)
        peak_measured = rate * 2.0 / 1e12
    except Exception:
        peak_measured = None
    traffic, traffic_source = None, None
    tfile = ROOT / "profiles" / "roofline_traffic.csv"      # dram bytes per launch of the dominant kernel, from ncu --set full
    if tfile.exists():
        import csv
        with open(tfile, newline="") as fh:
            for row in csv.DictReader(fh):
                if row["workload"] == spec.name:
                    traffic = float(row["force_sweep_dram_bytes_per_launch"])
                    traffic_source = "committed ncu reading, not measured in this run: " + row["source"]
    if m["one_launch"] and newton3:
        kernel = "n3_loop_kernel (whole step loop: Newton's-third-law sweeps, their finalize phases with the integrator, grid barriers; one launch)"
    elif m["one_launch"]:
        kernel = "small_step_kernel (whole step loop: both sweeps + integrator, one launch)"
    elif newton3:
        kernel = ("allpairs_n3_kernel" if spec.prec == "fp64" else "allpairs_n3p_kernel") + \
                 "<force+energy> (every unordered pair once) + n3_finalize_kernel"
    elif spec.r_cut > 0:
        kernel = f"nlist_kernel<force+energy, {spec.prec}>"
    else:
        kernel = ("allpairs64_kernel" if spec.prec == "fp64" else "allpairs32_kernel") + "<force+energy>"
    pipe = "FP64" if spec.prec == "fp64" else "FP32"
    roofline = {"bound": "alu", "kernel": kernel, "achieved": achieved,
                "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak, "traffic": traffic,
                "traffic_source": traffic_source,
                "peak_source": f"nominal: 148 SM x {LANES[spec.prec]} {pipe} lanes x 2 x 1.965 GHz (DESIGN.md section 6); "
                               "MEASURED_PEAKS.json has no CUDA-core figure",
                "peak_measured_fma_probe": peak_measured,
                "frac_vs_probe": achieved / peak_measured if peak_measured else None,
                "alu_inst_per_pair": i_f, "ms_force_sweep": t_force * 1e3, "ms_density_sweep": t_density * 1e3,
                "density_sweep_frac": i_d * 2.0 * pairs_per_step / t_density / 1e12 / peak,
                "both_sweeps_frac": (i_d + i_f) * 2.0 * pairs_per_step / (t_force + t_density) / 1e12 / peak}
    roofline["sweep_timing"] = ("whole MD step of the one-launch loop, split between the sweeps by instruction count" if m["one_launch"]
                                else "library events inside the timed region")
    if newton3:
        # the same time measured against the ONE-SIDED instruction count (22 per ordered pair, the formulation
        # BASELINE.json's north_star names): a speed-up figure (> 1 = faster than a one-sided sweep at FP64 peak),
        # never a fraction of peak
        roofline["speedup_vs_one_sided_at_peak"] = I_FORCE_ENERGY[spec.prec] * 2.0 * pairs_per_step / t_force / 1e12 / peak
        roofline["note"] = (f"frac counts the instructions this kernel must execute: {2 * i_f:g} per unordered pair = "
                            f"{i_f:g} per ordered pair (DESIGN.md 6.8)")
    if spec.r_cut > 0:
        # the list path's memory side: the method's own bytes are records in + forces out;
        # the neighbour rows are the data structure's cost
        hbm_peak, hbm_src = 6469.9, "fallback literal (MEASURED_PEAKS.json absent)"
        try:
            hbm_peak = json.loads((ROOT / "MEASURED_PEAKS.json").read_text())["hbm_gbs"]
            hbm_src = "MEASURED_PEAKS.json hbm_gbs (measured copy)"
        except Exception:
            pass
        alg_bytes = N * (32 + 8 + 24 + 32)                              # both sweeps: records, rho, forces
        t_sweeps = t_force + t_density
        hbm = {"algorithmic_bytes_per_step": alg_bytes, "peak_gbs": hbm_peak, "peak_source": hbm_src,
               "algorithmic_gbs": alg_bytes / t_sweeps / 1e9, "frac": alg_bytes / t_sweeps / 1e9 / hbm_peak,
               "rebuilds_in_timed_region": m["stats1"]["n_rebuilds"] - m["stats0"]["n_rebuilds"],
               "max_neighbours": m["stats1"]["max_neighbours"]}
        if traffic is not None:
            hbm["moved_gbs_force_sweep"] = traffic / t_force / 1e9
            hbm["moved_frac_force_sweep"] = traffic / t_force / 1e9 / hbm_peak
        roofline["hbm"] = hbm
    return roofline


def run_ours(args):
    import torch
    import paper_1210_3559_b200 as scmd

    rank, local_rank, world = dist_env()
    if world > 1:
        import torch.distributed as dist
        torch.cuda.set_device(local_rank)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    dev = torch.device("cuda", local_rank if world > 1 else 0)
    torch.cuda.set_device(dev)
    scmd.load_library()

    spec = Spec(args.workload)
    sampler = ClockSampler(dev.index or 0) if rank == 0 else None
    if sampler is not None:
        sampler.start()
    m = measure(scmd, spec, args.steps, args.warmup, rank, world, dev, args.one_sided, True, sampler)
    clocks = sampler.stop() if sampler is not None else None
    N, pairs_per_step, md_per_call = m["N"], m["pairs_per_step"], m["md_per_call"]
    total_ms, total_pairs = aggregate(m["local_ms"], pairs_per_step * args.steps * md_per_call, world)
    value = total_pairs / (total_ms * 1e-3)
    e2e_ms, e2e_pairs = aggregate(m["e2e_ms"], pairs_per_step * m["e2e_steps"], world)
    launches = m["launches"]

    # the other two variants of the same cluster (mixed all pairs, cutoff lists): 20 steps each, so that the
    # mixed >= 60 % and the neighbour-list figures are timed by whoever runs this file, not claimed
    also = []
    if args.also and world == 1 and args.workload == DEFAULT_WORKLOAD and not args.one_sided:
        for name in ALSO_WORKLOADS:
            s2 = Spec(name)
            m2 = measure(scmd, s2, 20, 3, rank, world, dev, False, False, None)
            ms2 = m2["local_ms"] / 20
            launches += m2["launches"]
            also.append({"workload": name, "steps": 20, "warmup": 3, "ms_per_step": ms2,
                         "value": m2["pairs_per_step"] * m2["md_per_call"] / (ms2 * 1e-3), "unit": UNIT,
                         "md_steps_per_s": m2["md_per_call"] / (ms2 * 1e-3),
                         "dtype": "f64" if s2.prec == "fp64" else "f32 pair math, f64 accumulation",
                         "path": PATH_NAMES[m2["sweep_path"]], "pairs_per_step": m2["pairs_per_step"],
                         "gpu_launches": m2["launches"], "roofline": roofline_block(scmd, s2, m2, 20)})
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank != 0:
        return
    roofline = roofline_block(scmd, spec, m, args.steps)
    frac_pairs = pairs_per_step / (float(N) * (N - 1)) if N > 1 else 1.0
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64" if spec.prec == "fp64" else "f32 pair math, f64 accumulation",
            "data": "synthetic",
            "md_steps_per_s": world * args.steps * md_per_call / (total_ms * 1e-3),
            "config": config_dict(spec, N, pairs_per_step, world, md_per_call),
            "path": PATH_NAMES[m["sweep_path"]],
            "clocks": clocks, "gpu_launches": launches,
            "e2e": {"value": e2e_pairs / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": 24 * N,
                    "d2h_bytes_per_step": 24 * N + 16, "call": "sc_eval_host (pinned host buffers)",
                    "ms_per_call": e2e_ms / m["e2e_steps"]},
            "roofline": roofline, "cpu_baseline": cpu_baseline(m["w"], spec.r_cut, frac_pairs)}
    if also:
        line["also"] = also
    print(json.dumps(line), flush=True)


ALSO_WORKLOADS = ["Ni65536-fcc-allpairs-mixed", "Ni65536-fcc-cutoff10-fp64"]


def run_rows(args):
    """`--parallel rows`: ONE cluster split by rows over the ranks (paper_1210_3559_b200/distributed.py):
    strong scaling.  Per step two all-gathers (positions, densities) on NCCL; every rank runs the one-sided sweeps on
    its rows.  All pairs only."""
    import torch
    import torch.distributed as dist
    import paper_1210_3559_b200 as scmd

    rank, local_rank, world = dist_env()
    spec = Spec(args.workload)
    if spec.r_cut > 0:
        raise SystemExit("--parallel rows is the all-pairs split; the list path runs as replicas")
    torch.cuda.set_device(local_rank if world > 1 else 0)
    dev = torch.device("cuda", torch.cuda.current_device())
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    scmd.load_library()
    w = spec.generate(0)                                               # the same cluster on every rank
    N = w.n_atoms
    prec = scmd.SC_PREC_MIXED if spec.prec == "mixed" else scmd.SC_PREC_FP64
    rs = scmd.RowSplitSuttonChen(N, rank, world, precision=prec)
    h_pos, h_vel = torch.as_tensor(w.pos).pin_memory(), torch.as_tensor(w.vel).pin_memory()
    rs.set_state(h_pos.to(dev), h_vel.to(dev))
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()
    sampler = ClockSampler(dev.index or 0) if rank == 0 else None
    if sampler is not None:
        sampler.start()
    for _ in range(max(args.warmup, 3)):
        rs.step(1.0, 1)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    if sampler is not None:
        sampler.mark()
    launches0 = rs.ctx.sc_launch_count()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for k in range(args.steps):
        flush.zero_()
        ev[k][0].record(stream)
        rs.step(1.0, 1)
        ev[k][1].record(stream)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    launches = rs.ctx.sc_launch_count() - launches0
    clocks = sampler.stop() if sampler is not None else None
    local_ms = sum(a.elapsed_time(b) for a, b in ev)
    rows = rs.end - rs.begin
    total_ms, total_pairs = aggregate(local_ms, float(rows) * (N - 1) * args.steps, world)
    # end to end: positions from pinned host memory, one force evaluation (both sweeps + the density all-gather),
    # this rank's forces back to the host
    h_force = torch.empty(rows, 3, dtype=torch.float64).pin_memory()
    e2e_steps, t_e2e = max(3, min(args.steps, 10)), 0.0
    for k in range(e2e_steps + 1):
        flush.zero_()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        rs.set_state(h_pos.to(dev, non_blocking=True), h_vel.to(dev, non_blocking=True))
        h_force.copy_(rs.own_forces(), non_blocking=True)
        torch.cuda.synchronize()
        if k > 0:
            t_e2e += time.perf_counter() - t0
    e2e_ms, e2e_pairs = aggregate(t_e2e * 1e3, float(rows) * (N - 1) * e2e_steps, world)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank != 0:
        return
    i_both = I_FORCE_ENERGY[spec.prec] + I_DENSITY[spec.prec]
    peak = PEAK_TFLOPS[spec.prec] * world
    achieved = i_both * 2.0 * float(N) * (N - 1) / (total_ms * 1e-3 / args.steps) / 1e12
    cfg = config_dict(spec, N, float(N) * (N - 1), world, 1)
    cfg["parallelism"] = f"rows{world}: one cluster, contiguous row ranges, 2 all-gathers per step (positions, densities)"
    line = {"metric": METRIC, "value": total_pairs / (total_ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None,
            "dtype": "f64" if spec.prec == "fp64" else "f32 pair math, f64 accumulation", "data": "synthetic",
            "md_steps_per_s": args.steps / (total_ms * 1e-3), "config": cfg, "path": "one-sided rows",
            "clocks": clocks, "gpu_launches": launches,
            "e2e": {"value": e2e_pairs / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": 48 * N,
                    "d2h_bytes_per_step": 24 * rows, "call": "RowSplitSuttonChen.set_state + own_forces (pinned host buffers)",
                    "ms_per_call": e2e_ms / e2e_steps},
            "roofline": {"bound": "alu", "kernel": "allpairs kernels, both sweeps, whole step incl. the two all-gathers",
                         "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak, "traffic": None,
                         "alu_inst_per_pair": i_both,
                         "peak_source": f"nominal per GPU x {world} (DESIGN.md section 6)"},
            "exchanges_per_step": 2, "exchange_bytes_per_step": 32 * N,
            "cpu_baseline": cpu_baseline(w, 0.0, 1.0)}
    print(json.dumps(line), flush=True)


def launcher_command(args, argv: list[str], port: int) -> list[str]:
    """`--gpus N` without a torchrun environment: the command that starts the N ranks (one per GPU, NCCL)."""
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
            "--master-addr", "127.0.0.1", "--master-port", str(port), str(Path(__file__).resolve()), *argv]


def main(argv=None):
    argv = list(sys.argv[1:] if argv is None else argv)
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD)
    ap.add_argument("--one-sided", action="store_true",
                    help="all pairs: force the one-sided sweeps (SC_OPT_NEWTON3 = 2) where Newton's third law is the default")
    ap.add_argument("--parallel", default="replicas", choices=["replicas", "rows"],
                    help="N > 1 GPUs: independent replicas (weak scaling, the paper's use) or ONE cluster split by rows "
                         "(strong scaling, two all-gathers per step)")
    ap.add_argument("--no-also", dest="also", action="store_false",
                    help="default workload only: skip the mixed and cutoff-list variants reported in `also`")
    args = ap.parse_args(argv)
    if args.gpus < 1:
        raise SystemExit("--gpus must be >= 1")
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl == "ours":
        # not under torchrun: start the ranks ourselves and hand over (rank 0 prints the line)
        import socket
        with socket.socket() as s:
            s.bind(("127.0.0.1", 0))
            port = s.getsockname()[1]
        env = dict(os.environ)
        env.setdefault("NCCL_DEBUG", "WARN")
        raise SystemExit(subprocess.run(launcher_command(args, argv, port), env=env).returncode)
    _, _, world = dist_env()
    if args.impl == "ours" and world != args.gpus:
        raise SystemExit(f"--gpus {args.gpus} but WORLD_SIZE = {world}: launch with --nproc-per-node {args.gpus}")
    if args.impl == "reference":
        run_reference(args)
    elif args.parallel == "rows":
        run_rows(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
