#!/usr/bin/env python
"""bench.py -- throughput of the bemcub hot path on B200 (driver contract: one JSON line on rank 0).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload cfg4|cfg1|cfg2|cfg3|cfg5|solve|table3|accuracy|few] [--scale S] [--no-secondary]

Metric (BASELINE.json): FP64 Phi+E element.point interactions/s.  One step = one pass of the whole
hot path (a1 preprocessing, a2 rule binning, a3 point-charge sum, a4 analytic near field, a6
reduction + scaling) over one batch of synthetic input.  Default workload =
config 4 (`configs[3]`, "the 10^6-element config" the north_star target is quoted on): 8e5
rectangles + 2e5 triangles, 10^6 helical-track field points, distance-ratio-adaptive rules.  The
default line also carries a `secondary` list: short device-timed runs of the other configs (matrix
fill of config 3, configs 1, 2, 5), each with its own roofline, clocks and oracle timing.
The other `--workload` values time one workload alone (profiling); `--workload accuracy` runs the
paper's random-element accuracy study (Figs. 8-10) through bemcub_eval_pairs and writes its
table to `--out`.

Multi-GPU (torchrun): field points shard across ranks with no data-path collective; every rank
holds the full mesh and its own 10^6 field points (weak scaling).

`--impl reference` times the CPU oracle (oracle/, as it stands) on the host cores, rank 0 only.
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

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

FLOP_PER_INTERACTION = 26       # 8 DFMA + 6 DMUL + 4 DADD per point charge, Phi + E
FLOP_PER_INTERACTION_PHI = 18   # 6 DFMA + 3 DMUL + 3 DADD, potential only (matrix fill)
FLOP_PER_INTERACTION_GRAD = 41  # + 5 DFMA + 4 DMUL + 1 DADD for the gradient sums (28 FP64 instructions)
FP64_LANES_PER_SM = 64          # B200: one FP64 warp instruction per scheduler every 2 cycles (profiles/r2_issue_model.md)
METRIC = "FP64 Phi+E element.point interactions/s"
UNIT = "element.point interactions/s"
# committed ncu capture of ONE launch of the bench's own launch configuration (hardware counters; not measured by this run)
NCU_CAPTURE = {"cfg4": ("profiles/r3_cfg4_full_eval_paired_counters.csv", "eval_paired_kernel")}
NCU_PIPE_METRIC = "sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_elapsed"
LINE_LIMIT = 4096               # bytes of the stdout record (the driver keeps a tail of stdout: round 2's 20 KB line did not parse)


def ncu_capture(workload: str, kernel: str):
    """{metric: value} of the committed counter capture of this workload's dominant kernel, or None."""
    import csv
    ent = NCU_CAPTURE.get(workload)
    if not ent or not kernel.startswith(ent[1]):
        return None
    out = {}
    try:
        with open(os.path.join(ROOT, ent[0]), newline="") as f:
            for row in csv.reader(f):
                if len(row) >= 3 and ent[1] in " ".join(row[:-3]):
                    try:
                        out[row[-3]] = float(row[-1].replace(",", ""))
                    except ValueError:
                        pass
    except OSError:
        return None
    return {"file": ent[0], "metrics": out} if out else None


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg4",
                    choices=["cfg4", "cfg1", "cfg2", "cfg3", "cfg5", "solve", "table3", "accuracy", "few"])
    ap.add_argument("--scale", type=float, default=1.0, help="config-4 size factor (profiling only)")
    ap.add_argument("--rule", type=int, default=1, help="fixed rule level of --workload cfg2 / cfg5 / table3 (-1 = adaptive)")
    ap.add_argument("--precision", default="f64", choices=["f64", "f32"],
                    help="f32: the FP32 variant (adaptive workloads then use the BEMCUB_POLICY_FIELD_F32 limits); not the bench line")
    ap.add_argument("--gradient", action="store_true",
                    help="also compute the field gradient (bemcub_eval_gradient; cubature levels only) - not the bench line")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-secondary", action="store_true", help="default workload only: skip the secondary block")
    ap.add_argument("--store-matrix", action="store_true",
                    help="--workload solve: let the solve keep the matrix (bemcub_solve_storage): one matrix fill, GEMV mat-vecs")
    ap.add_argument("--out", default=None, help="--workload accuracy: text file for the tables")
    ap.add_argument("--detail-out", default=os.path.join("gpurun_out", "bench_detail.json"),
                    help="file for the full record (peak sweep, definitions, the secondary runs with their rooflines); the "
                         "stdout line is the compact contract record only")
    return ap.parse_args()


# --------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""

    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int, period_ms: int = 200):
        self.gpu = gpu_index
        self.period = period_ms
        self.proc = None
        self.lines = []
        self.thread = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", str(self.period),
                 "-i", str(self.gpu)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        def pump():
            for line in self.proc.stdout:
                self.lines.append(line.strip())
        self.thread = threading.Thread(target=pump, daemon=True)
        self.thread.start()

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        if self.thread:
            self.thread.join(timeout=2)
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1]))
                smax.append(float(f[2]))
                power.append(float(f[3]))
            except ValueError:
                continue
            for name, val in zip(names, f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


# --------------------------------------------------------------------------------------------
def make_workload(name: str, args, rank: int):
    """Seeded synthetic inputs.  Rank r > 0 draws its own field points."""
    from paper_1606_03743_b200 import synth
    if name == "cfg4":
        c = synth.config4(scale=args.scale)
        if rank > 0:  # weak scaling: same mesh, another 10^6 track points per rank
            c["pts"] = synth.helical_tracks(c["ntracks"], c["npts_per_track"], seed=synth.SEED_CFG4_TRACKS + 1000 * rank)
        c["rule"] = -1
        c["desc"] = ("config 4: cylinder R=5 m L=20 m (%d rectangles) + two end cones (%d triangles), sigma = 8 "
                     "Fourier modes, %d helical-track field points, DR-adaptive rules, Phi+E"
                     % (int((c["etype"] == 1).sum()), int((c["etype"] == 0).sum()), len(c["pts"])))
    elif name == "cfg1":
        c = synth.config1()
        c["rule"] = 1
        c["desc"] = "config 1: level-3 icosphere (1280 triangles), 1000 field points, Table A2 (N = 7), Phi+E"
    elif name == "cfg2":
        c = synth.config2()
        c["rule"] = args.rule
        c["desc"] = "config 2: unit-cube surface 6144 squares, 10^4 field points, fixed rule level %d, %s" % (
            args.rule, args.precision)
    elif name == "cfg5":
        c = synth.config5(synth.TRI)
        c["rule"] = args.rule
        c["desc"] = "config 5: single triangle, 10^6 field points at log-uniform distance ratios 1..1e6, rule level %d, %s" % (
            args.rule, args.precision)
    elif name == "table3":
        # the SHAPE of the paper's GPU timing (Table 3: 1.5 M rectangles, 10^4 field points) on a
        # synthetic cylinder; --rule 1 = the 7-point rule, --rule -1 = distance-ratio dependent
        et, vt = synth.cylinder_rects(5.0, -10.0, 10.0, 1500, 1000)
        c = dict(etype=et, verts=vt, sigma=synth.fourier_sigma(synth.element_centroids(et, vt)),
                 pts=synth.helical_tracks(100, 100), rule=args.rule)
        c["desc"] = ("Table-3 shape: cylinder of 1.5e6 rectangles, 1e4 helical-track field points, rule %s, Phi+E"
                     % ("adaptive" if args.rule == -1 else "level %d" % args.rule))
    elif name == "solve":
        c = synth.config3()
        c["pts"] = np.zeros((len(c["etype"]), 3))
        c["rule"] = None
        c["desc"] = ("matrix-free BEM solve of the level-5 icosphere (20480 triangles) at unit potential: GMRES(30), "
                     "right Jacobi, rel. residual 1e-12; every mat-vec = potential-only adaptive evaluation at the centroids")
    else:
        c = synth.config3()
        c["pts"] = np.zeros((len(c["etype"]), 3))
        c["rule"] = None
        c["desc"] = "config 3: level-5 icosphere 20480 x 20480 collocation matrix, L159 limits"
    c["workload"] = name
    return c


def oracle_rate(c, target_seconds: float, full: bool = False, min_units: int = 8, max_units: int = 65536):
    """Times the CPU oracle (double-precision instantiation where it has one, OpenMP over field points /
    rows, all host cores, as it stands) on a bounded seeded sample of the workload's field points /
    matrix rows - or on all of them (`full`).  The sample is a multiple of the thread count, so every
    thread is busy.  Returns dict(value, cores, threads_busy, sample, seconds, units[, points_per_pair])."""
    import oracle
    cores = oracle.num_threads()
    n = len(c["etype"])
    is_matrix = c["workload"] == "cfg3"
    rng = np.random.default_rng(160603751)
    counts = {}
    if is_matrix:
        dr = oracle.default_policy(False)
        run = lambda idx: oracle.assemble_rows(c["etype"], c["verts"], idx, dr)
        total = n
    else:
        dr = oracle.default_policy(True)
        def run(idx):
            r = oracle.evaluate(c["etype"], c["verts"], c["sigma"], c["pts"][idx], c["rule"], dr=dr, precision="double",
                                want_counts=True)
            counts["npi"] = int(r["npi"].sum())
        total = len(c["pts"])
    if full:
        k = total
    else:
        probe = min(total, max(min_units, cores))
        idx = np.sort(rng.choice(total, probe, replace=False))
        t0 = time.perf_counter()
        run(idx)
        t_probe = time.perf_counter() - t0
        k = int(min(max_units, total, max(probe, probe * target_seconds / max(t_probe, 1e-6))))
        k = min(total, max(cores, k // cores * cores))
    idx = np.sort(rng.choice(total, k, replace=False)) if k < total else np.arange(total)
    t0 = time.perf_counter()
    run(idx)
    dt = time.perf_counter() - t0
    what = "matrix rows" if is_matrix else "field points"
    which = "long-double (its only matrix path)" if is_matrix else "double-precision"
    out = {"value": n * len(idx) / dt, "unit": "matrix entries/s" if is_matrix else UNIT, "cores": cores,
           "threads_busy": min(cores, len(idx)), "kind": "oracle",
           "sample": f"all {n} elements x {len(idx)} {'(all) ' if k == total else 'seeded '}{what} of the workload, oracle "
                     f"{which} path, {cores} OpenMP threads, one field point / row per task",
           "seconds": dt, "units": len(idx)}
    if "npi" in counts:
        out["points_per_pair"] = counts["npi"] / (float(n) * len(idx))
    return out


def run_reference(args, rank: int):
    """--impl reference: the oracle as it stands on the host cores, rank 0 only."""
    if rank != 0:
        return
    name = args.workload if args.workload in ("cfg1", "cfg2", "cfg3", "cfg4", "cfg5", "table3") else "cfg4"
    c = make_workload(name, args, 0)
    # each step a bounded sample (~4 s) so that warmup + steps end within a few minutes
    probe = oracle_rate(c, target_seconds=4.0)
    import oracle
    n, k = len(c["etype"]), probe["units"]
    is_matrix = name == "cfg3"
    rng = np.random.default_rng(160603752)
    total = n if is_matrix else len(c["pts"])
    dr = oracle.default_policy(not is_matrix)

    def step():
        idx = np.sort(rng.choice(total, k, replace=False)) if k < total else np.arange(total)
        if is_matrix:
            oracle.assemble_rows(c["etype"], c["verts"], idx, dr)
        else:
            oracle.evaluate(c["etype"], c["verts"], c["sigma"], c["pts"][idx], c["rule"], dr=dr, precision="double")

    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = (time.perf_counter() - t0) / max(args.steps, 1)
    value = n * k / dt
    unit = UNIT if not is_matrix else "matrix entries/s"
    line = {
        "impl": "reference", "metric": METRIC if not is_matrix else "FP64 collocation-matrix entries/s",
        "value": value, "unit": unit, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": c["desc"], "elements": n, "sampled_units_per_step": k},
        "cpu_baseline": {"value": value, "unit": unit, "cores": probe["cores"], "threads_busy": probe["threads_busy"],
                         "kind": "oracle", "sample": probe["sample"]},
        "e2e": {"value": value, "unit": unit, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(contract_line(line)), flush=True)


# --------------------------------------------------------------------------------------------
def measure_peak(b, h, num_sms: int, seconds: float = 3.6) -> dict:
    """Roofline denominator: the FP64 issue-rate sweep (DFMA / DADD / DMUL / the Eq. 4.1 mix at 8, 16, 32
    warps per SM, plus the two issue-model mixes; `seconds` / 18 each), its maximum, and the nominal rate."""
    rates, mhz = b.bemcub_fp64_issue_sweep(h, seconds / b.PEAK_VARIANTS)
    best = int(np.argmax(rates))
    table = [{"mix": b.PEAK_MIXES[i // 3], "warps_per_sm": b.PEAK_WARPS[i % 3], "fp64_inst_per_s": float(rates[i]),
              "sm_mhz": float(mhz[i]), "of_nominal": float(rates[i] / (FP64_LANES_PER_SM * num_sms * mhz[i] * 1e6)) if mhz[i] else None}
             for i in range(b.PEAK_VARIANTS)]
    return {"fp64_inst_per_s": float(rates[best]), "tflops": 2.0 * float(rates[best]) / 1e12,
            "best": f"{b.PEAK_MIXES[best // 3]}, {b.PEAK_WARPS[best % 3]} warps/SM", "sm_mhz": float(mhz[best]),
            "sweep": table,
            "source": "bemcub_fp64_issue_sweep in this run: max FP64 instruction issue rate over 6 mixes x 3 occupancies, "
                      f"{seconds / b.PEAK_VARIANTS:.2f} s each (x2 flop per instruction); MEASURED_PEAKS.json has no FP64 entry"}


def nominal_tflops(num_sms: int, sm_mhz: float) -> float:
    return FP64_LANES_PER_SM * num_sms * 2.0 * sm_mhz * 1e6 / 1e12


def roofline_block(kernel: str, k_ms: float, step_ms: float, inter: float, inter_own, fpi: int, ipi: float, peak: dict,
                   num_sms: int, kernel_mhz, smi_mhz) -> dict:
    """The dominant kernel against the FP64-ALU roofline.  `achieved` / `frac` count the ALGORITHMIC work (SURVEY.md
    section 8(d)): the point-charge interactions the per-pair distance-ratio policy asks for (`inter_own`; a fixed rule:
    all of them) x `fpi` flop each.  `frac_executed` counts the interactions the tiles really evaluated (a few per cent
    more: upgraded tiles), `fp64_issue_frac` the FP64 instructions really executed against the measured issue rate."""
    sec = k_ms * 1e-3
    base = inter if inter_own is None else inter_own
    ach = base * fpi / sec / 1e12
    ach_exec = inter * fpi / sec / 1e12
    clock = kernel_mhz or smi_mhz or peak["sm_mhz"]
    nom = nominal_tflops(num_sms, clock)
    return {"bound": "alu", "achieved": ach, "peak": peak["tflops"], "unit": "TFLOP/s", "frac": ach / peak["tflops"],
            "traffic": None,
            "traffic_source": "not measured by this run; ALU-bound (the bytes do not set the time); ncu captures are under profiles/",
            "kernel": kernel, "kernel_ms": k_ms, "kernel_share_of_step": k_ms / step_ms if step_ms else None,
            "work": "own" if inter_own is not None else "executed",
            "work_def": "point-charge interactions of the per-pair distance-ratio policy (device counter of one untimed call with "
                        "allow_upgrade = 0; fixed rule: every interaction) x flop_per_interaction: algorithm-equivalent flop, whatever "
                        "instruction sequence the kernel used for them",
            "interactions_per_launch": base, "interactions_executed_per_launch": inter,
            "flop_per_interaction": fpi, "fp64_inst_per_interaction": ipi,
            "achieved_executed": ach_exec, "frac_executed": ach_exec / peak["tflops"],
            "frac_nominal": ach / nom, "frac_executed_nominal": ach_exec / nom, "nominal_tflops": nom,
            "nominal_def": f"{num_sms} SMs x {FP64_LANES_PER_SM} FP64 lanes x 2 flop x {clock:.0f} MHz "
                           f"({'SM clock read inside the kernel: cycle counter / global timer' if kernel_mhz else 'nvidia-smi median'})",
            "peak_over_nominal": peak["tflops"] / nom, "peak_source": peak["source"], "peak_best_variant": peak["best"],
            "kernel_sm_mhz": kernel_mhz,
            "fp64_issue_frac": inter * ipi / sec / peak["fp64_inst_per_s"],
            "fp64_issue_frac_def": "FP64 instructions executed (interactions executed x instructions per interaction, device tally) "
                                   "/ kernel time / measured FP64 issue rate"}


def kernel_clock_mhz(st: dict):
    return 1e3 * st["kernel_cycles"] / st["kernel_ns"] if st.get("kernel_ns") else None


class Runner:
    """One bemcub ctx on this rank's GPU, device-resident inputs of one workload, a timed loop."""

    def __init__(self, b, torch, dev_index: int, c: dict):
        self.b, self.torch, self.c = b, torch, c
        self.dev = torch.device("cuda", dev_index)
        self.ctx = b.Context(dev_index)
        self.h = self.ctx.handle
        self.n, self.m = len(c["etype"]), len(c["pts"])
        self.h_type = torch.as_tensor(c["etype"]).pin_memory()
        self.h_verts = torch.as_tensor(c["verts"]).pin_memory()
        self.h_sigma = torch.as_tensor(np.ascontiguousarray(c["sigma"])).pin_memory()
        self.h_pts = torch.as_tensor(c["pts"]).pin_memory()
        self.d_type, self.d_verts = self.h_type.to(self.dev), self.h_verts.to(self.dev)
        self.d_sigma, self.d_pts = self.h_sigma.to(self.dev), self.h_pts.to(self.dev)
        b.bemcub_set_elements(self.h, self.n, self.d_type, self.d_verts)
        b.bemcub_set_timing(self.h, True)

    def timed(self, step, steps: int, warmup: int, barrier, gpu_index: int, period_ms: int = 200):
        """W untimed + K timed steps: CUDA events around the K steps, the dominant kernel's own event
        time per step, nvidia-smi clocks sampled during the timed region."""
        b, torch = self.b, self.torch
        for _ in range(warmup):
            step()
        barrier()
        b.bemcub_reset_stats(self.h)
        sampler = ClockSampler(gpu_index, period_ms)
        sampler.start()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        kernel_ms = []
        ev0.record()
        for _ in range(steps):
            step()
            kernel_ms.append(b.bemcub_get_timing(self.h)[1])   # waits for this step's events only
        ev1.record()
        barrier()
        clocks = sampler.stop()
        st = b.bemcub_get_stats(self.h)
        return {"ms": ev0.elapsed_time(ev1) / max(steps, 1), "kernel_ms": sum(kernel_ms) / max(len(kernel_ms), 1),
                "clocks": clocks, "stats": st}

    def close(self):
        self.ctx.close()


def steps_for(ms_estimate: float, seconds: float = 1.5, lo: int = 20, hi: int = 5000) -> int:
    return int(min(hi, max(lo, seconds * 1e3 / max(ms_estimate, 1e-3))))


def secondary_block(args, b, torch, dev_index: int, peak: dict, num_sms: int, barrier):
    """Short device-timed runs of the other configs: matrix fill of config 3,
    configs 1, 2 (B2 and B5, FP64 and FP32) and 5, each with roofline, clocks and the oracle beside it."""
    out = []

    def fixed_rule_entry(name, rule, precision_name):
        a2 = argparse.Namespace(**vars(args))
        a2.rule, a2.precision, a2.scale = rule, precision_name, 1.0
        c = make_workload(name, a2, 0)
        r = Runner(b, torch, dev_index, c)
        prec = b.F32 if precision_name == "f32" else b.F64
        phi = torch.empty(r.m, dtype=torch.float64, device=r.dev)
        E = torch.empty((r.m, 3), dtype=torch.float64, device=r.dev)
        step = lambda: b.bemcub_eval(r.h, r.d_sigma, c["rule"], None, r.m, r.d_pts, phi, E, prec)
        probe = r.timed(step, 5, 3, barrier, dev_index)
        t = r.timed(step, steps_for(probe["ms"]), 3, barrier, dev_index, period_ms=100)
        st = t["stats"]
        inter = float(st["point_interactions"])
        entry = {"name": "%s rule level %d %s" % (name, rule, precision_name),
                 "workload": c["desc"], "dtype": precision_name, "ms_per_step": t["ms"], "kernel_ms": t["kernel_ms"],
                 "value": float(r.n) * r.m / (t["ms"] * 1e-3), "unit": UNIT, "clocks": t["clocks"],
                 "points_per_pair": inter / (float(r.n) * r.m)}
        if prec == b.F64:
            entry["roofline"] = roofline_block("eval_fixed_kernel", t["kernel_ms"], t["ms"], inter, inter, FLOP_PER_INTERACTION, 18,
                                               peak, num_sms, kernel_clock_mhz(st), t["clocks"].get("sm_mhz"))
        else:
            entry["roofline"] = {"bound": "alu", "achieved": inter * FLOP_PER_INTERACTION / (t["kernel_ms"] * 1e-3) / 1e12,
                                 "unit": "TFLOP/s", "peak": None, "frac": None, "traffic": None,
                                 "note": "FP32 variant: reported, no FP32 peak measured (the FP32 pipe has twice the lanes)"}
        if not args.no_cpu_baseline and prec == b.F64:
            # configs 1, 2, 5 "in full" where that is a few seconds of oracle time
            entry["cpu_baseline"] = oracle_rate(c, target_seconds=3.0, full=inter <= 1.5e9)
        r.close()
        return entry

    # matrix fill, config 3
    c3 = make_workload("cfg3", args, 0)
    r = Runner(b, torch, dev_index, c3)
    pol0 = b.bemcub_default_policy(False)
    A = torch.empty((r.n, r.n), dtype=torch.float64, device=r.dev)
    step = lambda: b.bemcub_assemble(r.h, pol0, A, r.n)
    t = r.timed(step, 300, 5, barrier, dev_index, period_ms=100)
    st = t["stats"]
    inter = float(st["point_interactions"])
    pol_pp = b.bemcub_default_policy(False)
    pol_pp.allow_upgrade = 0
    b.bemcub_assemble(r.h, pol_pp, A, r.n)             # untimed: the per-pair policy's own work
    own = float(b.bemcub_get_stats(r.h)["point_interactions"])
    roof = roofline_block("assemble_kernel", t["kernel_ms"], t["ms"], inter, own, FLOP_PER_INTERACTION_PHI, 12, peak, num_sms,
                          kernel_clock_mhz(st), t["clocks"].get("sm_mhz"))
    roof["store_stream_gb_s"] = float(r.n) * r.n * 8 / (t["kernel_ms"] * 1e-3) / 1e9
    entry = {"name": "cfg3 matrix fill 20480^2", "workload": c3["desc"], "dtype": "f64", "ms_per_step": t["ms"], "kernel_ms": t["kernel_ms"],
             "value": float(r.n) * r.n / (t["ms"] * 1e-3), "unit": "matrix entries/s", "steps": 300, "clocks": t["clocks"],
             "points_per_entry": inter / (float(r.n) * r.n), "points_per_entry_own_work": own / (float(r.n) * r.n),
             "analytic_entries_per_row": st["analytic_pairs"] / float(r.n), "roofline": roof}
    if not args.no_cpu_baseline:
        entry["cpu_baseline"] = oracle_rate(c3, target_seconds=6.0, min_units=64)
    del A
    r.close()
    out.append(entry)

    out.append(fixed_rule_entry("cfg1", 1, "f64"))
    for rule in (1, 4):
        for prec in ("f64", "f32"):
            out.append(fixed_rule_entry("cfg2", rule, prec))
    out.append(fixed_rule_entry("cfg5", 1, "f64"))
    return out


# --------------------------------------------------------------------------------------------
def _pick(d, keys):
    return None if d is None else {k: d[k] for k in keys if k in d}


def _clip(v, n: int):
    return v if not isinstance(v, str) or len(v) <= n else v[:n - 3] + "..."


def _sig(v, digits: int = 6):
    """Floats to `digits` significant digits (the record is read by people and by a tail-limited log)."""
    if isinstance(v, float):
        return float(f"{v:.{digits}g}")
    if isinstance(v, dict):
        return {k: _sig(x, digits) for k, x in v.items()}
    if isinstance(v, list):
        return [_sig(x, digits) for x in v]
    return v


def contract_line(full: dict, detail_path=None) -> dict:
    """The ONE stdout record of the driver contract from the full record: the contract keys, short strings, no
    sweeps, no definitions; the secondary runs as one short row each.  Stays below LINE_LIMIT bytes."""
    top = ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
           "vs_baseline", "dtype", "data", "pct_fp64_peak", "gpu_launches")
    line = {k: full[k] for k in top if k in full}
    cfg = dict(full.get("config") or {})
    for k in cfg:
        cfg[k] = _clip(cfg[k], 230 if k == "workload" else 90)
    line["config"] = cfg
    line["clocks"] = _pick(full.get("clocks"), ("sm_mhz", "sm_max_mhz", "power_w_max", "samples", "reasons"))
    line["e2e"] = _pick(full.get("e2e"), ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step", "ms_per_step", "api", "note"))
    if line["e2e"] and "api" in line["e2e"]:
        line["e2e"]["api"] = _clip(line["e2e"]["api"], 80)
    roof = _pick(full.get("roofline"), ("bound", "achieved", "peak", "unit", "frac", "traffic", "traffic_source", "kernel",
                                         "kernel_ms", "kernel_share_of_step", "work", "flop_per_interaction",
                                         "fp64_inst_per_interaction", "frac_executed", "frac_nominal", "fp64_issue_frac",
                                         "fp64_pipe_pct_ncu", "store_stream_gb_s", "peak_source", "note"))
    if roof:
        for k, n in (("traffic_source", 150), ("peak_source", 100), ("note", 120)):
            if k in roof:
                roof[k] = _clip(roof[k], n)
    line["roofline"] = roof
    cpu = _pick(full.get("cpu_baseline"), ("value", "unit", "cores", "threads_busy", "kind", "sample", "value_single_thread"))
    if cpu and "sample" in cpu:
        cpu["sample"] = _clip(cpu["sample"], 120)
    line["cpu_baseline"] = cpu
    if full.get("solve"):
        line["solve"] = _pick(full["solve"], ("matvecs", "rel_residual", "converged", "capacitance_over_4pi_eps0_R"))
    if full.get("secondary"):
        rows = []
        for e in full["secondary"][:8]:
            rf = e.get("roofline") or {}
            rows.append({"name": _clip(e.get("name") or e.get("workload", ""), 40), "ms_per_step": e.get("ms_per_step"),
                         "value": e.get("value"), "frac": rf.get("frac")})
        line["secondary"] = rows
        line["secondary_def"] = "other configs, device-timed: value in matrix entries/s (fill) or element.point/s; frac as roofline.frac"
    if detail_path:
        line["detail"] = detail_path
    line = _sig(line)
    if len(json.dumps(line)) >= LINE_LIMIT:      # never print a record the driver cannot keep: drop the optional parts
        for k in ("secondary", "secondary_def", "solve"):
            line.pop(k, None)
    return line


def emit(full: dict, detail_path=None):
    """Full record -> `detail_path` (best effort), compact record -> the one stdout line."""
    wrote = None
    if detail_path:
        try:
            os.makedirs(os.path.dirname(os.path.abspath(detail_path)) or ".", exist_ok=True)
            with open(detail_path, "w") as f:
                json.dump(full, f, indent=1)
            wrote = detail_path
        except OSError:
            wrote = None
    print(json.dumps(contract_line(full, wrote)), flush=True)


# --------------------------------------------------------------------------------------------
def run_ours(args, rank: int, world: int, local_rank: int):
    import torch
    import torch.distributed as dist
    from paper_1606_03743_b200 import bemcub as b   # fails loudly if libbemcub.so is missing

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the bemcub path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    num_sms = torch.cuda.get_device_properties(local_rank).multi_processor_count

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    if args.workload == "accuracy":
        return run_accuracy(args, b, torch, local_rank, barrier)
    if args.workload == "few":
        return run_few(args, b, torch, local_rank)

    c = make_workload(args.workload, args, rank)
    r = Runner(b, torch, local_rank, c)
    h, dev, n, m = r.h, r.dev, r.n, r.m
    is_matrix = args.workload in ("cfg3", "solve")
    is_solve = args.workload == "solve"
    precision = b.F32 if (args.precision == "f32" and not is_matrix and not args.gradient) else b.F64
    adaptive = c["rule"] == -1
    solve_info = {}
    if is_solve:
        pol = b.bemcub_default_policy(False)
        d_V = torch.ones(n, dtype=torch.float64, device=dev)
        d_s = torch.zeros(n, dtype=torch.float64, device=dev)
        if args.store_matrix:
            b.bemcub_solve_storage(h, 8 * n * n)
            c["desc"] = c["desc"].replace("matrix-free BEM solve", "BEM solve with the matrix kept in HBM (bemcub_solve_storage)") \
                                 .replace("every mat-vec = potential-only adaptive evaluation at the centroids",
                                          "one matrix fill, every mat-vec = bemcub_matvec")

        def step():
            d_s.zero_()
            mv, res, ok = b.bemcub_solve(h, pol, d_V, d_s, 1e-12, 500)
            solve_info.update(matvecs=mv, rel_residual=res, converged=ok)
    elif is_matrix:
        pol = b.bemcub_default_policy(False)
        out = torch.empty((n, n), dtype=torch.float64, device=dev)
        step = lambda: b.bemcub_assemble(h, pol, out, n)
    else:
        # FP32 with the distance-ratio choice takes the limits made for it (BEMCUB_POLICY_FIELD_F32)
        pol = b.bemcub_default_policy(b.POLICY_FIELD_F32 if precision == b.F32 else b.POLICY_FIELD) if adaptive else None
        phi = torch.empty(m, dtype=torch.float64, device=dev)
        E = torch.empty((m, 3), dtype=torch.float64, device=dev)
        if args.gradient:
            if pol is not None:
                pol.use_levels_mask = 0b011111          # derivatives exist for the point charges only (L273)
            G = torch.empty((m, 6), dtype=torch.float64, device=dev)
            step = lambda: b.bemcub_eval_gradient(h, r.d_sigma, c["rule"], pol, m, r.d_pts, phi, E, G)
        else:
            step = lambda: b.bemcub_eval(h, r.d_sigma, c["rule"], pol, m, r.d_pts, phi, E, precision)

    # roofline denominator: FP64 issue rate of this GPU, measured in this run
    peak = measure_peak(b, h, num_sms)
    # second reference: the kernels' own inner loop on resident data (what the 18-instruction mix allows)
    loop_rate = b.bemcub_inner_loop_rate(h, 1.0)

    t = r.timed(step, args.steps, args.warmup, barrier, local_rank)
    st, clocks, ms, k_ms = t["stats"], t["clocks"], t["ms"], t["kernel_ms"]
    tt = torch.tensor([ms], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    ms_max = float(tt.item())
    units_per_step = float(n) * float(n if is_matrix else m) * (solve_info.get("matvecs", 1) if is_solve else 1)
    if is_solve:
        areas = 0.5 * np.linalg.norm(np.cross(c["verts"][:, 1] - c["verts"][:, 0], c["verts"][:, 2] - c["verts"][:, 0]), axis=1)
        q_tot = float((d_s.cpu().numpy() * areas).sum())
        solve_info["capacitance_over_4pi_eps0_R"] = q_tot / (4 * np.pi * 8.8541878128e-12)
        if args.store_matrix:
            # the mat-vec of this mode on its own: HBM-bound, 8 n^2 bytes per call against the measured copy rate
            b.bemcub_solve_storage(h, 0)
            A = torch.empty((n, n), dtype=torch.float64, device=dev)
            y = torch.empty(n, dtype=torch.float64, device=dev)
            b.bemcub_assemble(h, pol, A, n)
            for _ in range(3):
                b.bemcub_matvec(h, A, n, d_s, y)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize(dev)
            e0.record()
            for _ in range(50):
                b.bemcub_matvec(h, A, n, d_s, y)
            e1.record()
            torch.cuda.synchronize(dev)
            g_ms = e0.elapsed_time(e1) / 50
            hbm = None
            try:
                hbm = float(json.load(open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "MEASURED_PEAKS.json")))["hbm_gbs"])
            except Exception:
                pass
            peak_gbs = hbm if hbm else 6500.0
            solve_info["matvec_roofline"] = {
                "bound": "hbm", "kernel": "gemv_rows_kernel", "ms": g_ms, "achieved": 8.0 * n * n / (g_ms * 1e-3) / 1e9,
                "peak": peak_gbs, "unit": "GB/s", "frac": 8.0 * n * n / (g_ms * 1e-3) / 1e9 / peak_gbs,
                "peak_source": "MEASURED_PEAKS.json hbm_gbs (copy: read + write)" if hbm else "fallback 6500 GB/s (B200_PROFILING.md)",
                "bytes_per_call": 8.0 * n * n, "l2": "matrix (3.36 GB) larger than L2"}
            del A
    value = units_per_step * world / (ms_max * 1e-3)

    # dominant kernel against the FP64-ALU roofline
    inter = float(st["point_interactions"])          # point-charge interactions of the last step
    fpi = FLOP_PER_INTERACTION_PHI if is_matrix else (FLOP_PER_INTERACTION_GRAD if args.gradient else FLOP_PER_INTERACTION)
    ipi = 12 if is_matrix else (28 if args.gradient else 18)   # FP64 instructions per interaction
    inter_own = None
    if (adaptive and not args.gradient and precision == b.F64) or args.workload == "cfg3":
        # the method's own work: one untimed call with the exact per-pair policy, counted on the device
        pol_pp = b.bemcub_default_policy(not is_matrix)
        pol_pp.allow_upgrade = 0
        if is_matrix:
            b.bemcub_assemble(h, pol_pp, out, n)
        else:
            b.bemcub_eval(h, r.d_sigma, -1, pol_pp, m, r.d_pts, phi, E, precision)
        inter_own = float(b.bemcub_get_stats(h)["point_interactions"])
    elif not is_matrix and not adaptive:
        inter_own = inter
    paired = (not is_matrix) and b.bemcub_last_path(h) == b.PATH_PAIRED
    kernel = ("assemble_kernel" if (is_solve and args.store_matrix) else "eval_adaptive_kernel<kModePhi>" if is_solve else
              "assemble_kernel" if is_matrix else
              ("eval_paired_kernel" if paired else "eval_adaptive_kernel" if adaptive else "eval_fixed_kernel"))
    # FP64 instructions the kernel executed per interaction (device tally): 18 / 12 / 28, fewer in paired form
    if st.get("fp64_instructions") and inter:
        ipi = st["fp64_instructions"] / inter
    if precision == b.F32:
        roof = {"bound": "alu", "achieved": inter * fpi / (k_ms * 1e-3) / 1e12, "peak": None, "unit": "TFLOP/s", "frac": None,
                "traffic": None, "note": "FP32 variant: reported, no FP32 peak measured"}
    else:
        roof = roofline_block(kernel, k_ms, ms, inter, inter_own, fpi, ipi, peak, num_sms, kernel_clock_mhz(st), clocks.get("sm_mhz"))
        roof["inner_loop_ceiling"] = {
            "interactions_per_s": loop_rate,
            "frac_of_peak": loop_rate * FLOP_PER_INTERACTION / peak["tflops"] / 1e12,
            "kernel_over_ceiling": None if is_matrix else (inter / (k_ms * 1e-3)) / loop_rate,
            "source": "bemcub_inner_loop_rate: Eq. 4.1 loop (18 FP64 instr + MUFU, 8 of 18 are FMAs => at most 26/36 = 72.2% "
                      "of the FLOP peak), resident data"}
        if paired:
            roof["paired_form"] = ("rectangle rules evaluated in +- point pairs and the 7-point triangle rule on its medians "
                                   "(kernels_paired.cuh): the same point-charge interactions of Eq. 4.1, %.2f instead of 18 FP64 "
                                   "instructions each, so the 26/36 = 72.2 %% cap of the plain instruction mix does not bind `frac`; "
                                   "fp64_issue_frac uses the executed count; inner_loop_ceiling is the PLAIN loop's rate" % ipi)
        roof["peak_sweep"] = peak["sweep"]
        if is_matrix:
            roof["store_stream_gb_s"] = float(n) * n * 8 / (k_ms * 1e-3) / 1e9
        cap = ncu_capture(args.workload, kernel) if (args.scale == 1.0 and not args.gradient) else None
        if cap:
            mt = cap["metrics"]
            if "dram__bytes_read.sum" in mt and "dram__bytes_write.sum" in mt:
                roof["traffic"] = mt["dram__bytes_read.sum"] + mt["dram__bytes_write.sum"]
                roof["traffic_source"] = ("dram__bytes_read.sum + dram__bytes_write.sum of one launch, committed ncu capture "
                                          f"{cap['file']} (same launch configuration; not this run)")
            if NCU_PIPE_METRIC in mt:
                roof["fp64_pipe_pct_ncu"] = mt[NCU_PIPE_METRIC]
                roof["ncu_fp64_pipe_counter"] = {"file": cap["file"], "metric": NCU_PIPE_METRIC,
                                                 "note": "hardware counter of a committed capture of this launch configuration, "
                                                         "not of this run"}

    # end to end through the host-buffer C-ABI calls: H2D of the inputs, compute, D2H of Phi/E
    e2e = None
    if not args.no_e2e and not is_matrix and not args.gradient:
        o_phi = torch.empty(m, dtype=torch.float64).pin_memory()
        o_E = torch.empty((m, 3), dtype=torch.float64).pin_memory()
        ctx2 = b.Context(local_rank)

        def step_host():
            b.bemcub_set_elements_host(ctx2.handle, n, r.h_type, r.h_verts)
            b.bemcub_eval_host(ctx2.handle, r.h_sigma, c["rule"], pol, m, r.h_pts, o_phi, o_E, precision)

        step_host()
        barrier()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        for _ in range(args.steps):
            step_host()
        ev1.record()
        barrier()
        ms_e = ev0.elapsed_time(ev1) / max(args.steps, 1)
        tt = torch.tensor([ms_e], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        e2e = {"value": units_per_step * world / (float(tt.item()) * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": int(n * 1 + n * 72 + n * 8 + m * 24), "d2h_bytes_per_step": int(m * 32),
               "ms_per_step": float(tt.item()), "api": "bemcub_set_elements_host + bemcub_eval_host (pinned host buffers)"}
        assert bool(torch.isfinite(o_phi).all())
        ctx2.close()
    elif is_matrix:
        e2e = {"value": None, "unit": "matrix entries/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
               "note": "matrix stays on the device (3.36 GB); no host leg"}
    launches = int(st["kernel_launches"])

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline and not is_solve:
        cpu = oracle_rate(c, target_seconds=15.0)
        if not is_matrix:   # the paper's CPU numbers are single-threaded (Table 2): one thread on a smaller sample
            import oracle
            k1 = max(4, int(cpu["units"] / max(cpu["cores"], 1) / 4))
            idx1 = np.sort(np.random.default_rng(160603753).choice(m, min(k1, m), replace=False))
            t0 = time.perf_counter()
            oracle.evaluate(c["etype"], c["verts"], c["sigma"], c["pts"][idx1], c["rule"], dr=oracle.default_policy(True),
                            precision="double", nthreads=1)
            cpu["value_single_thread"] = n * len(idx1) / (time.perf_counter() - t0)

    secondary = None
    if rank == 0 and world == 1 and args.workload == "cfg4" and not args.no_secondary and not args.gradient:
        r.close()
        r = None
        del phi, E
        torch.cuda.empty_cache()
        try:
            secondary = secondary_block(args, b, torch, local_rank, peak, num_sms, barrier)
        except Exception as exc:     # the contract record does not depend on the side runs
            secondary = [{"workload": "secondary block failed", "error": repr(exc)[:200]}]

    if rank == 0:
        line = {
            "metric": METRIC if not is_matrix else "FP64 collocation-matrix entries/s",
            "value": value, "unit": UNIT if not is_matrix else "matrix entries/s",
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_max,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32" if precision == b.F32 else "f64", "data": "synthetic",
            "config": {"workload": c["desc"], "elements": n, "field_points_per_gpu": (n if is_matrix else m),
                       "parallelism": f"field points sharded over {world} GPU(s), no collective",
                       "l2": "inputs larger than L2 (expanded point arrays %.0f MB; compute-bound kernel)"
                             % (n * (7 + 12 + 19 + 33) * 32 / 1e6) if args.workload == "cfg4" else "compute-bound; not flushed",
                       "points_per_pair": inter / units_per_step if units_per_step else None,
                       "points_per_pair_own_work": inter_own / units_per_step if (inter_own and units_per_step) else None},
            "pct_fp64_peak": 100.0 * roof["frac"] if roof.get("frac") else None,
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches,
            "roofline": roof, "cpu_baseline": cpu,
        }
        if secondary is not None:
            line["secondary"] = secondary
        if is_solve:
            line["metric"] = "FP64 potential-only element.point interactions/s inside bemcub_solve"
            line["unit"] = "element.point interactions/s"
            line["solve"] = solve_info
            line["roofline"]["note"] = ("kernel_ms / interactions are those of the solve's one matrix fill; the mat-vecs are "
                                        "solve.matvec_roofline (HBM-bound); value counts every mat-vec as n^2 element.point pairs"
                                        if args.store_matrix else
                                        "kernel_ms / interactions are those of the LAST mat-vec of the solve")
        emit(line, args.detail_out)
    if r is not None:
        r.close()


# --------------------------------------------------------------------------------------------
def run_few(args, b, torch, dev_index: int):
    """Tracking-style calls (the field at one point after the other): bemcub_eval with 1 ... 64
    field points on the config-4 mesh (10^6 elements at --scale 1), distance-ratio choice, Phi + E, with a
    new sigma every call and with the sigma of the previous call (sigma = NULL).  One line: microseconds per
    call (CUDA events around 200 back-to-back calls) and the bytes of element data a call reads per second."""
    from paper_1606_03743_b200 import synth
    dev = torch.device("cuda", dev_index)
    c = synth.config4(args.scale, ntracks=1, npts_per_track=64)
    n = len(c["etype"])
    pol = b.bemcub_default_policy(b.POLICY_FIELD)
    rows = []
    with b.Context(dev_index) as ctx:
        h = ctx.handle
        b.bemcub_set_elements(h, n, torch.as_tensor(c["etype"]).to(dev), torch.as_tensor(c["verts"]).to(dev))
        d_sigma = torch.as_tensor(c["sigma"]).to(dev)
        for m in (1, 2, 4, 8, 16, 64):
            pts = torch.as_tensor(c["pts"][:m].copy()).to(dev)
            phi = torch.empty(m, dtype=torch.float64, device=dev)
            E = torch.empty((m, 3), dtype=torch.float64, device=dev)
            row = {"field_points": m}
            for sig, key in ((d_sigma, "us_per_call_new_sigma"), (None, "us_per_call_sigma_kept")):
                for _ in range(max(args.warmup, 3)):
                    b.bemcub_eval(h, sig, -1, pol, m, pts, phi, E, b.F64)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize(dev)
                e0.record()
                for _ in range(200):
                    b.bemcub_eval(h, sig, -1, pol, m, pts, phi, E, b.F64)
                e1.record()
                torch.cuda.synchronize(dev)
                row[key] = e0.elapsed_time(e1) / 200 * 1e3
            passes = 1 if m <= 2 else (m + 3) // 4
            row["element_bytes_read_gb_s"] = 121.0 * n * passes / (row["us_per_call_sigma_kept"] * 1e-6) / 1e9
            st = b.bemcub_get_stats(h)
            row["points_per_pair"] = st["point_interactions"] / (float(n) * m)
            row["launches_per_call"] = st["last_eval_launches"]
            rows.append(row)
    print(json.dumps({"metric": "microseconds per bemcub_eval call with few field points", "unit": "us", "higher_is_better": False,
                      "n_gpus": 1, "dtype": "f64", "data": "synthetic",
                      "config": {"workload": "config-4 mesh (%d elements), 1 ... 64 field points of one helical track, DR-adaptive "
                                             "rules per pair, Phi+E; eval_few_kernel (121 bytes of element data per element and pass)" % n},
                      "calls": rows}), flush=True)


# --------------------------------------------------------------------------------------------
def run_accuracy(args, b, torch, dev_index: int, barrier):
    """The paper's accuracy study on the GPU (Sec. 2 and 4: L68, L80, L149; Figs. 8-10; L163-169): random
    triangles / rectangles with corners in the unit cube, a field point in a random direction at each of
    500 distance ratios from 2 to 1e4, 2000 elements per ratio (10^6 pairs per element type), every rule
    of App. A/B, the Duffy-mapped rectangle rules on triangles and the closed form, FP64 and FP32, all
    through bemcub_eval_pairs.  The exact reference is this run's cpu_baseline leg: the oracle in long
    double (closed form below DR = 12, 33-point rule above), timed.  Tables go to --out."""
    import oracle
    from paper_1606_03743_b200 import synth
    dev = torch.device("cuda", dev_index)
    ctx = b.Context(dev_index)
    h = ctx.handle
    n_ratio, per_ratio = 500, 2000
    grid = np.geomspace(2.0, 1.0e4, n_ratio)
    ratio = np.repeat(grid, per_ratio)
    K = len(ratio)
    lines, gpu_ms, gpu_pairs, cpu_s, cpu_pairs, launches = [], 0.0, 0, 0.0, 0, 0
    sampler = ClockSampler(dev_index)
    sampler.start()
    summary = {}
    for kind, kname in ((synth.TRI, "triangles"), (synth.RECT, "rectangles")):
        et, verts, pts = synth.random_pairs(kind, K, ratio, 160603790 + kind)
        t0 = time.perf_counter()
        lo = oracle.evaluate_pairs(et, verts, pts, 5)
        hi = oracle.evaluate_pairs(et, verts, pts, 4)
        cpu_s += time.perf_counter() - t0
        cpu_pairs += 2 * K
        near = ratio < 12.0
        phi_x = np.where(near, lo["phi"], hi["phi"])
        E_x = np.where(near[:, None], lo["E"], hi["E"])
        d = lambda a: torch.as_tensor(np.ascontiguousarray(a)).to(dev)
        d_et, d_verts, d_pts = d(et), d(verts), d(pts)
        phi = torch.empty(K, dtype=torch.float64, device=dev)
        E = torch.empty((K, 3), dtype=torch.float64, device=dev)
        methods = [(f"N={oracle.rule_info(kind, l)[0]}", l, b.F64) for l in range(5)]
        methods += [(f"N={oracle.rule_info(kind, l)[0]} f32", l, b.F32) for l in range(5)]
        if kind == synth.TRI:
            methods += [(f"Duffy N={oracle.rule_info(1, l)[0]}", b.METHOD_DUFFY_L0 + l, b.F64) for l in range(5)]
        methods += [("closed form", b.METHOD_ANALYTIC, b.F64)]
        cols = {}
        for name, method, prec in methods:
            for rep in range(2):     # first call warms up
                ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                ev0.record()
                b.bemcub_eval_pairs(h, K, d_et, d_verts, None, method, None, d_pts, phi, E, prec)
                ev1.record()
                torch.cuda.synchronize()
            gpu_ms += ev0.elapsed_time(ev1)
            gpu_pairs += K
            launches += 1
            e_phi = np.abs(phi.cpu().numpy() - phi_x) / np.abs(phi_x)
            e_E = np.abs(E.cpu().numpy() - E_x).sum(axis=1) / np.linalg.norm(E_x, axis=1)
            cols[name] = (e_phi.reshape(n_ratio, per_ratio).mean(axis=1), e_E.reshape(n_ratio, per_ratio).mean(axis=1))
        # first distance ratio from which a rule's mean error stays at the paper's level (L159)
        for name in [m_[0] for m_ in methods[:5]]:
            ok_phi = cols[name][0] <= 2e-15
            ok_E = cols[name][1] <= 3e-15
            def first_from(ok):
                bad = np.flatnonzero(~ok)
                return float(grid[0]) if len(bad) == 0 else (None if bad[-1] == len(ok) - 1 else float(grid[bad[-1] + 1]))
            summary[f"{kname} {name}"] = {"phi_2e-15_from_dr": first_from(ok_phi), "field_3e-15_from_dr": first_from(ok_E)}
        lines.append(f"## {kname}: mean relative error over {per_ratio} random elements per distance ratio (every 10th of {n_ratio} ratios)")
        lines.append("# err(Phi) = |dPhi/Phi|, err(E) = sum_j |dE_j| / |E| (PAPER.md L80); columns: Phi / E per method")
        lines.append("DR        " + "  ".join(f"{name:>19s}" for name in cols))
        for i in range(0, n_ratio, 10):
            lines.append(f"{grid[i]:9.3f} " + "  ".join(f"{cols[nm][0][i]:9.2e}/{cols[nm][1][i]:9.2e}" for nm in cols))
        lines.append("")
    # Fig. 10: aspect-ratio dependence of the 7-point rule at DR = 300
    lines.append("## Fig. 10: 7-point rule at DR = 300, mean field / potential error per aspect-ratio bin (4e5 random elements per type)")
    edges = [1, 1.5, 2, 3, 5, 10, 20, 50, 100, 1e9]
    for kind, kname in ((synth.TRI, "triangles"), (synth.RECT, "rectangles")):
        Kar = 400_000
        et, verts, pts = synth.random_pairs(kind, Kar, 300.0, 160603795 + kind)
        ar = synth.aspect_ratio(et, verts)
        t0 = time.perf_counter()
        ref = oracle.evaluate_pairs(et, verts, pts, 4)
        cpu_s += time.perf_counter() - t0
        cpu_pairs += Kar
        d = lambda a: torch.as_tensor(np.ascontiguousarray(a)).to(dev)
        phi = torch.empty(Kar, dtype=torch.float64, device=dev)
        E = torch.empty((Kar, 3), dtype=torch.float64, device=dev)
        b.bemcub_eval_pairs(h, Kar, d(et), d(verts), None, 1, None, d(pts), phi, E, b.F64)
        torch.cuda.synchronize()
        launches += 1
        e_phi = np.abs(phi.cpu().numpy() - ref["phi"]) / np.abs(ref["phi"])
        e_E = np.abs(E.cpu().numpy() - ref["E"]).sum(axis=1) / np.linalg.norm(ref["E"], axis=1)
        for lo_, hi_ in zip(edges[:-1], edges[1:]):
            sel = (ar >= lo_) & (ar < hi_)
            if sel.any():
                lines.append(f"{kname:10s} AR [{lo_:5g},{hi_:7g})  n={int(sel.sum()):7d}  Phi {e_phi[sel].mean():9.2e}  E {e_E[sel].mean():9.2e}")
    clocks = sampler.stop()
    if args.out:
        os.makedirs(os.path.dirname(os.path.abspath(args.out)) or ".", exist_ok=True)
        with open(args.out, "w") as f:
            f.write("# bench.py --workload accuracy: the accuracy study of arXiv 1606.03743 (Figs. 8-10, L163-169) on one B200,\n"
                    "# GPU results of bemcub_eval_pairs against the long-double oracle (closed form below DR = 12, N = 33 above).\n")
            f.write("\n".join(lines) + "\n")
    ctx.close()
    value = gpu_pairs / (gpu_ms * 1e-3)
    line = {"metric": "single-element (element, point) pairs/s, all methods of the accuracy study", "value": value,
            "unit": "element.point pairs/s", "n_gpus": 1, "steps": 1, "warmup": 1, "ms_per_step": gpu_ms,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64+f32", "data": "synthetic",
            "config": {"workload": f"accuracy study: {n_ratio} distance ratios 2..1e4 x {per_ratio} random elements, triangles and "
                                   "rectangles, 5 rules x FP64/FP32 + Duffy + closed form; Fig. 10 at DR = 300"},
            "clocks": clocks, "gpu_launches": launches,
            "e2e": {"value": None, "unit": "element.point pairs/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
                    "note": "study mode; errors are reduced on the host"},
            "roofline": {"bound": "alu", "achieved": None, "peak": None, "unit": "TFLOP/s", "frac": None, "traffic": None,
                         "note": "one thread per pair with on-the-fly geometry: a study tool, not a throughput kernel"},
            "cpu_baseline": {"value": cpu_pairs / cpu_s, "unit": "element.point pairs/s", "cores": oracle.num_threads(),
                             "kind": "oracle", "sample": "the exact references of the whole study (long double)", "seconds": cpu_s},
            "limits": summary, "table": args.out}
    print(json.dumps(line), flush=True)


def main():
    args = parse_args()
    from paper_1606_03743_b200 import build as _libbuild
    if args.impl == "ours" and _libbuild.override_refused():
        raise SystemExit("bench.py: BEMCUB_LIB is set (%s): the bench times the library built from csrc/; unset it, or set "
                         "BEMCUB_LIB_ALLOW=1 to time that binary on purpose" % os.environ["BEMCUB_LIB"])
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if world > 1:
        import torch
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("NCCL_DEBUG", "INFO")      # the communicator log shows the ranks (and NVLS) of the barrier
        torch.cuda.set_device(local_rank)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    try:
        run_ours(args, rank, world, local_rank)
    finally:
        if world > 1:
            import torch.distributed as dist
            dist.destroy_process_group()


if __name__ == "__main__":
    main()
