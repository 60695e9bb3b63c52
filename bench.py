#!/usr/bin/env python
"""bench.py -- throughput of the bemcub hot path on B200 (driver contract: one JSON line on rank 0).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg4|cfg2|cfg3]
                    [--scale S]

Metric (BASELINE.json): FP64 Phi+E element.point interactions/s.  One step = one pass of the whole
hot path (a1 preprocessing, a2 rule binning, a3 point-charge sum, a4 analytic near field, a6
reduction + scaling) over one batch of synthetic input.  Default workload =
config 4 (`configs[3]`, "the 10^6-element config" the north_star target is quoted on): 8e5
rectangles + 2e5 triangles, 10^6 helical-track field points, distance-ratio-adaptive rules.
`--workload cfg2 / cfg3` and `--scale` exist for profiling smaller cases; they are not bench lines.

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

FLOP_PER_INTERACTION = 26      # 8 DFMA + 6 DMUL + 4 DADD per point charge, Phi + E
FLOP_PER_INTERACTION_PHI = 18  # 6 DFMA + 3 DMUL + 3 DADD, potential only (matrix fill)
FLOP_PER_INTERACTION_GRAD = 41  # + 5 DFMA + 4 DMUL + 1 DADD for the gradient sums (28 FP64 instructions)
METRIC = "FP64 Phi+E element.point interactions/s"
UNIT = "element.point interactions/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg4", choices=["cfg4", "cfg2", "cfg3", "solve", "table3"])
    ap.add_argument("--scale", type=float, default=1.0, help="config-4 size factor (profiling only)")
    ap.add_argument("--rule", type=int, default=1, help="fixed rule level of --workload cfg2")
    ap.add_argument("--precision", default="f64", choices=["f64", "f32"], help="--workload cfg2 only")
    ap.add_argument("--gradient", action="store_true",
                    help="also compute the field gradient (bemcub_eval_gradient; cubature levels only) - not the bench line")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


# --------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""

    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu = gpu_index
        self.proc = None
        self.lines = []
        self.thread = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200",
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
def make_workload(args, rank: int):
    """Seeded synthetic inputs.  Rank r > 0 draws its own field points."""
    from paper_1606_03743_b200 import synth
    if args.workload == "cfg4":
        c = synth.config4(scale=args.scale)
        if rank > 0:  # weak scaling: same mesh, another 10^6 track points per rank
            c["pts"] = synth.helical_tracks(c["ntracks"], c["npts_per_track"], seed=synth.SEED_CFG4_TRACKS + 1000 * rank)
        c["rule"] = -1
        c["desc"] = ("config 4: cylinder R=5 m L=20 m (%d rectangles) + two end cones (%d triangles), sigma = 8 "
                     "Fourier modes, %d helical-track field points, DR-adaptive rules, Phi+E"
                     % (int((c["etype"] == 1).sum()), int((c["etype"] == 0).sum()), len(c["pts"])))
    elif args.workload == "cfg2":
        c = synth.config2()
        c["rule"] = args.rule
        c["desc"] = "config 2: unit-cube surface 6144 squares, 10^4 field points, fixed rule level %d, %s" % (
            args.rule, args.precision)
    elif args.workload == "table3":
        # the SHAPE of the paper's GPU timing (Table 3: 1.5 M rectangles, 10^4 field points) on a
        # synthetic cylinder; --rule 1 = the 7-point rule, --rule -1 = distance-ratio dependent
        et, vt = synth.cylinder_rects(5.0, -10.0, 10.0, 1500, 1000)
        c = dict(etype=et, verts=vt, sigma=synth.fourier_sigma(synth.element_centroids(et, vt)),
                 pts=synth.helical_tracks(100, 100), rule=args.rule)
        c["desc"] = ("Table-3 shape: cylinder of 1.5e6 rectangles, 1e4 helical-track field points, rule %s, Phi+E"
                     % ("adaptive" if args.rule == -1 else "level %d" % args.rule))
    elif args.workload == "solve":
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
    return c


def oracle_rate(c, args, target_seconds: float, min_pts: int = 8, max_pts: int = 65536):
    """Times the CPU oracle (double-precision instantiation, OpenMP over field points, all host
    cores, as it stands) on a bounded seeded sample of the workload's field points / matrix rows.
    Returns (units per second, cores, sample description, seconds, sampled units)."""
    import oracle
    cores = oracle.num_threads()
    n = len(c["etype"])
    rng = np.random.default_rng(160603751)
    if args.workload == "cfg3":
        dr = oracle.default_policy(False)
        run = lambda idx: oracle.assemble_rows(c["etype"], c["verts"], idx, dr)
        total = n
    else:
        dr = oracle.default_policy(True)
        run = lambda idx: oracle.evaluate(c["etype"], c["verts"], c["sigma"], c["pts"][idx], c["rule"], dr=dr,
                                          precision="double")
        total = len(c["pts"])
    probe = min(total, max(min_pts, 4 * cores))
    idx = np.sort(rng.choice(total, probe, replace=False))
    t0 = time.perf_counter()
    run(idx)
    t_probe = time.perf_counter() - t0
    k = int(min(max_pts, total, max(probe, probe * target_seconds / max(t_probe, 1e-6))))
    k = max(cores, k // cores * cores)
    idx = np.sort(rng.choice(total, min(k, total), replace=False))
    t0 = time.perf_counter()
    run(idx)
    dt = time.perf_counter() - t0
    what = "matrix rows" if args.workload == "cfg3" else "field points"
    sample = f"all {n} elements x {len(idx)} seeded {what} of the workload, oracle double-precision path, {cores} OpenMP threads"
    return n * len(idx) / dt, cores, sample, dt, len(idx)


def run_reference(args, rank: int):
    """--impl reference: the oracle as it stands on the host cores, rank 0 only."""
    if rank != 0:
        return
    c = make_workload(args, 0)
    # each step a bounded sample (~4 s) so that warmup + steps end within a few minutes
    rate0, cores, sample, dt, k = oracle_rate(c, args, target_seconds=4.0)
    import oracle
    n = len(c["etype"])
    rng = np.random.default_rng(160603752)
    total = n if args.workload == "cfg3" else len(c["pts"])
    dr = oracle.default_policy(args.workload != "cfg3")

    def step():
        idx = np.sort(rng.choice(total, k, replace=False))
        if args.workload == "cfg3":
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
    unit = UNIT if args.workload != "cfg3" else "matrix entries/s"
    line = {
        "impl": "reference", "metric": METRIC if args.workload != "cfg3" else "FP64 collocation-matrix entries/s",
        "value": value, "unit": unit, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": c["desc"], "elements": n, "sampled_units_per_step": k},
        "cpu_baseline": {"value": value, "unit": unit, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": unit, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------------
def run_ours(args, rank: int, world: int, local_rank: int):
    import torch
    import torch.distributed as dist
    from paper_1606_03743_b200 import bemcub as b   # fails loudly if libbemcub.so is missing

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the bemcub path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    c = make_workload(args, rank)
    n, m = len(c["etype"]), len(c["pts"])
    is_matrix = args.workload in ("cfg3", "solve")
    is_solve = args.workload == "solve"
    precision = b.F32 if (args.workload == "cfg2" and args.precision == "f32") else b.F64

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    ctx = b.Context(local_rank)
    h = ctx.handle
    # pinned host copies (the e2e leg reads them), device-resident copies (the kernel-only leg)
    h_type = torch.as_tensor(c["etype"]).pin_memory()
    h_verts = torch.as_tensor(c["verts"]).pin_memory()
    h_sigma = torch.as_tensor(np.ascontiguousarray(c["sigma"])).pin_memory()
    h_pts = torch.as_tensor(c["pts"]).pin_memory()
    d_type, d_verts = h_type.to(dev), h_verts.to(dev)
    d_sigma, d_pts = h_sigma.to(dev), h_pts.to(dev)
    b.bemcub_set_elements(h, n, d_type, d_verts)
    solve_info = {}
    if is_solve:
        pol = b.bemcub_default_policy(False)
        d_V = torch.ones(n, dtype=torch.float64, device=dev)
        d_s = torch.zeros(n, dtype=torch.float64, device=dev)

        def step():
            d_s.zero_()
            mv, res, ok = b.bemcub_solve(h, pol, d_V, d_s, 1e-12, 500)
            solve_info.update(matvecs=mv, rel_residual=res, converged=ok)
    elif is_matrix:
        pol = b.bemcub_default_policy(False)
        out = torch.empty((n, n), dtype=torch.float64, device=dev)
        step = lambda: b.bemcub_assemble(h, pol, out, n)
    else:
        pol = b.bemcub_default_policy(True) if c["rule"] == -1 else None
        phi = torch.empty(m, dtype=torch.float64, device=dev)
        E = torch.empty((m, 3), dtype=torch.float64, device=dev)
        if args.gradient:
            if pol is not None:
                pol.use_levels_mask = 0b011111          # derivatives exist for the point charges only (L273)
            G = torch.empty((m, 6), dtype=torch.float64, device=dev)
            step = lambda: b.bemcub_eval_gradient(h, d_sigma, c["rule"], pol, m, d_pts, phi, E, G)
        else:
            step = lambda: b.bemcub_eval(h, d_sigma, c["rule"], pol, m, d_pts, phi, E, precision)

    # roofline denominator: sustained DFMA rate of this GPU, measured in this run
    dfma_per_s = b.bemcub_fp64_peak(h, 2.0)
    peak_tflops = 2.0 * dfma_per_s / 1e12
    # second reference: the kernels' own inner loop on resident data (what the 18-instruction mix allows)
    loop_rate = b.bemcub_inner_loop_rate(h, 1.0)

    b.bemcub_set_timing(h, True)
    for _ in range(args.warmup):
        step()
    barrier()
    b.bemcub_reset_stats(h)
    sampler = ClockSampler(local_rank)
    sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    kernel_ms = []
    ev0.record()
    for _ in range(args.steps):
        step()
        kernel_ms.append(b.bemcub_get_timing(h)[1])   # waits for this step's events only
    ev1.record()
    barrier()
    clocks = sampler.stop()
    st = b.bemcub_get_stats(h)
    ms = ev0.elapsed_time(ev1) / max(args.steps, 1)
    t = torch.tensor([ms], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_max = float(t.item())
    units_per_step = float(n) * float(n if is_matrix else m) * (solve_info.get("matvecs", 1) if is_solve else 1)
    if is_solve:
        areas = 0.5 * np.linalg.norm(np.cross(c["verts"][:, 1] - c["verts"][:, 0], c["verts"][:, 2] - c["verts"][:, 0]), axis=1)
        q_tot = float((d_s.cpu().numpy() * areas).sum())
        solve_info["capacitance_over_4pi_eps0_R"] = q_tot / (4 * np.pi * 8.8541878128e-12)
    value = units_per_step * world / (ms_max * 1e-3)

    # dominant kernel against the FP64-ALU roofline
    k_ms = sum(kernel_ms) / max(len(kernel_ms), 1)
    inter = float(st["point_interactions"])          # point-charge interactions of the last step
    fpi = FLOP_PER_INTERACTION_PHI if is_matrix else (FLOP_PER_INTERACTION_GRAD if args.gradient else FLOP_PER_INTERACTION)
    ipi = 12 if is_matrix else (28 if args.gradient else 18)   # FP64 instructions per interaction
    flop = inter * fpi
    if precision == b.F32:
        roof = {"bound": "alu", "achieved": flop / (k_ms * 1e-3) / 1e12, "peak": None, "unit": "TFLOP/s", "frac": None,
                "traffic": None, "note": "FP32 variant: reported, no FP32 peak measured"}
    else:
        ach = flop / (k_ms * 1e-3) / 1e12
        # DRAM bytes of ONE launch of the dominant kernel from the committed ncu capture of this very
        # workload (profiles/r1_cfg4_full_eval_adaptive_counters.csv: 3.28 GB read + 0.55 GB written)
        traffic = 3277495040 + 549181696 if (args.workload == "cfg4" and args.scale == 1.0 and not args.gradient) else None
        roof = {"bound": "alu", "achieved": ach, "peak": peak_tflops, "unit": "TFLOP/s", "frac": ach / peak_tflops,
                "traffic": traffic, "kernel": "eval_adaptive_kernel<kModePhi>" if is_solve else "assemble_kernel" if is_matrix else
                ("eval_adaptive_kernel" if c["rule"] == -1 else "eval_fixed_kernel"),
                "kernel_ms": k_ms, "kernel_share_of_step": k_ms / ms,
                "point_interactions_per_launch": inter,
                "flop_per_interaction": fpi,
                "peak_source": "bemcub_fp64_peak: sustained all-SM DFMA-only loop (best of 16 / 32 warps per SM), 2 s, same run (x2 flop/FMA); "
                               "MEASURED_PEAKS.json has no FP64 entry",
                "fp64_pipe_frac": (inter * ipi / (k_ms * 1e-3)) / dfma_per_s,
                "inner_loop_ceiling": {"interactions_per_s": loop_rate,
                                       "frac_of_peak": loop_rate * FLOP_PER_INTERACTION / (2.0 * dfma_per_s),
                                       "kernel_over_ceiling": None if is_matrix else (inter / (k_ms * 1e-3)) / loop_rate,
                                       "source": "bemcub_inner_loop_rate: Eq. 4.1 loop (18 FP64 instr + MUFU, 8 of 18 "
                                                 "are FMAs => at most 26/36 = 72.2% of the DFMA peak), resident data"}}

    # end to end through the host-buffer C-ABI calls: H2D of the inputs, compute, D2H of Phi/E
    e2e = None
    if not args.no_e2e and not is_matrix and not args.gradient:
        o_phi = torch.empty(m, dtype=torch.float64).pin_memory()
        o_E = torch.empty((m, 3), dtype=torch.float64).pin_memory()
        ctx2 = b.Context(local_rank)

        def step_host():
            b.bemcub_set_elements_host(ctx2.handle, n, h_type, h_verts)
            b.bemcub_eval_host(ctx2.handle, h_sigma, c["rule"], pol, m, h_pts, o_phi, o_E, precision)

        step_host()
        barrier()
        t0 = time.perf_counter()
        ev0.record()
        for _ in range(args.steps):
            step_host()
        ev1.record()
        barrier()
        ms_e = ev0.elapsed_time(ev1) / max(args.steps, 1)
        t = torch.tensor([ms_e], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e = {"value": units_per_step * world / (float(t.item()) * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": int(n * 1 + n * 72 + n * 8 + m * 24), "d2h_bytes_per_step": int(m * 32),
               "ms_per_step": float(t.item()), "api": "bemcub_set_elements_host + bemcub_eval_host (pinned host buffers)"}
        assert bool(torch.isfinite(o_phi).all())
        ctx2.close()
    elif is_matrix:
        e2e = {"value": None, "unit": "matrix entries/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
               "note": "matrix stays on the device (3.36 GB); no host leg"}

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline and not is_solve:
        rate, cores, sample, dt, k = oracle_rate(c, args, target_seconds=15.0)
        cpu = {"value": rate, "unit": UNIT if not is_matrix else "matrix entries/s", "cores": cores, "kind": "oracle",
               "sample": sample, "seconds": dt}
        if not is_matrix:   # the paper's CPU numbers are single-threaded (Table 2): one thread on a smaller sample
            import oracle
            k1 = max(4, int(k / max(cores, 1) / 4))
            idx1 = np.sort(np.random.default_rng(160603753).choice(m, min(k1, m), replace=False))
            t0 = time.perf_counter()
            oracle.evaluate(c["etype"], c["verts"], c["sigma"], c["pts"][idx1], c["rule"], dr=oracle.default_policy(True),
                            precision="double", nthreads=1)
            cpu["value_single_thread"] = n * len(idx1) / (time.perf_counter() - t0)

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
                       "points_per_pair": inter / units_per_step if units_per_step else None},
            "pct_fp64_peak": 100.0 * roof["frac"] if roof.get("frac") else None,
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(st["kernel_launches"]),
            "roofline": roof, "cpu_baseline": cpu,
        }
        if is_solve:
            line["metric"] = "FP64 potential-only element.point interactions/s inside bemcub_solve"
            line["unit"] = "element.point interactions/s"
            line["solve"] = solve_info
            line["roofline"]["note"] = "kernel_ms / interactions are those of the LAST mat-vec of the solve"
        print(json.dumps(line), flush=True)
    ctx.close()


def main():
    args = parse_args()
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
