"""bench.py's stdout record (no GPU): the driver keeps a tail of stdout and parses ONE JSON line from it.
Round 2's line had grown to 20 KB (peak sweep, definitions, secondary rooflines) and did not parse; the
record is now built by bench.contract_line from the full record, which goes to a side file.  Canned
numbers of the size and shape of a real config-4 run."""
import json

import bench


def _full_record():
    sweep = [{"mix": "mix 8 DFMA : 6 DMUL : 4 DADD", "warps_per_sm": w, "fp64_inst_per_s": 1.85e13, "sm_mhz": 1965.0,
              "of_nominal": 0.995} for _ in range(6) for w in (8, 16, 32)]
    peak = {"fp64_inst_per_s": 1.852e13, "tflops": 37.04, "best": "DFMA, 16 warps/SM", "sm_mhz": 1965.0, "sweep": sweep,
            "source": "bemcub_fp64_issue_sweep in this run: max FP64 instruction issue rate over 6 mixes x 3 occupancies, "
                      "0.20 s each (x2 flop per instruction); MEASURED_PEAKS.json has no FP64 entry"}
    inter, own = 7.629e12, 7.381e12
    roof = bench.roofline_block("eval_paired_kernel", 7181.6, 7185.6, inter, own, bench.FLOP_PER_INTERACTION, 14.92, peak, 148,
                                1964.8, 1965.0)
    roof["peak_sweep"] = sweep
    roof["inner_loop_ceiling"] = {"interactions_per_s": 1.03e12, "source": "x" * 200}
    roof["paired_form"] = "y" * 400
    roof["traffic"] = 4696823808.0
    roof["traffic_source"] = "dram__bytes_read.sum + dram__bytes_write.sum of one launch, committed ncu capture " + "z" * 120
    roof["fp64_pipe_pct_ncu"] = 85.51
    sec_roof = bench.roofline_block("eval_fixed_kernel", 0.66, 0.7, 4.3e8, 4.3e8, 26, 18, peak, 148, 1960.0, 1965.0)
    secondary = [{"name": "cfg2 rule level %d f64" % i, "workload": "config %d: " % i + "w" * 150, "dtype": "f64", "ms_per_step": 0.7, "kernel_ms": 0.66,
                  "value": 8.7e10, "unit": bench.UNIT, "clocks": {"sm_mhz": 1965.0, "reasons": []}, "roofline": dict(sec_roof),
                  "cpu_baseline": {"value": 1e8, "sample": "s" * 200}} for i in range(7)]
    return {
        "metric": bench.METRIC, "value": 1.3916e11, "unit": bench.UNIT, "n_gpus": 1, "steps": 20, "warmup": 5,
        "ms_per_step": 7185.6, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": "config 4: " + "c" * 300, "elements": 1000000, "field_points_per_gpu": 1000000,
                   "parallelism": "field points sharded over 1 GPU(s), no collective", "l2": "inputs larger than L2 " + "l" * 100,
                   "points_per_pair": 7.629, "points_per_pair_own_work": 7.381},
        "pct_fp64_peak": 100.0 * roof["frac"],
        "clocks": {"sm_mhz": 1965.0, "sm_max_mhz": 1965.0, "power_w_max": 736.2, "samples": 700, "reasons": []},
        "e2e": {"value": 1.391e11, "unit": bench.UNIT, "h2d_bytes_per_step": 105000000, "d2h_bytes_per_step": 32000000,
                "ms_per_step": 7189.0, "api": "bemcub_set_elements_host + bemcub_eval_host (pinned host buffers)"},
        "gpu_launches": 260, "roofline": roof,
        "cpu_baseline": {"value": 9.95e7, "unit": bench.UNIT, "cores": 16, "threads_busy": 16, "kind": "oracle",
                         "sample": "all 1000000 elements x 192 seeded field points of the workload, " + "o" * 150,
                         "seconds": 15.2, "units": 192, "value_single_thread": 7.1e6},
        "secondary": secondary,
    }


def test_stdout_record_is_compact_and_complete():
    full = _full_record()
    assert len(json.dumps(full)) > 3 * bench.LINE_LIMIT           # the shape that broke round 2
    line = bench.contract_line(full, "gpurun_out/bench_detail.json")
    text = json.dumps(line)
    assert len(text) < bench.LINE_LIMIT, len(text)
    assert "\n" not in text
    back = json.loads(text)
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline"):
        assert key in back, key
    assert back["value"] > 0 and back["config"]["workload"].startswith("config 4")
    for key in ("bound", "achieved", "peak", "unit", "frac", "traffic", "kernel", "kernel_ms", "frac_executed", "fp64_issue_frac"):
        assert key in back["roofline"], key
    for key in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step"):
        assert key in back["e2e"], key
    for key in ("value", "unit", "cores", "kind", "sample"):
        assert key in back["cpu_baseline"], key
    assert "peak_sweep" not in back["roofline"] and "inner_loop_ceiling" not in back["roofline"]
    assert len(text) < 3400, len(text)                                # headroom for longer numbers / names
    assert len(back["secondary"]) == 7 and set(back["secondary"][0]) == {"name", "ms_per_step", "value", "frac"}


def test_roofline_frac_is_the_methods_own_work():
    """achieved = algorithmic flop / kernel time: 26 flop per point-charge interaction of the
    per-pair policy; upgraded tiles (executed > own) and the paired form's shorter instruction sequence do not enter."""
    full = _full_record()
    r = full["roofline"]
    assert abs(r["achieved"] - 7.381e12 * 26 / 7.1816 / 1e12) < 1e-9
    assert abs(r["frac"] - r["achieved"] / 37.04) < 1e-12 and 0.72 < r["frac"] < 0.7225
    assert abs(r["frac_executed"] - 7.629e12 * 26 / 7.1816 / 1e12 / 37.04) < 1e-12 and r["frac_executed"] > r["frac"]
    assert abs(r["fp64_issue_frac"] - 7.629e12 * 14.92 / 7.1816 / 1.852e13) < 1e-12
    assert abs(full["pct_fp64_peak"] - 100 * r["frac"]) < 1e-12


def test_a_record_that_would_not_fit_drops_its_optional_parts(monkeypatch):
    full = _full_record()
    full["secondary"] = full["secondary"] * 6            # 42 rows: contract_line keeps 8
    full["config"]["extra"] = "e" * 3000                  # an oversized field somebody adds later: clipped
    line = bench.contract_line(full)
    assert len(line["secondary"]) == 8 and len(json.dumps(line)) < bench.LINE_LIMIT
    monkeypatch.setattr(bench, "LINE_LIMIT", 2500)
    line = bench.contract_line(full)
    assert "secondary" not in line and "value" in line and "roofline" in line and len(json.dumps(line)) < 2500


def test_committed_ncu_capture_is_readable():
    cap = bench.ncu_capture("cfg4", "eval_paired_kernel")
    assert cap and cap["metrics"]["dram__bytes_read.sum"] > 0 and cap["metrics"]["dram__bytes_write.sum"] > 0
    assert 50.0 < cap["metrics"][bench.NCU_PIPE_METRIC] <= 100.0
    assert bench.ncu_capture("cfg4", "eval_adaptive_kernel") is None
