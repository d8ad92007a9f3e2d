"""bench.py's stdout contract (host only, no CUDA): ONE compact JSON line, the last thing printed, under 4 KB.

Round 2's line carried every leg of the report (21.6 KB) and the driver could not parse it; the builders are imported
here and fed a report at least that large."""
from __future__ import annotations

import io
import json

import bench


def big_report():
    filler = {f"leg{i}": {"note": "x" * 400, "values": list(range(50))} for i in range(40)}
    return {
        "metric": bench.METRIC, "value": 7367375095.335045, "unit": bench.UNIT, "n_gpus": 1, "steps": 20000, "warmup": 50,
        "ms_per_step": 0.045563473510742185, "ms_per_event": 0.045563473510742185, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": bench.WORKLOAD, "events_per_step": 1, "pool_events_per_gpu": 40, "l2": "inputs and outputs rotate " * 30,
                   "call_signature": "y" * 300, "grid": {"dims": 4, "bits": 5}, "edge_capacity": 960000,
                   "parallelism": "events sharded over 1 GPU(s), no collective"},
        "edges_per_event": 335683.2,
        "roofline": {"bound": "alu", "what": "w" * 200, "kernel": "search", "achieved": 441.93391486339436, "peak": 1163.28,
                     "unit": "Gwarp-inst/s", "frac": 0.37990330347241796, "peak_source": "148 SMs x 4 schedulers x 1965 MHz " * 10,
                     "traffic": 7616000.0, "dram_frac_of_hbm_peak": 0.0557, "kernel_us": 21.17632000000001,
                     "algorithmic_bytes_per_launch": 245368921.6, "model_frac_hbm_equivalent": 1.79,
                     "counters": "profiles/r02_counters.csv (ncu, one launch, cold cache)", "counters_stale": True,
                     "ncu_cold": {"note": "z" * 500}},
        "roofline_model": filler, "path_roofline": filler, "phases_us": filler, "timeline_us": filler, "varying_n": filler,
        "k_binding": filler, "radius_sweep": [filler], "next_rows": filler, "other_configs": filler, "two_streams": filler,
        "cpu_baseline": {"value": 4738627.7, "unit": bench.UNIT, "cores": 16, "kind": "oracle", "sample": "120 whole config-2 events " * 20,
                         "ms_per_event": 70.87, "one_thread": filler, "brute_force_mode_once": filler, "note": "n" * 300},
        "e2e": {"value": 3314918511.871542, "unit": bench.UNIT, "h2d_bytes_per_step": 3840000, "d2h_bytes_per_step": 4031096,
                "ms_per_step": 0.10133703099999991, "steps": 1000, "api": "a" * 300, "e2e_verified": True, "events_verified": 5,
                "band_report": filler, "copy_floor_ms": 0.0961, "varying_n": filler, "one_call_at_a_time": filler},
        "gpu_launches": 120000, "gpu_launches_per_step": 6,
        "clocks": {"sm_mhz": 1965.0, "sm_max_mhz": 1965, "reasons": [], "samples": 182, "how": "h" * 300},
        "host_wall_ms_per_step": 0.0455, "paper_context": "p" * 200,
    }


def test_compact_line_holds_the_contract_and_stays_small():
    full = big_report()
    assert len(json.dumps(full)) > 20000
    line = bench.compact_line(full)
    text = json.dumps(line)
    assert len(text) < bench.COMPACT_LIMIT == 4096, len(text)
    back = json.loads(text)
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
                "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "clocks", "gpu_launches"):
        assert key in back, key
    assert back["value"] > 0 and back["metric"] == bench.METRIC
    assert set(("bound", "achieved", "peak", "unit", "frac", "traffic")) <= set(back["roofline"])
    assert abs(back["roofline"]["frac"] - back["roofline"]["achieved"] / back["roofline"]["peak"]) < 1e-4
    assert back["roofline"]["counters_stale"] is True
    assert set(("value", "unit", "cores", "kind", "sample")) <= set(back["cpu_baseline"])
    assert set(("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step")) <= set(back["e2e"])
    assert set(("sm_mhz", "sm_max_mhz", "reasons")) <= set(back["clocks"])
    assert "workload" in back["config"] and "model" not in back["config"]
    for dropped in ("other_configs", "radius_sweep", "k_binding", "roofline_issue", "roofline_model"):
        assert dropped not in back
    # nothing the driver computes from the line loses more than rounding
    assert abs(back["value"] / full["value"] - 1) < 1e-5 and abs(back["ms_per_step"] / full["ms_per_step"] - 1) < 1e-5


def test_emit_prints_the_compact_line_last_and_the_full_report_elsewhere(tmp_path, monkeypatch):
    monkeypatch.setattr(bench, "ROOT", str(tmp_path))
    out, err = io.StringIO(), io.StringIO()
    text = bench.emit(big_report(), out=out, err=err, path="gpurun_out/bench_full.json")
    lines = out.getvalue().splitlines()
    assert len(lines) == 1 and lines[-1] == text and len(text) < bench.COMPACT_LIMIT
    assert json.loads(lines[-1])["full_report"] == "gpurun_out/bench_full.json"
    on_disk = json.load(open(tmp_path / "gpurun_out" / "bench_full.json"))
    assert "other_configs" in on_disk and "radius_sweep" in on_disk
    assert "other_configs" in json.loads(err.getvalue())["full_report"]


def test_counters_file_names_the_kernel_source_it_was_captured_on():
    rows, name, stale = bench.ncu_counters()
    assert rows and name.startswith("profiles/r0")
    assert ("cfg2", "search") in rows and rows[("cfg2", "search")]["warp_inst"] > 0
    assert isinstance(stale, bool)
    h = bench.blob_hash(bench.KERNELS_SOURCE)
    assert h and len(h) == 40
    import subprocess
    try:
        git = subprocess.run(["git", "hash-object", bench.KERNELS_SOURCE], capture_output=True, text=True, cwd=bench.ROOT)
    except OSError:
        return
    if git.returncode == 0:
        assert git.stdout.strip() == h
