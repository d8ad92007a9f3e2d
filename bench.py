#!/usr/bin/env python
"""bench.py -- FRNN graph building at tracking scale (BASELINE.json: 120k hits, D=8, r=0.1, K=256).

One "step" = one pass of the whole hot path (S2..S10: bin, cell scan, scatter, search, degree scan + emit)
over ONE seeded synthetic event of config 2 through the C ABI (frnn_build_ex) on a non-default
stream.  Steps rotate over a pool of distinct events and distinct output buffers whose total size
exceeds the 126 MB L2, so every step reads its input cold from HBM and every call differs from the previous one
in its pointers (the library rewrites the graph's node parameters every step: nothing is a replay of an identical call).

Prints ONE compact JSON line (rank 0) as the last thing on stdout: the contract keys only (metric, value, config,
roofline, cpu_baseline, e2e, clocks, gpu_launches; under 4 KB -- the round-2 line carried every leg, grew to 21.6 KB
and the driver could not read it).  The FULL report goes to gpurun_out/bench_full.json and, as one line, to stderr:
  roofline      the dominant kernel against the bound that actually binds it: warp instructions per launch (committed
                ncu counters, profiles/r0N_counters.csv; `counters_stale` says whether they belong to the kernel source
                in the tree) / its in-graph duration vs the issue peak 148 SMs x 4 schedulers x measured SM clock
                ("bound": "alu"); `traffic` = measured DRAM bytes of that launch, `dram_frac_of_hbm_peak` their rate
                against MEASURED_PEAKS.json; `model_frac_hbm_equivalent` = north_star's byte model (not physical)
  roofline_model  north_star's figure for the same kernel: candidate-row bytes of the grid run / duration vs the measured
                HBM peak.  These bytes are served by L2/L1: an HBM-EQUIVALENT rate, not a physical fraction (can exceed 1)
  path_roofline north_star's whole-path figure: (candidate rows * 32 B + 12 B * edges) / ms_per_event
  varying_n     every step a different n in [90k, 120k] and different buffers, through frnn_build_ex and through the
                host pipeline; cost of a cold first call
  k_binding     the K cap when it binds (config 2 at K = 2, 4, 16; one cluster; a dense event of mean degree ~170)
  radius_sweep  config-2 recipe at r = 0.02 .. 0.2 with the grid frnn_suggest_grid picks, beside the default grid
  cpu_baseline  the oracle (cell-list mode) on this box's host cores on a bounded sample, all cores and one thread;
                brute-force mode once on configs 0-2
  e2e           the same metric through frnn_host_pipeline_*: pinned host buffers, H2D + D2H inside; a bare-copy floor
                (the same bytes, no build) beside it; events of the timed loop checked against the oracle
`--impl reference` times the oracle alone (rank 0 only) on the same metric/config.
`--legs a,b,..` restricts the run to some legs (for ncu captures): headline is always run.
"""
from __future__ import annotations

import argparse
import csv
import dataclasses
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2202_06929_b200 import events  # noqa: E402

CFG = events.CONFIGS[2]
METRIC = "frnn_edges_per_s_120k_hits_d8"
UNIT = "edges/s"
WORKLOAD = "configs[2]: single event N=120000 D=8 fp32, 11000 tracks Poisson(10), sigma 0.03, 8% noise, r=0.1, K=256"
POOL = 40                      # 40 x 3.84 MB inputs = 154 MB > 126 MB L2 (+ 40 x 11.5 MB outputs)
EDGE_CAP_PER_ROW = 8           # output room: 8 edges per row (mean degree is 2.8; overflow is reported, not fatal)
FALLBACK_HBM_GBS = 6650.0      # /opt/skills/guides/B200_PROFILING.md fallback
N_SMS, SCHEDULERS_PER_SM = 148, 4
ALL_LEGS = ("varying_n", "two_streams", "phases", "timeline", "k_binding", "radius_sweep", "next", "other", "e2e", "cpu")


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            j = json.load(f)
        return float(j["hbm_gbs"]), float(j.get("sm_max_mhz", 1965.0)), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return FALLBACK_HBM_GBS, 1965.0, "fallback (B200_PROFILING.md)"


KERNELS_SOURCE = os.path.join(ROOT, "paper_2202_06929_b200", "csrc", "frnn_kernels.cuh")
COUNTER_FILES = ("r03_counters.csv", "r02_counters.csv")      # the newest capture that is committed wins
FULL_REPORT = os.path.join("gpurun_out", "bench_full.json")   # every leg in full; the stdout line holds the contract keys only
COMPACT_LIMIT = 4096                                           # bytes; tests/test_bench_line.py holds the line to it


def blob_hash(path: str) -> str | None:
    """What `git hash-object <path>` prints (sha1 of "blob <size>\\0" + content); None if the file is absent."""
    import hashlib
    try:
        data = open(path, "rb").read()
    except OSError:
        return None
    return hashlib.sha1(b"blob %d\0" % len(data) + data).hexdigest()


def ncu_counters():
    """profiles/r0N_counters.csv: per (workload, kernel) the ncu figures of ONE launch (see the .md beside it).
    Returns (rows, file name, stale): `stale` says that the kernel source the counters were captured on (column
    `kernels_blob` = git hash-object of csrc/frnn_kernels.cuh at capture time) is not the one in the tree now."""
    for name in COUNTER_FILES:
        out, blobs = {}, set()
        try:
            with open(os.path.join(ROOT, "profiles", name)) as f:
                for row in csv.DictReader(f):
                    blobs.add(row.get("kernels_blob") or "")
                    out[(row["workload"], row["kernel"])] = {k: float(v) for k, v in row.items()
                                                             if k not in ("workload", "kernel", "profile", "kernels_blob")}
        except Exception:
            continue
        if out:
            return out, "profiles/" + name, blobs != {blob_hash(KERNELS_SOURCE)}
    return {}, None, True


def _round(v, digits=8):
    """Floats to `digits` significant digits (the compact line is for reading and parsing, the full report keeps everything)."""
    if isinstance(v, float):
        return float(f"{v:.{digits}g}")
    if isinstance(v, dict):
        return {k: _round(x, digits) for k, x in v.items()}
    if isinstance(v, (list, tuple)):
        return [_round(x, digits) for x in v]
    return v


def _pick(d, keys):
    return {k: d[k] for k in keys if isinstance(d, dict) and k in d}


def _short(text, limit=160):
    return text if not isinstance(text, str) or len(text) <= limit else text[: limit - 3] + "..."


def compact_line(full: dict) -> dict:
    """The ONE stdout line: the keys of the bench contract and nothing else (the round-2 line carried every leg, grew to
    21.6 KB and the driver could not read it).  Everything else stays in the full report (FULL_REPORT, stderr)."""
    line = _pick(full, ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                        "vs_baseline", "dtype", "data", "impl", "gpu_launches", "gpu_launches_per_step", "edges_per_event"))
    cfg = _pick(full.get("config"), ("workload", "events_per_step", "pool_events_per_gpu", "l2", "grid", "edge_capacity", "parallelism", "sample"))
    line["config"] = {k: _short(v) for k, v in cfg.items()}
    if full.get("roofline"):
        line["roofline"] = _pick(full["roofline"], ("bound", "kernel", "achieved", "peak", "unit", "frac", "traffic", "peak_source", "kernel_us",
                                                    "dram_frac_of_hbm_peak", "algorithmic_bytes_per_launch", "own_bytes_per_launch",
                                                    "model_frac_hbm_equivalent", "counters", "counters_stale"))
        line["roofline"]["peak_source"] = _short(line["roofline"].get("peak_source"), 120)
    if full.get("cpu_baseline"):
        line["cpu_baseline"] = _pick(full["cpu_baseline"], ("value", "unit", "cores", "kind", "sample", "ms_per_event"))
        line["cpu_baseline"]["sample"] = _short(line["cpu_baseline"].get("sample"))
    if full.get("e2e"):
        line["e2e"] = _pick(full["e2e"], ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step", "ms_per_step", "steps", "copy_floor_ms",
                                          "e2e_verified", "events_verified"))
    if full.get("clocks"):
        line["clocks"] = _pick(full["clocks"], ("sm_mhz", "sm_max_mhz", "reasons", "samples"))
    if "full_report" in full:
        line["full_report"] = full["full_report"]
    return _round(line)


def emit(full: dict, out=None, err=None, path: str | None = FULL_REPORT) -> str:
    """Full report to `path` (if it can be written) and to stderr, then the compact line as the LAST thing on stdout."""
    out, err = out or sys.stdout, err or sys.stderr
    full = dict(full)
    if path:
        try:
            os.makedirs(os.path.dirname(os.path.join(ROOT, path)) or ".", exist_ok=True)
            with open(os.path.join(ROOT, path), "w") as f:
                json.dump(full, f)
            full["full_report"] = path
        except OSError:
            full["full_report"] = "stderr"
    else:
        full["full_report"] = "stderr"
    print(json.dumps({"full_report": full}), file=err, flush=True)
    text = json.dumps(compact_line(full))
    print(text, file=out, flush=True)
    return text


def candidate_rows(x: np.ndarray, r: float, dims: int, bits: int) -> int:
    """ACCOUNTING ONLY (not on the product path): sum over queries of the rows in the 3^dims cells
    around the query's cell, for the grid the library reports it runs (cell side r*(1+2^-7),
    toroidal extent 2^bits, the first `dims` coordinates).  This is the 'bytes of candidate rows' of north_star / 32."""
    from scipy.ndimage import convolve1d
    m = 1 << bits
    side = float(np.float32(r) * np.float32(1.0078125))
    c = np.floor(x[:, :dims].astype(np.float64) / side).astype(np.int64) & (m - 1)
    lin = np.zeros(len(x), np.int64)
    for d in range(dims):
        lin = lin * m + c[:, d]
    occ = np.bincount(lin, minlength=m ** dims).reshape((m,) * dims).astype(np.int64)
    nb = occ
    for ax in range(dims):
        nb = convolve1d(nb, np.ones(3, np.int64), axis=ax, mode="wrap")
    return int(nb.reshape(-1)[lin].sum())


REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
           0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x100: "display_clock_setting"}


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons with NVML while the timed region runs; `sample_now` takes one reading
    synchronously (called right before and right after the timed loop, so that a short run still has a clock record)."""

    def __init__(self, uuid: str | None, index: int, period_s: float = 0.005):
        super().__init__(daemon=True)
        self.period, self.samples, self.stop_flag = period_s, [], False
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            try:
                self.h = pynvml.nvmlDeviceGetHandleByUUID(uuid)
            except Exception:
                self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.max_mhz = None

    def sample_now(self):
        if not self.ok:
            return
        try:
            mhz = self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM)
            reasons = self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
            self.samples.append((time.perf_counter(), mhz, reasons))
        except Exception:
            pass

    def run(self):
        while self.ok and not self.stop_flag:
            self.sample_now()
            time.sleep(self.period)

    def summary(self, t0: float, t1: float) -> dict:
        sel = [s for s in self.samples if t0 <= s[0] <= t1] or self.samples[-3:]
        if not sel:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0}
        mask = 0
        for s in sel:
            mask |= s[2]
        return {"sm_mhz": float(np.median([s[1] for s in sel])), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(n for b, n in REASONS.items() if mask & b), "samples": len(sel),
                "how": "NVML: one reading while the warm-up steps are in flight, one right after the last timed step was submitted (GPU busy at both), and every 5 ms in between"}


def oracle_sample_run(n_events: int, threads: int = 0):
    """The oracle as it stands (cell-list mode) on whole events of the workload."""
    import oracle
    total_e, total_t, used = 0, 0.0, 0
    for s in range(n_events):
        x = events.make_event(CFG, 1000 + s)
        t = time.perf_counter()
        res = oracle.frnn(x, CFG.r, CFG.k_max, oracle.CELLS, threads=threads)
        total_t += time.perf_counter() - t
        total_e += res.count
        used = res.threads
    return total_e, total_t, used


def run_reference(args, rank) -> None:
    """--impl reference: the CPU oracle (as it stands, cell-list mode) on the same metric.

    Each step is a bounded sample of the workload: a slab of one config-2 event along coordinate 0
    (queries = the rows inside the slab, candidates = those rows plus a halo of one radius on each
    side, so every query sees exactly the neighbours it has in the whole event).  The slab width is
    sized from one calibration run so that the K+W steps end within about two minutes; with few
    steps the slab is the whole event."""
    if not rank.is_main:
        return
    import oracle
    x = events.make_event(CFG, CFG.seed0)
    t = time.perf_counter()
    full = oracle.frnn(x, CFG.r, CFG.k_max, oracle.CELLS)
    t_event = time.perf_counter() - t
    frac = min(1.0, 120.0 / ((args.steps + args.warmup) * t_event))
    order = np.argsort(x[:, 0], kind="stable")
    xs = x[order]
    rows = max(int(frac * CFG.n), 64)
    n_slabs = max(CFG.n // rows, 1)
    edges, elapsed, threads, cand_rows = 0, 0.0, full.threads, 0
    for step in range(args.warmup + args.steps):
        lo = (step % n_slabs) * rows
        hi = min(lo + rows, CFG.n)
        c_lo = np.searchsorted(xs[:, 0], xs[lo, 0] - 1.01 * CFG.r, "left")
        c_hi = np.searchsorted(xs[:, 0], xs[hi - 1, 0] + 1.01 * CFG.r, "right")
        sub = np.ascontiguousarray(xs[c_lo:c_hi])
        q = np.arange(lo - c_lo, hi - c_lo, dtype=np.int64)
        t = time.perf_counter()
        res = oracle.frnn(sub, CFG.r, CFG.k_max, oracle.CELLS, queries=q)
        dt = time.perf_counter() - t
        if step >= args.warmup:
            edges += res.count
            elapsed += dt
            cand_rows += len(sub)
    value = edges / elapsed
    sample = (f"per step: a slab of {rows} query rows ({100.0 * rows / CFG.n:.1f}% of one config-2 event) along coordinate 0 "
              f"with a one-radius halo (mean {cand_rows / max(args.steps, 1):.0f} candidate rows), cell-list mode")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * elapsed / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": {"workload": WORKLOAD, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0, "whole_event_ms": 1e3 * t_event,
    }
    print(json.dumps(line), flush=True)


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20000)
    ap.add_argument("--warmup", type=int, default=50)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--pool", type=int, default=POOL)
    ap.add_argument("--legs", default="all", help="comma-separated subset of: " + ",".join(ALL_LEGS) + " (or all / none)")
    ap.add_argument("--cpu-events", type=int, default=120, help="events the cpu_baseline leg runs the oracle on (all cores)")
    ap.add_argument("--e2e-steps", type=int, default=1000)
    ap.add_argument("--varying-steps", type=int, default=4000)
    ap.add_argument("--profile-steps", type=int, default=200)
    ap.add_argument("--timeline-steps", type=int, default=100)
    ap.add_argument("--two-stream-steps", type=int, default=4000, help="steps of the two-events-in-flight throughput figure")
    ap.add_argument("--other-reps", type=int, default=50, help="repetitions for the other configs / N sweep / K and radius legs")
    ap.add_argument("--next-steps", type=int, default=300, help="timed repetitions of the two edge-list consumers")
    ap.add_argument("--other-configs", default="0,1,3,4,sweep", help="which parts of the `other` leg run (for ncu captures of one config)")
    ap.add_argument("--k-cases", default="config2,cluster,dense", help="which cases of the k_binding leg run (for ncu captures of one case)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    legs = set(ALL_LEGS) if args.legs == "all" else set(v for v in args.legs.split(",") if v and v != "none")
    assert legs <= set(ALL_LEGS), f"unknown leg in {legs}"
    if args.no_cpu_baseline:
        legs.discard("cpu")

    import torch
    from paper_2202_06929_b200 import dist as D

    if args.impl == "reference":
        rank = D.Rank(int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")))
        run_reference(args, rank)
        return

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the FRNN path has no CPU fallback")
    rank = D.init_from_env()
    torch.cuda.set_device(rank.local_rank)
    dev = torch.device("cuda", rank.local_rank)
    from paper_2202_06929_b200 import frnn as F
    import ctypes as C
    L = F.lib()

    n, k_max, r = CFG.n, CFG.k_max, CFG.r
    cap = n * EDGE_CAP_PER_ROW
    seeds = D.shard(list(range(args.pool * rank.world_size)), rank)       # events sharded round-robin across ranks
    host_events = [events.make_event(CFG, s) for s in seeds]
    stream = torch.cuda.Stream(dev)

    # ---- cost of a cold first call (graph build) on a fresh workspace, then of a second call with other buffers
    cold = {}
    p0 = torch.from_numpy(host_events[0]).to(dev)
    w_cold = F.Workspace(n, 1, k_max, cap, dev)
    torch.cuda.synchronize()
    for name in ("first_call_ms", "second_call_ms"):
        t = time.perf_counter()
        F.frnn_build_ex(p0, r, k_max, ws=w_cold, stream=stream)
        stream.synchronize()
        cold[name] = 1e3 * (time.perf_counter() - t)
    cold["note"] = ("host wall clock from the call to the end of the stream: first call on a new workspace (graph built and instantiated) "
                    "and the call after it (node parameters rewritten, graph replayed); includes module loading on the very first call of the process")
    del w_cold

    pts = [torch.from_numpy(x).to(dev) for x in host_events]
    outs = [F.Workspace(n, 1, k_max, cap, dev) for _ in seeds]
    shared = outs[0].buf                                                 # scratch is reused; only outputs rotate
    for w in outs[1:]:
        w.buf = shared
    call_args = [(C.c_void_p(p.data_ptr()), n, 8, C.c_float(r), k_max, C.c_void_p(w.src.data_ptr()), C.c_void_p(w.dst.data_ptr()),
                  C.c_void_p(w.d2.data_ptr()), cap, C.c_void_p(w.count.data_ptr()), C.c_void_p(w.status.data_ptr()), None,
                  C.c_void_p(shared.data_ptr()), shared.numel(), C.c_void_p(stream.cuda_stream)) for p, w in zip(pts, outs)]
    build_ex = L.frnn_build_ex

    def step(i: int):
        st = build_ex(*call_args[i % len(call_args)])
        if st != 0:
            raise RuntimeError(F.frnn_status_string(st))

    # one validated pass over the pool: per-event edge counts and status
    for i in range(len(call_args)):
        step(i)
    stream.synchronize()
    edges_per_event = [int(w.count.item()) for w in outs]
    assert all(int(w.status.item()) == 0 for w in outs), "edge capacity exceeded"
    launches_per_step = F.frnn_last_launch_count()

    try:
        uuid = "GPU-" + str(torch.cuda.get_device_properties(dev).uuid)
    except Exception:
        uuid = None
    sampler = ClockSampler(uuid, rank.local_rank)
    sampler.start()
    with torch.cuda.stream(stream):
        t_clk0 = time.perf_counter()
        for i in range(args.warmup):
            step(i)
        sampler.sample_now()                          # clocks under load, taken OUTSIDE the timed region: the warm-up steps are in flight
        stream.synchronize()
        D.barrier(rank)
        torch.cuda.synchronize()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        ev0.record(stream)
        for i in range(args.steps):                   # nothing but the calls between the two events: a synchronous NVML reading
            step(i)                                   # inside this loop would leave the GPU idle for longer than a 20-step run lasts
        ev1.record(stream)
        sampler.sample_now()                          # the last steps are still in flight
        torch.cuda.synchronize()
        t1 = time.perf_counter()
        D.barrier(rank)
    sampler.stop_flag = True
    ms_local = ev0.elapsed_time(ev1)
    my_edges = sum(edges_per_event[i % len(edges_per_event)] for i in range(args.steps))
    ms = D.reduce_max(ms_local, rank)
    total_edges = D.reduce_sum(my_edges, rank)
    value = total_edges / (ms * 1e-3)
    ms_per_step = ms / args.steps
    clocks = sampler.summary(t_clk0, t1)
    e_mean_all = float(np.mean(edges_per_event))
    peak, sm_max_mhz, peak_src = measured_peaks()
    sm_mhz = clocks.get("sm_mhz") or sm_max_mhz
    issue_peak = N_SMS * SCHEDULERS_PER_SM * sm_mhz * 1e6          # warp instructions per second

    def timed(fn, reps, warm=5):
        """mean ms per call of fn(i) on `stream`, CUDA events around `reps` back-to-back calls"""
        with torch.cuda.stream(stream):
            for i in range(warm):
                fn(i)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            for i in range(reps):
                fn(i)
            b.record(stream)
            stream.synchronize()
        return a.elapsed_time(b) / reps

    # ---- every step a different n and different buffers (events differ in size)
    varying = None
    if "varying_n" in legs:
        rng = np.random.default_rng(12345)
        n_lo = 90000
        steps_v = args.varying_steps
        sizes = rng.choice(np.arange(n_lo, n + 1), size=min(steps_v, n + 1 - n_lo), replace=False)     # all distinct
        v_args = []
        for i in range(steps_v):
            a = call_args[i % len(call_args)]
            v_args.append((a[0], int(sizes[i % len(sizes)])) + a[2:])
        for i in range(min(200, steps_v)):                          # warm-up (and the edge counts of these sizes are not needed)
            assert build_ex(*v_args[i]) == 0
        stream.synchronize()
        a_, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        tw = time.perf_counter()
        a_.record(stream)
        for i in range(steps_v):
            st = build_ex(*v_args[i])
            assert st == 0
        b_.record(stream)
        stream.synchronize()
        tw = time.perf_counter() - tw
        ms_v = a_.elapsed_time(b_) / steps_v
        mean_n = float(np.mean([v[1] for v in v_args]))
        # the same stream of sizes, but every size replayed on the fixed-N path for comparison: per-point time
        varying = {"ms_per_event": ms_v, "steps": steps_v, "distinct_n": int(len(set(v[1] for v in v_args))),
                   "n_range": [n_lo, n], "mean_n": mean_n, "distinct_buffer_sets": len(call_args),
                   "host_wall_ms_per_event": 1e3 * tw / steps_v,
                   "vs_fixed_n": ms_v / ms_per_step, "launches_per_call": F.frnn_last_launch_count(),
                   "cold_first_call": cold,
                   "note": "frnn_build_ex, one stream, one workspace; every call has its own n (a prefix of a pool event: the rows of an "
                           "event are permuted, so a prefix is an event of the same recipe with fewer hits) and other in/out buffers"}

    # throughput with two events in flight (two streams, two scratch workspaces): the fixed latency of one event's six
    # dependent graph nodes overlaps the other event's work.  Reported beside the headline, which stays one stream.
    two_streams = None
    if "two_streams" in legs and args.two_stream_steps > 0:
        def in_flight(n_streams: int) -> float:
            """ms per event with `n_streams` events in flight: events go round-robin to n_streams streams, each with its own scratch"""
            extra = [torch.cuda.Stream(dev) for _ in range(n_streams - 1)]
            scratch = [torch.empty_like(shared) for _ in extra]
            per_stream = [call_args] + [[a[:12] + (C.c_void_p(sc.data_ptr()), sc.numel(), C.c_void_p(st.cuda_stream)) for a in call_args]
                                        for st, sc in zip(extra, scratch)]
            for lst in per_stream[1:]:                            # build the graphs of the other workspaces
                for i in range(min(len(lst), 4)):
                    assert build_ex(*lst[i]) == 0
            torch.cuda.synchronize()
            ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ea.record(stream)
            for st in extra:
                st.wait_event(ea)
            for i in range(args.two_stream_steps):
                st = build_ex(*per_stream[i % n_streams][i % len(call_args)])     # outputs i % pool are only touched by step i
                assert st == 0
            for st in extra:
                done = torch.cuda.Event()
                done.record(st)
                stream.wait_event(done)
            eb.record(stream)
            torch.cuda.synchronize()
            return ea.elapsed_time(eb) / args.two_stream_steps

        ms2 = in_flight(2)
        ms4 = in_flight(4)
        two_streams = {"ms_per_event": ms2, "edges_per_s": e_mean_all / (ms2 * 1e-3), "steps": args.two_stream_steps,
                       "four_streams": {"ms_per_event": ms4, "edges_per_s": e_mean_all / (ms4 * 1e-3)},
                       "note": "same call, events go round-robin to 2 (4) streams with their own scratch workspace: the fixed latency of "
                               "one event's six dependent graph nodes overlaps the other events' work"}

    # per-phase device times (separate loop: event records between kernels perturb the main timing)
    phases_us = None
    if "phases" in legs and args.profile_steps > 0:
        phases = {}
        F.frnn_set_profiling(True)
        with torch.cuda.stream(stream):
            for i in range(args.profile_steps):
                step(i)
                for name, v in F.frnn_get_profile().items():
                    phases[name] = phases.get(name, 0.0) + v
        F.frnn_set_profiling(False)
        phases_us = {k: 1e3 * v / max(args.profile_steps, 1) for k, v in phases.items()}

    def timeline_of(step_fn, ws_buf, n_total, n_events, reps, group=8):
        """in-graph timeline (%globaltimer stamps written by the kernels themselves; the graph replay is untouched)"""
        F.frnn_set_profiling(2)
        acc = {}
        try:
            with torch.cuda.stream(stream):
                for rep in range(reps):
                    for k in range(group):                  # back to back, as in the timed loop; the stamps of the last call stay
                        step_fn(rep * group + k)
                    stream.synchronize()
                    for name, (b0, e0) in F.frnn_get_timeline(ws_buf, n_total, n_events).items():
                        a = acc.setdefault(name, [0.0, 0.0])
                        a[0] += b0
                        a[1] += e0
        finally:
            F.frnn_set_profiling(0)
        return {k: {"begin": v[0] / reps, "end": v[1] / reps, "dur": (v[1] - v[0]) / reps} for k, v in acc.items()}

    timeline_us = None
    if "timeline" in legs and args.timeline_steps > 0:
        timeline_us = timeline_of(step, shared, n, 1, args.timeline_steps)

    # ---- rooflines of the dominant kernel (the search pass)
    counters, counters_file, counters_stale = ncu_counters()
    dims, bits = F.frnn_get_grid(n, 1, 8)
    acct = [0, 1, 2, 3][: len(host_events)]
    cand = float(np.mean([candidate_rows(host_events[i], r, dims, bits) for i in acct]))
    cand_g3 = float(np.mean([candidate_rows(host_events[i], r, 3, bits) for i in acct]))
    e_mean = float(np.mean(edges_per_event))

    def rooflines(workload_key, kernel, dur_us, model_bytes):
        """(issue roofline, model-bytes figure) of one kernel launch of `dur_us` microseconds"""
        c = counters.get((workload_key, kernel))
        issue = None
        if c and dur_us:
            ach = c["warp_inst"] / (dur_us * 1e-6)
            issue = {"bound": "alu", "what": "warp-instruction issue (the kernel is bound by issue slots and dependent L2 latency, not by DRAM)",
                     "kernel": kernel, "achieved": ach / 1e9, "peak": issue_peak / 1e9, "unit": "Gwarp-inst/s", "frac": ach / issue_peak,
                     "peak_source": f"{N_SMS} SMs x {SCHEDULERS_PER_SM} schedulers x {sm_mhz:.0f} MHz (SM clock sampled during the timed loop)",
                     "warp_instructions_per_launch": c["warp_inst"], "threads_per_instruction": c.get("threads_per_inst"),
                     "l2_bytes_per_launch": c.get("l2_bytes"), "traffic": c.get("dram_bytes"),
                     "dram_gbs": (c["dram_bytes"] / (dur_us * 1e-6) / 1e9) if c.get("dram_bytes") else None,
                     "dram_frac_of_hbm_peak": (c["dram_bytes"] / (dur_us * 1e-6) / 1e9 / peak) if c.get("dram_bytes") else None,
                     "kernel_us": dur_us, "counters": f"{counters_file} (ncu, one launch, cold cache)", "counters_stale": counters_stale,
                     "ncu_cold": {"issue_active_pct": c.get("issue_active_pct"), "l1tex_pct_of_peak": c.get("l1tex_pct"), "l2_hit_pct": c.get("l2_hit_pct"),
                                  "occupancy_pct": c.get("occupancy_pct"), "sm_active_over_elapsed": (c["sm_active_cycles"] / c["sm_elapsed_cycles"]) if c.get("sm_elapsed_cycles") else None,
                                  "note": "the L1 data pipe (one wavefront per lane for the survivors' random 32-byte rows) is the busiest unit; neither it nor the "
                                          "issue slots saturate: the kernel is a chain of ~27 dependent memory round trips per warp (profiles/r02_summary.md)"}}
        model = None
        if dur_us and model_bytes:
            ach = model_bytes / (dur_us * 1e-6) / 1e9
            model = {"bound": "model_hbm_equivalent", "kernel": kernel, "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                     "physical": False, "peak_source": peak_src, "algorithmic_bytes_per_launch": model_bytes, "kernel_us": dur_us,
                     "traffic": c.get("dram_bytes") if c else None,
                     "note": "north_star's definition (bytes of candidate rows of the grid run + hit records over the HBM peak).  The rows are served by "
                             "L2/L1 and ~85 % of the candidates are rejected on a 4-byte key without touching their row, so this is an HBM-EQUIVALENT "
                             "rate, NOT a fraction of a physical limit (it can exceed 1); the physical bound is `roofline`"}
        return issue, model

    dom = "search"
    dom_us = (timeline_us or {}).get(dom, {}).get("dur") or (phases_us or {}).get(dom)
    roofline, roofline_model = rooflines("cfg2", dom, dom_us, cand * 32.0 + 8.0 * e_mean)
    if roofline is None:          # no counters file: still report the model figure as the roofline entry, flagged
        roofline = dict(roofline_model or {}, note2="no profiles/r0N_counters.csv: issue roofline unavailable")
    if roofline is not None and dom_us:
        roofline["kernel_us_source"] = "in-graph %globaltimer timeline" if (timeline_us or {}).get(dom) else "per-phase CUDA events (upper bound)"
        roofline["kernel_us_cuda_events"] = (phases_us or {}).get(dom)
        if roofline_model and roofline is not roofline_model:      # north_star's byte model beside the physical bound, flagged as what it is
            roofline["algorithmic_bytes_per_launch"] = roofline_model["algorithmic_bytes_per_launch"]
            roofline["model_frac_hbm_equivalent"] = roofline_model["frac"]
    path_bytes = cand * 32.0 + 12.0 * e_mean
    path_bytes_g3 = cand_g3 * 32.0 + 12.0 * e_mean
    t_event = ms_local / args.steps * 1e-3          # this rank's seconds per event
    path_roofline = {"bound": "model_hbm_equivalent", "physical": False, "grid_dims": dims, "grid_bits": bits, "model_bytes": path_bytes,
                     "frac": path_bytes / t_event / 1e9 / peak,
                     "model_bytes_g3": path_bytes_g3, "frac_vs_g3_grid": path_bytes_g3 / t_event / 1e9 / peak,
                     "compulsory_dram_bytes": n * 32.0 + 12.0 * e_mean,
                     "compulsory_frac": (n * 32.0 + 12.0 * e_mean) / t_event / 1e9 / peak,
                     "note": "north_star's target metric (>= 0.60): candidate rows of the grid actually run x 32 B + 12 B x edges per event over the "
                             "measured HBM peak; HBM-equivalent, see roofline_model"}

    def time_single(x_np, cfg_r, cfg_k, reps, opt=None, cap_rows=EDGE_CAP_PER_ROW, cap_edges=None):
        p = torch.from_numpy(x_np).to(dev)
        ecap = cap_edges if cap_edges is not None else max(len(x_np) * cap_rows, 64)
        w = F.Workspace(len(x_np), 1, cfg_k, ecap, dev, opt=opt)
        ms_ = timed(lambda i: F.frnn_build_ex(p, cfg_r, cfg_k, ws=w, stream=stream, opt=opt), reps)
        assert int(w.status.item()) == 0, "edge capacity exceeded"
        return ms_, int(w.count.item()), w, p

    # ---- the K cap when it binds (the paper's Faiss path asks for k neighbours and cuts at r)
    k_binding = None
    if "k_binding" in legs and args.other_reps > 0:
        reps = 4 * args.other_reps
        x2 = host_events[0]
        rows = {}
        k_cases = set(args.k_cases.split(","))
        for kk in (256, 16, 4, 2) if "config2" in k_cases else ():
            ms_, e_, _, _ = time_single(x2, r, kk, reps)
            rows[f"config2_K{kk}"] = {"k_max": kk, "ms_per_event": ms_, "edges": e_}
        for kk in (256, 4) if "config2" in k_cases else ():
            rows[f"config2_K{kk}"]["vs_K256"] = rows[f"config2_K{kk}"]["ms_per_event"] / rows["config2_K256"]["ms_per_event"]
        if "cluster" in k_cases:
            xc = events.one_cluster(2000, 0.01, 3)
            ms_, e_, _, _ = time_single(xc, 0.1, 64, reps, cap_rows=64)
            rows["one_cluster_n2000_K64"] = {"k_max": 64, "ms_per_event": ms_, "edges": e_, "note": "every row has 1999 neighbours: the bisection fallback (count > 512)"}
        xd = events.dense_tracks(n, 200.0, 0.02, 5) if "dense" in k_cases else None
        for kk in (64, 512) if "dense" in k_cases else ():
            ms_, e_, _, _ = time_single(xd, 0.1, kk, max(reps // 8, 3), cap_rows=min(kk, 256))
            rows[f"dense_event_n120k_K{kk}"] = {"k_max": kk, "ms_per_event": ms_, "edges": e_, "edges_per_s": e_ / (ms_ * 1e-3),
                                                "note": "120k points in tracks of Poisson(200) hits, sigma 0.02: mean degree ~170; "
                                                        + ("every row selected by the staged bitonic top-K" if kk == 64 else "K does not bind: rows collected and ordered")}
        k_binding = rows

    # ---- radius sweep with the data-driven grid
    radius_sweep = None
    if "radius_sweep" in legs and args.other_reps > 0:
        reps = 4 * args.other_reps
        radius_sweep = []
        p_dev = pts[0]
        for rr in (0.02, 0.05, 0.1, 0.2):
            opt, rep = F.frnn_suggest_grid(p_dev, rr, measure=True)
            ecap = n * (64 if rr > 0.15 else EDGE_CAP_PER_ROW)
            ms_s, e_s, _, _ = time_single(host_events[0], rr, k_max, reps, opt=opt, cap_edges=ecap)
            ms_d, e_d, _, _ = time_single(host_events[0], rr, k_max, reps, cap_edges=ecap)
            assert e_s == e_d
            row = {"r": rr, "edges": e_s, "suggested": {"grid_dims": opt.grid_dims, "grid_bits": opt.grid_bits, "reordered": bool(rep.reordered),
                                                        "ms_per_event": ms_s, "predicted_candidates_per_query": rep.predicted_candidates,
                                                        "predicted_us": rep.predicted_us, "measured_us_capacity0": rep.measured_us,
                                                        "shortlist": rep.tried()},
                   "default": {"grid": list(F.frnn_get_grid(n, 1, 8)), "ms_per_event": ms_d},
                   "extent_cells": rep.extent_cells[0]}
            if not rep.reordered:
                row["suggested"]["candidates_per_query"] = candidate_rows(host_events[0], rr, opt.grid_dims, opt.grid_bits) / n
            row["default"]["candidates_per_query"] = candidate_rows(host_events[0], rr, *F.frnn_get_grid(n, 1, 8)) / n
            radius_sweep.append(row)

    # the two steps that consume the edge list, timed on the outputs of the pool
    next_rows = None
    if "next" in legs and args.next_steps > 0:
        e_cap = max(edges_per_event)
        rows_out = [torch.empty((e_cap, 16), dtype=torch.float32, device=dev) for _ in range(4)]      # 4 x 21.5 MB
        labels = torch.empty(n, dtype=torch.int32, device=dev)
        ncomp = torch.zeros(1, dtype=torch.int32, device=dev)
        scores = torch.from_numpy(events.edge_scores(e_cap, 1)).to(dev)

        def gather(i):
            k = i % len(outs)
            F.frnn_gather_edge_rows(pts[k], outs[k].src, outs[k].dst, edge_count=outs[k].count, e_max=e_cap,
                                    out=rows_out[i % 4], stream=stream)

        def label(i):
            k = i % len(outs)
            F.frnn_label_components(n, outs[k].src, outs[k].dst, score=scores, threshold=0.5, edge_count=outs[k].count,
                                    edge_max=e_cap, labels=labels, n_components=ncomp, stream=stream)

        def dense(i):
            k = i % len(outs)
            F.frnn_build_dense_ex(pts[k], r, k_max, ws=outs[k], stream=stream)

        g_us, l_us = 1e3 * timed(gather, args.next_steps), 1e3 * timed(label, args.next_steps)
        d_us = 1e3 * timed(dense, max(args.next_steps // 50, 3), warm=2)
        stream.synchronize()
        assert [int(w.count.item()) for w in outs[:3]] == edges_per_event[:3], "brute-force variant disagrees with the grid path"
        g_bytes = e_mean * (8 + 64 + 64)
        g_dram = n * 32 + e_mean * (8 + 64)              # physical: every point row once (the event fits L2) + indices + the rows written
        next_rows = {
            "gather_edge_rows": {"us_per_event": g_us, "edges": e_mean, "algorithmic_bytes": g_bytes,
                                 "achieved_gbs": g_bytes / (g_us * 1e-6) / 1e9, "frac_of_hbm_peak": g_bytes / (g_us * 1e-6) / 1e9 / peak,
                                 "physical_dram_bytes": g_dram, "physical_dram_gbs": g_dram / (g_us * 1e-6) / 1e9,
                                 "physical_frac_of_hbm_peak": g_dram / (g_us * 1e-6) / 1e9 / peak, "bound": "hbm",
                                 "note": "per edge: 8 B indices + 2 x 32 B rows read + 64 B written (streaming stores).  The row reads are served by L2 "
                                         "(one event = 3.84 MB), so the PHYSICAL DRAM traffic is the event once + indices + the written rows"},
            "label_components": {"us_per_event": l_us, "nodes": n, "edges": e_mean, "threshold": 0.5,
                                 "components": int(ncomp.item()), "note": "3 kernels (init, hook: CAS union-find, flatten) replayed as one graph"},
            "dense_bruteforce": {"ms_per_event": d_us * 1e-3, "pair_evaluations": n * (n - 1) / 2,
                                 "pairs_per_s": n * (n - 1) / 2 / (d_us * 1e-6), "slower_than_grid_path": d_us * 1e-3 / ms_per_step,
                                 "bound": "alu", "fp32_lane_instr_per_s": 16 * n * (n - 1) / 2 / (d_us * 1e-6),
                                 "fp32_peak_lane_instr_per_s": N_SMS * 128 * sm_mhz * 1e6,
                                 "frac_of_fp32_issue_peak": 16 * n * (n - 1) / 2 / (d_us * 1e-6) / (N_SMS * 128 * sm_mhz * 1e6),
                                 "note": "frnn_build_dense_ex: every unordered pair once, same R3 chain; the paper's own ratio "
                                         "flat-index kNN + cut : grid FRNN is 0.54 s : 0.04 s (PAPER.md:77, V100)"},
        }
        del rows_out

    # the other BASELINE configs and the N sweep ("inference time depends almost linearly on the number
    # of spacepoints"): same call, CUDA events around back-to-back replays of ONE input (so L2 is warm for the small ones)
    other = None
    if "other" in legs and args.other_reps > 0:
        other = {}
        which = set(args.other_configs.split(","))
        for idx, reps in ((0, 20 * args.other_reps), (1, 20 * args.other_reps), (4, args.other_reps)):
            if str(idx) not in which:
                continue
            c = events.CONFIGS[idx]
            xe = events.make_event(c)
            ms_, e_, w_, p_ = time_single(xe, c.r, c.k_max, reps)
            g_ = F.frnn_get_grid(c.n, 1, 8)
            other[c.name] = {"n": c.n, "ms_per_event": ms_, "edges": e_, "edges_per_s": e_ / (ms_ * 1e-3), "grid": g_}
            if idx == 4:
                tl = timeline_of(lambda i: F.frnn_build_ex(p_, c.r, c.k_max, ws=w_, stream=stream), w_.buf, c.n, 1, max(args.other_reps // 5, 2), group=2)
                cand4 = candidate_rows(xe, c.r, *g_)
                ri, rm = rooflines("cfg4", "search", tl.get("search", {}).get("dur"), cand4 * 32.0 + 8.0 * e_)
                other[c.name].update({"timeline_us": tl, "roofline_issue": ri, "roofline_model": rm,
                                      "path_model_frac": (cand4 * 32.0 + 12.0 * e_) / (ms_ * 1e-3) / 1e9 / peak})
            del w_, p_
        if "3" in which:
            c3 = events.CONFIGS[3]
            xb, offs = events.make_batch(c3)
            pb = torch.from_numpy(xb).to(dev)
            wb = F.Workspace(len(xb), c3.n_events, c3.k_max, len(xb) * 4, dev)
            ms3 = timed(lambda i: F.frnn_build_batched(pb, offs, c3.r, c3.k_max, ws=wb, stream=stream), args.other_reps, warm=3)
            assert int(wb.status.item()) == 0
            e3 = int(wb.count[-1].item())
            g3 = F.frnn_get_grid(len(xb), c3.n_events, 8)
            tl3 = timeline_of(lambda i: F.frnn_build_batched(pb, offs, c3.r, c3.k_max, ws=wb, stream=stream), wb.buf, len(xb), c3.n_events,
                              max(args.other_reps // 5, 2), group=2)
            cand3 = sum(candidate_rows(xb[offs[e]:offs[e + 1]], c3.r, *g3) for e in range(2)) * c3.n_events / 2.0
            ri3, rm3 = rooflines("cfg3", "search", tl3.get("search", {}).get("dur"), cand3 * 32.0 + 8.0 * e3)
            other[c3.name] = {"n": len(xb), "events": c3.n_events, "ms_per_batch": ms3, "ms_per_event": ms3 / c3.n_events, "edges": e3,
                              "edges_per_s": e3 / (ms3 * 1e-3), "grid": g3, "workspace_bytes": F.frnn_workspace_bytes(len(xb), c3.n_events, 8, c3.k_max),
                              "timeline_us": tl3, "roofline_issue": ri3, "roofline_model": rm3,
                              "path_model_frac": (cand3 * 32.0 + 12.0 * e3) / (ms3 * 1e-3) / 1e9 / peak}
            del pb, wb
        if "sweep" in which:
            sweep = []
            for nn in (15000, 30000, 60000, 120000):
                c = dataclasses.replace(CFG, n=nn, n_tracks=CFG.n_tracks * nn // CFG.n)
                ms_, e_, _, _ = time_single(events.make_event(c, 77), c.r, c.k_max, 10 * args.other_reps)
                sweep.append({"n": nn, "ms_per_event": ms_, "edges": e_, "us_per_1k_points": 1e3 * ms_ / (nn / 1000)})
            other["n_sweep_config2_recipe"] = sweep

    # end to end through the host-buffer entry points: pinned host buffers, copies inside the timed region
    e2e = None
    if "e2e" in legs and args.e2e_steps > 0:
        import oracle
        n_pin = min(len(host_events), 8)
        pin_in = [torch.from_numpy(x).pin_memory() for x in host_events[:n_pin]]
        def out_block():
            """src | dst | d2 in ONE page-locked block: equally spaced arrays travel as one 2-D copy (include/frnn.h)"""
            blk = torch.empty(3 * cap, dtype=torch.int32).pin_memory()
            return blk[:cap], blk[cap:2 * cap], blk[2 * cap:].view(torch.float32)
        hs, hd, hq = out_block()
        for i in range(3):
            F.frnn_build_host(pin_in[i % n_pin], r, k_max, hs, hd, hq)
        torch.cuda.synchronize()
        D.barrier(rank)
        e_edges = 0
        sync_steps = max(args.e2e_steps // 4, 1)
        t = time.perf_counter()
        for i in range(sync_steps):
            e_edges += F.frnn_build_host(pin_in[i % n_pin], r, k_max, hs, hd, hq)
        torch.cuda.synchronize()
        dt_sync = D.reduce_max(time.perf_counter() - t, rank)
        e_total_sync = D.reduce_sum(e_edges, rank)
        # the host pipeline: the same copies per event, but H2D of event i+1, build of event i and D2H of event i-1
        # overlap (4 slots); every event's edges land in one of 5 rotating sets of pinned host buffers
        depth = 4
        pipe = F.HostPipeline(n, k_max, cap, depth=depth)
        hb = [out_block() + (torch.zeros(1, dtype=torch.int64).pin_memory(),) for _ in range(depth + 1)]

        def run_pipeline(sizes_):
            """submit len(sizes_) events (event i = the first sizes_[i] rows of pinned event i % n_pin); returns (seconds, edges)"""
            for i in range(2 * depth):
                pipe.submit(pin_in[i % n_pin][:sizes_[i % len(sizes_)]], r, *hb[i % len(hb)])
            pipe.wait()
            D.barrier(rank)
            got_edges = 0
            t_ = time.perf_counter()
            for i in range(len(sizes_)):
                slot = hb[i % len(hb)]
                if i >= len(hb):
                    got_edges += int(slot[3][0])      # the result of step i - (depth + 1): complete, since only `depth` events are in flight
                pipe.submit(pin_in[i % n_pin][:sizes_[i]], r, *slot)
            pipe.wait()
            dt_ = time.perf_counter() - t_
            for i in range(max(len(sizes_) - len(hb), 0), len(sizes_)):
                got_edges += int(hb[i % len(hb)][3][0])
            return dt_, got_edges

        dt, p_edges = run_pipeline([n] * args.e2e_steps)
        # the last depth + 1 events of the timed loop against the oracle (outside the timed region): every host buffer set
        # still holds the result of the last event that was written into it
        last = args.e2e_steps - 1
        verified, events_verified = True, 0
        for ev in range(max(last - len(hb) + 1, 0), last + 1):
            s_, d_, q_, c_ = hb[ev % len(hb)]
            e_last = int(c_[0])
            exp = oracle.frnn(host_events[ev % n_pin], r, k_max, oracle.CELLS)
            verified = verified and bool(e_last == exp.count and np.array_equal(s_[:e_last].numpy(), exp.src)
                                         and np.array_equal(d_[:e_last].numpy(), exp.dst)
                                         and np.array_equal(q_[:e_last].numpy().view(np.uint32), exp.d2.view(np.uint32)))
            events_verified += 1
        # (the band report below is that of the last event: s_, d_, q_, e_last and exp are left at it)
        # north_star's acceptance rule: membership may differ only for pairs with |d2 - r2| <= 1e-6 r2, and those must be reported
        r2f = float(np.float32(r) * np.float32(r))
        got_keys = s_[:e_last].numpy().astype(np.int64) << 32 | d_[:e_last].numpy().astype(np.int64)
        exp_keys = exp.src.astype(np.int64) << 32 | exp.dst.astype(np.int64)
        only = np.setxor1d(got_keys, exp_keys)
        band_report = {"event_seed": int(seeds[last % n_pin]), "edges_in_band": int((np.abs(exp.d2.astype(np.float64) - r2f) <= 1e-6 * r2f).sum()),
                       "membership_differences": int(len(only)), "differing_pairs": [[int(k >> 32), int(k & 0xffffffff)] for k in only[:20]],
                       "d2_bitwise_differences": int((q_[:min(e_last, exp.count)].numpy().view(np.uint32) != exp.d2[:min(e_last, exp.count)].view(np.uint32)).sum()) if e_last == exp.count else None,
                       "rule": "pairs with |d2 - r2| <= 1e-6 r2 may differ and must be listed; with r2 and the summation order pinned the expected number is 0"}
        rng = np.random.default_rng(777)
        v_sizes = [int(v) for v in rng.choice(np.arange(90000, n + 1), size=min(args.e2e_steps, n + 1 - 90000), replace=False)]
        dt_v, p_edges_v = run_pipeline(v_sizes)
        pipe.close()
        # bare-copy floor: the same bytes per event over the same number of streams, no build (torch copies)
        e_avg = int(p_edges / args.e2e_steps)
        streams_c = [torch.cuda.Stream(dev) for _ in range(depth)]
        d_in = [torch.empty((n, 8), dtype=torch.float32, device=dev) for _ in range(depth)]
        d_out = [torch.empty(3 * e_avg, dtype=torch.int32, device=dev) for _ in range(depth)]
        h_out = [torch.empty(3 * e_avg, dtype=torch.int32).pin_memory() for _ in range(depth + 1)]

        def copy_loop(steps_):
            for i in range(steps_):
                s = streams_c[i % depth]
                with torch.cuda.stream(s):
                    d_in[i % depth].copy_(pin_in[i % n_pin], non_blocking=True)
                    h_out[i % (depth + 1)].copy_(d_out[i % depth], non_blocking=True)
            torch.cuda.synchronize()
        copy_loop(2 * depth)
        t = time.perf_counter()
        copy_loop(args.e2e_steps)
        dt_copy = time.perf_counter() - t
        dt = D.reduce_max(dt, rank)
        e_total = D.reduce_sum(p_edges, rank)
        e2e = {"value": e_total / dt, "unit": UNIT, "h2d_bytes_per_step": n * 32,
               "d2h_bytes_per_step": int(8 + 12 * p_edges / args.e2e_steps), "ms_per_step": 1e3 * dt / args.e2e_steps,
               "steps": args.e2e_steps, "api": f"frnn_host_pipeline_submit/wait, depth {depth}: pinned host buffers in and out (src | dst | d2 of an event in one "
               "block: one 2-D copy per event), copies of consecutive events overlap", "timer": "host wall clock around the submit loop + wait",
               "e2e_verified": verified, "events_verified": events_verified, "band_report": band_report,
               "verified_how": f"the last {events_verified} events of the timed loop (one per host buffer set), edges and d2 bit for bit against the oracle (outside the timed region)",
               "copy_floor_ms": 1e3 * dt_copy / args.e2e_steps,
               "copy_floor_note": f"the same H2D ({n * 32} B) + D2H ({12 * e_avg} B) per event over {depth} streams, pinned buffers, no build: what the "
                                  "box's PCIe link allows",
               "varying_n": {"ms_per_step": 1e3 * dt_v / len(v_sizes), "value": p_edges_v / dt_v, "steps": len(v_sizes),
                             "distinct_n": len(set(v_sizes)), "n_range": [90000, n], "mean_n": float(np.mean(v_sizes)),
                             "h2d_bytes_per_step": float(np.mean(v_sizes)) * 32, "vs_fixed_n": (dt_v / len(v_sizes)) / (dt / args.e2e_steps)},
               "one_call_at_a_time": {"value": e_total_sync / dt_sync, "ms_per_step": 1e3 * dt_sync / sync_steps,
                                      "api": "frnn_build_host (synchronous: H2D, build, D2H, nothing overlaps)"}}

    cpu_baseline = None
    if "cpu" in legs and rank.is_main and rank.world_size == 1 and args.cpu_events > 0:
        import oracle
        ce, ct, cores = oracle_sample_run(args.cpu_events)
        c1e, c1t, _ = oracle_sample_run(max(args.cpu_events // 60, 1), threads=1)
        brute = {}
        for idx in (0, 1, 2):
            c = events.CONFIGS[idx]
            xe = events.make_event(c)
            t = time.perf_counter()
            res = oracle.frnn(xe, c.r, c.k_max, oracle.BRUTE)
            brute[c.name] = {"ms_per_event": 1e3 * (time.perf_counter() - t), "edges": res.count, "pair_evaluations": c.n * (c.n - 1)}
        cpu_baseline = {"value": ce / ct, "unit": UNIT, "cores": cores, "kind": "oracle",
                        "sample": f"{args.cpu_events} whole config-2 events (seeds 1000..), cell-list mode, {ct:.1f} s of CPU work",
                        "ms_per_event": 1e3 * ct / args.cpu_events,
                        "one_thread": {"value": c1e / c1t, "ms_per_event": 1e3 * c1t / max(args.cpu_events // 60, 1), "cores": 1,
                                       "sample": f"{max(args.cpu_events // 60, 1)} whole config-2 event(s), cell-list mode"},
                        "brute_force_mode_once": brute,
                        "note": "PAPER.md:43 contrasts one CPU core with 48: the same oracle at all cores and at one thread; mode A (brute force) "
                                "timed once per config where it is run in full (SURVEY.md 8(d))"}

    if rank.is_main:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": rank.world_size, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "ms_per_event": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": WORKLOAD, "events_per_step": 1, "pool_events_per_gpu": len(seeds),
                       "l2": f"inputs and outputs rotate over {len(seeds)} events ({len(seeds) * n * 32 / 1e6:.0f} MB in + "
                             f"{len(seeds) * cap * 12 / 1e6:.0f} MB out > 126 MB L2); no explicit flush",
                       "call_signature": "every step differs from the previous one in its input and output pointers: the graph's node parameters are rewritten every step",
                       "grid": {"dims": dims, "bits": bits}, "edge_capacity": cap, "parallelism": f"events sharded over {rank.world_size} GPU(s), no collective"},
            "edges_per_event": e_mean, "roofline": roofline,
            "roofline_model": roofline_model, "path_roofline": path_roofline, "phases_us": phases_us, "timeline_us": timeline_us,
            "varying_n": varying, "k_binding": k_binding, "radius_sweep": radius_sweep,
            "cpu_baseline": cpu_baseline, "e2e": e2e, "next_rows": next_rows, "other_configs": other, "two_streams": two_streams, "gpu_launches": launches_per_step * args.steps,
            "gpu_launches_per_step": launches_per_step, "clocks": clocks,
            "host_wall_ms_per_step": 1e3 * (t1 - t0) / args.steps,
            "paper_context": "paper: 0.04 +- 0.01 s/event on V100 16 GB (PAPER.md:77 Table 1 'FRNN' column), TrackML events; other machine, other data",
        }
        emit(line)
    D.finalize(rank)


if __name__ == "__main__":
    main()
