#!/usr/bin/env python
"""bench.py -- FRNN graph building at tracking scale (BASELINE.json: 120k hits, D=8, r=0.1, K=256).

One "step" = one pass of the whole hot path (S2..S10: bin, cell scan, scatter, search, degree scan + emit)
over ONE seeded synthetic event of config 2 through the C ABI (frnn_build_ex) on a non-default
stream.  Steps rotate over a pool of distinct events and distinct output buffers whose total size
exceeds the 126 MB L2, so every step reads its input cold from HBM.

Prints ONE JSON line (rank 0).  Keys beyond the base contract:
  roofline      dominant kernel: algorithmic bytes per launch / its CUDA-event duration vs the
                measured HBM peak (MEASURED_PEAKS.json, else the profiling guide's fallback)
  path_roofline north_star's whole-path figure: (candidate rows * 32 B + 12 B * edges) / ms_per_event
  cpu_baseline  the oracle (cell-list mode) timed on this box's host cores on a bounded sample
  e2e           the same metric through frnn_build_host: pinned host buffers, H2D + D2H inside
  phases_us     mean device time per phase of the path
`--impl reference` times the oracle alone (rank 0 only) on the same metric/config.
"""
from __future__ import annotations

import argparse
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


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def candidate_rows(x: np.ndarray, r: float, dims: int, bits: int) -> int:
    """ACCOUNTING ONLY (not on the product path): sum over queries of the rows in the 3^dims cells
    around the query's cell, for the grid the library reports it runs (cell side r*(1+2^-7),
    toroidal extent 2^bits).  This is the 'bytes of candidate rows' of north_star / 32."""
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


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""

    def __init__(self, uuid: str | None, index: int, period_s: float = 0.02):
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

    def run(self):
        while self.ok and not self.stop_flag:
            try:
                mhz = self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM)
                reasons = self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                self.samples.append((time.perf_counter(), mhz, reasons))
            except Exception:
                pass
            time.sleep(self.period)

    def summary(self, t0: float, t1: float) -> dict:
        names = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
                 0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x100: "display_clock_setting"}
        sel = [s for s in self.samples if t0 <= s[0] <= t1] or self.samples[-3:]
        if not sel:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0}
        mask = 0
        for s in sel:
            mask |= s[2]
        return {"sm_mhz": float(np.median([s[1] for s in sel])), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(n for b, n in names.items() if mask & b), "samples": len(sel)}


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
    ap.add_argument("--cpu-events", type=int, default=160, help="events the cpu_baseline leg runs the oracle on")
    ap.add_argument("--e2e-steps", type=int, default=1000)
    ap.add_argument("--profile-steps", type=int, default=200)
    ap.add_argument("--timeline-steps", type=int, default=100)
    ap.add_argument("--two-stream-steps", type=int, default=4000, help="steps of the two-events-in-flight throughput figure (0: skip)")
    ap.add_argument("--other-reps", type=int, default=50, help="repetitions for the other configs / N sweep (0: skip)")
    ap.add_argument("--next-steps", type=int, default=300, help="timed repetitions of the two edge-list consumers (0: skip)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)

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
    F.lib()

    n, k_max, r = CFG.n, CFG.k_max, CFG.r
    cap = n * EDGE_CAP_PER_ROW
    seeds = D.shard(list(range(args.pool * rank.world_size)), rank)       # events sharded round-robin across ranks
    host_events = [events.make_event(CFG, s) for s in seeds]
    pts = [torch.from_numpy(x).to(dev) for x in host_events]
    outs = [F.Workspace(n, 1, k_max, cap, dev) for _ in seeds]
    shared = outs[0].buf                                                 # scratch is reused; only outputs rotate
    for w in outs[1:]:
        w.buf = shared
    stream = torch.cuda.Stream(dev)
    L = F.lib()
    import ctypes as C
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
        for i in range(args.warmup):
            step(i)
        stream.synchronize()
        D.barrier(rank)
        torch.cuda.synchronize()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        ev0.record(stream)
        for i in range(args.steps):
            step(i)
        ev1.record(stream)
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
    clocks = sampler.summary(t0, t1)
    e_mean_all = float(np.mean(edges_per_event))

    # throughput with two events in flight (two streams, two scratch workspaces): the fixed latency of one event's six
    # dependent graph nodes overlaps the other event's work.  Reported beside the headline, which stays one stream.
    two_streams = None
    if args.two_stream_steps > 0:
        stream_b = torch.cuda.Stream(dev)
        scratch_b = torch.empty_like(shared)
        args_b = [a[:12] + (C.c_void_p(scratch_b.data_ptr()), scratch_b.numel(), C.c_void_p(stream_b.cuda_stream)) for a in call_args]
        for i in range(len(call_args)):                       # build the graphs of the second stream
            assert build_ex(*args_b[i]) == 0
        torch.cuda.synchronize()
        ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ea.record(stream)
        stream_b.wait_event(ea)
        for i in range(args.two_stream_steps):
            k = i % len(call_args)
            st = build_ex(*(call_args[k] if i % 2 == 0 else args_b[k]))     # outputs k are only touched by step i
            assert st == 0
        done_b = torch.cuda.Event()
        done_b.record(stream_b)
        stream.wait_event(done_b)
        eb.record(stream)
        torch.cuda.synchronize()
        ms2 = ea.elapsed_time(eb) / args.two_stream_steps
        two_streams = {"ms_per_event": ms2, "edges_per_s": e_mean_all / (ms2 * 1e-3), "steps": args.two_stream_steps,
                       "note": "same call, events alternate between two streams with their own scratch workspace"}

    # per-phase device times (separate loop: event records between kernels perturb the main timing)
    phases = {}
    F.frnn_set_profiling(True)
    with torch.cuda.stream(stream):
        for i in range(args.profile_steps):
            step(i)
            for name, v in F.frnn_get_profile().items():
                phases[name] = phases.get(name, 0.0) + v
    F.frnn_set_profiling(False)
    phases_us = {k: 1e3 * v / max(args.profile_steps, 1) for k, v in phases.items()}

    # in-graph timeline (%globaltimer stamps written by the kernels themselves; the graph replay is untouched)
    timeline_us = None
    if args.timeline_steps > 0:
        F.frnn_set_profiling(2)
        acc = {}
        with torch.cuda.stream(stream):
            for rep in range(args.timeline_steps):
                for k in range(8):                      # back to back, as in the timed loop; the stamps of the last call stay
                    step(rep * 8 + k)
                stream.synchronize()
                for name, (b0, e0) in F.frnn_get_timeline(shared, n, 1).items():
                    a = acc.setdefault(name, [0.0, 0.0])
                    a[0] += b0
                    a[1] += e0
        F.frnn_set_profiling(0)
        timeline_us = {k: {"begin": v[0] / args.timeline_steps, "end": v[1] / args.timeline_steps,
                           "dur": (v[1] - v[0]) / args.timeline_steps} for k, v in acc.items()}

    # roofline of the dominant kernel
    peak, peak_src = measured_peak()
    dims, bits = F.frnn_get_grid(n, 1)
    acct = [0, 1, 2, 3]
    cand = float(np.mean([candidate_rows(host_events[i], r, dims, bits) for i in acct]))
    cand_g3 = float(np.mean([candidate_rows(host_events[i], r, 3, bits) for i in acct]))
    e_mean = float(np.mean(edges_per_event))
    # dominant kernel = the search pass (one launch per step): candidate rows read + (j, d2) hit records written
    dom = "search"
    alg_bytes = cand * 32.0 + 8.0 * e_mean
    dom_us = phases_us.get(dom, float("nan"))
    achieved = alg_bytes / (dom_us * 1e-6) / 1e9 if dom_us and dom_us == dom_us else float("nan")
    traffic = None
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.csv")) as f:      # ncu dram bytes per launch (see profiles/traffic.md)
            for row in f.read().splitlines()[1:]:
                k, v = row.split(",")[:2]
                if k == dom:
                    traffic = int(v)
    except Exception:
        pass
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic, "peak_source": peak_src, "algorithmic_bytes_per_launch": alg_bytes,
                "kernel_us": dom_us, "kernel_us_in_graph": (timeline_us or {}).get(dom, {}).get("dur"), "note": "candidate rows are served by L2/L1, so this is an HBM-equivalent rate"}
    path_bytes = cand * 32.0 + 12.0 * e_mean
    path_bytes_g3 = cand_g3 * 32.0 + 12.0 * e_mean
    t_event = ms_local / args.steps * 1e-3          # this rank's seconds per event
    path_roofline = {"grid_dims": dims, "grid_bits": bits, "model_bytes": path_bytes, "frac": path_bytes / t_event / 1e9 / peak,
                     "model_bytes_g3": path_bytes_g3, "frac_vs_g3_grid": path_bytes_g3 / t_event / 1e9 / peak,
                     "compulsory_dram_bytes": n * 32.0 + 12.0 * e_mean,
                     "compulsory_frac": (n * 32.0 + 12.0 * e_mean) / t_event / 1e9 / peak}

    # the two steps that consume the edge list, timed on the outputs of the pool
    next_rows = None
    if args.next_steps > 0:
        e_cap = max(edges_per_event)
        rows_out = [torch.empty((e_cap, 16), dtype=torch.float32, device=dev) for _ in range(4)]      # 4 x 21.5 MB
        labels = torch.empty(n, dtype=torch.int32, device=dev)
        ncomp = torch.zeros(1, dtype=torch.int32, device=dev)
        scores = torch.from_numpy(events.edge_scores(e_cap, 1)).to(dev)

        def t_loop(fn, reps):
            with torch.cuda.stream(stream):
                for i in range(5):
                    fn(i)
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream)
                for i in range(reps):
                    fn(i)
                b.record(stream)
                stream.synchronize()
            return 1e3 * a.elapsed_time(b) / reps

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

        g_us, l_us = t_loop(gather, args.next_steps), t_loop(label, args.next_steps)
        d_us = t_loop(dense, max(args.next_steps // 50, 3))
        assert [int(w.count.item()) for w in outs[:3]] == edges_per_event[:3], "brute-force variant disagrees with the grid path"
        g_bytes = e_mean * (8 + 64 + 64)
        next_rows = {
            "gather_edge_rows": {"us_per_event": g_us, "edges": e_mean, "algorithmic_bytes": g_bytes,
                                 "achieved_gbs": g_bytes / (g_us * 1e-6) / 1e9, "frac_of_hbm_peak": g_bytes / (g_us * 1e-6) / 1e9 / peak,
                                 "note": "per edge: 8 B indices + 2 x 32 B rows read (L2) + 64 B written (streaming stores)"},
            "label_components": {"us_per_event": l_us, "nodes": n, "edges": e_mean, "threshold": 0.5,
                                 "components": int(ncomp.item()), "note": "3 kernels: init, hook (CAS union-find), flatten"},
            "dense_bruteforce": {"ms_per_event": d_us * 1e-3, "pair_evaluations": n * (n - 1) / 2,
                                 "pairs_per_s": n * (n - 1) / 2 / (d_us * 1e-6), "slower_than_grid_path": d_us * 1e-3 / ms_per_step,
                                 "bound": "alu", "fp32_lane_instr_per_s": 16 * n * (n - 1) / 2 / (d_us * 1e-6),
                                 "fp32_peak_lane_instr_per_s": 148 * 128 * 1.965e9,
                                 "frac_of_fp32_issue_peak": 16 * n * (n - 1) / 2 / (d_us * 1e-6) / (148 * 128 * 1.965e9),
                                 "note": "frnn_build_dense_ex: every unordered pair once, same R3 chain; the paper's own ratio "
                                         "flat-index kNN + cut : grid FRNN is 0.54 s : 0.04 s (PAPER.md:77, V100)"},
        }

    # the other BASELINE configs and the N sweep ("inference time depends almost linearly on the number
    # of spacepoints"): same call, CUDA events around back-to-back replays of ONE input (so L2 is warm for the small ones)
    other = None
    if args.other_reps > 0:
        import dataclasses

        def time_single(x_np, cfg_r, cfg_k, reps):
            p = torch.from_numpy(x_np).to(dev)
            w = F.Workspace(len(x_np), 1, cfg_k, max(len(x_np) * EDGE_CAP_PER_ROW, 64), dev)
            with torch.cuda.stream(stream):
                for _ in range(5):
                    F.frnn_build_ex(p, cfg_r, cfg_k, ws=w, stream=stream)
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream)
                for _ in range(reps):
                    F.frnn_build_ex(p, cfg_r, cfg_k, ws=w, stream=stream)
                b.record(stream)
                stream.synchronize()
            assert int(w.status.item()) == 0
            return a.elapsed_time(b) / reps, int(w.count.item())

        other = {}
        for idx, reps in ((0, 20 * args.other_reps), (1, 20 * args.other_reps), (4, args.other_reps)):
            c = events.CONFIGS[idx]
            ms, e = time_single(events.make_event(c), c.r, c.k_max, reps)
            other[c.name] = {"n": c.n, "ms_per_event": ms, "edges": e, "edges_per_s": e / (ms * 1e-3), "grid": F.frnn_get_grid(c.n, 1)}
        c3 = events.CONFIGS[3]
        xb, offs = events.make_batch(c3)
        pb = torch.from_numpy(xb).to(dev)
        wb = F.Workspace(len(xb), c3.n_events, c3.k_max, len(xb) * 4, dev)
        with torch.cuda.stream(stream):
            for _ in range(3):
                F.frnn_build_batched(pb, offs, c3.r, c3.k_max, ws=wb, stream=stream)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            for _ in range(args.other_reps):
                F.frnn_build_batched(pb, offs, c3.r, c3.k_max, ws=wb, stream=stream)
            b.record(stream)
            stream.synchronize()
        assert int(wb.status.item()) == 0
        ms3 = a.elapsed_time(b) / args.other_reps
        e3 = int(wb.count[-1].item())
        other[c3.name] = {"n": len(xb), "events": c3.n_events, "ms_per_batch": ms3, "ms_per_event": ms3 / c3.n_events, "edges": e3,
                          "edges_per_s": e3 / (ms3 * 1e-3), "grid": F.frnn_get_grid(len(xb), c3.n_events)}
        del pb, wb
        sweep = []
        for nn in (15000, 30000, 60000, 120000):
            c = dataclasses.replace(CFG, n=nn, n_tracks=CFG.n_tracks * nn // CFG.n)
            ms, e = time_single(events.make_event(c, 77), c.r, c.k_max, 10 * args.other_reps)
            sweep.append({"n": nn, "ms_per_event": ms, "edges": e, "us_per_1k_points": 1e3 * ms / (nn / 1000)})
        other["n_sweep_config2_recipe"] = sweep

    # end to end through the host-buffer entry point: pinned host buffers, copies inside the timed region
    e2e = None
    if args.e2e_steps > 0:
        n_pin = min(len(host_events), 8)
        pin_in = [torch.from_numpy(x).pin_memory() for x in host_events[:n_pin]]
        hs = torch.empty(cap, dtype=torch.int32).pin_memory()
        hd = torch.empty(cap, dtype=torch.int32).pin_memory()
        hq = torch.empty(cap, dtype=torch.float32).pin_memory()
        for i in range(3):
            F.frnn_build_host(pin_in[i % n_pin], r, k_max, hs, hd, hq)
        torch.cuda.synchronize()
        D.barrier(rank)
        e_edges = 0
        t = time.perf_counter()
        for i in range(args.e2e_steps):
            e_edges += F.frnn_build_host(pin_in[i % n_pin], r, k_max, hs, hd, hq)
        torch.cuda.synchronize()
        dt_sync = D.reduce_max(time.perf_counter() - t, rank)
        e_total_sync = D.reduce_sum(e_edges, rank)
        # the host pipeline: the same copies per event, but H2D of event i+1, build of event i and D2H of event i-1
        # overlap (4 slots); every event's edges land in one of 5 rotating sets of pinned host buffers
        depth = 4
        pipe = F.HostPipeline(n, k_max, cap, depth=depth)
        hb = [(torch.empty(cap, dtype=torch.int32).pin_memory(), torch.empty(cap, dtype=torch.int32).pin_memory(),
               torch.empty(cap, dtype=torch.float32).pin_memory(), torch.zeros(1, dtype=torch.int64).pin_memory())
              for _ in range(depth + 1)]
        for i in range(2 * depth):
            pipe.submit(pin_in[i % n_pin], r, *hb[i % len(hb)])
        pipe.wait()
        D.barrier(rank)
        p_edges = 0
        t = time.perf_counter()
        for i in range(args.e2e_steps):
            slot = hb[i % len(hb)]
            if i >= len(hb):
                p_edges += int(slot[3][0])        # the result of step i - (depth + 1): complete, since only `depth` events are in flight
            pipe.submit(pin_in[i % n_pin], r, *slot)
        pipe.wait()
        dt = time.perf_counter() - t
        for i in range(max(args.e2e_steps - len(hb), 0), args.e2e_steps):
            p_edges += int(hb[i % len(hb)][3][0])
        pipe.close()
        dt = D.reduce_max(dt, rank)
        e_total = D.reduce_sum(p_edges, rank)
        e2e = {"value": e_total / dt, "unit": UNIT, "h2d_bytes_per_step": n * 32,
               "d2h_bytes_per_step": int(8 + 12 * p_edges / args.e2e_steps), "ms_per_step": 1e3 * dt / args.e2e_steps,
               "steps": args.e2e_steps, "api": f"frnn_host_pipeline_submit/wait, depth {depth}: pinned host buffers in and out, copies of "
               "consecutive events overlap", "timer": "host wall clock around the submit loop + wait",
               "one_call_at_a_time": {"value": e_total_sync / dt_sync, "ms_per_step": 1e3 * dt_sync / args.e2e_steps,
                                      "api": "frnn_build_host (synchronous: H2D, build, D2H, nothing overlaps)"}}

    cpu_baseline = None
    if rank.is_main and rank.world_size == 1 and not args.no_cpu_baseline and args.cpu_events > 0:
        ce, ct, cores = oracle_sample_run(args.cpu_events)
        cpu_baseline = {"value": ce / ct, "unit": UNIT, "cores": cores, "kind": "oracle",
                        "sample": f"{args.cpu_events} whole config-2 events (seeds 1000..), cell-list mode, {ct:.1f} s of CPU work",
                        "ms_per_event": 1e3 * ct / args.cpu_events}

    if rank.is_main:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": rank.world_size, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "ms_per_event": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": WORKLOAD, "events_per_step": 1, "pool_events_per_gpu": len(seeds),
                       "l2": f"inputs and outputs rotate over {len(seeds)} events ({len(seeds) * n * 32 / 1e6:.0f} MB in + "
                             f"{len(seeds) * cap * 12 / 1e6:.0f} MB out > 126 MB L2); no explicit flush",
                       "grid": {"dims": dims, "bits": bits}, "edge_capacity": cap, "parallelism": f"events sharded over {rank.world_size} GPU(s), no collective"},
            "edges_per_event": e_mean, "roofline": roofline, "path_roofline": path_roofline, "phases_us": phases_us, "timeline_us": timeline_us,
            "cpu_baseline": cpu_baseline, "e2e": e2e, "next_rows": next_rows, "other_configs": other, "two_streams": two_streams, "gpu_launches": launches_per_step * args.steps,
            "gpu_launches_per_step": launches_per_step, "clocks": clocks,
            "host_wall_ms_per_step": 1e3 * (t1 - t0) / args.steps,
            "paper_context": "paper: 0.04 +- 0.01 s/event on V100 16 GB (PAPER.md:77 Table 1 'FRNN' column), TrackML events; other machine, other data",
        }
        print(json.dumps(line), flush=True)
    D.finalize(rank)


if __name__ == "__main__":
    main()
