"""GPU parity of what a STREAM of real events exercises (section 3: the latency "depends almost linearly
on the number of spacepoints" -- no two events have the same size; 500 different events):

  * one workspace, one graph, > 128 calls that all differ in n and in their input / output buffers;
  * the K cap when it binds (section 3.1: the paper's Faiss path asks for k neighbours, then cuts at r):
    rows resolved from their slot buffer (K < count <= 32), rows collected once and selected by a bitonic network
    (32 < count <= 512), rows beyond the staging capacity;
  * two host threads, each with its own stream and workspace;
  * the end-to-end entry points (frnn_host_pipeline_*, frnn_build_host) at the size bench.py times them;
  * per-call options instead of process-wide setters, and the data-driven grid (frnn_suggest_grid).

Every comparison is bit for bit against the CPU oracle through the C ABI.
"""
from __future__ import annotations

import dataclasses
import threading

import numpy as np
import pytest

import oracle
from paper_2202_06929_b200 import events
from tests import helpers as H
from tests.test_parity_gpu import Got, assert_same

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def F():
    from paper_2202_06929_b200 import frnn
    frnn.lib()
    frnn.frnn_set_grid(0, 0)
    frnn.frnn_set_bin_order(None)
    return frnn


def host_result(res):
    s, d, q = (t.cpu().numpy() for t in res.trimmed())
    return Got(s, d, q)


def tight_clusters(sizes, seed, spread=0.004, dim=8):
    """Clusters so tight (spread << r = 0.1) and so far apart that every row's neighbours are exactly its cluster mates:
    the count of a row is its cluster size - 1."""
    rng = np.random.default_rng(seed)
    parts = []
    for k, m in enumerate(sizes):
        centre = rng.uniform(-1, 1, dim)
        centre[0] = -0.9 + 1.8 * (k + 0.5) / len(sizes) if len(sizes) < 16 else centre[0]
        parts.append(centre + rng.normal(0, spread, (m, dim)))
    x = np.concatenate(parts).astype(np.float32)
    return np.ascontiguousarray(x[rng.permutation(len(x))])


# ---------------------------------------------------------------- item 1: the graph does not depend on the call
def test_more_than_128_distinct_sizes_through_one_workspace(F):
    """150 calls, each with its own n (all distinct), rotating over 5 input and 3 output buffer sets, ONE workspace and
    stream: the library must replay one graph (same launch count, no rebuild) and every result must equal the oracle."""
    cfg = events.CONFIGS[1]
    n_max = 24000
    rng = np.random.default_rng(11)
    sizes = rng.choice(np.arange(16500, n_max), size=150, replace=False)      # one grid class (16,384 <= n < 400,000)
    base = [events.make_event(dataclasses.replace(cfg, n=n_max, n_tracks=2150), 300 + s) for s in range(5)]
    dev_in = [torch.from_numpy(b).cuda() for b in base]
    cap = n_max * 8
    stream = torch.cuda.Stream()
    ws = F.Workspace(n_max, 1, cfg.k_max, cap)
    outs = [F.Workspace(64, 1, cfg.k_max, cap) for _ in range(3)]
    for o in outs:
        o.buf = ws.buf
    results = []
    launch_counts = set()
    builds = []
    for i, n in enumerate(sizes):
        o = outs[i % 3]
        res = F.frnn_build_ex(dev_in[i % 5][:n], cfg.r, cfg.k_max, ws=o, stream=stream)
        launch_counts.add(F.frnn_last_launch_count())
        builds.append(F.frnn_graph_builds())
        if i % 3 == 2 or i == len(sizes) - 1:                                  # the three output sets are full: check them
            stream.synchronize()
            for j in range(i - (i % 3), i + 1):
                r_ = outs[j % 3]
                e = int(r_.count.item())
                assert int(r_.status.item()) == 0
                results.append((j, r_.src[:e].cpu().numpy(), r_.dst[:e].cpu().numpy(), r_.d2[:e].cpu().numpy()))
    assert launch_counts == {6}, launch_counts                                 # memset + 5 kernels, every time
    assert builds[-1] == builds[0], "the graph was rebuilt although only n and the buffers changed"
    assert len(results) == 150
    for j, s, d, q in results:
        n = sizes[j]
        exp = oracle.frnn(base[j % 5][:n], cfg.r, cfg.k_max, oracle.CELLS)
        assert_same(Got(s, d, q), exp, cfg.r, f"call {j} n={n}")


def test_sizes_across_grid_classes_and_back(F):
    """n jumping between the grid classes (g = 3 below 16,384 rows, g = 4 above) on ONE workspace: two graphs, reused."""
    cfg = events.CONFIGS[1]
    x = events.make_event(cfg)
    pts = torch.from_numpy(x).cuda()
    ws = F.Workspace(cfg.n, 1, cfg.k_max, cfg.n * 8)
    need3 = F.frnn_workspace_bytes(16000, 1, 8, cfg.k_max)
    assert need3 <= ws.buf.numel()
    st = torch.cuda.Stream()
    b0 = F.frnn_graph_builds()
    for n in (20000, 5000, 17000, 16383, 16384, 1, 2, 300, 19999):
        res = F.frnn_build_ex(pts[:n], cfg.r, cfg.k_max, ws=ws, stream=st)
        st.synchronize()
        res.check()
        assert_same(host_result(res), oracle.frnn(x[:n], cfg.r, cfg.k_max, oracle.CELLS), cfg.r, f"n={n}")
    assert F.frnn_graph_builds() - b0 <= 2                                     # one graph per grid class, reused (none if an earlier
                                                                               # workspace at this address left them behind)


def test_batched_calls_with_changing_offsets_replay_one_graph(F):
    cfg = events.CONFIGS[0]
    evs = [events.make_event(cfg, 40 + e) for e in range(6)]
    st = torch.cuda.Stream()
    total_max = 6 * cfg.n
    ws = F.Workspace(total_max, 6, 5, total_max * 5)
    rng = np.random.default_rng(3)
    b0 = None
    for trial in range(5):
        sizes = rng.integers(0, cfg.n, 6)
        x = np.ascontiguousarray(np.concatenate([e[:m] for e, m in zip(evs, sizes)]))
        offs = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
        if len(x) == 0:
            continue
        need = F.frnn_workspace_bytes(len(x), 6, 8, 5)
        assert need <= ws.buf.numel()
        res = F.frnn_build_batched(torch.from_numpy(x).cuda(), offs, cfg.r, 5, ws=ws, stream=st)
        st.synchronize()
        res.check()
        exp, eoffs = oracle.frnn_batched(x, offs, cfg.r, 5)
        assert np.array_equal(res.count.cpu().numpy(), eoffs)
        s, d, q = (t.cpu().numpy() for t in res.trimmed())
        assert np.array_equal(s, exp.src) and np.array_equal(d, exp.dst) and np.array_equal(H.bits(q), H.bits(exp.d2))
        b0 = F.frnn_graph_builds() if b0 is None else b0
    assert F.frnn_graph_builds() == b0                                         # the offsets changed, the graph did not


def test_plain_launch_mode_and_graph_mode_agree(F):
    cfg = events.CONFIGS[0]
    x = events.make_event(cfg, 9)
    pts = torch.from_numpy(x).cuda()
    exp = oracle.frnn(x, cfg.r, 3)
    st = torch.cuda.Stream()
    for mode in (F.FRNN_LAUNCH_PLAIN, F.FRNN_LAUNCH_GRAPH):
        res = F.frnn_build_ex(pts, cfg.r, 3, stream=st, opt=F.frnn_options(launch_mode=mode))
        st.synchronize()
        res.check()
        assert_same(host_result(res), exp, cfg.r, f"launch mode {mode}")


# ---------------------------------------------------------------- item 2: S8 when K binds
@pytest.mark.parametrize("k", [1, 5, 15, 16, 17, 31, 32, 33, 64])
def test_counts_straddling_the_slot_buffer(F, k):
    """Rows with 7..44 neighbours (cluster sizes 8..45): counts on both sides of the 32 hit slots per row (and of 16, a layout that was tried), K on
    both sides of the counts -- small, medium (from the slot buffer) and big (recomputed, staged, selected) rows in the same tiles."""
    x = tight_clusters(list(range(8, 46)) * 2, 5)
    exp = oracle.frnn(x, 0.1, k, oracle.BRUTE)
    assert exp.uncapped.min() == 7 and exp.uncapped.max() == 44
    res = F.frnn_build_ex(torch.from_numpy(x).cuda(), 0.1, k)
    torch.cuda.synchronize()
    res.check()
    assert_same(host_result(res), exp, 0.1, f"straddle K={k}")


@pytest.mark.parametrize("k", [2, 4, 8])
def test_config1_with_a_binding_k(F, k):
    cfg = events.CONFIGS[1]
    x = events.make_event(cfg)
    exp = oracle.frnn(x, cfg.r, k, oracle.CELLS)
    assert (exp.uncapped > k).sum() > (100 if k == 8 else 1000)
    res = F.frnn_build_ex(torch.from_numpy(x).cuda(), cfg.r, k)
    torch.cuda.synchronize()
    res.check()
    assert_same(host_result(res), exp, cfg.r, f"cfg1 K={k}")


@pytest.mark.parametrize("k", [2, 4])
def test_config2_full_size_with_a_binding_k(F, k):
    """The K-binding bench leg's workload at its own size: 120,000 points, a quarter of the rows over K = 4."""
    cfg = events.CONFIGS[2]
    x = events.make_event(cfg)
    exp = oracle.frnn(x, cfg.r, k, oracle.CELLS)
    assert (exp.uncapped > k).sum() > 20000
    res = F.frnn_build_ex(torch.from_numpy(x).cuda(), cfg.r, k, edge_capacity=cfg.n * k, want_row_ptr=True)
    torch.cuda.synchronize()
    res.check()
    assert_same(host_result(res), exp, cfg.r, f"cfg2 K={k}")
    assert np.array_equal(np.diff(res.row_ptr.cpu().numpy()), np.minimum(exp.uncapped, k))


@pytest.mark.parametrize("k", [1, 64, 200, 512, 600])
def test_dense_rows_staged_and_beyond_staging(F, k):
    """Counts 99..699: up to 512 the row is collected once and selected by the bitonic network; beyond, the bisection
    fallback.  Heavy d2 ties are added by duplicating points (d2 = 0 many times: the index tie-break decides)."""
    x = tight_clusters([100, 257, 400, 513, 700, 33, 512], 8)
    x[:40] = x[40:80]                                       # exact duplicates: ties at d2 = 0 and equal d2 to third points
    exp = oracle.frnn(x, 0.1, k, oracle.BRUTE)
    assert exp.uncapped.max() > 600 and exp.uncapped.min() < 40
    for entry in (F.frnn_build_ex, F.frnn_build_dense_ex):
        res = entry(torch.from_numpy(x).cuda(), 0.1, k)
        torch.cuda.synchronize()
        res.check()
        assert_same(host_result(res), exp, 0.1, f"dense rows K={k} {entry.__name__}")


def test_dense_event_every_row_selected(F):
    """A dense event (mean degree ~200, K = 64: the regime BASELINE.json's config 4 parenthetical describes): 200 tracks
    of ~200 hits; every row goes through the staged selection."""
    rng = np.random.default_rng(21)
    sizes = rng.poisson(200, 100)
    x = tight_clusters(list(sizes), 22, spread=0.02)
    exp = oracle.frnn(x, 0.1, 64, oracle.CELLS)
    assert np.mean(exp.uncapped) > 120 and (exp.uncapped > 64).mean() > 0.9
    res = F.frnn_build_ex(torch.from_numpy(x).cuda(), 0.1, 64)
    torch.cuda.synchronize()
    res.check()
    assert_same(host_result(res), exp, 0.1, "dense event K=64")


def test_capacity_overflow_with_selected_rows(F):
    x = tight_clusters([40, 300, 600], 2)
    exp = oracle.frnn(x, 0.1, 20, oracle.BRUTE)
    cap = exp.count // 2
    pts = torch.from_numpy(x).cuda()
    ws = F.Workspace(len(x), 1, 20, cap)
    guard_lo = torch.full((1024,), -7, dtype=torch.int32, device="cuda")
    res = F.frnn_build_ex(pts, 0.1, 20, edge_capacity=cap, ws=ws)
    torch.cuda.synchronize()
    assert int(res.status.item()) == F.FRNN_ERR_CAPACITY and res.n_edges() == exp.count
    assert torch.all(guard_lo == -7)


# ---------------------------------------------------------------- item 6: threads, end-to-end entry points
def test_two_host_threads_with_their_own_stream_and_workspace(F):
    """include/frnn.h: calls on distinct workspaces may run concurrently from different host threads.  Two threads, 100
    interleaved calls each with different n, every result compared with the oracle afterwards."""
    cfg = events.CONFIGS[0]
    n_max = 6000
    base = [events.make_event(dataclasses.replace(cfg, n=n_max, n_tracks=540), 500 + t) for t in range(2)]
    exps, gots, errors = [{}, {}], [{}, {}], []

    def worker(t):
        try:
            torch.cuda.set_device(0)
            rng = np.random.default_rng(70 + t)
            st = torch.cuda.Stream()
            pts = torch.from_numpy(base[t]).cuda()
            ws = F.Workspace(n_max, 1, 7, n_max * 7)
            for i in range(100):
                n = int(rng.integers(2000, n_max))
                k = 7 if i % 2 else 2
                res = F.frnn_build_ex(pts[:n], cfg.r, k, ws=ws, stream=st)
                st.synchronize()
                res.check()
                gots[t][i] = (n, k, host_result(res))
        except Exception as exc:                         # noqa: BLE001
            errors.append(exc)

    threads = [threading.Thread(target=worker, args=(t,)) for t in range(2)]
    for th in threads:
        th.start()
    for th in threads:
        th.join()
    assert not errors, errors
    for t in range(2):
        assert len(gots[t]) == 100
        for i, (n, k, got) in gots[t].items():
            assert_same(got, oracle.frnn(base[t][:n], cfg.r, k, oracle.CELLS), cfg.r, f"thread {t} call {i}")


def test_host_pipeline_at_tracking_scale_with_ragged_events(F):
    """The path bench.py's e2e figure runs on: depth 4, 12 events of different sizes around 120k, pinned and pageable
    outputs, compared with the oracle bit for bit."""
    cfg = events.CONFIGS[2]
    cap = cfg.n * 8
    pipe = F.HostPipeline(cfg.n, cfg.k_max, cap, depth=4)
    rng = np.random.default_rng(4)
    full = [events.make_event(cfg, 60 + i) for i in range(3)]
    sizes = [int(v) for v in rng.integers(90000, cfg.n + 1, 12)]
    sizes[5] = cfg.n
    xs = [np.ascontiguousarray(full[i % 3][:m]) for i, m in enumerate(sizes)]
    pins = [torch.from_numpy(x).pin_memory() for x in xs]

    def bufs(pinned, packed):
        mk = (lambda t: t.pin_memory()) if pinned else (lambda t: t)
        if packed:                                         # src | dst | d2 in one block: the library sends them as one 2-D copy
            blk = mk(torch.empty(3 * cap + 64, dtype=torch.int32))
            return blk[:cap], blk[cap + 32:2 * cap + 32], blk[2 * cap + 64:].view(torch.float32), mk(torch.zeros(1, dtype=torch.int64))
        return (mk(torch.empty(cap, dtype=torch.int32)), mk(torch.empty(cap, dtype=torch.int32)), mk(torch.empty(cap, dtype=torch.float32)),
                mk(torch.zeros(1, dtype=torch.int64)))
    outs = [bufs(pinned=(i % 4 != 3), packed=(i % 3 != 0)) for i in range(12)]
    for p, o in zip(pins, outs):
        pipe.submit(p, cfg.r, *o)
    pipe.wait()
    pipe.close()
    for i, (x, (s, d, q, c)) in enumerate(zip(xs, outs)):
        exp = oracle.frnn(x, cfg.r, cfg.k_max, oracle.CELLS)
        e = int(c.item())
        assert e == exp.count
        assert_same(Got(s[:e].numpy(), d[:e].numpy(), q[:e].numpy()), exp, cfg.r, f"pipeline event {i} n={len(x)}")


def test_build_host_at_tracking_scale_and_unaligned_host_rows(F):
    cfg = events.CONFIGS[2]
    x = events.make_event(cfg, 77)
    exp = oracle.frnn(x, cfg.r, cfg.k_max, oracle.CELLS)
    cap = cfg.n * 8
    hs, hd, hq = torch.empty(cap, dtype=torch.int32), torch.empty(cap, dtype=torch.int32), torch.empty(cap, dtype=torch.float32)
    e = F.frnn_build_host(torch.from_numpy(x), cfg.r, cfg.k_max, hs, hd, hq)
    assert_same(Got(hs[:e].numpy(), hd[:e].numpy(), hq[:e].numpy()), exp, cfg.r, "frnn_build_host 120k")
    blk = torch.empty(3 * cap, dtype=torch.int32).pin_memory()         # equally spaced outputs: one 2-D copy
    ps, pd, pq = blk[:cap], blk[cap:2 * cap], blk[2 * cap:].view(torch.float32)
    e = F.frnn_build_host(torch.from_numpy(x).pin_memory(), cfg.r, cfg.k_max, ps, pd, pq)
    assert_same(Got(ps[:e].numpy(), pd[:e].numpy(), pq[:e].numpy()), exp, cfg.r, "frnn_build_host 120k, packed outputs")
    # a host array whose rows start 4 bytes past a 32-byte boundary: only the device fast path needs the alignment
    raw = torch.empty(cfg.n * 8 + 16, dtype=torch.float32)
    off = 1 + (-(raw.data_ptr() // 4)) % 8
    assert (raw.data_ptr() + 4 * off) % 32 == 4
    shifted = raw[off:off + cfg.n * 8].view(cfg.n, 8)
    shifted.copy_(torch.from_numpy(x))
    e2 = F.frnn_build_host(shifted, cfg.r, cfg.k_max, hs, hd, hq)
    assert e2 == exp.count and np.array_equal(hs[:e2].numpy(), exp.src) and np.array_equal(hd[:e2].numpy(), exp.dst)


# ---------------------------------------------------------------- item 3: options and the data-driven grid
@pytest.mark.parametrize("dims,bits,order", [(1, 8, None), (2, 7, None), (3, 6, [5, 1, 7]), (4, 4, None), (5, 3, [2, 3]), (6, 2, None),
                                             (2, 8, [7, 0]), (3, 3, None)])
def test_grid_invariance_through_options(F, dims, bits, order):
    cfg = events.CONFIGS[1]
    x = events.make_event(cfg)[:7000]
    exp = oracle.frnn(x, cfg.r, 6, oracle.CELLS)
    opt = F.frnn_options(dims, bits, order)
    res = F.frnn_build_ex(torch.from_numpy(x).cuda(), cfg.r, 6, opt=opt)
    torch.cuda.synchronize()
    res.check()
    assert_same(host_result(res), exp, cfg.r, f"options grid {dims}x{bits} order {order}")
    assert F.frnn_get_grid(len(x)) == (3, 5)                                   # the process defaults were not touched


def test_options_errors(F):
    pts = torch.zeros((16, 8), device="cuda")
    for bad in (F.frnn_options(7, 5), F.frnn_options(3, 9), F.frnn_options(3, 1), F.frnn_options(0, 0, [1, 1]), F.frnn_options(0, 0, [16])):
        with pytest.raises(F.FrnnError):
            F.frnn_build_ex(pts, 0.1, 4, opt=bad)
    small = F.frnn_options()
    small.struct_bytes = 8
    with pytest.raises(F.FrnnError):
        F.frnn_build_ex(pts, 0.1, 4, opt=small)
    # a workspace sized for the default grid is too small for a finer one: reported, nothing enqueued
    ws = F.Workspace(16, 1, 4, 64)
    with pytest.raises(F.FrnnError) as ei:
        F.frnn_build_ex(pts, 0.1, 4, ws=ws, opt=F.frnn_options(3, 8))
    assert ei.value.status == F.FRNN_ERR_WORKSPACE


def spread_event(n, extent, seed, offset=0.0, sigma=0.03):
    """Tracking-shaped clusters over [offset - extent/2, offset + extent/2]^8."""
    rng = np.random.default_rng(seed)
    tracks = n // 10
    c = rng.uniform(-extent / 2, extent / 2, (tracks, 8))
    x = c[rng.integers(0, tracks, n)] + rng.normal(0, sigma, (n, 8)) + offset
    return np.ascontiguousarray(x.astype(np.float32))


@pytest.mark.parametrize("extent,r,offset", [(20.0, 0.1, 0.0), (2.0, 0.1, 1001.0), (2.0, 0.02, 0.0), (2.0, 0.3, 0.0)])
def test_suggested_grid_on_wide_offset_and_fine_data(F, extent, r, offset):
    """extent / r = 200 (more cells than any table row holds: aliasing), data offset to [1000, 1002] (the torus needs no
    origin), r = 0.02 and r = 0.3 on the usual cube: the suggested grid gives the oracle's result, as does the default."""
    n = 40000
    x = spread_event(n, extent, 31, offset, sigma=0.3 * r)
    exp = oracle.frnn(x, r, 32, oracle.CELLS)
    assert exp.count > 1000
    pts = torch.from_numpy(x).cuda()
    tried_opts = [None]
    for measure in (False, True):
        opt, rep = F.frnn_suggest_grid(pts, r, measure=measure)
        assert 1 <= opt.grid_dims <= 6 and 2 <= opt.grid_bits <= 8
        assert (1 << (opt.grid_dims * opt.grid_bits)) <= 64 * n
        ext = extent / (np.float32(r) * np.float32(1.0078125))
        assert abs(rep.extent_cells[0] - ext) < 0.15 * ext + 2
        if measure:
            tried = rep.tried()
            assert 1 <= len(tried) <= 12 and rep.measured_us > 0
            assert rep.measured_us == min(t["measured_us"] for t in tried)         # the fastest of the shortlist was taken
            assert any(t["grid_dims"] == opt.grid_dims and t["grid_bits"] == opt.grid_bits for t in tried)
            print(f"[suggest] extent {extent} r {r}: ({opt.grid_dims},{opt.grid_bits}) {rep.measured_us:.1f} us of {tried}")
        else:
            assert rep.n_tried == 0
        tried_opts.append(opt)
    for o in tried_opts:
        res = F.frnn_build_ex(pts, r, 32, opt=o)
        torch.cuda.synchronize()
        res.check()
        assert_same(host_result(res), exp, r, f"extent {extent} r {r} offset {offset} opt {'suggested' if o else 'default'}")


def test_grid_chosen_per_call_from_the_event_itself(F):
    """grid_dims = FRNN_GRID_AUTO: every call looks at its own rows first.  One workspace (sized for any grid the call may
    pick), events whose extent / r differs by two orders of magnitude following each other: every result is the oracle's."""
    n = 30000
    opt = F.frnn_options(F.FRNN_GRID_AUTO)
    ws = F.Workspace(n, 1, 32, n * 40, opt=opt)
    assert ws.buf.numel() >= F.frnn_workspace_bytes(n, 1, 8, 32)
    st = torch.cuda.Stream()
    for extent, r, offset in ((2.0, 0.1, 0.0), (20.0, 0.1, 0.0), (2.0, 0.02, 0.0), (2.0, 0.3, 0.0), (2.0, 0.1, 1001.0), (2.0, 0.1, 0.0)):
        x = spread_event(n, extent, 77, offset, sigma=0.3 * r)
        exp = oracle.frnn(x, r, 32, oracle.CELLS)
        res = F.frnn_build_ex(torch.from_numpy(x).cuda(), r, 32, ws=ws, stream=st, opt=opt)
        st.synchronize()
        res.check()
        assert_same(host_result(res), exp, r, f"auto grid extent {extent} r {r} offset {offset}")
    # batched, and tiny events
    cfg = events.CONFIGS[0]
    xb = np.ascontiguousarray(np.concatenate([events.make_event(cfg, 3)[:900], events.make_event(cfg, 4)[:17], events.make_event(cfg, 5)]))
    offs = np.array([0, 900, 917, 917 + cfg.n], np.int64)
    expb, eoffs = oracle.frnn_batched(xb, offs, cfg.r, 6)
    resb = F.frnn_build_batched(torch.from_numpy(xb).cuda(), offs, cfg.r, 6, opt=opt)
    torch.cuda.synchronize()
    resb.check()
    assert np.array_equal(resb.count.cpu().numpy(), eoffs)
    s_, d_, q_ = (t.cpu().numpy() for t in resb.trimmed())
    assert np.array_equal(s_, expb.src) and np.array_equal(d_, expb.dst) and np.array_equal(H.bits(q_), H.bits(expb.d2))
    for m in (1, 2, 40):
        xs = events.make_event(cfg, 6)[:m]
        res = F.frnn_build_ex(torch.from_numpy(xs).cuda(), cfg.r, 4, opt=opt)
        torch.cuda.synchronize()
        res.check()
        assert_same(host_result(res), oracle.frnn(xs, cfg.r, 4, oracle.BRUTE), cfg.r, f"auto grid n={m}")


def test_batched_config3_subset_with_suggested_and_odd_grids(F):
    """Four of config 3's events in one batched call, through the measured suggestion and through two hand-picked grids."""
    cfg = events.CONFIGS[2]
    evs = [events.make_event(cfg, 100 + e)[: cfg.n - 1000 * e] for e in range(4)]
    x = np.ascontiguousarray(np.concatenate(evs))
    offs = np.concatenate([[0], np.cumsum([len(e) for e in evs])]).astype(np.int64)
    exp, eoffs = oracle.frnn_batched(x, offs, cfg.r, cfg.k_max)
    pts = torch.from_numpy(x).cuda()
    sug, rep = F.frnn_suggest_grid(pts, cfg.r, n_events=4, measure=True)
    assert rep.n_tried >= 1
    for opt in (sug, F.frnn_options(3, 6), F.frnn_options(5, 4, [7, 6, 5, 4, 3])):
        res = F.frnn_build_batched(pts, offs, cfg.r, cfg.k_max, edge_capacity=len(x) * 4, opt=opt)
        torch.cuda.synchronize()
        res.check()
        assert np.array_equal(res.count.cpu().numpy(), eoffs)
        s_, d_, q_ = (t.cpu().numpy() for t in res.trimmed())
        assert np.array_equal(s_, exp.src) and np.array_equal(d_, exp.dst) and np.array_equal(H.bits(q_), H.bits(exp.d2))


def test_suggest_grid_statistics_match_a_numpy_histogram(F):
    """The probabilities frnn_suggest_grid reports are those of the folded cell histogram of the points it sampled."""
    cfg = events.CONFIGS[1]
    x = events.make_event(cfg)
    r = cfg.r
    opt, rep = F.frnn_suggest_grid(torch.from_numpy(x).cuda(), r)
    assert rep.sampled == cfg.n
    side = float(np.float32(1.0) / (np.float32(1.0) / (np.float32(r) * np.float32(1.0078125))))
    for d in range(8):
        c = np.floor(x[:, d].astype(np.float64) / side).astype(np.int64)
        for bits, got in ((opt.grid_bits, rep.pair_probability[d]), (6, rep.key_probability[d])):
            m = 1 << bits
            p = np.bincount(c & (m - 1), minlength=m) / cfg.n
            s = float(np.sum(p * (np.roll(p, 1) + p + np.roll(p, -1))))
            assert abs(got - s) < 2e-3 * s + 1e-6, (d, bits, got, s)
    assert rep.pair_probability[8] == 1.0
