"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element.

Bar (BASELINE.json north_star): identical edge set after sorting with d2 in the same fixed fp32
order -- here the library's raw output must already be (src,dst)-sorted, so arrays are compared
as they are, d2 bitwise.  The only tolerated exception is pairs with |d2 - r2| <= 1e-6*r2, which
``compare_edges`` returns and the tests print; with the pinned order the expected number is zero.
"""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from paper_2202_06929_b200 import events
from tests import helpers as H

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def F():
    from paper_2202_06929_b200 import frnn
    frnn.lib()
    frnn.frnn_set_grid(0, 0)
    return frnn


class Got:
    def __init__(self, src, dst, d2):
        self.src, self.dst, self.d2 = src, dst, d2


def run_gpu(F, x, r, k, capacity=None, want_row_ptr=False):
    pts = torch.from_numpy(np.ascontiguousarray(x)).cuda()
    res = F.frnn_build_ex(pts, r, k, edge_capacity=capacity, want_row_ptr=want_row_ptr)
    torch.cuda.synchronize()
    res.check()
    s, d, q = res.trimmed()
    return Got(s.cpu().numpy(), d.cpu().numpy(), q.cpu().numpy()), res


def assert_same(got, exp, r, label):
    H.assert_sorted_unique(got.src, got.dst)
    band, n_d2 = H.compare_edges(got, exp, r, label)
    if band or n_d2:
        print(f"[band report] {label}: {len(band)} band edge(s) {band[:10]}, {n_d2} d2 value(s) differ within 1e-6")
    assert not band, f"{label}: membership differs inside the tolerance band (must be reported): {band[:10]}"
    assert n_d2 == 0, f"{label}: {n_d2} d2 values differ bitwise"
    assert np.array_equal(got.src, exp.src) and np.array_equal(got.dst, exp.dst)
    assert np.array_equal(H.bits(got.d2), H.bits(exp.d2))


# ---------------------------------------------------------------- BASELINE configs, full size
@pytest.mark.parametrize("cfg_idx", [0, 1, 2])
def test_config_single_event(F, cfg_idx):
    cfg = events.CONFIGS[cfg_idx]
    x = events.make_event(cfg)
    exp = oracle.frnn(x, cfg.r, cfg.k_max, oracle.CELLS)
    got, res = run_gpu(F, x, cfg.r, cfg.k_max, capacity=cfg.n * 8, want_row_ptr=True)
    assert_same(got, exp, cfg.r, cfg.name)
    rp = res.row_ptr.cpu().numpy()
    assert np.array_equal(np.diff(rp), np.minimum(exp.uncapped, cfg.k_max)) and rp[0] == 0


def test_config3_batched_16_events(F):
    cfg = events.CONFIGS[3]
    x, offs = events.make_batch(cfg)
    exp, eoffs = oracle.frnn_batched(x, offs, cfg.r, cfg.k_max)
    pts = torch.from_numpy(x).cuda()
    res = F.frnn_build_batched(pts, offs, cfg.r, cfg.k_max, edge_capacity=len(x) * 4)
    torch.cuda.synchronize()
    res.check()
    got_offs = res.count.cpu().numpy()
    assert np.array_equal(got_offs, eoffs)
    s, d, q = (t.cpu().numpy() for t in res.trimmed())
    for e in range(cfg.n_events):
        sl = slice(eoffs[e], eoffs[e + 1])
        assert_same(Got(s[sl], d[sl], q[sl]), Got(exp.src[sl], exp.dst[sl], exp.d2[sl]), cfg.r, f"{cfg.name}[{e}]")


def test_config4_dense_1m(F):
    cfg = events.CONFIGS[4]
    x = events.make_event(cfg)
    exp = oracle.frnn(x, cfg.r, cfg.k_max, oracle.CELLS)
    got, _ = run_gpu(F, x, cfg.r, cfg.k_max, capacity=cfg.n * 4)
    assert_same(got, exp, cfg.r, cfg.name)


# ---------------------------------------------------------------- fixtures and closed forms through the GPU
@pytest.mark.parametrize("section,k", [("uncapped", 4), ("uncapped", 64), ("k2", 2)])
def test_handcase_golden(F, section, k):
    src, dst, d2 = H.read_handcase(section)
    got, _ = run_gpu(F, H.HANDCASE_POINTS, 0.5, k)
    assert np.array_equal(got.src, src) and np.array_equal(got.dst, dst)
    assert np.array_equal(H.bits(got.d2), H.bits(d2))


@pytest.mark.parametrize("L", [2, 3])
@pytest.mark.parametrize("fac", [1.0, 1.1, 1.5, 1.8])
def test_lattice_closed_form(F, L, fac):
    from tests.test_oracle_pins import lattice_closed_form
    x = events.lattice(L, 8, 0.125)
    r = float(np.float32(fac * 0.125))
    got, _ = run_gpu(F, x, r, 1024)
    assert len(got.src) == lattice_closed_form(L, 8, fac)
    assert_same(got, oracle.frnn(x, r, 1024, oracle.BRUTE), r, f"lattice L={L} fac={fac}")


@pytest.mark.parametrize("k", [512, 100, 16, 1])
def test_lattice_k_truncation(F, k):
    """S8 with heavy d2 ties: 576 in-radius neighbours in three exact shells at the centre."""
    x = events.lattice(3, 8, 0.125)
    r = float(np.float32(1.8 * 0.125))
    got, _ = run_gpu(F, x, r, k)
    assert_same(got, oracle.frnn(x, r, k, oracle.BRUTE), r, f"lattice K={k}")


@pytest.mark.parametrize("k", [1, 7, 64, 4096])
def test_one_cluster_every_query_overflows(F, k):
    x = events.one_cluster(2000, 0.01, 3)
    exp = oracle.frnn(x, 0.1, k, oracle.BRUTE)
    if k <= 64:
        assert exp.uncapped.min() > k            # S8 on every row
    got, _ = run_gpu(F, x, 0.1, k)
    assert_same(got, exp, 0.1, f"one cluster K={k}")


@pytest.mark.parametrize("cfg_idx", [0, 1])
@pytest.mark.parametrize("k", [1, 2, 4])
def test_small_k_on_configs(F, cfg_idx, k):
    cfg = events.CONFIGS[cfg_idx]
    x = events.make_event(cfg)
    got, _ = run_gpu(F, x, cfg.r, k)
    assert_same(got, oracle.frnn(x, cfg.r, k, oracle.CELLS), cfg.r, f"{cfg.name} K={k}")


# ---------------------------------------------------------------- the result must not depend on the grid
@pytest.mark.parametrize("dims,bits", [(1, 5), (2, 5), (3, 5), (4, 5), (5, 5), (6, 4), (3, 2), (4, 3), (2, 8)])
def test_grid_invariance(F, dims, bits):
    cfg = events.CONFIGS[1]
    x = events.make_event(cfg)[:6000]
    exp = oracle.frnn(x, cfg.r, 5, oracle.CELLS)
    try:
        F.frnn_set_grid(dims, bits)
        assert F.frnn_get_grid(len(x)) == (dims, bits)
        got, _ = run_gpu(F, x, cfg.r, 5)
    finally:
        F.frnn_set_grid(0, 0)
    assert_same(got, exp, cfg.r, f"grid dims={dims} bits={bits}")


def test_far_from_origin_and_clamped_cells(F):
    """Coordinates beyond the +-2^15-cell clamp pile up in boundary cells: slower, still exact.
    The oracle sees the same fp32 inputs."""
    cfg = events.CONFIGS[0]
    base = events.make_event(cfg)
    for shift in (50.0, 5000.0):
        x = (base + np.float32(shift)).astype(np.float32)
        got, _ = run_gpu(F, x, cfg.r, cfg.k_max)
        assert_same(got, oracle.frnn(x, cfg.r, cfg.k_max, oracle.BRUTE), cfg.r, f"shift {shift}")
    x = (base * np.float32(1000.0)).astype(np.float32)
    got, _ = run_gpu(F, x, 100.0, cfg.k_max)
    assert_same(got, oracle.frnn(x, 100.0, cfg.k_max, oracle.BRUTE), 100.0, "scaled x1000")


# ---------------------------------------------------------------- degenerate inputs and error behaviour
def test_r_zero_finds_exact_duplicates(F):
    x = events.make_event(events.CONFIGS[0]).copy()
    x[100] = x[7]; x[2000] = x[7]; x[3000] = x[11]
    got, _ = run_gpu(F, x, 0.0, 4)
    assert_same(got, oracle.frnn(x, 0.0, 4, oracle.BRUTE), 0.0, "r=0")
    assert len(got.src) == 8


@pytest.mark.parametrize("n", [0, 1, 2, 31, 32, 33])
def test_tiny_n(F, n):
    x = np.zeros((n, 8), np.float32)
    got, _ = run_gpu(F, x, 0.1, 3, capacity=max(n * 3, 1))
    exp = oracle.frnn(x, 0.1, 3, oracle.BRUTE)
    assert np.array_equal(got.src, exp.src) and np.array_equal(got.dst, exp.dst)


def test_capacity_overflow_is_reported_not_fatal(F):
    cfg = events.CONFIGS[0]
    x = events.make_event(cfg)
    exp = oracle.frnn(x, cfg.r, cfg.k_max)
    pts = torch.from_numpy(x).cuda()
    cap = 1000
    ws = F.Workspace(cfg.n, 1, cfg.k_max, cap)
    guard = torch.full((64,), -7, dtype=torch.int32, device="cuda")
    res = F.frnn_build_ex(pts, cfg.r, cfg.k_max, edge_capacity=cap, ws=ws)
    torch.cuda.synchronize()
    assert int(res.status.item()) == F.FRNN_ERR_CAPACITY
    assert res.n_edges() == exp.count                    # the needed size
    assert torch.all(guard == -7)
    with pytest.raises(F.FrnnError):
        res.check()


def test_host_detectable_errors(F):
    pts = torch.zeros((16, 8), device="cuda")
    L = F.lib()
    ws = F.Workspace(16, 1, 4, 64)
    args = lambda **kw: dict(dict(p=pts.data_ptr(), n=16, dim=8, r=0.1, k=4, cap=64), **kw)

    def call(p, n, dim, r, k, cap, wsbytes=None):
        return L.frnn_build_ex(p, n, dim, r, k, ws.src.data_ptr(), ws.dst.data_ptr(), ws.d2.data_ptr(), cap,
                               ws.count.data_ptr(), ws.status.data_ptr(), None, ws.buf.data_ptr(),
                               ws.buf.numel() if wsbytes is None else wsbytes, None)
    assert call(**args()) == F.FRNN_OK
    assert call(**args(n=-1)) == F.FRNN_ERR_INVALID_ARG
    assert call(**args(r=-0.5)) == F.FRNN_ERR_INVALID_ARG
    assert call(**args(r=float("nan"))) == F.FRNN_ERR_INVALID_ARG
    assert call(**args(r=float("inf"))) == F.FRNN_ERR_INVALID_ARG
    assert call(**args(k=0)) == F.FRNN_ERR_INVALID_ARG
    assert call(**args(p=None)) == F.FRNN_ERR_INVALID_ARG
    assert call(**args(p=pts.data_ptr() + 16)) == F.FRNN_ERR_INVALID_ARG      # rows must be 32-byte aligned
    assert call(**args(dim=17)) == F.FRNN_ERR_UNSUPPORTED
    assert call(**args(dim=0)) == F.FRNN_ERR_UNSUPPORTED
    assert call(**args(), wsbytes=128) == F.FRNN_ERR_WORKSPACE
    torch.cuda.synchronize()
    assert "capacity" in F.frnn_status_string(F.FRNN_ERR_CAPACITY)


def test_sync_nine_argument_form_and_host_form(F):
    cfg = events.CONFIGS[0]
    x = events.make_event(cfg)
    exp = oracle.frnn(x, cfg.r, cfg.k_max)
    s, d, q = F.frnn_build(torch.from_numpy(x).cuda(), cfg.r, cfg.k_max)
    assert_same(Got(s.cpu().numpy(), d.cpu().numpy(), q.cpu().numpy()), exp, cfg.r, "frnn_build")
    hp = torch.from_numpy(x).pin_memory()
    cap = cfg.n * 8
    hs = torch.empty(cap, dtype=torch.int32).pin_memory()
    hd = torch.empty(cap, dtype=torch.int32).pin_memory()
    hq = torch.empty(cap, dtype=torch.float32).pin_memory()
    e = F.frnn_build_host(hp, cfg.r, cfg.k_max, hs, hd, hq)
    assert_same(Got(hs[:e].numpy(), hd[:e].numpy(), hq[:e].numpy()), exp, cfg.r, "frnn_build_host")


def test_batched_ragged_events_with_empty_ones(F):
    cfg = events.CONFIGS[0]
    parts = [events.make_event(cfg, 5)[:1000], np.zeros((0, 8), np.float32), events.make_event(cfg, 6)[:33],
             events.make_event(cfg, 7), np.zeros((1, 8), np.float32)]
    x = np.concatenate(parts)
    offs = np.concatenate([[0], np.cumsum([len(p) for p in parts])]).astype(np.int64)
    exp, eoffs = oracle.frnn_batched(x, offs, cfg.r, 3)
    res = F.frnn_build_batched(torch.from_numpy(x).cuda(), offs, cfg.r, 3)
    torch.cuda.synchronize()
    res.check()
    assert np.array_equal(res.count.cpu().numpy(), eoffs)
    s, d, q = (t.cpu().numpy() for t in res.trimmed())
    assert np.array_equal(s, exp.src) and np.array_equal(d, exp.dst) and np.array_equal(H.bits(q), H.bits(exp.d2))


def test_repeated_calls_reuse_workspace_and_are_deterministic(F):
    cfg = events.CONFIGS[1]
    x = events.make_event(cfg)
    pts = torch.from_numpy(x).cuda()
    ws = F.Workspace(cfg.n, 1, cfg.k_max, cfg.n * 8)
    outs = []
    for _ in range(3):
        res = F.frnn_build_ex(pts, cfg.r, cfg.k_max, ws=ws)
        torch.cuda.synchronize()
        outs.append(tuple(t.cpu().numpy().copy() for t in res.trimmed()))
    for o in outs[1:]:
        assert all(np.array_equal(a, b) for a, b in zip(o, outs[0]))
    assert F.frnn_last_launch_count() >= 6


def test_timeline_mode_gives_the_same_result_and_ordered_stamps(F):
    """Profiling mode 2: kernels stamp %globaltimer into the workspace; results are unchanged."""
    cfg = events.CONFIGS[1]
    x = events.make_event(cfg)
    exp = oracle.frnn(x, cfg.r, cfg.k_max, oracle.CELLS)
    pts = torch.from_numpy(x).cuda()
    ws = F.Workspace(cfg.n, 1, cfg.k_max, cfg.n * 8)
    st = torch.cuda.Stream()
    try:
        F.frnn_set_profiling(2)
        res = F.frnn_build_ex(pts, cfg.r, cfg.k_max, ws=ws, stream=st)
        st.synchronize()
        tl = F.frnn_get_timeline(ws.buf, cfg.n, 1)
    finally:
        F.frnn_set_profiling(0)
    s, d, q = (t.cpu().numpy() for t in res.trimmed())
    assert_same(Got(s, d, q), exp, cfg.r, "timeline mode")
    names = list(tl)
    assert names == ["bin", "scan_cells", "scatter", "search", "emit"]
    assert tl["bin"][0] == 0.0
    for a, b in zip(names, names[1:]):
        assert tl[a][0] <= tl[a][1] <= tl[b][0] + 1e-9, (a, b, tl)        # kernels of one call are serialised
    assert tl["emit"][1] < 1e5                                            # microseconds, not garbage


@pytest.mark.parametrize("how", ["grid_3x6", "grid_2x8_order", "auto"])
def test_timeline_of_calls_made_with_options(F, how):
    """The stamps sit at the head of the workspace, so frnn_get_timeline reads them whatever grid, coordinate order or
    launch options the call was made with (it used to derive their offset from the process defaults)."""
    cfg = events.CONFIGS[1]
    x = events.make_event(cfg)
    exp = oracle.frnn(x, cfg.r, cfg.k_max, oracle.CELLS)
    pts = torch.from_numpy(x).cuda()
    opt = {"grid_3x6": F.frnn_options(3, 6, timeline=True), "grid_2x8_order": F.frnn_options(2, 8, order=[5, 2, 7], timeline=True),
           "auto": F.frnn_options(F.FRNN_GRID_AUTO, timeline=True)}[how]
    assert F.frnn_workspace_bytes(cfg.n, 1, 8, cfg.k_max, opt) != F.frnn_workspace_bytes(cfg.n, 1, 8, cfg.k_max)
    ws = F.Workspace(cfg.n, 1, cfg.k_max, cfg.n * 8, opt=opt)
    st = torch.cuda.Stream()
    res = F.frnn_build_ex(pts, cfg.r, cfg.k_max, ws=ws, stream=st, opt=opt)
    st.synchronize()
    tl = F.frnn_get_timeline(ws.buf, cfg.n, 1)
    s, d, q = (t.cpu().numpy() for t in res.trimmed())
    assert_same(Got(s, d, q), exp, cfg.r, "timeline with options: " + how)
    names = list(tl)
    assert names == ["bin", "scan_cells", "scatter", "search", "emit"]
    assert tl["bin"][0] == 0.0
    for a, b in zip(names, names[1:]):
        assert tl[a][0] < tl[a][1] <= tl[b][0] + 1e-9, (a, b, tl)
    assert 1.0 < tl["emit"][1] < 1e5                                      # microseconds of a real call, not garbage


def test_host_pipeline_overlapped_events(F):
    """frnn_host_pipeline_*: seven events through three slots, results in pinned host buffers, count on the host."""
    cfg = events.CONFIGS[0]
    cap = cfg.n * 8
    pipe = F.HostPipeline(cfg.n, cfg.k_max, cap, depth=3)
    xs = [events.make_event(cfg, 20 + i)[: cfg.n - 37 * i] for i in range(7)]
    pins = [torch.from_numpy(x).pin_memory() for x in xs]
    outs = [(torch.empty(cap, dtype=torch.int32).pin_memory(), torch.empty(cap, dtype=torch.int32).pin_memory(),
             torch.empty(cap, dtype=torch.float32).pin_memory(), torch.zeros(1, dtype=torch.int64).pin_memory()) for _ in xs]
    for p, o in zip(pins, outs):
        pipe.submit(p, cfg.r, *o)
    pipe.wait()
    for x, (s, d, q, c) in zip(xs, outs):
        exp = oracle.frnn(x, cfg.r, cfg.k_max)
        e = int(c.item())
        assert e == exp.count
        assert_same(Got(s[:e].numpy(), d[:e].numpy(), q[:e].numpy()), exp, cfg.r, "host pipeline")
    # capacity overflow is reported through the count word; pageable outputs work too
    small = F.HostPipeline(cfg.n, cfg.k_max, 1000, depth=1)
    small.submit(pins[0], cfg.r, *outs[0])
    small.wait()
    assert int(outs[0][3].item()) == -oracle.frnn(xs[0], cfg.r, cfg.k_max).count - 1
    pageable = (torch.empty(cap, dtype=torch.int32), torch.empty(cap, dtype=torch.int32), torch.empty(cap, dtype=torch.float32),
                torch.zeros(1, dtype=torch.int64))
    pipe.submit(torch.from_numpy(xs[1]), cfg.r, *pageable)
    pipe.wait()
    exp1 = oracle.frnn(xs[1], cfg.r, cfg.k_max)
    e1 = int(pageable[3].item())
    assert e1 == exp1.count and np.array_equal(pageable[0][:e1].numpy(), exp1.src) and np.array_equal(pageable[1][:e1].numpy(), exp1.dst)
    small.close()
    pipe.close()


def test_canaries_around_workspace_and_outputs(F):
    """compute-sanitizer is closed on this GPU pool, so out-of-bounds WRITES are hunted with canaries: the workspace
    and the three output arrays sit inside larger buffers filled with a pattern that must survive every call."""
    L = F.lib()
    cases = [(events.make_event(events.CONFIGS[0]), 0.1, 64), (events.make_event(events.CONFIGS[1]), 0.1, 3),
             (events.one_cluster(2000, 0.01, 3), 0.1, 7), (events.lattice(3, 8, 0.125), float(np.float32(1.8 * 0.125)), 100)]
    pad = 4096
    for x, r, k in cases:
        n = len(x)
        exp = oracle.frnn(x, r, k, oracle.BRUTE if n <= 7000 else oracle.CELLS)
        cap = exp.count                                                   # exactly enough room
        wsb = F.frnn_workspace_bytes(n, 1, 8, k)
        big_ws = torch.full((wsb + 2 * pad,), 0xA5, dtype=torch.uint8, device="cuda")
        outs = [torch.full((cap + 2 * 1024,), -7, dtype=torch.int32, device="cuda") for _ in range(3)]
        pts = torch.from_numpy(x).cuda()
        cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
        stat = torch.zeros(1, dtype=torch.int32, device="cuda")
        for entry in (L.frnn_build_ex, L.frnn_build_dense_ex):
            rc = entry(pts.data_ptr(), n, 8, r, k, outs[0][1024:].data_ptr(), outs[1][1024:].data_ptr(), outs[2][1024:].data_ptr(), cap,
                       cnt.data_ptr(), stat.data_ptr(), None, big_ws[pad:].data_ptr(), wsb, None)
            torch.cuda.synchronize()
            assert rc == 0 and int(stat.item()) == 0 and int(cnt.item()) == cap
            assert bool((big_ws[:pad] == 0xA5).all()) and bool((big_ws[pad + wsb:] == 0xA5).all()), "write outside the workspace"
            for o in outs:
                assert bool((o[:1024] == -7).all()) and bool((o[1024 + cap:] == -7).all()), "write outside an output array"
            assert np.array_equal(outs[0][1024:1024 + cap].cpu().numpy(), exp.src)
            assert np.array_equal(outs[1][1024:1024 + cap].cpu().numpy(), exp.dst)


def test_non_finite_coordinates_cannot_fault(F):
    """include/frnn.h: non-finite coordinates are a precondition violation but can never cause an out-of-bounds
    access.  The result is unspecified for the affected rows; the call must complete, report a consistent count and
    leave the rows that are far from every poisoned point exactly right."""
    cfg = events.CONFIGS[0]
    x = events.make_event(cfg).copy()
    x[5, 0] = np.nan; x[77, 3] = np.inf; x[300, 7] = -np.inf; x[1000] = np.nan; x[2000, :4] = 3e38
    for entry in (F.frnn_build_ex, F.frnn_build_dense_ex):
        res = entry(torch.from_numpy(x).cuda(), cfg.r, cfg.k_max, edge_capacity=cfg.n * 8, want_row_ptr=True)
        torch.cuda.synchronize()
        res.check()
        e = res.n_edges()
        rp = res.row_ptr.cpu().numpy()
        assert rp[0] == 0 and rp[-1] == e and np.all(np.diff(rp) >= 0)
        s, d, _ = (t.cpu().numpy() for t in res.trimmed())
        assert s.min() >= 0 and s.max() < cfg.n and d.min() >= 0 and d.max() < cfg.n
        bad = np.zeros(cfg.n, bool); bad[[5, 77, 300, 1000, 2000]] = True
        clean = events.make_event(cfg)
        exp = oracle.frnn(clean, cfg.r, cfg.k_max)
        keep_e = ~(bad[exp.src] | bad[exp.dst])
        keep_g = ~(bad[s] | bad[d])
        assert np.array_equal(s[keep_g], exp.src[keep_e]) and np.array_equal(d[keep_g], exp.dst[keep_e])


# ---------------------------------------------------------------- embedding dimensions below 8
@pytest.mark.parametrize("dim", [1, 2, 3, 4, 5, 6, 7, 9, 12, 15, 16])
@pytest.mark.parametrize("entry", ["frnn_build_ex", "frnn_build_dense_ex"])
def test_other_dimensions(F, dim, entry):
    """Rows of dim != 8 floats (unaligned stride): padded with zeros internally (dim > 8: a second internal row for
    coordinates 8..15), d2 over dim terms bit for bit."""
    n = 3000
    x = events.uniform_points(n, dim, -1.0, 1.0, 40 + dim)
    r = {1: 0.002, 2: 0.03, 3: 0.1, 4: 0.2, 5: 0.3, 6: 0.4, 7: 0.5, 9: 0.65, 12: 1.05, 15: 1.35, 16: 1.4}[dim]
    for k in (3, 64):
        exp = oracle.frnn(x, r, k, oracle.BRUTE)
        assert exp.count > 500
        res = getattr(F, entry)(torch.from_numpy(x).cuda(), r, k)
        torch.cuda.synchronize()
        res.check()
        s_, d_, q_ = (t.cpu().numpy() for t in res.trimmed())
        assert_same(Got(s_, d_, q_), exp, r, f"dim={dim} K={k}")


@pytest.mark.parametrize("L,D,fac", [(4, 4, 1.0), (4, 4, 1.5), (4, 4, 1.8), (5, 3, 1.0), (5, 3, 1.5), (5, 3, 1.8)])
def test_lattice_closed_form_low_dim(F, L, D, fac):
    from tests.test_oracle_pins import lattice_closed_form
    x = events.lattice(L, D, 0.125)
    r = float(np.float32(fac * 0.125))
    got, _ = run_gpu(F, x, r, 1024)
    assert len(got.src) == lattice_closed_form(L, D, fac)
    assert_same(got, oracle.frnn(x, r, 1024, oracle.BRUTE), r, f"lattice L={L} D={D} fac={fac}")


@pytest.mark.parametrize("dim", [12, 16])
def test_clustered_event_in_higher_dimension(F, dim):
    """A tracking-shaped event in a 12- or 16-dimensional embedding: tight clusters + uniform noise, K binding on some rows."""
    rng = np.random.default_rng(dim)
    centres = rng.uniform(-1, 1, (1500, dim))
    sig = centres[rng.integers(0, 1500, 18000)] + rng.normal(0, 0.03, (18000, dim))
    x = np.ascontiguousarray(np.concatenate([sig, rng.uniform(-1, 1, (2000, dim))]).astype(np.float32)[rng.permutation(20000)])
    r = 0.03 * np.sqrt(2 * dim) * 0.9
    for k in (256, 4):
        exp = oracle.frnn(x, r, k, oracle.CELLS)
        assert exp.count > 20000
        got, _ = run_gpu(F, x, r, k, capacity=exp.count + 8)
        assert_same(got, exp, r, f"clustered dim={dim} K={k}")


# ---------------------------------------------------------------- which coordinates are binned
@pytest.mark.parametrize("order", [[7, 6, 5, 4, 3, 2, 1, 0], [4, 5, 6, 7], [3], [2, 9, 0, 15, 1], [1, 3, 5, 7, 0, 2, 4, 6]])
def test_bin_order_never_changes_the_result(F, order):
    cfg = events.CONFIGS[1]
    x = events.make_event(cfg)[:8000]
    exp = oracle.frnn(x, cfg.r, 6, oracle.CELLS)
    try:
        F.frnn_set_bin_order(order)
        got, _ = run_gpu(F, x, cfg.r, 6)
    finally:
        F.frnn_set_bin_order(None)
    assert_same(got, exp, cfg.r, f"bin order {order}")


def test_suggested_bin_order_on_an_anisotropic_embedding(F):
    """An embedding whose first four coordinates carry almost no spread: binning them prunes nothing.  The suggested
    order must rank the four wide coordinates first, give the same result, and be much faster than the default."""
    rng = np.random.default_rng(5)
    n, tracks = 60000, 6000
    centres = rng.uniform(-1, 1, (tracks, 8))
    centres[:, :4] *= 0.02                                               # squeezed coordinates
    x = centres[rng.integers(0, tracks, n)] + rng.normal(0, 0.02, (n, 8))
    x = np.ascontiguousarray(x.astype(np.float32))
    r, k = 0.08, 64
    exp = oracle.frnn(x, r, k, oracle.BRUTE)
    pts = torch.from_numpy(x).cuda()
    order, score = F.frnn_suggest_bin_order(pts, r)
    assert sorted(order[:4]) == [4, 5, 6, 7], (order, score)
    assert all(score[d] > 0.9 for d in range(4)) and all(score[d] < 0.3 for d in range(4, 8)) and score[8] == 2.0

    def timed():
        ws = F.Workspace(n, 1, k, exp.count + 8)
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            for _ in range(3):
                res = F.frnn_build_ex(pts, r, k, ws=ws, stream=st)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(st)
            for _ in range(10):
                res = F.frnn_build_ex(pts, r, k, ws=ws, stream=st)
            b.record(st)
            st.synchronize()
        res.check()
        s, d, q = (t.cpu().numpy() for t in res.trimmed())
        return a.elapsed_time(b) / 10, Got(s, d, q)

    t_default, got_default = timed()
    try:
        F.frnn_set_bin_order(order)
        t_suggested, got_suggested = timed()
    finally:
        F.frnn_set_bin_order(None)
    assert_same(got_default, exp, r, "anisotropic, default order")
    assert_same(got_suggested, exp, r, "anisotropic, suggested order")
    print(f"[bin order] default {t_default:.3f} ms, suggested {order} {t_suggested:.3f} ms")
    assert t_suggested < 0.5 * t_default


@pytest.mark.parametrize("dim,order", [(5, None), (12, None), (12, [9, 3, 11, 0, 5]), (8, [6, 2])])
def test_batched_other_dims_and_bin_orders(F, dim, order):
    """The batched entry point with dim != 8 and with a caller-chosen bin order (ragged events, an empty one)."""
    rng = np.random.default_rng(100 + dim)
    sizes = [1500, 0, 37, 2600, 1]
    parts = []
    for m in sizes:
        c = rng.uniform(-1, 1, (max(m // 8, 1), dim))
        parts.append((c[rng.integers(0, len(c), m)] + rng.normal(0, 0.03, (m, dim))).astype(np.float32))
    x = np.ascontiguousarray(np.concatenate(parts))
    offs = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    r = 0.03 * np.sqrt(2 * dim)
    exp, eoffs = oracle.frnn_batched(x, offs, r, 5)
    assert eoffs[-1] > 3000
    try:
        F.frnn_set_bin_order(order)
        res = F.frnn_build_batched(torch.from_numpy(x).cuda(), offs, r, 5)
        torch.cuda.synchronize()
    finally:
        F.frnn_set_bin_order(None)
    res.check()
    assert np.array_equal(res.count.cpu().numpy(), eoffs)
    s, d, q = (t.cpu().numpy() for t in res.trimmed())
    assert np.array_equal(s, exp.src) and np.array_equal(d, exp.dst) and np.array_equal(H.bits(q), H.bits(exp.d2))
