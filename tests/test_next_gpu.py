"""GPU parity of frnn_gather_edge_rows and frnn_label_components (through the C ABI) against oracle/next_oracle.py.
Integer / byte work: bit-exact.  Inputs of the oracle never come from the CUDA path: the edge lists are the
FRNN oracle's (or seeded random graphs)."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from oracle import next_oracle as NO
from paper_2202_06929_b200 import events
from tests.test_next_oracle_pins import read_components_hand

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def F():
    from paper_2202_06929_b200 import frnn
    frnn.lib()
    return frnn


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def gpu_labels(F, n, src, dst, score=None, thr=0.0, **kw):
    lab, nc = F.frnn_label_components(n, dev(src), dev(dst), None if score is None else dev(score), thr, **kw)
    torch.cuda.synchronize()
    return lab.cpu().numpy(), int(nc.item())


# ---------------------------------------------------------------- f2: components
def test_components_hand_fixture(F):
    src, dst, score, labels, ncomp = read_components_hand()
    got, nc = gpu_labels(F, 10, src, dst, score, 0.5)
    assert np.array_equal(got, labels) and nc == ncomp


@pytest.mark.parametrize("cfg_idx", [0, 1, 2])
@pytest.mark.parametrize("thr", [None, 0.3, 0.9])
def test_components_on_frnn_graphs(F, cfg_idx, thr):
    """The workload shape of the paper: the radius graph of an event, edge scores, a threshold."""
    cfg = events.CONFIGS[cfg_idx]
    x = events.make_event(cfg)
    g = oracle.frnn(x, cfg.r, cfg.k_max, oracle.CELLS)
    score = None if thr is None else events.edge_scores(g.count, 11)
    exp, nc_exp = NO.label_components(cfg.n, g.src, g.dst, score, thr or 0.0)
    got, nc = gpu_labels(F, cfg.n, g.src, g.dst, score, thr or 0.0)
    assert np.array_equal(got, exp) and nc == nc_exp


def test_components_long_path_star_and_random(F):
    n = 200_000
    rng = np.random.default_rng(3)
    a = np.arange(n - 1, dtype=np.int32)
    p = rng.permutation(n - 1)
    got, nc = gpu_labels(F, n, (a + 1)[p], a[p])                       # a 200k-node path in scrambled order
    assert nc == 1 and not got.any()
    hub = np.full(n - 1, n - 1, np.int32)                               # a star whose hub is the LARGEST index
    got, nc = gpu_labels(F, n, hub, a)
    assert nc == 1 and not got.any()
    src, dst = events.random_graph(1_000_000, 700_000, 5)               # many components of every size
    exp, nc_exp = NO.label_components(1_000_000, src, dst)
    got, nc = gpu_labels(F, 1_000_000, src, dst)
    assert np.array_equal(got, exp) and nc == nc_exp


def test_components_rotating_label_arrays_replay_one_graph(F):
    """A consumer that writes every event's labels into a different array (here 80 of them, more than the 64 graph
    executables the library keeps) must not pay a graph build per call: the graph belongs to the stream and the
    labels pointer is one more node parameter.  Results are checked for every array."""
    n = 5000
    graphs = [events.random_graph(n, 3000 + 10 * k, 100 + k) for k in range(4)]
    exps = [NO.label_components(n, s, d) for s, d in graphs]
    dg = [(dev(s), dev(d)) for s, d in graphs]
    st = torch.cuda.Stream()
    labels = [torch.empty(n, dtype=torch.int32, device="cuda") for _ in range(80)]
    ncs = torch.zeros(80, dtype=torch.int32, device="cuda")
    torch.cuda.synchronize()
    F.frnn_label_components(n, *dg[0], labels=labels[0], n_components=ncs[0:1], stream=st)     # first call on this stream: may build
    b0 = F.frnn_graph_builds()
    for k in range(80):
        F.frnn_label_components(n, *dg[k % 4], labels=labels[k], n_components=ncs[k:k + 1], stream=st)
    st.synchronize()
    assert F.frnn_graph_builds() == b0
    for k in range(80):
        assert np.array_equal(labels[k].cpu().numpy(), exps[k % 4][0]) and int(ncs[k].item()) == exps[k % 4][1], k


def test_components_degenerate_and_device_count(F):
    got, nc = gpu_labels(F, 7, np.zeros(0, np.int32), np.zeros(0, np.int32))
    assert np.array_equal(got, np.arange(7)) and nc == 7
    got, nc = gpu_labels(F, 0, np.zeros(0, np.int32), np.zeros(0, np.int32))
    assert len(got) == 0 and nc == 0
    got, nc = gpu_labels(F, 3, np.array([0, 1, 7, -1], np.int32), np.array([0, 5, 1, 2], np.int32))
    assert nc == 3
    # only the first *edge_count edges count (device-side count, as left by frnn_build_ex)
    src, dst = np.array([0, 2, 4], np.int32), np.array([1, 3, 5], np.int32)
    cnt = torch.tensor([2], dtype=torch.int64, device="cuda")
    got, nc = gpu_labels(F, 6, src, dst, edge_count=cnt)
    assert list(got) == [0, 0, 2, 2, 4, 5] and nc == 4
    L = F.lib()
    lab = torch.zeros(4, dtype=torch.int32, device="cuda")
    assert L.frnn_label_components(-1, None, None, None, 0.0, None, 0, lab.data_ptr(), None, None) == F.FRNN_ERR_INVALID_ARG
    assert L.frnn_label_components(4, None, None, None, 0.0, None, 3, lab.data_ptr(), None, None) == F.FRNN_ERR_INVALID_ARG
    assert L.frnn_label_components(4, None, None, None, float("nan"), None, 0, lab.data_ptr(), None, None) == F.FRNN_OK


# ---------------------------------------------------------------- f4: gather
@pytest.mark.parametrize("cfg_idx", [0, 1])
def test_gather_whole_event(F, cfg_idx):
    cfg = events.CONFIGS[cfg_idx]
    x = events.make_event(cfg)
    g = oracle.frnn(x, cfg.r, cfg.k_max, oracle.CELLS)
    exp = NO.gather_edge_rows(x, g.src, g.dst)
    got = F.frnn_gather_edge_rows(dev(x), dev(g.src), dev(g.dst))
    torch.cuda.synchronize()
    assert np.array_equal(got.cpu().numpy().view(np.uint32), exp.view(np.uint32))


def test_gather_config4_in_batches_of_800k(F):
    """the filter is fed in batches of 800,000 edges.  Full size: 1.11 M edges of config 4, two batches;
    expected rows sampled (the oracle's loop is slow) plus the library-indexing identity on everything."""
    cfg = events.CONFIGS[4]
    x = events.make_event(cfg)
    g = oracle.frnn(x, cfg.r, cfg.k_max, oracle.CELLS)
    dx, ds, dd = dev(x), dev(g.src), dev(g.dst)
    cnt = torch.tensor([g.count], dtype=torch.int64, device="cuda")
    rng = np.random.default_rng(0)
    for e0 in range(0, g.count, 800_000):
        out = torch.full((800_000, 16), float("nan"), device="cuda")
        F.frnn_gather_edge_rows(dx, ds, dd, edge_count=cnt, e_begin=e0, e_max=800_000, out=out)
        torch.cuda.synchronize()
        m = min(800_000, g.count - e0)
        got = out.cpu().numpy()
        assert np.isnan(got[m:]).all()                                   # nothing written beyond the count
        assert np.array_equal(got[:m], np.concatenate([x[g.src[e0:e0 + m]], x[g.dst[e0:e0 + m]]], axis=1))
        for e in rng.integers(0, m, 200):
            assert np.array_equal(got[e], NO.gather_edge_rows(x, g.src, g.dst, e_begin=e0 + int(e), e_max=1)[0])


def test_gather_row_base_chunks_and_errors(F):
    x = events.uniform_points(100, 8, -1, 1, 0)
    src, dst = events.random_graph(50, 333, 2)
    exp = NO.gather_edge_rows(x, src, dst, e_begin=7, e_max=100, row_base=50)
    got = F.frnn_gather_edge_rows(dev(x), dev(src), dev(dst), e_begin=7, e_max=100, row_base=50)
    torch.cuda.synchronize()
    assert np.array_equal(got.cpu().numpy(), exp)
    assert F.frnn_gather_edge_rows(dev(x), dev(src), dev(dst), e_begin=0, e_max=0).shape == (0, 16)
    L = F.lib()
    dx, ds, dd = dev(x), dev(src), dev(dst)
    out = torch.empty((10, 16), device="cuda")
    assert L.frnn_gather_edge_rows(dx.data_ptr(), 100, 3, ds.data_ptr(), dd.data_ptr(), None, 0, 10, 0, out.data_ptr(), None) == F.FRNN_ERR_UNSUPPORTED
    assert L.frnn_gather_edge_rows(dx.data_ptr(), 100, 8, None, dd.data_ptr(), None, 0, 10, 0, out.data_ptr(), None) == F.FRNN_ERR_INVALID_ARG
    assert L.frnn_gather_edge_rows(dx.data_ptr() + 16, 99, 8, ds.data_ptr(), dd.data_ptr(), None, 0, 10, 0, out.data_ptr(), None) == F.FRNN_ERR_INVALID_ARG
    assert L.frnn_gather_edge_rows(dx.data_ptr(), 100, 8, ds.data_ptr(), dd.data_ptr(), None, -1, 10, 0, out.data_ptr(), None) == F.FRNN_ERR_INVALID_ARG


def test_chain_build_gather_label_without_host_sync(F):
    """The three calls chained on one stream with the edge count staying on the device."""
    cfg = events.CONFIGS[1]
    x = events.make_event(cfg)
    g = oracle.frnn(x, cfg.r, cfg.k_max, oracle.CELLS)
    pts = dev(x)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        res = F.frnn_build_ex(pts, cfg.r, cfg.k_max, edge_capacity=cfg.n * 8, stream=st)
        rows = torch.zeros((cfg.n * 8, 16), device="cuda")
        F.frnn_gather_edge_rows(pts, res.src, res.dst, edge_count=res.count, e_max=cfg.n * 8, out=rows, stream=st)
        lab, nc = F.frnn_label_components(cfg.n, res.src, res.dst, edge_count=res.count, edge_max=cfg.n * 8, stream=st)
    st.synchronize()
    assert res.n_edges() == g.count
    assert np.array_equal(rows[:g.count].cpu().numpy(), NO.gather_edge_rows(x, g.src, g.dst))
    exp, nc_exp = NO.label_components(cfg.n, g.src, g.dst)
    assert np.array_equal(lab.cpu().numpy(), exp) and int(nc.item()) == nc_exp


# ---------------------------------------------------------------- f1: the brute-force variant
def run_dense(F, x, r, k, capacity=None, want_row_ptr=False):
    pts = dev(x)
    res = F.frnn_build_dense_ex(pts, r, k, edge_capacity=capacity, want_row_ptr=want_row_ptr)
    torch.cuda.synchronize()
    return res


def same_as_oracle(res, exp):
    res.check()
    s, d, q = (t.cpu().numpy() for t in res.trimmed())
    assert np.array_equal(s, exp.src) and np.array_equal(d, exp.dst)
    assert np.array_equal(q.view(np.uint32), exp.d2.view(np.uint32))


@pytest.mark.parametrize("cfg_idx", [0, 1, 2])
def test_dense_configs(F, cfg_idx):
    """Config 2 at full size: 7.2e9 pair evaluations on the GPU against the cell-list oracle."""
    cfg = events.CONFIGS[cfg_idx]
    x = events.make_event(cfg)
    exp = oracle.frnn(x, cfg.r, cfg.k_max, oracle.CELLS)
    res = run_dense(F, x, cfg.r, cfg.k_max, capacity=cfg.n * 8, want_row_ptr=True)
    same_as_oracle(res, exp)
    rp = res.row_ptr.cpu().numpy()
    assert np.array_equal(np.diff(rp), np.minimum(exp.uncapped, cfg.k_max)) and rp[0] == 0


@pytest.mark.parametrize("k", [1, 7, 64, 4096])
def test_dense_one_cluster_k_cap(F, k):
    x = events.one_cluster(2000, 0.01, 3)
    same_as_oracle(run_dense(F, x, 0.1, k), oracle.frnn(x, 0.1, k, oracle.BRUTE))


@pytest.mark.parametrize("fac,k", [(1.0, 1024), (1.8, 1024), (1.8, 100), (1.8, 1)])
def test_dense_lattice_ties(F, fac, k):
    x = events.lattice(3, 8, 0.125)
    r = float(np.float32(fac * 0.125))
    same_as_oracle(run_dense(F, x, r, k), oracle.frnn(x, r, k, oracle.BRUTE))


@pytest.mark.parametrize("n", [0, 1, 2, 127, 128, 129, 300])
def test_dense_ragged_sizes_and_duplicates(F, n):
    x = events.uniform_points(max(n, 1), 8, -0.2, 0.2, n)[:n].copy()
    if n > 5:
        x[3] = x[0]; x[n - 1] = x[0]
    exp = oracle.frnn(x, 0.15, 5, oracle.BRUTE)
    res = run_dense(F, x, 0.15, 5, capacity=max(n * 5, 1))
    same_as_oracle(res, exp)
    same_as_oracle(run_dense(F, x, 0.0, 5, capacity=max(n * 5, 1)), oracle.frnn(x, 0.0, 5, oracle.BRUTE))


def test_dense_equals_grid_and_reports_capacity(F):
    cfg = events.CONFIGS[1]
    x = events.make_event(cfg, 9)
    pts = dev(x)
    a = F.frnn_build_ex(pts, cfg.r, 3)
    b = F.frnn_build_dense_ex(pts, cfg.r, 3)
    torch.cuda.synchronize()
    for u, v in zip(a.trimmed(), b.trimmed()):
        assert torch.equal(u, v)
    ws = F.Workspace(cfg.n, 1, cfg.k_max, 1000)
    res = F.frnn_build_dense_ex(pts, cfg.r, cfg.k_max, edge_capacity=1000, ws=ws)
    torch.cuda.synchronize()
    assert int(res.status.item()) == F.FRNN_ERR_CAPACITY and res.n_edges() == oracle.frnn(x, cfg.r, cfg.k_max).count
