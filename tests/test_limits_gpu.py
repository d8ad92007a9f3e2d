"""GPU parity at the edges of the size range (the brief's "maximum sizes"): an event several times larger than
BASELINE.json's largest config, checked on sampled queries the oracle computes one by one, and batched calls with more
events than one offsets chunk carries (500 events; the batched call takes them in one go).

Every comparison is bit for bit against the CPU oracle through the C ABI.
"""
from __future__ import annotations

import dataclasses

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
    frnn.frnn_set_bin_order(None)
    return frnn


def rows_of(res, queries):
    """(src, dst, d2) of the given query rows out of a device result that carries its CSR row_ptr"""
    rp = res.row_ptr.cpu().numpy()
    s, d, q = (t.cpu().numpy() for t in res.trimmed())
    sel = np.concatenate([np.arange(rp[i], rp[i + 1]) for i in queries]) if len(queries) else np.zeros(0, np.int64)
    return s[sel], d[sel], q[sel], rp


def test_six_million_point_event_on_sampled_queries(F):
    """config 4's recipe at six times its size (300,000 tracks): row indices, slot-buffer offsets (6 M x 256 B) and the
    2^25-cell table are far beyond anything the timed configs reach.  The oracle answers 3,000 sampled queries against
    all six million points; the device result is compared on exactly those rows, and its global invariants are checked."""
    base = events.CONFIGS[4]
    cfg = dataclasses.replace(base, n=6_000_000, n_tracks=300_000)
    x = events.make_event(cfg, 11)
    k = 4                                               # binds on some rows (mean degree 1.1, maximum about 11)
    pts = torch.from_numpy(x).cuda()
    res = F.frnn_build_ex(pts, cfg.r, k, edge_capacity=cfg.n * 4, want_row_ptr=True)
    torch.cuda.synchronize()
    res.check()
    rng = np.random.default_rng(3)
    queries = np.sort(rng.choice(cfg.n, 3000, replace=False))
    queries = np.concatenate([[0], queries[(queries > 0) & (queries < cfg.n - 1)], [cfg.n - 1]])
    exp = oracle.frnn(x, cfg.r, k, oracle.CELLS, queries=queries)
    s, d, q, rp = rows_of(res, queries)
    assert np.array_equal(s, exp.src) and np.array_equal(d, exp.dst), "edges of the sampled rows differ from the oracle"
    assert np.array_equal(H.bits(q), H.bits(exp.d2)), "d2 of the sampled rows differs from the oracle"
    assert np.array_equal(np.diff(rp)[queries], np.minimum(exp.uncapped, k))
    # properties that hold at any size: sorted, no self pairs, within the radius, degrees capped, count = last offset
    sa, da, qa = (t.cpu().numpy() for t in res.trimmed())
    assert rp[0] == 0 and rp[-1] == len(sa) == res.n_edges()
    assert np.all(np.diff(rp) <= k) and np.all(np.diff(rp) >= 0)
    key = sa.astype(np.int64) * cfg.n + da
    assert np.all(np.diff(key) > 0), "raw output is not strictly (src, dst)-sorted"
    assert np.all(sa != da) and np.all(qa <= np.float32(cfg.r) * np.float32(cfg.r))
    assert np.array_equal(np.repeat(np.arange(cfg.n, dtype=np.int32), np.diff(rp)), sa)


@pytest.mark.parametrize("n_events", [129, 300])
def test_batched_call_with_more_events_than_one_offsets_chunk(F, n_events):
    """Event offsets reach the device 128 at a time as kernel arguments: 129 and 300 events take two and three chunks.
    Ragged sizes (0 .. 900 rows), empty events at both ends and in the middle."""
    cfg = events.CONFIGS[0]
    rng = np.random.default_rng(n_events)
    sizes = rng.integers(0, 900, n_events)
    sizes[[0, n_events // 2, n_events - 1]] = 0
    sizes[1] = 1
    pool = [events.make_event(cfg, 40 + s) for s in range(4)]
    parts = [pool[e % 4][rng.integers(0, cfg.n - 900):][:sizes[e]] for e in range(n_events)]
    x = np.ascontiguousarray(np.concatenate(parts))
    offs = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    for k in (64, 2):
        exp, eoffs = oracle.frnn_batched(x, offs, cfg.r, k)
        res = F.frnn_build_batched(torch.from_numpy(x).cuda(), offs, cfg.r, k, want_row_ptr=True)
        torch.cuda.synchronize()
        res.check()
        assert np.array_equal(res.count.cpu().numpy(), eoffs)
        s, d, q = (t.cpu().numpy() for t in res.trimmed())
        assert np.array_equal(s, exp.src) and np.array_equal(d, exp.dst) and np.array_equal(H.bits(q), H.bits(exp.d2))
        rp = res.row_ptr.cpu().numpy()
        assert rp[-1] == exp.count and np.all(np.diff(rp) <= k)
