"""Pins for the CPU oracle (oracle/frnn_oracle.c) against things other than itself.

Each pin is chosen so that a plausible mistake in the oracle (strict instead of inclusive radius,
a dropped coordinate, wrong summation order, no fused multiply-add, self pairs kept, wrong K order,
a missed neighbour cell) fails at least one of them.  SURVEY.md section 8(c) P1..P7.
"""
from __future__ import annotations

import math
from itertools import product

import numpy as np
import pytest

import oracle
from paper_2202_06929_b200 import events
from tests import helpers as H

MODES = [oracle.BRUTE, oracle.CELLS]
H_LAT = 0.125


# ---------------------------------------------------------------- hand-worked fixture (tests/golden)
@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("section,k", [("uncapped", 4), ("uncapped", 64), ("k2", 2)])
def test_handcase_golden(mode, section, k):
    src, dst, d2 = H.read_handcase(section)
    res = oracle.frnn(H.HANDCASE_POINTS, 0.5, k, mode)
    assert np.array_equal(res.src, src)
    assert np.array_equal(res.dst, dst)
    assert np.array_equal(H.bits(res.d2), H.bits(d2))
    assert res.uncapped.tolist() == [3, 4, 4, 2, 3, 0]


# ---------------------------------------------------------------- summation order (R3), exact rationals
def test_d2_order_matches_exact_rational_fma_chain():
    rng = np.random.default_rng(123)
    n_diff_muladd = n_diff_rev = 0
    for _ in range(300):
        a = rng.uniform(-1, 1, 8).astype(np.float32)
        b = (a + rng.normal(0, 0.03, 8)).astype(np.float32)
        got = oracle.d2(a, b)
        exp = H.d2_exact_chain(a, b)
        assert H.bits(got) == H.bits(exp), (a, b, got, exp)
        n_diff_muladd += H.bits(H.d2_exact_mul_add(a, b)) != H.bits(exp)
        n_diff_rev += H.bits(H.d2_exact_chain(a[::-1], b[::-1])) != H.bits(exp)
    # the sample must be able to tell the pinned order from the two plausible wrong ones
    assert n_diff_muladd > 20 and n_diff_rev > 20


def test_d2_symmetric_bitwise():
    rng = np.random.default_rng(5)
    for _ in range(200):
        a = rng.uniform(-1, 1, 8).astype(np.float32)
        b = rng.uniform(-1, 1, 8).astype(np.float32)
        assert H.bits(oracle.d2(a, b)) == H.bits(oracle.d2(b, a))


# ---------------------------------------------------------------- closed-form lattice counts (P3)
def lattice_closed_form(L, D, fac):
    e1 = 2 * D * (L - 1) * L ** (D - 1)
    e2 = 4 * math.comb(D, 2) * (L - 1) ** 2 * L ** (D - 2)
    e3 = 8 * math.comb(D, 3) * (L - 1) ** 3 * L ** (D - 3) if D >= 3 else 0
    return e1 + (e2 if fac * fac >= 2 else 0) + (e3 if fac * fac >= 3 else 0)


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("L,D", [(2, 8), (3, 8), (4, 4), (5, 3)])
@pytest.mark.parametrize("fac", [1.0, 1.1, 1.5, 1.8])
def test_lattice_edge_counts(mode, L, D, fac):
    """r = h EXACTLY must count the axis neighbours (pins <=); r in [h*sqrt2, h*sqrt3) adds the face
    diagonals; r in [h*sqrt3, 2h) adds the cube diagonals.  Counts are closed forms."""
    x = events.lattice(L, D, H_LAT)
    r = np.float32(fac * H_LAT)
    res = oracle.frnn(x, r, 10 ** 6, mode)
    assert res.count == lattice_closed_form(L, D, fac)
    # every d2 is an exact small multiple of h^2
    m = res.d2 / np.float32(H_LAT * H_LAT)
    assert np.array_equal(m, np.round(m)) and m.min() >= 1 and m.max() <= 3
    if L == 2:      # every point of the 2^D lattice is a corner: uniform degree
        per = {1.0: D, 1.1: D, 1.5: D + math.comb(D, 2), 1.8: D + math.comb(D, 2) + math.comb(D, 3)}[fac]
        assert np.all(res.uncapped == per)
    H.assert_sorted_unique(res.src, res.dst)


def lattice_integer_reference(L, D, max_sq, k):
    """Independent integer brute force on lattice indices: in radius iff sum (ci-cj)^2 <= max_sq;
    keep the k smallest by (integer d2, j); list by j."""
    g = np.array(list(product(range(L), repeat=D)), dtype=np.int64)
    n = len(g)
    src, dst, dsq = [], [], []
    for i in range(n):
        q = ((g - g[i]) ** 2).sum(1)
        j = np.flatnonzero((q <= max_sq) & (np.arange(n) != i))
        if len(j) > k:
            order = np.lexsort((j, q[j]))[:k]
            j = np.sort(j[order])
        src.append(np.full(len(j), i)); dst.append(j); dsq.append(q[j])
    return np.concatenate(src), np.concatenate(dst), np.concatenate(dsq)


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("k", [512, 100, 16, 1])
def test_lattice_k_truncation_order(mode, k):
    """P4: D=8, L=3, r=1.8h.  The centre point has 576 in-radius neighbours in three exact distance
    shells (16, 112, 448): heavy ties, so the (d2, j) order decides.  Expected values come from an
    integer computation on lattice indices."""
    L, D = 3, 8
    x = events.lattice(L, D, H_LAT)
    res = oracle.frnn(x, np.float32(1.8 * H_LAT), k, mode)
    s, d, q = lattice_integer_reference(L, D, 3, k)
    assert np.array_equal(res.src, s) and np.array_equal(res.dst, d)
    assert np.array_equal(res.d2, (q * (H_LAT * H_LAT)).astype(np.float32))
    centre = (3 ** 8 - 1) // 2
    assert res.uncapped[centre] == 576 and res.uncapped.max() == 576


# ---------------------------------------------------------------- float64 library routine (cKDTree)
@pytest.mark.parametrize("cfg_idx", [0, 1])
def test_against_ckdtree_float64(cfg_idx):
    """The uncapped radius graph from scipy's k-d tree in float64 must equal the oracle's edge set
    except for pairs inside the 1e-6*r2 band; d2 within 1e-6 relative."""
    from scipy.spatial import cKDTree
    cfg = events.CONFIGS[cfg_idx]
    x = events.make_event(cfg)
    res = oracle.frnn(x, cfg.r, cfg.k_max, oracle.CELLS)
    assert res.uncapped.max() <= cfg.k_max          # K does not bind: capped == uncapped
    x64 = x.astype(np.float64)
    r2 = float(np.float32(cfg.r) * np.float32(cfg.r))
    pairs = cKDTree(x64).query_pairs(cfg.r * 1.001, output_type="ndarray")
    d64 = ((x64[pairs[:, 0]] - x64[pairs[:, 1]]) ** 2).sum(1)
    sure_in = d64 < r2 * (1 - 1e-6)
    sure_out = d64 > r2 * (1 + 1e-6)
    have = set(H.edge_keys(res.src, res.dst).tolist())
    for a, b in ((0, 1), (1, 0)):
        k = H.edge_keys(pairs[:, a].astype(np.int32), pairs[:, b].astype(np.int32))
        assert all(int(v) in have for v in k[sure_in])
        assert not any(int(v) in have for v in k[sure_out])
    n_band = int((~sure_in & ~sure_out).sum())
    assert res.count >= 2 * sure_in.sum() and res.count <= 2 * (sure_in.sum() + n_band)
    # distances
    lut = {int(k): v for k, v in zip(H.edge_keys(pairs[:, 0].astype(np.int32), pairs[:, 1].astype(np.int32)), d64)}
    sel = np.flatnonzero(res.src < res.dst)[:5000]
    ref = np.array([lut[int(k)] for k in H.edge_keys(res.src[sel], res.dst[sel])])
    assert np.max(np.abs(res.d2[sel] - ref) / ref) < 1e-6


# ---------------------------------------------------------------- tiny random sets vs numpy float64 (P6)
@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("seed", range(6))
def test_tiny_random_vs_numpy(mode, seed):
    rng = np.random.default_rng(1000 + seed)
    n = int(rng.integers(8, 65))
    x = rng.uniform(-0.2, 0.2, (n, 8)).astype(np.float32)
    r = 0.4
    res = oracle.frnn(x, r, 10 ** 6, mode)
    x64 = x.astype(np.float64)
    d = ((x64[:, None, :] - x64[None, :, :]) ** 2).sum(-1)
    r2 = float(np.float32(r) * np.float32(r))
    np.fill_diagonal(d, np.inf)
    assert not np.any(np.abs(d - r2) <= 1e-6 * r2), "band pair in a tiny set: change the seed"
    i, j = np.nonzero(d <= r2)
    assert np.array_equal(res.src, i) and np.array_equal(res.dst, j)
    assert 0 < len(i) < n * (n - 1), "degenerate sample: change the seed"
    assert np.max(np.abs(res.d2 - d[i, j]) / d[i, j]) < 1e-6


# ---------------------------------------------------------------- mode A == mode B bitwise (P2)
def same(a, b):
    return (np.array_equal(a.src, b.src) and np.array_equal(a.dst, b.dst)
            and np.array_equal(H.bits(a.d2), H.bits(b.d2)) and np.array_equal(a.uncapped, b.uncapped))


@pytest.mark.parametrize("r", [0.0, 0.05, 0.1, 0.3])
@pytest.mark.parametrize("k", [1, 4, 64])
def test_brute_equals_cells_cfg0(r, k):
    x = events.make_event(events.CONFIGS[0]).copy()
    x[100] = x[7]; x[2000] = x[7]; x[3000] = x[11]        # exact duplicates: the only r = 0 edges
    a = oracle.frnn(x, r, k, oracle.BRUTE)
    b = oracle.frnn(x, r, k, oracle.CELLS)
    assert same(a, b)
    if r == 0.0:
        assert a.count == (8 if k >= 2 else 5) and np.all(a.d2 == 0)   # triple {7,100,2000} + pair {11,3000}


def test_brute_equals_cells_cfg1():
    cfg = events.CONFIGS[1]
    x = events.make_event(cfg)
    assert same(oracle.frnn(x, cfg.r, cfg.k_max, oracle.BRUTE), oracle.frnn(x, cfg.r, cfg.k_max, oracle.CELLS))


@pytest.mark.slow
def test_brute_equals_cells_cfg2_sampled_queries():
    cfg = events.CONFIGS[2]
    x = events.make_event(cfg)
    q = np.sort(np.random.default_rng(0).choice(cfg.n, 4000, replace=False))
    assert same(oracle.frnn(x, cfg.r, cfg.k_max, oracle.BRUTE, queries=q),
                oracle.frnn(x, cfg.r, cfg.k_max, oracle.CELLS, queries=q))


@pytest.mark.slow
def test_brute_equals_cells_cfg3_event0_sampled_queries():
    """SURVEY.md 8(c) P1/P2 at config 3's size: event 0 of the 16-event batch (the event the batched GPU parity leans on),
    the definition (section 3.4, quadratic) against the cell list on 4,000 sampled queries."""
    cfg = events.CONFIGS[3]
    xb, off = events.make_batch(cfg)
    x = np.ascontiguousarray(xb[off[0]:off[1]])
    assert len(x) == cfg.n
    q = np.sort(np.random.default_rng(3).choice(len(x), 4000, replace=False))
    a = oracle.frnn(x, cfg.r, cfg.k_max, oracle.BRUTE, queries=q)
    assert a.count > 4000                                       # mean degree ~2.8: the sample is not empty
    assert same(a, oracle.frnn(x, cfg.r, cfg.k_max, oracle.CELLS, queries=q))


@pytest.mark.slow
def test_brute_equals_cells_cfg4_sampled_queries():
    """The same at config 4's parameters (N = 10^6, r = 0.12, sigma = 0.05, K = 512: the dense regime), 2,000 sampled
    queries = 2 * 10^9 pair evaluations of the definition; and once with a K that binds on most of these rows."""
    cfg = events.CONFIGS[4]
    x = events.make_event(cfg)
    assert len(x) == 1000000
    q = np.sort(np.random.default_rng(4).choice(cfg.n, 2000, replace=False))
    a = oracle.frnn(x, cfg.r, cfg.k_max, oracle.BRUTE, queries=q)
    b = oracle.frnn(x, cfg.r, cfg.k_max, oracle.CELLS, queries=q)
    assert a.count > 2000 and same(a, b)
    k = 2
    assert int((a.uncapped > k).sum()) > 50                      # the cap decides on these rows
    qk = q[a.uncapped > k]
    assert same(oracle.frnn(x, cfg.r, k, oracle.BRUTE, queries=qk), oracle.frnn(x, cfg.r, k, oracle.CELLS, queries=qk))


def test_low_dimensional_inputs_and_other_dims():
    for dim in (1, 2, 3, 5):
        x = events.uniform_points(500, dim, -1, 1, 3)
        assert same(oracle.frnn(x, 0.2, 7, oracle.BRUTE), oracle.frnn(x, 0.2, 7, oracle.CELLS))


# ---------------------------------------------------------------- invariants (P5)
@pytest.mark.parametrize("cfg_idx", [0, 1])
def test_invariants(cfg_idx):
    cfg = events.CONFIGS[cfg_idx]
    x = events.make_event(cfg)
    res = oracle.frnn(x, cfg.r, 10 ** 6, oracle.CELLS)
    r2 = np.float32(cfg.r) * np.float32(cfg.r)
    assert not np.any(res.src == res.dst)
    H.assert_sorted_unique(res.src, res.dst)
    assert np.all(res.d2 <= r2)
    assert res.count == int(res.uncapped.sum())
    assert np.array_equal(np.bincount(res.src, minlength=cfg.n), res.uncapped)
    # symmetry of the uncapped graph with bitwise-equal d2 in both directions
    fwd = H.edge_keys(res.src, res.dst)
    rev = H.edge_keys(res.dst, res.src)
    order = np.argsort(rev)
    assert np.array_equal(rev[order], fwd)
    assert np.array_equal(H.bits(res.d2[order]), H.bits(res.d2))
    # K-prefix property: the capped list of i is the first K of i's uncapped list under (d2, j)
    for k in (1, 2, 4):
        capped = oracle.frnn(x, cfg.r, k, oracle.CELLS)
        assert capped.count == int(np.minimum(res.uncapped, k).sum())
        exp_s, exp_d = [], []
        starts = np.concatenate([[0], np.cumsum(res.uncapped)])
        for i in np.flatnonzero(res.uncapped > 0)[:3000]:
            sl = slice(starts[i], starts[i + 1])
            o = np.lexsort((res.dst[sl], res.d2[sl]))[:k]
            exp_d.append(np.sort(res.dst[sl][o])); exp_s.append(np.full(len(o), i))
        exp_s, exp_d = np.concatenate(exp_s), np.concatenate(exp_d)
        m = capped.src <= exp_s.max()
        assert np.array_equal(capped.src[m], exp_s) and np.array_equal(capped.dst[m], exp_d)


def test_row_permutation_invariance():
    cfg = events.CONFIGS[0]
    x = events.make_event(cfg)
    p = np.random.default_rng(9).permutation(cfg.n)
    a = oracle.frnn(x, cfg.r, 3, oracle.CELLS)
    b = oracle.frnn(x[p], cfg.r, 3, oracle.CELLS)          # row t of x[p] is row p[t] of x
    # K=3 with index tiebreak is NOT permutation invariant under d2 ties; the uncapped graph is
    a = oracle.frnn(x, cfg.r, 10 ** 6, oracle.CELLS)
    b = oracle.frnn(x[p], cfg.r, 10 ** 6, oracle.CELLS)
    kb = H.edge_keys(p[b.src].astype(np.int32), p[b.dst].astype(np.int32))
    order = np.argsort(kb)
    assert np.array_equal(kb[order], H.edge_keys(a.src, a.dst))
    assert np.array_equal(H.bits(b.d2[order]), H.bits(a.d2))


def test_degenerate_sizes_and_bad_arguments():
    for n in (0, 1):
        res = oracle.frnn(np.zeros((n, 8), np.float32), 0.1, 4)
        assert res.count == 0 and len(res.uncapped) == n
    two = np.zeros((2, 8), np.float32)
    assert oracle.frnn(two, 0.0, 4).count == 2          # duplicates at r = 0
    with pytest.raises(ValueError):
        oracle.frnn(two, -1.0, 4)
    with pytest.raises(ValueError):
        oracle.frnn(two, float("nan"), 4)
    with pytest.raises(ValueError):
        oracle.frnn(two, 0.1, 0)


def test_batched_events_are_independent():
    cfg = events.CONFIGS[0]
    evs = [events.make_event(cfg, s) for s in (0, 1, 2)]
    x = np.concatenate(evs)
    offs = np.array([0, 4096, 8192, 12288], np.int64)
    res, eoffs = oracle.frnn_batched(x, offs, cfg.r, cfg.k_max)
    for e in range(3):
        single = oracle.frnn(evs[e], cfg.r, cfg.k_max)
        sl = slice(eoffs[e], eoffs[e + 1])
        assert np.array_equal(res.src[sl], single.src) and np.array_equal(res.dst[sl], single.dst)
        assert res.src[sl].max() < 4096                  # indices are local to the event
