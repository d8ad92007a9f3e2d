"""Pins of oracle/next_oracle.py (gather of edge rows, weakly connected components) against things other than
itself: a hand-worked fixture, closed forms, a library routine (scipy), brute-force search on tiny graphs."""
from __future__ import annotations

import os

import numpy as np
import pytest

from oracle import next_oracle as NO
from paper_2202_06929_b200 import events

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def read_components_hand():
    sec, edges, labels, ncomp = None, [], None, None
    for line in open(os.path.join(GOLDEN, "components_hand.txt")):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        if line.startswith("["):
            sec = line.strip("[]")
        elif sec == "edges":
            a, b, c = line.split()
            edges.append((int(a), int(b), float(c)))
        elif sec == "labels":
            labels = np.array(line.split(), dtype=np.int32)
        elif sec == "n_components":
            ncomp = int(line)
    e = np.array(edges)
    return e[:, 0].astype(np.int32), e[:, 1].astype(np.int32), e[:, 2].astype(np.float32), labels, ncomp


def bfs_labels(n, src, dst, keep):
    """Brute force: breadth-first search from every node, label = min reached (tiny graphs only)."""
    adj = [[] for _ in range(n)]
    for s, d, k in zip(src, dst, keep):
        if k and 0 <= s < n and 0 <= d < n:
            adj[s].append(d)
            adj[d].append(s)
    out = np.empty(n, np.int32)
    for i in range(n):
        seen, todo = {i}, [i]
        while todo:
            a = todo.pop()
            for b in adj[a]:
                if b not in seen:
                    seen.add(b)
                    todo.append(b)
        out[i] = min(seen)
    return out


def test_components_hand_fixture():
    src, dst, score, labels, ncomp = read_components_hand()
    got, n = NO.label_components(10, src, dst, score, 0.5)
    assert np.array_equal(got, labels) and n == ncomp
    # just above the boundary score the edge 6->1 goes and {1},{6} split: the threshold is inclusive
    got2, n2 = NO.label_components(10, src, dst, score, float(np.nextafter(np.float32(0.5), np.float32(1))))
    assert got2[6] == 6 and n2 == ncomp + 1


def test_components_closed_forms():
    n = 1000
    # a path given in scrambled order and arbitrary directions: one component, label 0
    rng = np.random.default_rng(1)
    a = np.arange(n - 1, dtype=np.int32)
    flip = rng.random(n - 1) < 0.5
    src, dst = np.where(flip, a + 1, a), np.where(flip, a, a + 1)
    p = rng.permutation(n - 1)
    lab, nc = NO.label_components(n, src[p], dst[p])
    assert nc == 1 and np.all(lab == 0)
    # k disjoint cycles of length m: label = first node of the cycle
    k, m = 37, 11
    base = np.repeat(np.arange(k) * m, m)
    src = (base + np.tile(np.arange(m), k)).astype(np.int32)
    dst = (base + np.tile((np.arange(m) + 1) % m, k)).astype(np.int32)
    lab, nc = NO.label_components(k * m, src, dst)
    assert nc == k and np.array_equal(lab, base)
    # no edges / all edges dropped: every node its own component
    lab, nc = NO.label_components(5, np.zeros(0, np.int32), np.zeros(0, np.int32))
    assert nc == 5 and np.array_equal(lab, np.arange(5))
    lab, nc = NO.label_components(5, np.array([0, 1], np.int32), np.array([1, 2], np.int32), np.array([0.1, 0.2], np.float32), 0.3)
    assert nc == 5
    # direction is ignored: only (j, i) present
    lab, nc = NO.label_components(3, np.array([2], np.int32), np.array([0], np.int32))
    assert list(lab) == [0, 1, 0] and nc == 2
    # out-of-range end points and self loops are ignored
    lab, nc = NO.label_components(3, np.array([0, 1, 7, -1], np.int32), np.array([0, 5, 1, 2], np.int32))
    assert nc == 3


@pytest.mark.parametrize("seed", range(6))
def test_components_vs_brute_force_bfs(seed):
    n, e = 40, 30 + 5 * seed
    src, dst = events.random_graph(n, e, seed)
    score = events.edge_scores(e, 100 + seed)
    got, nc = NO.label_components(n, src, dst, score, 0.4)
    exp = bfs_labels(n, src, dst, score >= np.float32(0.4))
    assert np.array_equal(got, exp) and nc == len(set(exp.tolist()))


@pytest.mark.parametrize("n,e,thr", [(5000, 4000, 0.0), (20000, 30000, 0.5), (20000, 15000, 0.2)])
def test_components_vs_scipy(n, e, thr):
    from scipy.sparse import coo_matrix
    from scipy.sparse.csgraph import connected_components
    src, dst = events.random_graph(n, e, 7)
    score = events.edge_scores(e, 8)
    got, nc = NO.label_components(n, src, dst, score, thr)
    keep = score >= np.float32(thr)
    g = coo_matrix((np.ones(int(keep.sum())), (src[keep], dst[keep])), shape=(n, n))
    nc_ref, part = connected_components(g, directed=True, connection="weak")
    assert nc == nc_ref
    # same partition, and the label is the minimum index of its part
    first = np.full(nc_ref, n, np.int64)
    np.minimum.at(first, part, np.arange(n))
    assert np.array_equal(got, first[part].astype(np.int32))


def test_gather_hand_and_library():
    x = np.arange(6 * 8, dtype=np.float32).reshape(6, 8)
    src = np.array([5, 0, 3], np.int32)
    dst = np.array([1, 0, 2], np.int32)
    got = NO.gather_edge_rows(x, src, dst)
    assert got.shape == (3, 16)
    assert list(got[0]) == list(range(40, 48)) + list(range(8, 16))          # worked by hand: rows 5 and 1
    assert list(got[1]) == list(range(0, 8)) * 2
    assert np.array_equal(got, np.concatenate([x[src], x[dst]], axis=1))    # the library's fancy indexing
    # chunking and a row base
    assert np.array_equal(NO.gather_edge_rows(x, src, dst, e_begin=1, e_max=1), got[1:2])
    assert np.array_equal(NO.gather_edge_rows(x, src, dst, e_begin=2, e_max=10), got[2:])
    assert np.array_equal(NO.gather_edge_rows(x, np.array([1], np.int32), np.array([0], np.int32), row_base=2)[0],
                          np.concatenate([x[3], x[2]]))
