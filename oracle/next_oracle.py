"""CPU oracle of the two steps that consume the edge list.

TEST INFRASTRUCTURE ONLY (same rule as oracle/__init__.py): plain numpy, obviously correct, slow; imports
nothing from ``paper_2202_06929_b200``.

gather_edge_rows   PAPER.md:31 (section 2: the filter classifies EDGES from the features of their end points),
                   PAPER.md:37 (section 3: fed in batches of 800,000 edges).  The plain definition: row e of the
                   output is x[src[e]] followed by x[dst[e]].
label_components   PAPER.md:33 (section 2: edges whose score passes a threshold are kept, the connected
                   components are the track candidates), PAPER.md:61 (section 3.2: WEAKLY connected components).
                   The plain definition of the canonical labelling: label[i] = the smallest node index that can
                   be reached from i over kept edges, direction ignored.  Computed as the fixed point of
                   "every node takes the minimum label among itself and its neighbours", which is that
                   definition iterated (at most diameter + 1 sweeps).
Readings: an edge is kept when score >= threshold (inclusive); self loops and edges with
an end point outside [0, n) are ignored; isolated nodes are components of their own.
"""
from __future__ import annotations

import numpy as np


def gather_edge_rows(x: np.ndarray, src: np.ndarray, dst: np.ndarray, e_begin: int = 0, e_max: int | None = None,
                     row_base: int = 0) -> np.ndarray:
    e_end = len(src) if e_max is None else min(len(src), e_begin + e_max)
    out = np.empty((max(e_end - e_begin, 0), 2 * x.shape[1]), dtype=x.dtype)
    for k, e in enumerate(range(e_begin, e_end)):
        out[k, : x.shape[1]] = x[int(src[e]) + row_base]
        out[k, x.shape[1]:] = x[int(dst[e]) + row_base]
    return out


def label_components(n: int, src: np.ndarray, dst: np.ndarray, score: np.ndarray | None = None, threshold: float = 0.0):
    src = np.asarray(src, dtype=np.int64)
    dst = np.asarray(dst, dtype=np.int64)
    keep = np.ones(len(src), dtype=bool) if score is None else (np.asarray(score, dtype=np.float32) >= np.float32(threshold))
    keep &= (src >= 0) & (src < n) & (dst >= 0) & (dst < n) & (src != dst)
    u, v = src[keep], dst[keep]
    label = np.arange(n, dtype=np.int64)
    while True:
        new = label.copy()
        np.minimum.at(new, u, label[v])
        np.minimum.at(new, v, label[u])
        if np.array_equal(new, label):
            break
        label = new
    return label.astype(np.int32), int(np.count_nonzero(label == np.arange(n)))
