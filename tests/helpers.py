"""Test-side helpers: fixture parsing, exact rational fp32 emulation, edge-list comparison.

None of this is used by the product path or by the oracle itself.
"""
from __future__ import annotations

import os
from fractions import Fraction

import numpy as np

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")

HANDCASE_POINTS = np.array([
    [0, 0, 0, 0, 0, 0, 0, 0],
    [0.5, 0, 0, 0, 0, 0, 0, 0],
    [0.25, 0.25, 0.25, 0.25, 0, 0, 0, 0],
    [0.5, 0.25, 0, 0, 0, 0, 0, 0],
    [0, 0, 0, 0, 0, 0, 0, 0],
    [2, 2, 2, 2, 2, 2, 2, 2],
], dtype=np.float32)


def read_handcase(section: str):
    src, dst, d2 = [], [], []
    cur = None
    with open(os.path.join(GOLDEN, "handcase_8d.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            if line.startswith("["):
                cur = line.strip("[]")
                continue
            if cur == section:
                a, b, c = line.split()
                src.append(int(a)); dst.append(int(b)); d2.append(float(c))
    return np.array(src, np.int32), np.array(dst, np.int32), np.array(d2, np.float32)


def round_f32(q: Fraction) -> Fraction:
    """Round an exact rational to the nearest fp32 (ties to even), normal range only."""
    if q == 0:
        return Fraction(0)
    sign = -1 if q < 0 else 1
    q = abs(q)
    e = q.numerator.bit_length() - q.denominator.bit_length()
    if Fraction(2) ** e > q:
        e -= 1
    assert Fraction(2) ** e <= q < Fraction(2) ** (e + 1)
    assert -126 <= e <= 127, "outside the normal fp32 range"
    ulp = Fraction(2) ** (e - 23)
    m = q / ulp                                  # in [2^23, 2^24)
    lo = m.numerator // m.denominator
    rem = m - lo
    if rem > Fraction(1, 2) or (rem == Fraction(1, 2) and lo % 2 == 1):
        lo += 1
    return sign * lo * ulp


def d2_exact_chain(a: np.ndarray, b: np.ndarray) -> np.float32:
    """DESIGN.md R3 in exact rational arithmetic: t = fl32(a_d - b_d); acc = fl32(t*t + acc)."""
    acc = Fraction(0)
    for d in range(len(a)):
        t = round_f32(Fraction(float(a[d])) - Fraction(float(b[d])))
        acc = round_f32(t * t + acc)
    return np.float32(float(acc))


def d2_exact_mul_add(a: np.ndarray, b: np.ndarray) -> np.float32:
    """A plausible WRONG order: round the square, then round the sum (no fused multiply-add)."""
    acc = Fraction(0)
    for d in range(len(a)):
        t = round_f32(Fraction(float(a[d])) - Fraction(float(b[d])))
        acc = round_f32(round_f32(t * t) + acc)
    return np.float32(float(acc))


def bits(a: np.ndarray) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float32).view(np.uint32)


def assert_sorted_unique(src: np.ndarray, dst: np.ndarray):
    key = src.astype(np.int64) << 32 | dst.astype(np.int64)
    assert np.all(np.diff(key) > 0), "edge list is not strictly (src,dst)-sorted (or has duplicates)"


def edge_keys(src, dst) -> np.ndarray:
    return src.astype(np.int64) << 32 | dst.astype(np.int64)


def compare_edges(got, exp, r: float, label: str = ""):
    """Exact edge-set + bitwise-d2 comparison; the ONLY tolerated differences are pairs with
    |d2 - r2| <= 1e-6 * r2 (north_star), which are returned (and must be reported by the caller).

    ``got`` / ``exp`` expose .src .dst .d2.  Raises AssertionError on any other difference.
    """
    r2 = np.float32(r) * np.float32(r)
    kg, ke = edge_keys(got.src, got.dst), edge_keys(exp.src, exp.dst)
    only_g = np.setdiff1d(kg, ke, assume_unique=True)
    only_e = np.setdiff1d(ke, kg, assume_unique=True)
    band = []
    for keys, side in ((only_g, got), (only_e, exp)):
        if len(keys):
            k_side = edge_keys(side.src, side.dst)
            d = side.d2[np.searchsorted(k_side, keys)]
            bad = np.abs(d.astype(np.float64) - float(r2)) > 1e-6 * float(r2)
            assert not bad.any(), f"{label}: {bad.sum()} edge(s) differ outside the 1e-6*r2 band, e.g. key {keys[bad][0]}"
            band.extend(keys.tolist())
    common_g = np.isin(kg, ke, assume_unique=True)
    common_e = np.isin(ke, kg, assume_unique=True)
    dg, de = got.d2[common_g], exp.d2[common_e]
    neq = bits(dg) != bits(de)
    if neq.any():
        rel = np.abs(dg[neq].astype(np.float64) - de[neq].astype(np.float64)) / np.maximum(de[neq].astype(np.float64), 1e-300)
        assert rel.max() <= 1e-6, f"{label}: d2 differs by more than 1e-6 relative (max {rel.max():.3e})"
    return band, int(neq.sum())
