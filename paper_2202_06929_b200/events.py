"""Seeded synthetic tracking events (the ONLY module shared by the oracle tests and the CUDA path).

Holds no arithmetic of the FRNN method: no distances, no cells, no radius tests.  It only
draws random point sets.  The recipe stands in for "one TrackML event after the embedding
MLP" (§2: same-track spacepoints are close in the embedded space and away from
others; the dataset and the trained weights are not available here), with the shapes and
sizes of BASELINE.json's five configs.  The recipe is restated in DESIGN.md §5.

RNG: numpy ``default_rng(seed)`` (PCG64), calls in exactly this order:
  1. hits per track            Poisson(lam) clipped below at ``min_hits`` (or a fixed count)
  2. track centres             U[-1, 1]^(T x D)
  3. padding track ids         only if the tracks hold fewer hits than the signal slots
  4. signal offsets            N(0, sigma^2) per dim
  5. noise hits                U[-1, 1]^D
  6. row permutation           so that same-track hits are not adjacent in memory
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

DIM = 8


@dataclass(frozen=True)
class EventConfig:
    """One BASELINE.json config line (``configs[idx]``)."""

    idx: int
    name: str
    n: int              # points per event
    n_tracks: int
    lam: float | None   # Poisson mean of hits per track; None = fixed_hits
    fixed_hits: int | None
    min_hits: int
    sigma: float
    noise_frac: float
    r: float
    k_max: int
    n_events: int = 1   # >1: batched call, seeds seed0..seed0+n_events-1
    seed0: int = 0


CONFIGS = (
    EventConfig(0, "cfg0_4k", 4096, 370, None, 10, 0, 0.03, 0.10, 0.1, 64),
    EventConfig(1, "cfg1_20k", 20000, 1800, 10.0, None, 3, 0.03, 0.10, 0.1, 128),
    EventConfig(2, "cfg2_120k", 120000, 11000, 10.0, None, 3, 0.03, 0.08, 0.1, 256),
    EventConfig(3, "cfg3_16x120k", 120000, 11000, 10.0, None, 3, 0.03, 0.08, 0.1, 256, n_events=16),
    EventConfig(4, "cfg4_1m_dense", 1000000, 50000, 20.0, None, 3, 0.05, 0.05, 0.12, 512),
)


def make_event(cfg: EventConfig, seed: int | None = None) -> np.ndarray:
    """Return one event as a C-contiguous float32 array of shape (cfg.n, 8)."""
    if seed is None:
        seed = cfg.seed0
    rng = np.random.default_rng(seed)
    n = cfg.n
    n_noise = int(round(cfg.noise_frac * n))
    n_sig = n - n_noise
    t = cfg.n_tracks
    if cfg.fixed_hits is not None:
        counts = np.full(t, cfg.fixed_hits, dtype=np.int64)
    else:
        counts = np.maximum(rng.poisson(cfg.lam, t), cfg.min_hits).astype(np.int64)
    total = int(counts.sum())
    centres = rng.uniform(-1.0, 1.0, (t, DIM))
    tid = np.repeat(np.arange(t), counts)
    if total >= n_sig:
        tid = tid[:n_sig]                       # N is binding; the track count is nominal
    else:
        tid = np.concatenate([tid, rng.integers(0, t, n_sig - total)])
    sig = centres[tid] + rng.normal(0.0, cfg.sigma, (n_sig, DIM))
    noise = rng.uniform(-1.0, 1.0, (n_noise, DIM))
    x = np.concatenate([sig, noise]).astype(np.float32)
    return np.ascontiguousarray(x[rng.permutation(n)])


def make_batch(cfg: EventConfig) -> tuple[np.ndarray, np.ndarray]:
    """Concatenated events of a batched config and their int64 row offsets (n_events+1)."""
    evs = [make_event(cfg, cfg.seed0 + e) for e in range(cfg.n_events)]
    offs = np.zeros(cfg.n_events + 1, dtype=np.int64)
    offs[1:] = np.cumsum([len(e) for e in evs])
    return np.ascontiguousarray(np.concatenate(evs)), offs


def one_cluster(n: int, sigma: float, seed: int) -> np.ndarray:
    """A single tight cluster: every query overflows a small K (SURVEY.md §8(c) pin P4)."""
    rng = np.random.default_rng(seed)
    return np.ascontiguousarray(rng.normal(0.0, sigma, (n, DIM)).astype(np.float32))


def dense_tracks(n: int, hits_per_track: float, sigma: float, seed: int) -> np.ndarray:
    """A dense event: ``n`` points in tracks of Poisson(hits_per_track) hits (min 3) around U[-1,1]^8 centres with
    N(0, sigma^2) spread, rows permuted.  With hits_per_track = 200, sigma = 0.02 and r = 0.1 the mean degree is about
    170: the regime BASELINE.json's config-4 parenthetical "(mean degree ~200)" describes and its recipe does not reach
    (R14); used for the K-binding bench leg and parity tests."""
    rng = np.random.default_rng(seed)
    t = max(int(round(n / hits_per_track)), 1)
    counts = np.maximum(rng.poisson(hits_per_track, t), 3).astype(np.int64)
    centres = rng.uniform(-1.0, 1.0, (t, DIM))
    tid = np.repeat(np.arange(t), counts)
    if len(tid) >= n:
        tid = tid[:n]
    else:
        tid = np.concatenate([tid, rng.integers(0, t, n - len(tid))])
    x = (centres[tid] + rng.normal(0.0, sigma, (n, DIM))).astype(np.float32)
    return np.ascontiguousarray(x[rng.permutation(n)])


def lattice(length: int, dim: int, h: float) -> np.ndarray:
    """Cubic lattice of ``length**dim`` points, spacing ``h``, centred on the origin.

    With h = 0.125 and small ``length`` every coordinate and every squared distance is exact
    in fp32 (SURVEY.md §8(c) pin P3).  Row order: the last coordinate varies fastest.
    """
    axes = [np.arange(length, dtype=np.float64)] * dim
    g = np.stack(np.meshgrid(*axes, indexing="ij"), axis=-1).reshape(-1, dim)
    return np.ascontiguousarray(((g - (length - 1) / 2.0) * h).astype(np.float32))


def uniform_points(n: int, dim: int, lo: float, hi: float, seed: int) -> np.ndarray:
    rng = np.random.default_rng(seed)
    return np.ascontiguousarray(rng.uniform(lo, hi, (n, dim)).astype(np.float32))


def shard_events(n_events: int, world_size: int, rank: int) -> list[int]:
    """Round-robin event -> rank assignment (events are independent units)."""
    return list(range(rank, n_events, world_size))


def edge_scores(n_edges: int, seed: int) -> np.ndarray:
    """Stand-in for the GNN's per-edge scores (the trained GNN is not available): seeded U[0,1) fp32."""
    rng = np.random.default_rng(seed)
    return np.ascontiguousarray(rng.random(n_edges, dtype=np.float32))


def random_graph(n: int, n_edges: int, seed: int):
    """Seeded random directed edge list (src, dst int32) with possible self loops and duplicates."""
    rng = np.random.default_rng(seed)
    return (np.ascontiguousarray(rng.integers(0, n, n_edges, dtype=np.int32)),
            np.ascontiguousarray(rng.integers(0, n, n_edges, dtype=np.int32)))
