"""ctypes front end of the CPU oracle (oracle/frnn_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference leg, never by the product package.  It imports nothing from
``paper_2202_06929_b200`` and nothing under ``include/``.

``frnn(x, r, k_max, mode=...)`` returns ``OracleResult(src, dst, d2, uncapped)`` following the
definition in the C header: PAPER.md:31 (section 2) and PAPER.md:69 (section 3.4), with the
readings R1..R10 of DESIGN.md section 2.
"""
from __future__ import annotations

import ctypes
from dataclasses import dataclass

import numpy as np

from . import build as _build

BRUTE = 0   # mode A: O(n^2), the plain definition
CELLS = 1   # mode B: cell list on the first 3 coordinates, double binning


class _CResult(ctypes.Structure):
    _fields_ = [
        ("n_queries", ctypes.c_int64),
        ("count", ctypes.c_int64),
        ("src", ctypes.POINTER(ctypes.c_int32)),
        ("dst", ctypes.POINTER(ctypes.c_int32)),
        ("d2", ctypes.POINTER(ctypes.c_float)),
        ("uncapped", ctypes.POINTER(ctypes.c_int64)),
        ("threads", ctypes.c_int),
    ]


@dataclass
class OracleResult:
    src: np.ndarray        # int32 [E]
    dst: np.ndarray        # int32 [E]
    d2: np.ndarray         # float32 [E]
    uncapped: np.ndarray   # int64 [n_queries]: |S_i| before the K cap
    threads: int

    @property
    def count(self) -> int:
        return int(self.src.shape[0])


_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(_build.build())
        _lib.frnn_oracle_run.restype = ctypes.POINTER(_CResult)
        _lib.frnn_oracle_run.argtypes = [
            ctypes.c_int, ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_float, ctypes.c_int,
            ctypes.c_void_p, ctypes.c_int64, ctypes.c_int]
        _lib.frnn_oracle_free.restype = None
        _lib.frnn_oracle_free.argtypes = [ctypes.POINTER(_CResult)]
        _lib.frnn_oracle_d2.restype = ctypes.c_float
        _lib.frnn_oracle_d2.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int]
    return _lib


def frnn(x: np.ndarray, r: float, k_max: int, mode: int = CELLS, queries=None, threads: int = 0) -> OracleResult:
    """Directed, K-capped, (src,dst)-sorted radius graph of one event ``x`` (n x D float32)."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    assert x.ndim == 2
    n, dim = x.shape
    q_ptr, n_q = None, 0
    if queries is not None:
        queries = np.ascontiguousarray(queries, dtype=np.int64)
        q_ptr, n_q = queries.ctypes.data, len(queries)
    res = lib().frnn_oracle_run(mode, x.ctypes.data, n, dim, np.float32(r), int(k_max), q_ptr, n_q, threads)
    if not res:
        raise ValueError("frnn_oracle_run: invalid arguments")
    try:
        c = res.contents
        e, nq = c.count, c.n_queries
        out = OracleResult(
            np.ctypeslib.as_array(c.src, (max(e, 1),))[:e].copy(),
            np.ctypeslib.as_array(c.dst, (max(e, 1),))[:e].copy(),
            np.ctypeslib.as_array(c.d2, (max(e, 1),))[:e].copy(),
            np.ctypeslib.as_array(c.uncapped, (max(nq, 1),))[:nq].copy(),
            c.threads,
        )
    finally:
        lib().frnn_oracle_free(res)
    return out


def frnn_batched(x: np.ndarray, event_offsets: np.ndarray, r: float, k_max: int, mode: int = CELLS,
                 threads: int = 0) -> tuple[OracleResult, np.ndarray]:
    """B independent events (R10): no cross-event edges, src/dst LOCAL to the event.

    Returns the concatenated result and the int64 edge offsets (B+1).
    """
    parts = [frnn(x[event_offsets[e]:event_offsets[e + 1]], r, k_max, mode, threads=threads)
             for e in range(len(event_offsets) - 1)]
    offs = np.zeros(len(parts) + 1, dtype=np.int64)
    offs[1:] = np.cumsum([p.count for p in parts])
    cat = OracleResult(*(np.concatenate([getattr(p, f) for p in parts]) for f in ("src", "dst", "d2", "uncapped")),
                       threads=parts[0].threads if parts else 0)
    return cat, offs


def d2(a: np.ndarray, b: np.ndarray) -> np.float32:
    """The pinned-order fp32 squared distance of two rows (R3)."""
    a = np.ascontiguousarray(a, dtype=np.float32)
    b = np.ascontiguousarray(b, dtype=np.float32)
    return np.float32(lib().frnn_oracle_d2(a.ctypes.data, b.ctypes.data, a.shape[0]))
