"""B200-native fixed-radius nearest-neighbour (FRNN) graph building.

The Exa.TrkX graph-building hot path (§2, §3.4) as hand-written CUDA for
sm_100a behind the C ABI declared in ``include/frnn.h``.  ``frnn`` is the thin ctypes binding,
``events`` the seeded synthetic input generators.  Nothing here imports ``oracle/``.
"""
from . import events  # noqa: F401

__all__ = ["events"]
