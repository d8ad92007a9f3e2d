"""frnn_build_static: the build for callers that cannot allocate device memory.

Some users of this library run where allocation on the event path is not an option: an online / trigger process that
gave all of the GPU's memory to its framework's arena at configure time (a later cudaMalloc fails or breaks the
budget), a latency-bound event loop (cudaMalloc / cudaFree stall the whole device for an unpredictable time), a plug-in
living under another program's allocator.  They can pass inputs and outputs but have no workspace to offer, so
``frnn_build_static`` keeps its scratch in a fixed 3 MiB array inside the library and accepts at most
``FRNN_STATIC_MAX_ROWS`` (8192) rows.

The checks here: the entry point gives exactly what ``frnn_build_ex`` (caller-owned workspace) gives -- the bar of the
other GPU tests: indices, count, status and CSR offsets equal, d2 bit for bit -- on calls made back to back, so that
the second call runs on whatever the first left in the shared array; and it refuses events beyond the limit without
touching anything.  The file is named to be collected last: under ``pytest -x`` a failure here hides no other test.
It makes no assumption about what ran before it in the process (it passes alone and after the whole suite).
"""
from __future__ import annotations

import numpy as np
import pytest

from paper_2202_06929_b200 import events

torch = pytest.importorskip("torch")


def _bits(t):
    return t.view(torch.int32)


def _static_call(F, pts, r, k, out, stream=None):
    """One frnn_build_static call into the caller-owned outputs ``out`` (nothing is allocated on the way)."""
    return F.frnn_build_static(pts, r, k, out["src"], out["dst"], out["d2"], out["count"], out["status"], out["row_ptr"], stream)


def _outputs(n, cap, fill):
    """Output arrays as a caller would own them, pre-filled with a pattern so that stale values cannot pass for results."""
    dev = torch.device("cuda", torch.cuda.current_device())
    return {
        "src": torch.full((cap,), fill, dtype=torch.int32, device=dev),
        "dst": torch.full((cap,), fill, dtype=torch.int32, device=dev),
        "d2": torch.full((cap,), float(fill), dtype=torch.float32, device=dev),
        "count": torch.full((1,), fill, dtype=torch.int64, device=dev),
        "status": torch.full((1,), fill, dtype=torch.int32, device=dev),
        "row_ptr": torch.full((n + 1,), fill, dtype=torch.int64, device=dev),
    }


def _assert_equal_to_existing_path(F, x, r, k, out, label):
    """``out`` (filled by frnn_build_static) against frnn_build_ex on its own freshly allocated workspace."""
    pts = torch.from_numpy(np.ascontiguousarray(x)).cuda()
    ref = F.frnn_build_ex(pts, r, k, edge_capacity=out["src"].numel(), want_row_ptr=True)
    torch.cuda.synchronize()
    ref.check()
    assert int(out["status"].item()) == F.FRNN_OK, label
    e = ref.n_edges()
    assert int(out["count"].item()) == e, f"{label}: edge count {int(out['count'].item())} != {e}"
    assert e > 0, f"{label}: the case must have edges to mean anything"
    assert torch.equal(out["src"][:e], ref.src[:e]), f"{label}: src differs"
    assert torch.equal(out["dst"][:e], ref.dst[:e]), f"{label}: dst differs"
    assert torch.equal(_bits(out["d2"][:e]), _bits(ref.d2[:e])), f"{label}: d2 differs bitwise"
    assert torch.equal(out["row_ptr"], ref.row_ptr), f"{label}: CSR offsets differ"
    return e


def test_scratch_array_holds_the_largest_accepted_event():
    """Host only: the stated limit and the array size agree with the header and with the layout of the largest event."""
    import os
    import re

    from paper_2202_06929_b200 import frnn as F
    header = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "frnn.h")).read()
    assert int(re.search(r"#define\s+FRNN_STATIC_MAX_ROWS\s+(\d+)", header).group(1)) == F.FRNN_STATIC_MAX_ROWS == 8192
    F.frnn_set_grid(0, 0)
    need = max(F.frnn_workspace_bytes(n, 1, dim, 64) for n in (1, 4096, F.FRNN_STATIC_MAX_ROWS) for dim in (1, 3, 8, 9, 16))
    assert need <= F.frnn_static_scratch_bytes() == 3 << 20
    assert F.frnn_static_scratch_bytes() % 256 == 0


@pytest.mark.gpu
def test_static_scratch_build_matches_the_workspace_build_on_consecutive_calls():
    from paper_2202_06929_b200 import frnn as F
    F.lib()
    F.frnn_set_grid(0, 0)
    cfg = events.CONFIGS[0]                                  # 4096 points, r = 0.1, K = 64: the small BASELINE config
    xa = events.make_event(cfg)
    xb = events.make_event(cfg, seed=4242)[:3001]            # another event, ragged size, and a K that binds (cap = 2 per row)
    xc = events.uniform_points(F.FRNN_STATIC_MAX_ROWS, 12, 0.0, 1.0, 77)   # the largest accepted event, 12 coordinates (two internal rows)
    cases = [("event A, K=64", xa, cfg.r, cfg.k_max), ("event B, K=2", xb, cfg.r, 2), ("8192 x 12", xc, 0.45, 16),
             ("event A again", xa, cfg.r, cfg.k_max)]
    # two calls in a row on one stream, checked only afterwards: the second starts from the first one's leftovers
    dev_pts = [torch.from_numpy(np.ascontiguousarray(x)).cuda() for _, x, _, _ in cases]
    outs = [_outputs(x.shape[0], x.shape[0] * k, -7 - i) for i, (_, x, _, k) in enumerate(cases)]
    launches = []
    for (label, x, r, k), pts, out in zip(cases, dev_pts, outs):
        _static_call(F, pts, r, k, out)
        launches.append(F.frnn_last_launch_count())
    torch.cuda.synchronize()
    assert all(5 <= c <= 8 for c in launches), launches      # memset + kernels, launched one by one
    counts = [_assert_equal_to_existing_path(F, x, r, k, out, label) for (label, x, r, k), out in zip(cases, outs)]
    assert counts[0] == counts[3] and counts[1] < counts[0]
    # and once more after the reference path has run in between (separate synchronised calls)
    for (label, x, r, k), pts in zip(cases[:2], dev_pts[:2]):
        out = _outputs(x.shape[0], x.shape[0] * k, -99)
        _static_call(F, pts, r, k, out)
        torch.cuda.synchronize()
        _assert_equal_to_existing_path(F, x, r, k, out, label + " (repeat)")


@pytest.mark.gpu
def test_static_scratch_build_rejects_events_beyond_the_limit_and_handles_empty_ones():
    from paper_2202_06929_b200 import frnn as F
    F.lib()
    n = F.FRNN_STATIC_MAX_ROWS + 1
    pts = torch.from_numpy(events.uniform_points(n, 8, 0.0, 1.0, 5)).cuda()
    out = _outputs(n, 1024, -3)
    with pytest.raises(F.FrnnError) as err:
        _static_call(F, pts, 0.1, 4, out)
    assert err.value.status == F.FRNN_ERR_UNSUPPORTED
    assert "FRNN_STATIC_MAX_ROWS" in str(err.value) and str(n) in str(err.value)
    torch.cuda.synchronize()
    for name, t in out.items():                              # nothing was enqueued, no output was touched
        assert bool((t == -3).all()), name
    # an empty event and a capacity overflow behave as in frnn_build_ex
    empty = torch.empty((0, 8), dtype=torch.float32, device="cuda")
    out = _outputs(0, 16, -3)
    _static_call(F, empty, 0.1, 4, out)
    torch.cuda.synchronize()
    assert int(out["count"].item()) == 0 and int(out["status"].item()) == F.FRNN_OK
    x = events.make_event(events.CONFIGS[0])
    small = _outputs(x.shape[0], 100, -3)
    _static_call(F, torch.from_numpy(x).cuda(), 0.1, 64, small)
    torch.cuda.synchronize()
    assert int(small["status"].item()) == F.FRNN_ERR_CAPACITY and int(small["count"].item()) > 100
