"""Thin ctypes binding of include/frnn.h (argument marshalling only).

Every step of the path runs in the CUDA kernels of ``libfrnn_b200.so``; PyTorch is used for device
memory and streams.  There is no CPU fallback: a missing library or a missing CUDA device raises.
Function names mirror the C ABI.  Operation: PAPER.md:31 (section 2), PAPER.md:69 (section 3.4).
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

import torch

from . import build as _build

FRNN_OK = 0
FRNN_ERR_INVALID_ARG = -1
FRNN_ERR_UNSUPPORTED = -2
FRNN_ERR_CAPACITY = -3
FRNN_ERR_WORKSPACE = -4
FRNN_ERR_CUDA = -5

_c = ctypes


class FrnnOptions(_c.Structure):
    """``frnn_options`` of include/frnn.h (per-call grid / bin order / launch mode)."""
    _fields_ = [("struct_bytes", _c.c_uint32), ("grid_dims", _c.c_int32), ("grid_bits", _c.c_int32), ("order_count", _c.c_int32),
                ("order", _c.c_int32 * 8), ("launch_mode", _c.c_int32), ("timeline", _c.c_int32), ("reserved", _c.c_int32 * 4)]


class FrnnGridReport(_c.Structure):
    """``frnn_grid_report`` of include/frnn.h (what frnn_suggest_grid saw and predicts)."""
    _fields_ = [("grid_dims", _c.c_int32), ("grid_bits", _c.c_int32), ("reordered", _c.c_int32), ("n_tried", _c.c_int32),
                ("sampled", _c.c_int64),
                ("predicted_candidates", _c.c_float), ("predicted_survivors", _c.c_float), ("predicted_us", _c.c_float),
                ("measured_us", _c.c_float),
                ("extent_cells", _c.c_float * 16), ("pair_probability", _c.c_float * 16), ("key_probability", _c.c_float * 16),
                ("tried_dims", _c.c_int32 * 12), ("tried_bits", _c.c_int32 * 12), ("tried_reordered", _c.c_int32 * 12),
                ("tried_predicted_us", _c.c_float * 12), ("tried_measured_us", _c.c_float * 12)]

    def tried(self):
        """The measured shortlist as a list of dicts (empty when measure was off)."""
        return [{"grid_dims": self.tried_dims[k], "grid_bits": self.tried_bits[k], "reordered": bool(self.tried_reordered[k]),
                 "predicted_us": self.tried_predicted_us[k], "measured_us": self.tried_measured_us[k]} for k in range(self.n_tried)]


FRNN_LAUNCH_DEFAULT, FRNN_LAUNCH_GRAPH, FRNN_LAUNCH_PLAIN = 0, 1, 2
FRNN_GRID_AUTO = -1
_OPT = _c.POINTER(FrnnOptions)
_BUILD_ARGS = [_c.c_void_p, _c.c_int64, _c.c_int, _c.c_float, _c.c_int,
               _c.c_void_p, _c.c_void_p, _c.c_void_p, _c.c_int64,
               _c.c_void_p, _c.c_void_p, _c.c_void_p,
               _c.c_void_p, _c.c_size_t, _c.c_void_p]
_BATCHED_ARGS = [_c.c_void_p, _c.POINTER(_c.c_int64), _c.c_int, _c.c_int, _c.c_float, _c.c_int,
                 _c.c_void_p, _c.c_void_p, _c.c_void_p, _c.c_int64,
                 _c.c_void_p, _c.c_void_p, _c.c_void_p,
                 _c.c_void_p, _c.c_size_t, _c.c_void_p]
_SIGNATURES = {
    "frnn_version": (_c.c_int, []),
    "frnn_status_string": (_c.c_char_p, [_c.c_int]),
    "frnn_last_error_string": (_c.c_char_p, []),
    "frnn_options_init": (None, [_OPT]),
    "frnn_workspace_bytes": (_c.c_size_t, [_c.c_int64, _c.c_int, _c.c_int, _c.c_int]),
    "frnn_workspace_bytes_opt": (_c.c_size_t, [_OPT, _c.c_int64, _c.c_int, _c.c_int, _c.c_int]),
    "frnn_set_grid": (_c.c_int, [_c.c_int, _c.c_int]),
    "frnn_get_grid": (None, [_c.c_int64, _c.c_int, _c.c_int, _c.POINTER(_c.c_int), _c.POINTER(_c.c_int)]),
    "frnn_get_grid_opt": (None, [_OPT, _c.c_int64, _c.c_int, _c.c_int, _c.POINTER(_c.c_int), _c.POINTER(_c.c_int)]),
    "frnn_suggest_grid": (_c.c_int, [_c.c_void_p, _c.c_int64, _c.c_int, _c.c_int, _c.c_float, _c.c_int, _OPT, _c.POINTER(FrnnGridReport),
                                     _c.c_void_p]),
    "frnn_build_opt": (_c.c_int, [_OPT] + _BUILD_ARGS),
    "frnn_build_batched_opt": (_c.c_int, [_OPT] + _BATCHED_ARGS),
    "frnn_host_pipeline_create_opt": (_c.c_int, [_OPT, _c.c_int64, _c.c_int, _c.c_int, _c.c_int64, _c.c_int, _c.POINTER(_c.c_void_p)]),
    "frnn_build": (_c.c_int, [_c.c_void_p, _c.c_int64, _c.c_int, _c.c_float, _c.c_int,
                              _c.c_void_p, _c.c_void_p, _c.c_void_p, _c.POINTER(_c.c_int64)]),
    "frnn_build_ex": (_c.c_int, _BUILD_ARGS),
    "frnn_build_dense_ex": (_c.c_int, _BUILD_ARGS),
    "frnn_static_scratch_bytes": (_c.c_size_t, []),
    "frnn_build_static": (_c.c_int, _BUILD_ARGS[:12] + [_c.c_void_p]),
    "frnn_build_batched": (_c.c_int, _BATCHED_ARGS),
    "frnn_build_host": (_c.c_int, [_c.c_void_p, _c.c_int64, _c.c_int, _c.c_float, _c.c_int,
                                   _c.c_void_p, _c.c_void_p, _c.c_void_p, _c.c_int64, _c.POINTER(_c.c_int64)]),
    "frnn_last_launch_count": (_c.c_int, []),
    "frnn_set_graph_mode": (_c.c_int, [_c.c_int]),
    "frnn_graph_builds": (_c.c_longlong, []),
    "frnn_set_profiling": (_c.c_int, [_c.c_int]),
    "frnn_get_profile": (_c.c_int, [_c.POINTER(_c.c_float), _c.c_int]),
    "frnn_phase_name": (_c.c_char_p, [_c.c_int]),
    "frnn_get_timeline": (_c.c_int, [_c.c_void_p, _c.c_int64, _c.c_int, _c.c_int, _c.POINTER(_c.c_double), _c.POINTER(_c.c_double), _c.c_int]),
    "frnn_timeline_name": (_c.c_char_p, [_c.c_int]),
    "frnn_gather_edge_rows": (_c.c_int, [_c.c_void_p, _c.c_int64, _c.c_int, _c.c_void_p, _c.c_void_p, _c.c_void_p,
                                         _c.c_int64, _c.c_int64, _c.c_int64, _c.c_void_p, _c.c_void_p]),
    "frnn_label_components": (_c.c_int, [_c.c_int64, _c.c_void_p, _c.c_void_p, _c.c_void_p, _c.c_float, _c.c_void_p,
                                         _c.c_int64, _c.c_void_p, _c.c_void_p, _c.c_void_p]),
    "frnn_host_pipeline_create": (_c.c_int, [_c.c_int64, _c.c_int, _c.c_int, _c.c_int64, _c.c_int, _c.POINTER(_c.c_void_p)]),
    "frnn_host_pipeline_submit": (_c.c_int, [_c.c_void_p, _c.c_void_p, _c.c_int64, _c.c_float, _c.c_void_p, _c.c_void_p,
                                             _c.c_void_p, _c.c_void_p]),
    "frnn_host_pipeline_wait": (_c.c_int, [_c.c_void_p]),
    "frnn_host_pipeline_destroy": (None, [_c.c_void_p]),
    "frnn_set_bin_order": (_c.c_int, [_c.POINTER(_c.c_int), _c.c_int]),
    "frnn_suggest_bin_order": (_c.c_int, [_c.c_void_p, _c.c_int64, _c.c_int, _c.c_float, _c.POINTER(_c.c_int), _c.POINTER(_c.c_float),
                                          _c.c_void_p]),
    "frnn_release_cached": (None, []),
}
EXPORTED_SYMBOLS = tuple(_SIGNATURES)

_lib = None


def library_path() -> str:
    return _build.LIB


def lib() -> ctypes.CDLL:
    """Load (building first if the sources are newer) the C-ABI shared library.  Raises if absent."""
    global _lib
    if _lib is None:
        path = _build.build() if os.path.exists(_build.SOURCES[0]) else _build.LIB
        if not os.path.exists(path):
            raise RuntimeError(f"{path} is missing: the CUDA extension is required (no CPU fallback)")
        handle = ctypes.CDLL(path)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(handle, name)
            fn.restype, fn.argtypes = res, args
        _lib = handle
    return _lib


class FrnnError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        detail = f" [{frnn_last_error_string()}]" if status == FRNN_ERR_CUDA else ""
        super().__init__(f"{where}: {frnn_status_string(status)} ({status}){detail}")


def _check(status: int, where: str):
    if status != FRNN_OK:
        raise FrnnError(status, where)


def frnn_version() -> int:
    return lib().frnn_version()


def frnn_status_string(status: int) -> str:
    return lib().frnn_status_string(int(status)).decode()


def frnn_last_error_string() -> str:
    return lib().frnn_last_error_string().decode()


def frnn_options(grid_dims: int = 0, grid_bits: int = 0, order=None, launch_mode: int = FRNN_LAUNCH_DEFAULT,
                 timeline: bool = False) -> FrnnOptions:
    """An initialised ``frnn_options`` (frnn_options_init + the given fields)."""
    o = FrnnOptions()
    lib().frnn_options_init(_c.byref(o))
    o.grid_dims, o.grid_bits, o.launch_mode, o.timeline = int(grid_dims), int(grid_bits), int(launch_mode), int(bool(timeline))
    order = [int(v) for v in (order or [])]
    o.order_count = len(order)
    for k, v in enumerate(order):
        o.order[k] = v
    return o


def _opt_ref(opt):
    return None if opt is None else _c.byref(opt)


def frnn_workspace_bytes(n_total: int, n_events: int = 1, dim: int = 8, k_max: int = 1, opt: FrnnOptions | None = None) -> int:
    if opt is not None:
        return int(lib().frnn_workspace_bytes_opt(_c.byref(opt), int(n_total), int(n_events), int(dim), int(k_max)))
    return int(lib().frnn_workspace_bytes(int(n_total), int(n_events), int(dim), int(k_max)))


def frnn_set_grid(grid_dims: int = 0, grid_bits: int = 0) -> None:
    _check(lib().frnn_set_grid(int(grid_dims), int(grid_bits)), "frnn_set_grid")


def frnn_get_grid(n_total: int, n_events: int = 1, dim: int = 8) -> tuple[int, int]:
    d, b = _c.c_int(0), _c.c_int(0)
    lib().frnn_get_grid(int(n_total), int(n_events), int(dim), _c.byref(d), _c.byref(b))
    return d.value, b.value


def frnn_get_grid_opt(opt: FrnnOptions | None, n_total: int, n_events: int = 1, dim: int = 8) -> tuple[int, int]:
    """(grid_dims, grid_bits) a call made with ``opt`` runs on; (0, 0) for FRNN_GRID_AUTO (chosen per call)."""
    d, b = _c.c_int(0), _c.c_int(0)
    lib().frnn_get_grid_opt(_opt_ref(opt), int(n_total), int(n_events), int(dim), _c.byref(d), _c.byref(b))
    return d.value, b.value


def frnn_suggest_grid(points: torch.Tensor, r: float, n_events: int = 1, opt: FrnnOptions | None = None,
                      stream: torch.cuda.Stream | None = None, measure: bool = False) -> tuple[FrnnOptions, FrnnGridReport]:
    """Data-driven choice of (grid_dims, grid_bits, order) for ``points`` (device, n x dim); synchronous.
    ``measure``: time the model's shortlist on the sample and take the fastest."""
    _require_cuda(points)
    n, dim = points.shape
    opt = opt if opt is not None else frnn_options()
    rep = FrnnGridReport()
    stream = stream or torch.cuda.current_stream(points.device)
    _check(lib().frnn_suggest_grid(_ptr(points), n, int(n_events), dim, float(r), int(bool(measure)), _c.byref(opt), _c.byref(rep),
                                   _c.c_void_p(stream.cuda_stream)), "frnn_suggest_grid")
    return opt, rep


def frnn_set_graph_mode(enabled: bool) -> None:
    _check(lib().frnn_set_graph_mode(int(bool(enabled))), "frnn_set_graph_mode")


def frnn_graph_builds() -> int:
    return int(lib().frnn_graph_builds())


def frnn_last_launch_count() -> int:
    return lib().frnn_last_launch_count()


def frnn_set_profiling(enabled) -> None:
    """0/False: off; 1/True: one CUDA event after every phase; 2: in-graph %globaltimer timeline."""
    _check(lib().frnn_set_profiling(int(enabled)), "frnn_set_profiling")


def frnn_get_timeline(workspace: torch.Tensor, n_total: int, n_events: int = 1, dim: int = 8) -> dict[str, tuple[float, float]]:
    """(begin_us, end_us) per kernel of the last call on ``workspace`` made in profiling mode 2
    (the caller synchronises first)."""
    b, e = (_c.c_double * 8)(), (_c.c_double * 8)()
    n = lib().frnn_get_timeline(_ptr(workspace), int(n_total), int(n_events), int(dim), b, e, 8)
    if n < 0:
        raise FrnnError(n, "frnn_get_timeline")
    return {lib().frnn_timeline_name(i).decode(): (float(b[i]), float(e[i])) for i in range(n)}


def frnn_get_profile() -> dict[str, float]:
    """Per-phase milliseconds of the last profiled call (synchronises on it)."""
    buf = (_c.c_float * 16)()
    n = lib().frnn_get_profile(buf, 16)
    if n < 0:
        raise FrnnError(n, "frnn_get_profile")
    return {lib().frnn_phase_name(i).decode(): float(buf[i]) for i in range(n)}


def frnn_release_cached() -> None:
    lib().frnn_release_cached()


def _require_cuda(points: torch.Tensor):
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2202_06929_b200 needs a CUDA device (no CPU fallback)")
    if not (points.is_cuda and points.dtype == torch.float32 and points.is_contiguous() and points.dim() == 2):
        raise ValueError("points must be a contiguous CUDA float32 tensor of shape (n, dim)")


def _ptr(t):
    return None if t is None else _c.c_void_p(t.data_ptr())


@dataclass
class EdgeList:
    """Device-resident result.  ``src/dst/d2`` have ``edge_capacity`` entries; the first ``count``
    (device scalar; ``n_edges()`` synchronises) are valid and (src,dst)-sorted."""
    src: torch.Tensor
    dst: torch.Tensor
    d2: torch.Tensor
    count: torch.Tensor             # int64[1] (single event) or int64[B+1] edge offsets (batched)
    status: torch.Tensor            # int32[1]
    row_ptr: torch.Tensor | None

    def n_edges(self) -> int:
        return int(self.count[-1].item())

    def check(self):
        st = int(self.status.item())
        if st != FRNN_OK:
            raise FrnnError(st, "device status")
        return self

    def trimmed(self):
        e = self.n_edges()
        return self.src[:e], self.dst[:e], self.d2[:e]


class Workspace:
    """Reusable device scratch + output buffers for repeated calls of one shape."""

    def __init__(self, n_total: int, n_events: int, k_max: int, edge_capacity: int, device=None, want_row_ptr: bool = False,
                 dim: int = 8, opt: FrnnOptions | None = None):
        device = device or torch.device("cuda", torch.cuda.current_device())
        self.bytes = frnn_workspace_bytes(n_total, n_events, dim, k_max, opt)
        self.buf = torch.empty(max(self.bytes, 256), dtype=torch.uint8, device=device)
        self.edge_capacity = int(edge_capacity)
        cap = max(self.edge_capacity, 1)
        self.src = torch.empty(cap, dtype=torch.int32, device=device)
        self.dst = torch.empty(cap, dtype=torch.int32, device=device)
        self.d2 = torch.empty(cap, dtype=torch.float32, device=device)
        self.count = torch.zeros(n_events + 1 if n_events > 1 else 1, dtype=torch.int64, device=device)
        self.status = torch.zeros(1, dtype=torch.int32, device=device)
        self.row_ptr = torch.empty(n_total + 1, dtype=torch.int64, device=device) if want_row_ptr else None


def frnn_build_dense_ex(points: torch.Tensor, r: float, k_max: int, edge_capacity: int | None = None,
                        ws: Workspace | None = None, stream: torch.cuda.Stream | None = None,
                        want_row_ptr: bool = False) -> EdgeList:
    """The brute-force variant of ``frnn_build_ex``: same result, O(n^2)."""
    return frnn_build_ex(points, r, k_max, edge_capacity, ws, stream, want_row_ptr, _entry="frnn_build_dense_ex")


def frnn_build_ex(points: torch.Tensor, r: float, k_max: int, edge_capacity: int | None = None,
                  ws: Workspace | None = None, stream: torch.cuda.Stream | None = None,
                  want_row_ptr: bool = False, _entry: str = "frnn_build_ex", opt: FrnnOptions | None = None) -> EdgeList:
    """Asynchronous single-event build on ``stream`` (default: torch's current stream); ``opt``: frnn_build_opt."""
    _require_cuda(points)
    n, dim = points.shape
    if edge_capacity is None:
        edge_capacity = ws.edge_capacity if ws is not None else n * k_max
    if ws is None:
        ws = Workspace(n, 1, k_max, edge_capacity, points.device, want_row_ptr, dim, opt)
    stream = stream or torch.cuda.current_stream(points.device)
    args = (_ptr(points), n, dim, float(r), int(k_max), _ptr(ws.src), _ptr(ws.dst), _ptr(ws.d2),
            int(edge_capacity), _ptr(ws.count), _ptr(ws.status), _ptr(ws.row_ptr),
            _ptr(ws.buf), ws.buf.numel(), _c.c_void_p(stream.cuda_stream))
    if opt is not None:
        assert _entry == "frnn_build_ex"
        _entry = "frnn_build_opt"
        st = lib().frnn_build_opt(_c.byref(opt), *args)
    else:
        st = getattr(lib(), _entry)(*args)
    _check(st, _entry)
    return EdgeList(ws.src, ws.dst, ws.d2, ws.count, ws.status, ws.row_ptr)


FRNN_STATIC_MAX_ROWS = 8192


def frnn_static_scratch_bytes() -> int:
    """Size of the library's built-in scratch array (held by every GPU that loads the library)."""
    return int(lib().frnn_static_scratch_bytes())


def frnn_build_static(points: torch.Tensor, r: float, k_max: int, out_src: torch.Tensor, out_dst: torch.Tensor,
                      out_d2: torch.Tensor, out_count: torch.Tensor, out_status: torch.Tensor,
                      out_row_ptr: torch.Tensor | None = None, stream: torch.cuda.Stream | None = None) -> EdgeList:
    """``frnn_build_static`` of include/frnn.h: the single-event build for callers that cannot allocate device
    memory on their event path (all memory handed to a framework arena at configure time, a latency-bound loop where
    ``cudaMalloc`` would stall the device, a plug-in under a foreign allocator).  The scratch is a 3 MiB array inside
    the library, so ``points`` may have at most ``FRNN_STATIC_MAX_ROWS`` rows; the caller passes every output
    (``out_src/out_dst/out_d2``: equally long device arrays = the edge capacity; ``out_count`` int64[1];
    ``out_status`` int32[1]; optional ``out_row_ptr`` int64[n+1]) and this wrapper allocates no tensor either.
    All calls on a device share the one scratch array: keep them ordered on the GPU (one stream, or events);
    make the first call on a device outside any stream capture.  Asynchronous on ``stream``."""
    _require_cuda(points)
    n, dim = points.shape
    cap = min(out_src.numel(), out_dst.numel(), out_d2.numel())
    stream = stream or torch.cuda.current_stream(points.device)
    st = lib().frnn_build_static(_ptr(points), n, dim, float(r), int(k_max), _ptr(out_src), _ptr(out_dst), _ptr(out_d2), int(cap),
                                 _ptr(out_count), _ptr(out_status), _ptr(out_row_ptr), _c.c_void_p(stream.cuda_stream))
    if st == FRNN_ERR_UNSUPPORTED and n > FRNN_STATIC_MAX_ROWS:
        raise FrnnError(st, f"frnn_build_static [{frnn_last_error_string()}]")
    _check(st, "frnn_build_static")
    return EdgeList(out_src, out_dst, out_d2, out_count, out_status, out_row_ptr)


def frnn_build_opt(opt: FrnnOptions | None, points: torch.Tensor, r: float, k_max: int, **kw) -> EdgeList:
    """frnn_build_ex with per-call options."""
    return frnn_build_ex(points, r, k_max, opt=opt, **kw)


def frnn_build_batched(points: torch.Tensor, event_offsets, r: float, k_max: int, edge_capacity: int | None = None,
                       ws: Workspace | None = None, stream: torch.cuda.Stream | None = None,
                       want_row_ptr: bool = False, opt: FrnnOptions | None = None) -> EdgeList:
    """Asynchronous batched build: ``event_offsets`` is a host sequence of B+1 ascending row offsets."""
    _require_cuda(points)
    n, dim = points.shape
    offs = [int(v) for v in event_offsets]
    n_events = len(offs) - 1
    if edge_capacity is None:
        edge_capacity = ws.edge_capacity if ws is not None else n * k_max
    if ws is None:
        ws = Workspace(n, n_events, k_max, edge_capacity, points.device, want_row_ptr, dim, opt)
    count = ws.count if ws.count.numel() == n_events + 1 else torch.zeros(n_events + 1, dtype=torch.int64, device=points.device)
    stream = stream or torch.cuda.current_stream(points.device)
    c_offs = (_c.c_int64 * (n_events + 1))(*offs)
    args = (_ptr(points), c_offs, n_events, dim, float(r), int(k_max), _ptr(ws.src), _ptr(ws.dst),
            _ptr(ws.d2), int(edge_capacity), _ptr(count), _ptr(ws.status), _ptr(ws.row_ptr),
            _ptr(ws.buf), ws.buf.numel(), _c.c_void_p(stream.cuda_stream))
    st = lib().frnn_build_batched_opt(_c.byref(opt), *args) if opt is not None else lib().frnn_build_batched(*args)
    _check(st, "frnn_build_batched")
    return EdgeList(ws.src, ws.dst, ws.d2, count, ws.status, ws.row_ptr)


def frnn_build(points: torch.Tensor, r: float, k_max: int):
    """The synchronous 9-argument form: returns trimmed (src, dst, d2) device tensors."""
    _require_cuda(points)
    n, dim = points.shape
    cap = max(n * k_max, 1)
    src = torch.empty(cap, dtype=torch.int32, device=points.device)
    dst = torch.empty(cap, dtype=torch.int32, device=points.device)
    d2 = torch.empty(cap, dtype=torch.float32, device=points.device)
    count = _c.c_int64(0)
    torch.cuda.current_stream(points.device).synchronize()      # the C call uses the legacy default stream
    st = lib().frnn_build(_ptr(points), n, dim, float(r), int(k_max), _ptr(src), _ptr(dst), _ptr(d2), _c.byref(count))
    _check(st, "frnn_build")
    e = count.value
    return src[:e], dst[:e], d2[:e]


def frnn_build_host(points_host: torch.Tensor, r: float, k_max: int, out_src: torch.Tensor, out_dst: torch.Tensor,
                    out_d2: torch.Tensor) -> int:
    """End-to-end call on HOST tensors (pinned recommended): H2D, build, D2H.  Returns the edge count."""
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2202_06929_b200 needs a CUDA device (no CPU fallback)")
    assert not points_host.is_cuda and points_host.dtype == torch.float32 and points_host.is_contiguous()
    n, dim = points_host.shape
    cap = min(out_src.numel(), out_dst.numel(), out_d2.numel())
    count = _c.c_int64(0)
    st = lib().frnn_build_host(_ptr(points_host), n, dim, float(r), int(k_max), _ptr(out_src), _ptr(out_dst), _ptr(out_d2),
                               cap, _c.byref(count))
    _check(st, "frnn_build_host")
    return count.value


def frnn_gather_edge_rows(points: torch.Tensor, src: torch.Tensor, dst: torch.Tensor, edge_count: torch.Tensor | None = None,
                          e_begin: int = 0, e_max: int | None = None, row_base: int = 0, out: torch.Tensor | None = None,
                          stream: torch.cuda.Stream | None = None) -> torch.Tensor:
    """[x_src || x_dst] rows of the edges [e_begin, min(e_begin + e_max, edge_count)) (the filter stage's input)."""
    _require_cuda(points)
    n, dim = points.shape
    if e_max is None:
        e_max = src.numel() - e_begin
    if out is None:
        out = torch.empty((max(e_max, 0), 2 * dim), dtype=torch.float32, device=points.device)
    stream = stream or torch.cuda.current_stream(points.device)
    st = lib().frnn_gather_edge_rows(_ptr(points), n, dim, _ptr(src), _ptr(dst), _ptr(edge_count), int(e_begin), int(e_max),
                                     int(row_base), _ptr(out), _c.c_void_p(stream.cuda_stream))
    _check(st, "frnn_gather_edge_rows")
    return out


def frnn_label_components(n: int, src: torch.Tensor, dst: torch.Tensor, score: torch.Tensor | None = None, threshold: float = 0.0,
                          edge_count: torch.Tensor | None = None, edge_max: int | None = None,
                          labels: torch.Tensor | None = None, n_components: torch.Tensor | None = None,
                          stream: torch.cuda.Stream | None = None):
    """labels[i] = smallest node index of the weakly connected component of i; returns (labels, n_components)."""
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2202_06929_b200 needs a CUDA device (no CPU fallback)")
    dev = src.device
    if edge_max is None:
        edge_max = src.numel()
    if labels is None:
        labels = torch.empty(max(n, 1), dtype=torch.int32, device=dev)[:n]
    if n_components is None:
        n_components = torch.zeros(1, dtype=torch.int32, device=dev)
    stream = stream or torch.cuda.current_stream(dev)
    st = lib().frnn_label_components(int(n), _ptr(src), _ptr(dst), _ptr(score), float(threshold), _ptr(edge_count), int(edge_max),
                                     _ptr(labels), _ptr(n_components), _c.c_void_p(stream.cuda_stream))
    _check(st, "frnn_label_components")
    return labels, n_components


class HostPipeline:
    """frnn_host_pipeline_*: a stream of host-resident events with copies and builds overlapped."""

    def __init__(self, n_max: int, k_max: int, edge_capacity: int, depth: int = 3, opt: FrnnOptions | None = None):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2202_06929_b200 needs a CUDA device (no CPU fallback)")
        self._h = _c.c_void_p()
        _check(lib().frnn_host_pipeline_create_opt(_opt_ref(opt), int(n_max), 8, int(k_max), int(edge_capacity), int(depth),
                                                   _c.byref(self._h)), "frnn_host_pipeline_create")

    def submit(self, points_host: torch.Tensor, r: float, out_src: torch.Tensor, out_dst: torch.Tensor, out_d2: torch.Tensor,
               out_count: torch.Tensor) -> None:
        n = points_host.shape[0]
        _check(lib().frnn_host_pipeline_submit(self._h, _ptr(points_host), n, float(r), _ptr(out_src), _ptr(out_dst), _ptr(out_d2),
                                               _ptr(out_count)), "frnn_host_pipeline_submit")

    def wait(self) -> None:
        _check(lib().frnn_host_pipeline_wait(self._h), "frnn_host_pipeline_wait")

    def close(self) -> None:
        if self._h:
            lib().frnn_host_pipeline_destroy(self._h)
            self._h = _c.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def frnn_set_bin_order(order=None) -> None:
    """Coordinates to bin (first) and to key (next four); None / empty restores the default."""
    order = [int(v) for v in (order or [])]
    arr = (_c.c_int * max(len(order), 1))(*order)
    _check(lib().frnn_set_bin_order(arr if order else None, len(order)), "frnn_set_bin_order")


def frnn_suggest_bin_order(points: torch.Tensor, r: float, stream: torch.cuda.Stream | None = None):
    """Data-driven ranking of the coordinates of ``points`` (device, n x dim): returns (order[8], score[16])."""
    _require_cuda(points)
    n, dim = points.shape
    order, score = (_c.c_int * 8)(), (_c.c_float * 16)()
    stream = stream or torch.cuda.current_stream(points.device)
    _check(lib().frnn_suggest_bin_order(_ptr(points), n, dim, float(r), order, score, _c.c_void_p(stream.cuda_stream)),
           "frnn_suggest_bin_order")
    return list(order), list(score)
