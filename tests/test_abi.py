"""The C-ABI library loads on a CPU-only box and exports every symbol include/frnn.h declares.
No compute entry point is called here (there is no GPU and no CPU fallback)."""
from __future__ import annotations

import ctypes
import os
import re

import pytest

from paper_2202_06929_b200 import frnn

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def header_functions():
    text = open(os.path.join(ROOT, "include", "frnn.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(frnn_[a-z_]+)\s*\(", text)))


def test_header_declares_the_north_star_entry_points():
    names = header_functions()
    for required in ("frnn_build", "frnn_build_ex", "frnn_build_batched", "frnn_workspace_bytes", "frnn_status_string"):
        assert required in names


def test_library_exports_every_declared_symbol():
    lib = frnn.lib()
    for name in header_functions():
        assert hasattr(lib, name), f"{name} is declared in include/frnn.h but not exported"
    assert sorted(frnn.EXPORTED_SYMBOLS) == header_functions()
    raw = ctypes.CDLL(frnn.library_path())
    assert raw.frnn_version() == frnn.frnn_version() >= 100


def test_host_only_entry_points():
    assert frnn.frnn_status_string(frnn.FRNN_OK) == "ok"
    assert "workspace" in frnn.frnn_status_string(frnn.FRNN_ERR_WORKSPACE)
    assert frnn.frnn_workspace_bytes(120000, 1, 8, 256) > 120000 * 32
    assert frnn.frnn_workspace_bytes(120000, 1, 17, 256) == 0         # dim outside 1..16
    assert frnn.frnn_workspace_bytes(120000, 1, 12, 256) == frnn.frnn_workspace_bytes(120000, 1, 8, 256) + 120000 * 32   # the second internal row
    assert 0 < frnn.frnn_workspace_bytes(120000, 1, 3, 256) < frnn.frnn_workspace_bytes(120000, 1, 8, 256)   # 3 binned coordinates: smaller table
    assert frnn.frnn_workspace_bytes(-1, 1, 8, 256) == 0
    big = frnn.frnn_workspace_bytes(16 * 120000, 16, 8, 256)
    assert big > 16 * 120000 * 32
    try:
        frnn.frnn_set_grid(3, 4)
        assert frnn.frnn_get_grid(1000) == (3, 4)
        with pytest.raises(frnn.FrnnError):
            frnn.frnn_set_grid(9, 4)
        with pytest.raises(frnn.FrnnError):
            frnn.frnn_set_grid(3, 1)
    finally:
        frnn.frnn_set_grid(0, 0)
    d, b = frnn.frnn_get_grid(120000)
    assert 1 <= d <= 6 and 2 <= b <= 8
    # options never inherit frnn_set_grid's default; frnn_get_grid_opt says what a call with options runs on
    try:
        frnn.frnn_set_grid(2, 7)
        assert frnn.frnn_get_grid(120000) == (2, 7)
        assert frnn.frnn_get_grid_opt(frnn.frnn_options(), 120000) == (d, b)
        assert frnn.frnn_get_grid_opt(frnn.frnn_options(3, 6), 120000) == (3, 6)
        assert frnn.frnn_get_grid_opt(None, 120000) == (2, 7)
        assert frnn.frnn_get_grid_opt(frnn.frnn_options(frnn.FRNN_GRID_AUTO), 120000) == (0, 0)
    finally:
        frnn.frnn_set_grid(0, 0)
    assert frnn.frnn_get_grid(120000, 1, 2)[0] == 2                    # never more binned coordinates than the rows have
    # the linear cell id (event, cell) must fit 32 bits for any batch size
    d, b = frnn.frnn_get_grid(120000 * 4096, 4096)
    assert d * b + 12 <= 31


def test_options_struct_and_sizing():
    """frnn_options: layout, defaults, validation and workspace sizing (host only)."""
    o = frnn.frnn_options()
    assert o.struct_bytes == ctypes.sizeof(frnn.FrnnOptions) == 72
    assert (o.grid_dims, o.grid_bits, o.order_count, o.launch_mode, o.timeline) == (0, 0, 0, 0, 0)
    base = frnn.frnn_workspace_bytes(120000, 1, 8, 256)
    assert frnn.frnn_workspace_bytes(120000, 1, 8, 256, o) == base
    assert frnn.frnn_workspace_bytes(120000, 1, 8, 256, frnn.frnn_options(4, 5)) == base
    assert frnn.frnn_workspace_bytes(120000, 1, 8, 256, frnn.frnn_options(2, 8)) < base          # 65k cells instead of 1M
    assert frnn.frnn_workspace_bytes(120000, 1, 8, 256, frnn.frnn_options(4, 6)) > base
    assert frnn.frnn_workspace_bytes(120000, 1, 8, 256, frnn.frnn_options(order=[3, 1])) == base + (120000 * 4 + 255) // 256 * 256   # slot -> cell array
    assert frnn.frnn_workspace_bytes(120000, 1, 8, 256, frnn.frnn_options(order=[0, 1, 2])) == base   # the default order written out
    assert frnn.frnn_workspace_bytes(120000, 1, 8, 256, frnn.frnn_options(9, 5)) == 0                # invalid options
    assert frnn.frnn_workspace_bytes(120000, 1, 8, 256, frnn.frnn_options(order=[4, 4])) == 0
    auto = frnn.frnn_options(frnn.FRNN_GRID_AUTO)
    assert frnn.frnn_workspace_bytes(120000, 1, 8, 256, auto) >= max(
        frnn.frnn_workspace_bytes(120000, 1, 8, 256, frnn.frnn_options(g, b)) for g, b in ((4, 5), (3, 7), (2, 8), (5, 4)))   # room for any pick
    assert frnn.frnn_workspace_bytes(120000, 1, 8, 256, frnn.frnn_options(-2)) == 0
    assert frnn.frnn_last_error_string() == ""


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(RuntimeError):
        frnn.frnn_build_ex(torch.zeros((4, 8)), 0.1, 4)
    with pytest.raises(RuntimeError):
        frnn.frnn_build_host(torch.zeros((4, 8)), 0.1, 4, torch.zeros(4, dtype=torch.int32),
                             torch.zeros(4, dtype=torch.int32), torch.zeros(4))
