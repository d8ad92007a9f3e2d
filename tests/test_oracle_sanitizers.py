"""The CPU oracle under AddressSanitizer + UndefinedBehaviorSanitizer ("ASan/UBSan on the CPU oracle").

``tests/oracle_sanitizer_driver.c`` includes ``oracle/frnn_oracle.c`` itself and is built with
``-fsanitize=address,undefined -fno-sanitize-recover=all``; every case below must run clean (exit code 0, nothing on
stderr) and give the same edges as the ordinary build of the oracle (count and checksums of src, dst, the d2 bit
patterns and the uncapped degrees)."""
from __future__ import annotations

import os
import struct
import subprocess

import numpy as np
import pytest

import oracle
from paper_2202_06929_b200 import events
from tests import helpers as H

HERE = os.path.dirname(os.path.abspath(__file__))
FLAGS = ["-O1", "-g", "-std=c11", "-fopenmp", "-mfma", "-ffp-contract=off", "-fno-fast-math", "-fno-omit-frame-pointer",
         "-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-Wall"]


@pytest.fixture(scope="module")
def driver(tmp_path_factory):
    exe = str(tmp_path_factory.mktemp("san") / "oracle_sanitizer_driver")
    res = subprocess.run(["gcc", *FLAGS, os.path.join(HERE, "oracle_sanitizer_driver.c"), "-o", exe, "-lm"], capture_output=True, text=True)
    if res.returncode != 0 and "sanitize" in res.stderr and ("cannot find" in res.stderr or "not supported" in res.stderr):
        pytest.skip("this gcc has no sanitizer runtime: " + res.stderr.strip().splitlines()[-1])
    assert res.returncode == 0, res.stderr
    assert res.stderr.strip() == "", "warnings from -Wall:\n" + res.stderr
    return exe


def run_case(driver, tmp_path, x, r, k, mode, queries=None):
    x = np.ascontiguousarray(x, dtype=np.float32)
    n, dim = x.shape
    path = str(tmp_path / "case.bin")
    with open(path, "wb") as f:
        f.write(struct.pack("<qiiifq", n, dim, k, mode, float(np.float32(r)), -1 if queries is None else len(queries)))
        f.write(x.tobytes())
        if queries is not None:
            f.write(np.ascontiguousarray(queries, dtype=np.int64).tobytes())
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1", OMP_NUM_THREADS="4")
    res = subprocess.run([driver, path], capture_output=True, text=True, env=env, timeout=300)
    assert res.returncode == 0 and res.stderr.strip() == "", f"sanitizer report (rc {res.returncode}):\n{res.stderr[-3000:]}"
    got = [int(v) for v in res.stdout.split()]
    exp = oracle.frnn(x, r, k, mode, queries=queries)
    xor = 0
    for b in H.bits(exp.d2).astype(np.uint32):
        xor ^= int(b)
    assert got == [exp.count, int(exp.src.astype(np.int64).sum()), int(exp.dst.astype(np.int64).sum()), xor, int(exp.uncapped.sum())]
    return exp.count


@pytest.mark.parametrize("mode", [oracle.BRUTE, oracle.CELLS])
def test_hand_fixture_runs_clean(driver, tmp_path, mode):
    assert run_case(driver, tmp_path, H.HANDCASE_POINTS, 0.5, 64, mode) > 0
    assert run_case(driver, tmp_path, H.HANDCASE_POINTS, 0.5, 2, mode) > 0
    assert run_case(driver, tmp_path, H.HANDCASE_POINTS, 0.0, 1, mode) == 2          # the two exact duplicates (rows 0 and 4)


@pytest.mark.parametrize("mode", [oracle.BRUTE, oracle.CELLS])
def test_config0_event_runs_clean(driver, tmp_path, mode):
    cfg = events.CONFIGS[0]
    x = events.make_event(cfg)
    assert run_case(driver, tmp_path, x, cfg.r, cfg.k_max, mode) > cfg.n
    assert run_case(driver, tmp_path, x, cfg.r, 1, mode) > 0                           # every row capped to its nearest
    q = np.sort(np.random.default_rng(1).choice(cfg.n, 300, replace=False))
    assert run_case(driver, tmp_path, x, cfg.r, cfg.k_max, mode, queries=q) > 0


@pytest.mark.parametrize("mode", [oracle.BRUTE, oracle.CELLS])
def test_degenerate_inputs_run_clean(driver, tmp_path, mode):
    assert run_case(driver, tmp_path, np.zeros((0, 8), np.float32), 0.1, 4, mode) == 0
    assert run_case(driver, tmp_path, np.ones((1, 8), np.float32), 0.1, 4, mode) == 0
    assert run_case(driver, tmp_path, np.zeros((40, 3), np.float32), 0.0, 5, mode) == 40 * 5      # one cluster of duplicates, K binds
    assert run_case(driver, tmp_path, events.uniform_points(300, 1, -50.0, 50.0, 2), 0.7, 8, mode) > 0     # negative cells, 1 coordinate
    assert run_case(driver, tmp_path, events.uniform_points(200, 16, 0.0, 1.0, 3), 0.9, 300, mode) > 0
