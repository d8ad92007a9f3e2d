"""The N>1 host logic on CPU: two gloo ranks shard events round-robin, reduce time by MAX and units by
SUM, gather per-rank counts (the path shards by event, no data-path collective)."""
from __future__ import annotations

import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.multiprocessing as mp  # noqa: E402

from paper_2202_06929_b200 import dist as D  # noqa: E402
from paper_2202_06929_b200 import events  # noqa: E402


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    r = D.init_from_env(backend="gloo")
    assert (r.rank, r.world_size, r.is_main) == (rank, world, rank == 0)
    seeds = D.shard(list(range(7)), r)
    assert seeds == events.shard_events(7, world, rank)
    # "work": the number of rows of each of my events (stands in for per-event edge counts)
    cfg = events.CONFIGS[0]
    units = sum(len(events.make_event(cfg, s)) for s in seeds)
    D.barrier(r)
    t_max = D.reduce_max(10.0 + rank, r)
    total = D.reduce_sum(units, r)
    counts = D.gather_counts(units, r)
    D.barrier(r)
    np.save(os.path.join(out_dir, f"r{rank}.npy"), np.array([t_max, total, *counts], dtype=np.float64))
    D.finalize(r)


def test_two_gloo_ranks_shard_reduce_and_gather(tmp_path):
    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    cfg = events.CONFIGS[0]
    res = [np.load(tmp_path / f"r{k}.npy") for k in range(world)]
    for k in range(world):
        assert res[k][0] == 10.0 + (world - 1)               # max over ranks
        assert res[k][1] == 7 * cfg.n                        # sum over ranks = all events
        assert res[k][2:].tolist() == [4 * cfg.n, 3 * cfg.n]  # rank 0 owns seeds 0,2,4,6; rank 1 owns 1,3,5
    assert np.array_equal(res[0], res[1])


def test_single_process_defaults():
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        os.environ.pop(k, None)
    r = D.init_from_env()
    assert (r.rank, r.world_size, r.is_main) == (0, 1, True)
    assert D.shard([1, 2, 3], r) == [1, 2, 3]
    assert D.reduce_max(3.5, r) == 3.5 and D.reduce_sum(2, r) == 2.0 and D.gather_counts(9, r) == [9]
    D.barrier(r)
    D.finalize(r)
