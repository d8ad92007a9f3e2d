"""Multi-GPU plumbing: one process per GPU, events sharded across ranks, no data-path collective.

SURVEY.md section 8(e): events are independent units (PAPER.md:73 averages over 500 independent
events), so the path shards by event with nothing to exchange; the only collectives are the
barrier and the two scalar reductions of the timing protocol (max time, summed units).
Backends: ``nccl`` on GPUs, ``gloo`` for the CPU tests of this host logic.
"""
from __future__ import annotations

import os
from dataclasses import dataclass

import torch
import torch.distributed as dist


@dataclass
class Rank:
    rank: int = 0
    local_rank: int = 0
    world_size: int = 1

    @property
    def is_main(self) -> bool:
        return self.rank == 0


def init_from_env(backend: str | None = None) -> Rank:
    """Join the process group torchrun describes (RANK / LOCAL_RANK / WORLD_SIZE / MASTER_*)."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world == 1:
        return Rank()
    rank = int(os.environ["RANK"])
    local = int(os.environ.get("LOCAL_RANK", rank))
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29511")
    if backend is None:
        backend = "nccl" if torch.cuda.is_available() else "gloo"
    if backend == "nccl":
        torch.cuda.set_device(local)
    if not dist.is_initialized():
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return Rank(rank, local, world)


def shard(items: list, r: Rank) -> list:
    """Round-robin assignment of independent work units (events) to ranks."""
    return items[r.rank::r.world_size]


def _device(r: Rank):
    return torch.device("cuda", r.local_rank) if dist.is_initialized() and dist.get_backend() == "nccl" else torch.device("cpu")


def barrier(r: Rank) -> None:
    if r.world_size > 1:
        dist.barrier()


def reduce_max(value: float, r: Rank) -> float:
    """Whole-job time = the slowest rank's device time."""
    if r.world_size == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=_device(r))
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def reduce_sum(value: float, r: Rank) -> float:
    """Whole-job units = the sum over ranks."""
    if r.world_size == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=_device(r))
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def gather_counts(value: int, r: Rank) -> list[int]:
    """Per-rank edge counts on every rank (what a caller would use to stitch global offsets)."""
    if r.world_size == 1:
        return [int(value)]
    t = torch.tensor([value], dtype=torch.int64, device=_device(r))
    out = [torch.zeros_like(t) for _ in range(r.world_size)]
    dist.all_gather(out, t)
    return [int(o.item()) for o in out]


def finalize(r: Rank) -> None:
    if r.world_size > 1 and dist.is_initialized():
        dist.destroy_process_group()
