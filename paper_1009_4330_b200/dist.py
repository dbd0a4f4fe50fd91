"""Rank bookkeeping for ``bench.py``: the MD hot path of this round runs on ONE GPU per problem
(BASELINE.json north_star: "Everything runs on one GPU"), so N GPUs run N independent replicas of
the workload -- no data-path collective.  ``torch.distributed`` is used only for the barrier that
brackets the timed region and for the max-over-ranks / sum-over-ranks of two scalars.

Works with ``nccl`` (GPU box) and ``gloo`` (CPU tests, world_size 2).
"""
from __future__ import annotations

import dataclasses
import os


@dataclasses.dataclass
class Rank:
    rank: int
    local_rank: int
    world: int
    backend: str | None     # None: single process, torch.distributed not initialised

    @property
    def is_root(self) -> bool:
        return self.rank == 0


def init(backend: str | None = None) -> Rank:
    """Reads RANK / LOCAL_RANK / WORLD_SIZE / MASTER_* from the environment (torchrun sets them)."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", str(rank)))
    if world <= 1:
        return Rank(0, local if "LOCAL_RANK" in os.environ else 0, 1, None)
    import torch
    import torch.distributed as dist
    if backend is None:
        backend = "nccl" if torch.cuda.is_available() else "gloo"
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29533")
    if backend == "nccl":
        torch.cuda.set_device(local)
    if not dist.is_initialized():
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return Rank(rank, local, world, backend)


def _device(r: Rank):
    import torch
    return torch.device("cuda", r.local_rank) if r.backend == "nccl" else torch.device("cpu")


def barrier(r: Rank) -> None:
    if r.backend is None:
        return
    import torch.distributed as dist
    if r.backend == "nccl":
        dist.barrier(device_ids=[r.local_rank])
    else:
        dist.barrier()


def all_max(r: Rank, value: float) -> float:
    if r.backend is None:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=_device(r))
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def all_sum(r: Rank, value: float) -> float:
    if r.backend is None:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=_device(r))
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def replica_seed_offset(r: Rank) -> int:
    """Each replica gets its own velocity seed (decorrelated trajectories, identical cost)."""
    return r.rank


def aggregate_throughput(r: Rank, units_this_rank: float, seconds_this_rank: float) -> tuple[float, float]:
    """(whole-job units / max-over-ranks time, max time): the contract's aggregate."""
    tmax = all_max(r, seconds_this_rank)
    total = all_sum(r, units_this_rank)
    return (total / tmax if tmax > 0 else 0.0), tmax


def finalize(r: Rank) -> None:
    if r.backend is None:
        return
    import torch.distributed as dist
    if dist.is_initialized():
        dist.destroy_process_group()
