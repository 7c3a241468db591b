"""Process-group plumbing for bench.py (one process per GPU, torch.distributed).

The hot path itself does not shard ("one B200, no sharding, no collectives",
BASELINE.json north_star): with N > 1 every rank runs an
independent replica of the layer on its own GPU and there is NO data-path collective.
torch.distributed is used only for the timing protocol: barrier, max-over-ranks of the
device time, sum of the units processed.  Works with backend "nccl" (GPU) and "gloo" (CPU
tests, world_size 2).
"""
from __future__ import annotations

import os
from typing import Optional

import torch
import torch.distributed as dist


class Group:
    def __init__(self, rank: int, world: int, local_rank: int, backend: Optional[str]):
        self.rank, self.world, self.local_rank, self.backend = rank, world, local_rank, backend

    @property
    def is_main(self) -> bool:
        return self.rank == 0

    def _dev(self):
        return torch.device("cuda", self.local_rank) if self.backend == "nccl" else torch.device("cpu")

    def barrier(self) -> None:
        if self.world > 1:
            if self.backend == "nccl":
                dist.barrier(device_ids=[self.local_rank])
            else:
                dist.barrier()

    def max_over_ranks(self, x: float) -> float:
        if self.world == 1:
            return float(x)
        t = torch.tensor([float(x)], dtype=torch.float64, device=self._dev())
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    def sum_over_ranks(self, x: float) -> float:
        if self.world == 1:
            return float(x)
        t = torch.tensor([float(x)], dtype=torch.float64, device=self._dev())
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        return float(t.item())

    def close(self) -> None:
        if self.world > 1 and dist.is_initialized():
            dist.destroy_process_group()


def init_from_env(backend: Optional[str] = None) -> Group:
    """Reads RANK / LOCAL_RANK / WORLD_SIZE / MASTER_ADDR / MASTER_PORT (torchrun)."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world == 1:
        return Group(0, 1, local, None)
    backend = backend or ("nccl" if torch.cuda.is_available() else "gloo")
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29511")
    if backend == "nccl":
        torch.cuda.set_device(local)
    dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return Group(rank, world, local, backend)


def aggregate_throughput(group: Group, units_this_rank: float, device_ms_this_rank: float):
    """Whole-job throughput for independent replicas: (sum of units) / (max time).
    Returns (units_per_s, max_ms)."""
    max_ms = group.max_over_ranks(device_ms_this_rank)
    total = group.sum_over_ranks(units_this_rank)
    return total / (max_ms * 1e-3), max_ms
