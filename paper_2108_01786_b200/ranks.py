"""Rank plumbing of ``bench.py --gpus N``.

The path has no inter-GPU exchange (north_star: one GPU, no sharding, no collective on the data path), so N
ranks are N independent replicas of the same step.  What the ranks share is only the measurement protocol:
a barrier on both sides of the timed region, the MAX over ranks of the device time, and the aggregate
``value`` = units all ranks processed / that time.  This module holds exactly that, backend-agnostic
(``nccl`` on the GPU box, ``gloo`` in the CPU tests), and none of the method's arithmetic.
"""
from __future__ import annotations

import os
from dataclasses import dataclass
from typing import Callable, Optional, Sequence


@dataclass
class Ranks:
    rank: int
    local_rank: int
    world: int
    backend: Optional[str]          # None when world == 1 (no process group at all)
    device: str                     # "cuda" or "cpu": where the reduction tensors live

    @property
    def is_root(self) -> bool:
        return self.rank == 0


def from_env(backend: str = "nccl") -> Ranks:
    """Reads RANK / LOCAL_RANK / WORLD_SIZE (torchrun) and creates the process group when WORLD_SIZE > 1."""
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    dev = "cuda" if backend == "nccl" else "cpu"
    if world > 1:
        import torch
        import torch.distributed as dist
        if not dist.is_initialized():
            if backend == "nccl":
                dist.init_process_group("nccl", device_id=torch.device("cuda", local))
            else:
                dist.init_process_group(backend)
        return Ranks(rank, local, world, backend, dev)
    return Ranks(rank, local, 1, None, dev)


def barrier(r: Ranks, device_sync: Optional[Callable[[], None]] = None) -> None:
    """Process-group barrier, then the device synchronisation (torch.cuda.synchronize on the GPU box)."""
    if r.world > 1:
        import torch.distributed as dist
        dist.barrier()
    if device_sync is not None:
        device_sync()


def max_over_ranks(r: Ranks, v: float) -> float:
    if r.world == 1:
        return float(v)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(v)], dtype=torch.float64, device=r.device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t[0])


def sum_over_ranks(r: Ranks, v: float) -> float:
    if r.world == 1:
        return float(v)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(v)], dtype=torch.float64, device=r.device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t[0])


def aggregate_value(r: Ranks, units_this_rank: float, seconds_this_rank: float) -> tuple:
    """Whole-job throughput of independent replicas: (sum of the units over ranks) / (max of the time over ranks).
    Returns (value, max_seconds, total_units); identical on every rank."""
    tmax = max_over_ranks(r, seconds_this_rank)
    total = sum_over_ranks(r, units_this_rank)
    return total / tmax, tmax, total


def assign_replicas(n_items: int, world: int) -> Sequence[range]:
    """Contiguous split of n_items independent problems (e.g. Runge-Kutta stages) over the ranks; the first
    n_items % world ranks get one more.  Rank i works on assign_replicas(n, w)[i]."""
    base, extra = divmod(n_items, world)
    out, lo = [], 0
    for i in range(world):
        hi = lo + base + (1 if i < extra else 0)
        out.append(range(lo, hi))
        lo = hi
    return out


def finish(r: Ranks) -> None:
    if r.world > 1:
        import torch.distributed as dist
        if dist.is_initialized():
            dist.destroy_process_group()
