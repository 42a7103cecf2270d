"""Multi-GPU plumbing for the replica mode (replicas only).

z-steps are sequential and every step is a global 2-D FFT, so one propagation does not
shard; independent propagations do.  Each rank runs its own propagations on its own GPU with
no data-path collective.  ``torch.distributed`` is used only to line the ranks up (barrier)
and to combine their timings (max) and unit counts (sum).  Works with ``nccl`` (GPU) and
``gloo`` (CPU tests).
"""
from __future__ import annotations

import os
from typing import Optional

import torch
import torch.distributed as dist


def env_world():
    """(rank, local_rank, world_size) from the torchrun environment (1 process if unset)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: Optional[str] = None) -> int:
    """Initialises the default process group when WORLD_SIZE > 1; returns world size."""
    rank, local_rank, world = env_world()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29500")
        if backend is None:
            backend = "nccl" if torch.cuda.is_available() else "gloo"
        kw = {}
        if backend == "nccl":
            torch.cuda.set_device(local_rank)
            kw["device_id"] = torch.device("cuda", local_rank)
        dist.init_process_group(backend=backend, rank=rank, world_size=world, **kw)
    return world


def _device():
    if dist.is_initialized() and dist.get_backend() == "nccl":
        return torch.device("cuda", torch.cuda.current_device())
    return torch.device("cpu")


def barrier():
    if dist.is_initialized():
        if dist.get_backend() == "nccl":
            dist.barrier(device_ids=[torch.cuda.current_device()])
        else:
            dist.barrier()


def max_over_ranks(x: float) -> float:
    if not dist.is_initialized():
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=_device())
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x: float) -> float:
    if not dist.is_initialized():
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=_device())
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def shard(n_units: int, rank: int, world: int):
    """Contiguous share [lo, hi) of n_units independent propagations for this rank."""
    lo = (n_units * rank) // world
    hi = (n_units * (rank + 1)) // world
    return lo, hi


def throughput(units_this_rank: float, seconds_this_rank: float) -> float:
    """Whole-job units per second: all ranks' units / the slowest rank's time."""
    total = sum_over_ranks(units_this_rank)
    t = max_over_ranks(seconds_this_rank)
    return total / t if t > 0 else float("nan")


def shutdown():
    if dist.is_initialized():
        dist.destroy_process_group()
