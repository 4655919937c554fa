"""Multi-GPU plumbing for bench.py: one process per GPU, independent observations per rank.

The path shards by observation / time span with no exchange step: there is no
data-path collective.  torch.distributed is used only for the barrier around the timed region and
the max-over-ranks of the measured time.  Backend-agnostic so the host logic is testable with gloo.
"""
from __future__ import annotations

import dataclasses
import os
from typing import Tuple


def env() -> Tuple[int, int, int]:
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def init(backend: str | None = None, device=None) -> bool:
    """Initialise the default process group if WORLD_SIZE > 1.  Returns True if distributed."""
    rank, world, local = env()
    if world <= 1:
        return False
    import torch
    import torch.distributed as dist
    if dist.is_initialized():
        return True
    if backend is None:
        backend = "nccl" if torch.cuda.is_available() else "gloo"
    kw = {}
    if backend == "nccl" and device is not None:
        kw["device_id"] = device
    dist.init_process_group(backend, **kw)
    return True


def barrier() -> None:
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def max_over_ranks(t: float) -> float:
    """The slowest rank's time: every multi-GPU number is the max over ranks."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(t)
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    x = torch.tensor([t], dtype=torch.float64, device=dev)
    dist.all_reduce(x, op=dist.ReduceOp.MAX)
    return float(x.item())


def sum_over_ranks(v: int) -> int:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return int(v)
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    x = torch.tensor([v], dtype=torch.int64, device=dev)
    dist.all_reduce(x, op=dist.ReduceOp.SUM)
    return int(x.item())


def rank_workload(w, rank: int):
    """Rank r searches its own observation: same shape and plan, its own noise seed."""
    return dataclasses.replace(w, noise_seed=w.noise_seed + 1000 * rank) if rank else w


def shutdown() -> None:
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()
        dist.destroy_process_group()
