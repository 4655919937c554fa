"""Multi-GPU plumbing: one process per GPU, no data-path collective.

Two ways to use several GPUs, both without an exchange step on the data path:
  * independent observations, one per rank (bench.py --gpus N: weak scaling);
  * ONE observation sharded by time (`time_shards`, `shard_workload`, `merge_shards`): rank r searches a
    contiguous run of whole normalisation blocks plus the DM-sweep / boxcar halo, keeps the candidates that
    start inside its blocks and rank 0 gathers and sorts the lists.  Because normalisation blocks live on the
    absolute sample index (A9) the merged list equals the single-GPU list exactly.
torch.distributed is used for the barrier around the timed region, the max-over-ranks of the measured time
and the gather of the candidate lists.  Backend-agnostic so the host logic is testable with gloo.
"""
from __future__ import annotations

import dataclasses
import os
from typing import Tuple


def env() -> Tuple[int, int, int]:
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def _parse_cpulist(text: str):
    cpus = []
    for part in text.strip().split(","):
        if not part:
            continue
        a, _, b = part.partition("-")
        cpus += list(range(int(a), int(b or a) + 1))
    return cpus


def gpu_numa_node(local: int):
    """NUMA node the GPU `local` hangs off (sysfs, through its PCI address), or None if the host does not say."""
    try:
        import torch
        p = torch.cuda.get_device_properties(local)
        addr = f"{p.pci_domain_id:04x}:{p.pci_bus_id:02x}:{p.pci_device_id:02x}.0"
        with open(f"/sys/bus/pci/devices/{addr}/numa_node") as f:
            node = int(f.read().strip())
        return node if node >= 0 else None
    except Exception:
        return None


def rank_cpus(local: int, world: int, node_cpus=None, allowed=None):
    """The host cores rank `local` of `world` ranks on this node should run on: the cores of its GPU's NUMA node
    (all allowed cores if unknown), split evenly among the ranks that share them.  Pure function of its arguments when
    `node_cpus` / `allowed` are given (tests)."""
    if allowed is None:
        allowed = sorted(os.sched_getaffinity(0))
    cpus = [c for c in (node_cpus or allowed) if c in set(allowed)] or list(allowed)
    if world <= 1:
        return cpus
    # ranks are spread over the nodes in order; the ranks of one node share its cores evenly
    per = max(1, len(cpus) // world) if node_cpus is None else max(1, len(cpus) * max(1, _nodes_hint(node_cpus, allowed)) // world)
    per = min(per, len(cpus))
    share = local % max(1, len(cpus) // per)
    return cpus[share * per:(share + 1) * per] or cpus


def _nodes_hint(node_cpus, allowed) -> int:
    """How many NUMA nodes the allowed cores span, guessed from the size of this one."""
    return max(1, round(len(allowed) / max(1, len(node_cpus))))


def place_rank(local: int, world: int) -> dict:
    """Bind this rank's host threads (the per-stream workers of aa_run, the generator's OpenMP team) to cores of its
    GPU's NUMA node and cap the OpenMP team at its share, BEFORE the pinned observation is allocated, so that
    first touch puts the pages next to the GPU.  With 8 ranks on one node that is 8 x 34 GB of pinned memory and
    8 x (n_streams + generator) threads which would otherwise all float over both sockets.  Best effort: a host
    that hides sysfs or forbids sched_setaffinity is left alone.  Returns what was done (bench.py logs it)."""
    info = {"numa_node": None, "cpus": None, "omp_threads": None}
    try:
        node = gpu_numa_node(local)
        node_cpus = None
        if node is not None:
            with open(f"/sys/devices/system/node/node{node}/cpulist") as f:
                node_cpus = _parse_cpulist(f.read())
        cpus = rank_cpus(local, world, node_cpus)
        if world > 1 or node_cpus:
            os.sched_setaffinity(0, cpus)
        info.update({"numa_node": node, "cpus": len(cpus)})
        # torchrun exports OMP_NUM_THREADS=1 to every rank unless the user set it: that would fill 34 GB per rank with one
        # thread; a value of 1 under torchrun is therefore read as "not chosen" and replaced by the rank's share of cores
        if "OMP_NUM_THREADS" not in os.environ or (world > 1 and os.environ["OMP_NUM_THREADS"] == "1"):
            os.environ["OMP_NUM_THREADS"] = str(max(1, len(cpus)))
        info["omp_threads"] = int(os.environ["OMP_NUM_THREADS"])
    except Exception as e:                                  # placement is an optimisation, never a failure
        info["error"] = f"{type(e).__name__}: {e}"
    return info


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


@dataclasses.dataclass(frozen=True)
class TimeShard:
    rank: int
    t_first: int      # first raw input sample of the shard
    nsamp: int        # raw input samples the shard reads (its blocks + DM sweep + boxcar tail); 0 = nothing to do
    keep: int         # candidates with local t_start < keep belong to this shard


def time_shards(nsamp: int, maxshift: int, norm_block: int, tail: int, world: int):
    """Split the valid output span [0, nsamp - maxshift) into `world` contiguous runs of whole normalisation
    blocks.  `tail` = (wmax - 1) * bin_max rounded up to a multiple of every bin: the samples past a shard's
    last block that its boxcars may touch (the halo of DESIGN.md section 5 is maxshift + tail)."""
    t_valid = nsamp - maxshift
    if t_valid <= 0:
        raise ValueError("observation shorter than the DM sweep")
    nblocks = -(-t_valid // norm_block)
    per = -(-nblocks // world)
    out = []
    for r in range(world):
        b0 = min(r * per, nblocks)
        b1 = min(b0 + per, nblocks)
        if b0 == b1:
            out.append(TimeShard(r, 0, 0, 0))
            continue
        t_first = b0 * norm_block
        keep = min(b1 * norm_block, t_valid) - t_first
        n_in = nsamp - t_first if b1 == nblocks else min(keep + maxshift + tail, nsamp - t_first)
        out.append(TimeShard(r, t_first, n_in, keep))
    return out


def shard_workload(w, shard: TimeShard):
    """The plan of one shard: same band, DM plan and widths on `shard.nsamp` samples (pulses are data, not plan)."""
    return dataclasses.replace(w, nsamp=shard.nsamp, pulses=(), name=f"{w.name}_shard{shard.rank}")


def merge_shards(cands, shard: TimeShard):
    """Keep this shard's own candidates, move them to absolute time, gather on rank 0 and sort by
    (dm_index, t_start).  Returns the merged structured array on rank 0 (every rank if not distributed),
    None elsewhere."""
    import numpy as np
    mine = cands[cands["t_start"] < shard.keep].copy()
    mine["t_start"] += np.uint32(shard.t_first)
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        rank, world = dist.get_rank(), dist.get_world_size()
        parts = [None] * world if rank == 0 else None
        dist.gather_object(mine, parts, dst=0)
        if rank != 0:
            return None
        mine = np.concatenate(parts)
    return mine[np.lexsort((mine["t_start"], mine["dm_index"]))]


def shutdown() -> None:
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()
        dist.destroy_process_group()
