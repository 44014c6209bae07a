"""Multi-GPU = independent replicas.

A batch-1 decode step is one dependent chain: it has nothing to shard and no exchange step, so
N GPUs run N independent replicas (own weights copy, own KV cache, own prompt stream) with NO
data-path collective.  The only cross-rank traffic is the timing protocol of bench.py: a barrier
before and after the timed region, the MAX over ranks of the device-timed duration, and the SUM
of the units (tokens) every rank processed.  This module holds that host logic so that it can be
tested with the gloo backend on CPU (tests/test_replicas.py).
"""
from __future__ import annotations

import os
from dataclasses import dataclass
from typing import Optional


@dataclass
class Rank:
    rank: int = 0
    world: int = 1
    local_rank: int = 0
    group: Optional[object] = None   # None when world == 1 (no process group is created)


def init_from_env(backend: Optional[str] = None) -> Rank:
    """Read RANK / LOCAL_RANK / WORLD_SIZE / MASTER_* (torchrun) and create the process group.
    backend None: 'nccl' when CUDA is available, else 'gloo'."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", str(rank)))
    if world == 1:
        return Rank(0, 1, local, None)
    import torch
    import torch.distributed as dist
    if backend is None:
        backend = "nccl" if torch.cuda.is_available() else "gloo"
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29531")
    if backend == "nccl":
        torch.cuda.set_device(local)
        dist.init_process_group(backend, rank=rank, world_size=world, device_id=torch.device("cuda", local))
    else:
        dist.init_process_group(backend, rank=rank, world_size=world)
    return Rank(rank, world, local, dist.group.WORLD)


def _device_for(r: Rank):
    import torch
    import torch.distributed as dist
    if r.group is not None and dist.get_backend(r.group) == "nccl":
        return torch.device("cuda", r.local_rank)
    return torch.device("cpu")


def barrier(r: Rank) -> None:
    if r.world == 1:
        return
    import torch
    import torch.distributed as dist
    # an all-reduce on the group's device instead of dist.barrier(): works for gloo and nccl alike
    t = torch.zeros(1, device=_device_for(r))
    dist.all_reduce(t, group=r.group)
    if t.is_cuda:
        torch.cuda.synchronize()


def replica_seed(base_seed: int, r: Rank) -> int:
    """Each replica decodes its own prompt stream (weak scaling: per-GPU work fixed)."""
    return base_seed + 7919 * r.rank


def aggregate(r: Rank, elapsed_ms: float, units: float):
    """-> (max over ranks of elapsed_ms, sum over ranks of units).  Every rank gets the result."""
    if r.world == 1:
        return float(elapsed_ms), float(units)
    import torch
    import torch.distributed as dist
    dev = _device_for(r)
    t = torch.tensor([elapsed_ms], dtype=torch.float64, device=dev)
    u = torch.tensor([units], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=r.group)
    dist.all_reduce(u, op=dist.ReduceOp.SUM, group=r.group)
    return float(t.item()), float(u.item())


def whole_job_throughput(r: Rank, elapsed_ms: float, units: float) -> float:
    """value = units all ranks processed / max-over-ranks time (units per second)."""
    t, u = aggregate(r, elapsed_ms, units)
    return u / (t * 1e-3)


def shutdown(r: Rank) -> None:
    if r.world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()
