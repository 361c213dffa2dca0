"""Replica plumbing for `bench.py --gpus N`.

The graded path runs all S emulated stages on ONE GPU and has no exchange step between GPUs
("without data parallelism", "No global flush or
cross-stage barrier"), so N GPUs run N independent replicas of the same job.  The only cross-rank
traffic is the benchmark's own bookkeeping: a barrier before and after the timed region, the MAX of
the per-rank times and the SUM of the per-rank work.  `torch.distributed` (NCCL on GPUs, gloo in the
CPU tests) carries it; there is no data-path collective.
"""
from __future__ import annotations

import os


def init_from_env(backend: str | None = None):
    """Initialise torch.distributed from RANK / WORLD_SIZE / MASTER_* if WORLD_SIZE > 1.
    Returns (rank, world_size, local_rank)."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch
        import torch.distributed as dist
        if not dist.is_initialized():
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29511")
            if backend is None:
                backend = "nccl" if torch.cuda.is_available() else "gloo"
            kw = {}
            if backend == "nccl":
                torch.cuda.set_device(local)
                kw["device_id"] = torch.device("cuda", local)
            dist.init_process_group(backend=backend, rank=rank, world_size=world, **kw)
    return rank, world, local


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def aggregate(local_ms: float, local_units: float, device=None):
    """(max over ranks of local_ms, sum over ranks of local_units).  Single process: identity."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(local_ms), float(local_units)
    if device is None:
        device = torch.device("cuda", torch.cuda.current_device()) if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([local_ms], dtype=torch.float64, device=device)
    u = torch.tensor([local_units], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def whole_job_throughput(local_ms: float, local_units: float, device=None):
    """units/s of the whole job: all ranks' units over the slowest rank's time."""
    ms, units = aggregate(local_ms, local_units, device)
    return units / (ms * 1e-3), ms
