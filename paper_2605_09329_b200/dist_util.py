"""Multi-process plumbing for bench.py and the multi-GPU paths: one process per GPU, torch.distributed (NCCL on GPUs,
gloo in the CPU tests).  Only rendezvous, barriers and the max-over-ranks / sum-over-ranks reductions of scalars
that the timing contract needs -- no tensor of the method travels through here (the step runs
as independent replicas, or vocabulary shards with their own tiny collectives in sharded.py)."""
from __future__ import annotations

import os

import torch
import torch.distributed as dist


def env_ranks():
    """(rank, world_size, local_rank) from the torchrun environment; (0, 1, 0) without it."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def init(backend: str, device: torch.device | None = None):
    """Joins the process group described by RANK / WORLD_SIZE / MASTER_ADDR / MASTER_PORT (no-op for one process)."""
    rank, world, _ = env_ranks()
    if world > 1 and not dist.is_initialized():
        kw = {}
        if backend == "nccl" and device is not None:
            kw["device_id"] = device
        dist.init_process_group(backend, **kw)
    return rank, world


def barrier(device: torch.device | None = None):
    """Process barrier, then (on a GPU) a device synchronise: both sides of every timed region."""
    if dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()
    if device is not None and device.type == "cuda":
        torch.cuda.synchronize(device)


def _reduce_scalar(x: float, op, device: torch.device | None):
    if not (dist.is_initialized() and dist.get_world_size() > 1):
        return float(x)
    dev = device if (device is not None and dist.get_backend() == "nccl") else torch.device("cpu")
    t = torch.tensor([x], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=op)
    return float(t.item())


def max_over_ranks(x: float, device: torch.device | None = None) -> float:
    return _reduce_scalar(x, dist.ReduceOp.MAX, device)


def sum_over_ranks(x: float, device: torch.device | None = None) -> float:
    return _reduce_scalar(x, dist.ReduceOp.SUM, device)


def job_throughput(units_this_rank: float, seconds_this_rank: float, device: torch.device | None = None) -> float:
    """Whole-job throughput: the units ALL ranks processed divided by the slowest rank's time."""
    total = sum_over_ranks(units_this_rank, device)
    worst = max_over_ranks(seconds_this_rank, device)
    return total / worst
