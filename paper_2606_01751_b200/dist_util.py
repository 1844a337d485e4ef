"""Multi-process plumbing for bench.py: one process per GPU, no data-path collective.

The Sparse-KV recomputation step has no exchange step: ranks run independent
replicas of the workload. The only cross-rank traffic is the timing reduction (max over ranks) and the
start/stop barriers; both work on the nccl (GPU) and gloo (CPU tests) backends.
"""
from __future__ import annotations

import os

import torch
import torch.distributed as dist


def env_rank():
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def init(backend: str, device=None):
    rank, world, _ = env_rank()
    if world > 1 and not dist.is_initialized():
        kw = {"device_id": device} if (backend == "nccl" and device is not None) else {}
        dist.init_process_group(backend, **kw)
    return rank, world


def barrier():
    if dist.is_initialized():
        dist.barrier()


def max_over_ranks(x: float, device="cpu") -> float:
    """Slowest rank's time: the job's time."""
    if not dist.is_initialized():
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(units_per_rank: float, ms: float, world: int) -> float:
    """Whole-job units/s: every rank processed units_per_rank in (max over ranks) ms."""
    return world * units_per_rank / (ms * 1e-3)
