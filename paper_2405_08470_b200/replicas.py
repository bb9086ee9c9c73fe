"""Multi-GPU plumbing for bench.py: N independent replicas, one process per GPU.

The hot path has no exchange step (BASELINE.json north_star: one GPU, no sharding, no
collectives), so `--gpus N` runs N replicas of the workload and the only
communication is the timing protocol: a barrier on both sides of the timed region and a MAX
over ranks of the device time.  `torch.distributed` (nccl on GPUs, gloo in the CPU tests) is
used for exactly that.
"""
from __future__ import annotations

import os
from typing import Tuple

import torch
import torch.distributed as dist


def env_ranks() -> Tuple[int, int, int]:
    """(rank, world_size, local_rank) from the torchrun environment (1 process: 0, 1, 0)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def init(backend: str, device=None) -> Tuple[int, int, int]:
    rank, world, local = env_ranks()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29533")
        if backend == "nccl":
            dist.init_process_group("nccl", device_id=device)
        else:
            dist.init_process_group(backend)
    return rank, world, local


def barrier(device=None) -> None:
    if dist.is_initialized():
        dist.barrier()
    if device is not None and torch.device(device).type == "cuda":
        torch.cuda.synchronize(device)


def max_over_ranks(x: float, device=None) -> float:
    if not dist.is_initialized():
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(units_per_rank: float, ms_local: float, device=None) -> Tuple[float, float]:
    """Whole-job throughput of `world` replicas: every rank processed `units_per_rank` units, the job
    took the slowest rank's time.  Returns (units per second over all ranks, max ms)."""
    world = dist.get_world_size() if dist.is_initialized() else 1
    ms = max_over_ranks(ms_local, device)
    return world * units_per_rank / (ms * 1e-3), ms


def finalize() -> None:
    if dist.is_initialized():
        dist.destroy_process_group()
