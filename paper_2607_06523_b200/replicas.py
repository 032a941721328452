"""Rank plumbing for `bench.py --gpus N`: the path is "replicas only" -- every rank runs the whole
hot path on its own GPU and its own cache; no data-path collective exists. Only the timing is reduced across ranks.
Works with any torch.distributed backend (NCCL on the GPU box, gloo in the CPU tests); world size 1 needs no process group."""
from __future__ import annotations

import os
from typing import Optional, Tuple

import torch


def env_rank() -> Tuple[int, int, int]:
    """(rank, world_size, local_rank) from the torchrun environment; (0, 1, 0) when launched plainly."""
    return int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0"))


def init(backend: str, device: Optional[torch.device] = None) -> bool:
    """Join the process group if WORLD_SIZE > 1. Returns True if a group was created."""
    _, world, _ = env_rank()
    if world <= 1:
        return False
    import torch.distributed as dist
    if backend == "nccl":
        dist.init_process_group("nccl", device_id=device)
    else:
        dist.init_process_group(backend)
    return True


def barrier() -> None:
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def max_over_ranks(value: float, device="cpu") -> float:
    """Slowest rank's time: every multi-GPU number is the max over ranks of a device-timed duration."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(units_per_rank: float, ms_per_step_max: float, world: int) -> float:
    """Whole-job throughput of `world` replicas that each process `units_per_rank` per step (weak scaling)."""
    return units_per_rank * world / (ms_per_step_max * 1e-3)
