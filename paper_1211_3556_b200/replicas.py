"""Multi-GPU host logic: "replicas only".

The hot path does not shard (BASELINE.json north_star: one GPU, no sharding, no collectives), so
`bench.py --gpus N` runs N independent replicas, one process per GPU.  The only cross-rank steps are
the timing barrier and the reduction of the per-rank device times (max) and unit counts (sum); they
live here so that the CPU `gloo` tests (world_size 2) can cover them.
"""
from __future__ import annotations

import os
from typing import Tuple


def env_world() -> Tuple[int, int, int]:
    """(rank, local_rank, world_size) from the torchrun environment (1 process: 0, 0, 1)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: str):
    """Initialise torch.distributed from the torchrun env if WORLD_SIZE > 1; returns the module or None."""
    rank, _, world = env_world()
    if world <= 1:
        return None
    import torch.distributed as dist
    if not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29500")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return dist


def barrier(dist) -> None:
    if dist is not None:
        dist.barrier()


def aggregate(dist, elapsed_ms: float, units: float, device=None) -> Tuple[float, float]:
    """Whole-job numbers of N replicas: (max over ranks of the device time, sum over ranks of units)."""
    if dist is None:
        return float(elapsed_ms), float(units)
    import torch
    t = torch.tensor([float(elapsed_ms)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def throughput(total_units: float, max_elapsed_ms: float) -> float:
    return total_units / (max_elapsed_ms * 1e-3)
