"""Multi-GPU host logic.  The path shards with NO exchange step: every (micro-step, layer)
instance is independent, so N GPUs run N independent shards (each rank its
own step of the same shape, seeded by its rank) and the only cross-rank traffic is the timing
reduction below.  Weak scaling: per-GPU work is fixed.
"""
from __future__ import annotations

import os
from typing import Tuple

import torch
import torch.distributed as dist


def env_rank() -> Tuple[int, int, int]:
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) without it."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def shard_seed(base_seed: int, rank: int) -> int:
    """Seed of the trace a rank generates: rank r handles its own RL step (data-parallel shard)."""
    return base_seed + 7919 * rank


def init(backend: str, device=None) -> bool:
    """Join the process group when launched under torchrun with world_size > 1."""
    _, _, world = env_rank()
    if world <= 1:
        return False
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    kw = {}
    if device is not None and backend == "nccl":
        kw["device_id"] = device
    dist.init_process_group(backend=backend, **kw)
    return True


def barrier(device=None) -> None:
    if dist.is_available() and dist.is_initialized():
        if device is not None and torch.device(device).type == "cuda":
            dist.barrier(device_ids=[torch.device(device).index])
        else:
            dist.barrier()


def aggregate(elapsed_ms: float, units: float, device="cpu") -> Tuple[float, float]:
    """(max over ranks of elapsed_ms, sum over ranks of units): whole-job throughput is
    units_total / max_time -- never an average of per-rank rates."""
    if not (dist.is_available() and dist.is_initialized()):
        return float(elapsed_ms), float(units)
    t = torch.tensor([float(elapsed_ms)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())
