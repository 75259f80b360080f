"""Multi-GPU plumbing: replicas only.

The demons iteration shards by z-slabs in principle, but BASELINE.json's north_star fixes one
GPU per registration, so N GPUs run N independent registrations (one process per GPU, no
data-path collective).  torch.distributed is used only for the barrier
and for the max-over-ranks of the timing; `value` = units all ranks processed / that time.
"""
from __future__ import annotations

import os


def env_world():
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) when absent."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: str):
    """Initialise the process group when launched under torchrun with WORLD_SIZE > 1."""
    import torch.distributed as dist
    rank, _, world = env_world()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, world


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def _reduce(x: float, op_name: str, device="cpu") -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=getattr(dist.ReduceOp, op_name))
    return float(t.item())


def max_over_ranks(x: float, device="cpu") -> float:
    return _reduce(x, "MAX", device)


def sum_over_ranks(x: float, device="cpu") -> float:
    return _reduce(x, "SUM", device)


def replica_seed(base_seed: int, rank: int) -> int:
    """Every replica registers its own phantom pair."""
    return int(base_seed) + 1000 * int(rank)


def aggregate(units_local: float, seconds_local: float, device="cpu"):
    """Whole-job throughput: units of all ranks / slowest rank's time."""
    seconds = max_over_ranks(seconds_local, device)
    units = sum_over_ranks(units_local, device)
    return {"units": units, "seconds": seconds, "value": units / seconds if seconds > 0 else 0.0}
