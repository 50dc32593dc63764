"""Multi-process plumbing for bench.py: one process per GPU, intrinsic points sharded with no data-path collective
("embarrassingly parallel").  torch.distributed is used only for the barrier and for the max-over-ranks
of the timed region; the backend is NCCL on GPUs and gloo in the CPU tests."""
from __future__ import annotations

import os
from typing import List, Tuple


def env_world() -> Tuple[int, int, int]:
    """(rank, world_size, local_rank) from the torchrun environment (1 process if unset)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def shard_points(n_points: int, rank: int, world: int) -> List[int]:
    """Weak scaling: every rank owns n_points intrinsic points of its own; global ids rank*n_points + i."""
    return [rank * n_points + i for i in range(n_points)]


def init(backend: str, device=None) -> None:
    import torch.distributed as dist
    if not dist.is_initialized():
        kw = {"device_id": device} if (device is not None and backend == "nccl") else {}
        dist.init_process_group(backend, **kw)


def barrier() -> None:
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def max_over_ranks(value: float, device="cpu") -> float:
    """Max of a per-rank scalar (the timed region's milliseconds)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(units_per_rank: int, ms_local: float, device="cpu") -> Tuple[float, float]:
    """(whole-job units/s, max ms) = (world * units_per_rank) / max-over-ranks time."""
    import torch.distributed as dist
    world = dist.get_world_size() if (dist.is_available() and dist.is_initialized()) else 1
    ms = max_over_ranks(ms_local, device)
    return world * units_per_rank / (ms * 1e-3), ms
