"""Multi-GPU plumbing: replicas only.

north_star runs the whole path on one GPU; with N ranks every rank tracks an independent bunch (its own
contiguous range of the counter-based particle stream) and there is NO data-path collective.  The only
exchanges are the barrier around the timed region and the max-over-ranks / sum-over-ranks of the
timing scalars, done with torch.distributed (NCCL on the GPU box, gloo in the CPU tests).
"""
from __future__ import annotations

import os
from typing import Optional, Tuple


def env_rank() -> Tuple[int, int, int]:
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) when absent."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def shard_start(rank: int, n_per_rank: int) -> int:
    """First particle index of rank's bunch in the counter-based stream (weak scaling: every rank
    gets n_per_rank fresh particles, ranks never overlap)."""
    if rank < 0 or n_per_rank < 0:
        raise ValueError("rank and n_per_rank must be >= 0")
    return rank * n_per_rank


def init_process_group(backend: Optional[str] = None):
    """Initialise torch.distributed from the environment when WORLD_SIZE > 1.  Returns world size."""
    rank, local_rank, world = env_rank()
    if world <= 1:
        return 1
    import torch
    import torch.distributed as dist
    if not dist.is_initialized():
        if backend is None:
            backend = "nccl" if torch.cuda.is_available() else "gloo"
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29531")
        if backend == "nccl":
            torch.cuda.set_device(local_rank)
            dist.init_process_group(backend, rank=rank, world_size=world,
                                    device_id=torch.device("cuda", local_rank))
        else:
            dist.init_process_group(backend, rank=rank, world_size=world)
    return world


def barrier() -> None:
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def aggregate(elapsed_ms: float, units: float, device=None) -> Tuple[float, float]:
    """(max over ranks of elapsed_ms, sum over ranks of units).  Identity without a process group."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(elapsed_ms), float(units)
    if device is None:
        device = torch.device("cuda", torch.cuda.current_device()) if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([elapsed_ms], dtype=torch.float64, device=device)
    u = torch.tensor([units], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())
