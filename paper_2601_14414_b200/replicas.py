"""Multi-GPU plumbing: the path shards only by INSTANCE (replicas only).

Every MPC instance has its own A_k, B_k, x0, its own residual c, alpha and accept/restart decision
(Algorithm 1, runs per instance), so ranks own disjoint instance ranges and no
data-path collective exists.  The only communication is the harness's: a barrier before/after the
timed region and a MAX over ranks of the device time.  Works with any torch.distributed backend
(nccl on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

import os


def env_rank():
    """(rank, local_rank, world_size) from the torchrun environment (1 process = 1 GPU)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def weak_instance_range(per_rank_batch: int, rank: int):
    """Weak scaling: rank r owns instances [r*B, (r+1)*B) of the global seeded instance stream."""
    return rank * per_rank_batch, (rank + 1) * per_rank_batch


def strong_instance_range(total: int, rank: int, world: int):
    """Strong scaling: contiguous, balanced split of `total` instances (first `total % world` get one more)."""
    base, rem = divmod(total, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def init(backend: str | None = None):
    """Initialise torch.distributed from the torchrun environment if WORLD_SIZE > 1."""
    import torch.distributed as dist
    rank, local_rank, world = env_rank()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29500")
        if backend is None:
            import torch
            backend = "nccl" if torch.cuda.is_available() else "gloo"
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def barrier(device=None):
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        if device is not None and dist.get_backend() == "nccl":
            dist.barrier(device_ids=[device])
        else:
            dist.barrier()


def max_over_ranks(value: float, device=None) -> float:
    """MAX over ranks of a per-rank scalar (the per-rank device time of the timed region)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    dev = "cpu" if dist.get_backend() != "nccl" else f"cuda:{device or 0}"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device=None) -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    dev = "cpu" if dist.get_backend() != "nccl" else f"cuda:{device or 0}"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())
