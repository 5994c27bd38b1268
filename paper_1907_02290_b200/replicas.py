"""Multi-GPU = independent replicas: the path is fixed to one GPU by the
north_star, so `bench.py --gpus N` runs N copies, one process per GPU, with no data-path collective.
This module holds the only cross-rank logic: the barrier and the max-over-ranks / sum-over-ranks
reduction of the timing, over torch.distributed (nccl on GPUs, gloo in the CPU tests)."""
from __future__ import annotations

import os


def init_from_env(backend: str | None = None):
    """Returns (rank, world_size, local_rank); initialises torch.distributed when WORLD_SIZE > 1."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch
        import torch.distributed as dist
        if not dist.is_initialized():
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29511")
            if backend is None:
                backend = "nccl" if torch.cuda.is_available() else "gloo"
            if backend == "nccl":
                torch.cuda.set_device(local)
            dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, world, local


def barrier(world: int) -> None:
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


def reduce_timing(units_local: float, ms_local: float, world: int, device=None):
    """Whole-job figures: (sum of units over ranks, max of elapsed ms over ranks)."""
    if world == 1:
        return float(units_local), float(ms_local)
    import torch
    import torch.distributed as dist
    if device is None:
        device = torch.device("cuda", torch.cuda.current_device()) if dist.get_backend() == "nccl" else torch.device("cpu")
    u = torch.tensor([float(units_local)], dtype=torch.float64, device=device)
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(u.item()), float(t.item())
