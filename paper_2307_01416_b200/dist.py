"""Multi-GPU plumbing: histories are independent and streams are keyed by (seed, history id), so
the dose path shards by giving every rank its own Philox key and the same plan; the only exchange is one
all-reduce of the dose grid.  One process per GPU, torch.distributed (NCCL on GPUs, gloo in the CPU tests)."""
from __future__ import annotations

import os


def env_world():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def init(backend: str | None = None):
    """Initialise torch.distributed from the torchrun environment; returns (rank, local_rank, world)."""
    rank, local_rank, world = env_world()
    if world > 1:
        import torch
        import torch.distributed as dist
        if not dist.is_initialized():
            if backend is None:
                backend = "nccl" if torch.cuda.is_available() else "gloo"
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def rank_seed(seed: int, rank: int) -> int:
    """Philox key of a rank: disjoint streams per rank (the key's high word carries the rank)."""
    return (int(seed) & 0xFFFFFFFF) | ((int(rank) + ((int(seed) >> 32) & 0xFFFFFFFF)) & 0xFFFFFFFF) << 32


def combine_dose(dose, world: int):
    """Mean of the ranks' dose grids: each rank ran N histories of the same plan, the result is the N*world
    estimate.  In place; one all-reduce, no other data-path collective."""
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(dose, op=dist.ReduceOp.SUM)
        dose /= world
    return dose


def barrier(world: int):
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


def max_over_ranks(value: float, world: int, device="cpu") -> float:
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
