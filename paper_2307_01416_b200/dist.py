"""Multi-GPU plumbing.  Histories are independent and random streams are keyed by (seed, history id), so
the path shards with no exchange inside the transport:

* dose: every rank transports shard `rank` of `world` of the SAME N-history run (vpmc_set_shard: the r-th part of every
  spot's id range, so all ranks hold the same mix of spots), then ONE all-reduce(SUM) of the dose grid.  The result is the
  dose of the one-GPU run of the same ids, up to the order of floating-point additions -- so the oracle checks it too;
* influence matrices: the (scenario, spot) columns are sharded by spot; each rank's CSR has its own rows filled and the others
  empty; the pieces are concatenated after an all-gather of the per-rank nnz (row_ptr offsets).

One process per GPU, torch.distributed (NCCL on GPUs, gloo in the CPU tests).  Nothing waits on another rank inside a kernel.
"""
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


def shard_range(lo: int, hi: int, index: int, count: int):
    """Part `index` of `count` of the integer range [lo, hi): the library's rule (include/vpmc.h, vpmc_set_shard)."""
    n = int(hi) - int(lo)
    return int(lo) + n * int(index) // int(count), int(lo) + n * (int(index) + 1) // int(count)


def sharded_dose(engine, n_total: int, seed: int, rank: int, world: int, out=None, stream=None):
    """This rank's share of the n_total-history dose, summed over the ranks: on return every rank holds the full dose."""
    engine.set_shard(rank, world)
    d = engine.dose(n_total, seed, out=out, stream=stream)
    return combine_dose(d, world)


def combine_dose(dose, world: int):
    """Sum of the ranks' partial dose grids (each already carries the scale W / N of the full run).  In place; the one
    data-path collective of the dose path."""
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(dose, op=dist.ReduceOp.SUM)
    return dose


def csr_offsets(nnz_local: int, rank: int, world: int, device="cpu"):
    """All-gather of the per-rank nnz: (offset of this rank's entries in the concatenated arrays, total nnz, list of nnz)."""
    if world <= 1:
        return 0, int(nnz_local), [int(nnz_local)]
    import torch
    import torch.distributed as dist
    mine = torch.tensor([int(nnz_local)], dtype=torch.int64, device=device)
    parts = [torch.zeros(1, dtype=torch.int64, device=device) for _ in range(world)]
    dist.all_gather(parts, mine)
    nnz = [int(p.item()) for p in parts]
    return sum(nnz[:rank]), sum(nnz), nnz


def global_row_ptr(row_ptr_local, n_rows: int, rank: int, world: int):
    """row_ptr of the concatenated matrix from a rank's row_ptr (rows of other ranks empty): own rows are shifted by the
    rank's offset, rows owned by rank r' start at the offset of r'.  Every rank gets the same array."""
    import torch
    rp = row_ptr_local.clone()
    if world <= 1:
        return rp
    import torch.distributed as dist
    nnz_local = int(rp[-1].item())
    off, total, nnz = csr_offsets(nnz_local, rank, world, device=rp.device)
    lo, hi = shard_range(0, n_rows, rank, world)
    own = torch.zeros_like(rp)
    own[lo:hi] = rp[lo:hi] + off                     # entries of this rank's rows; every other row is filled in by its owner
    dist.all_reduce(own, op=dist.ReduceOp.SUM)
    own[n_rows] = total
    return own


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
