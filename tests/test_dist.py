"""Multi-GPU host logic on CPU: world size 2, gloo backend.

The N > 1 path has no data-path collective but the final sum of the dose grids; what can be wrong on the host side is
the rank keys (streams must be disjoint), the reduction and the max-over-ranks timing.  The per-rank "dose" here is the
CPU oracle on a small case, so the test also checks the statistical claim the sharding rests on: the mean of the ranks'
N-history estimates is an N x world estimate of the same dose."""
import os
import socket

import numpy as np
import torch
import torch.distributed as td
import torch.multiprocessing as mp

from paper_2307_01416_b200 import dist, workloads as wl


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out_dir):
    os.environ.update({"RANK": str(rank), "LOCAL_RANK": str(rank), "WORLD_SIZE": str(world),
                       "MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port)})
    r, lr, w = dist.init(backend="gloo")
    assert (r, lr, w) == (rank, rank, world) and td.is_initialized()
    from oracle import vpmc_oracle as orc
    from tests.helpers import oracle_problem
    case = wl.small_water(n=(10, 10, 30), energy=70.0, sigma=2.0)
    pb = oracle_problem(case)
    N, seed = 4000, 5
    d, _ = orc.dose(pb, N, dist.rank_seed(seed, rank))
    dose = torch.from_numpy(d.copy())
    own = dose.clone()
    dist.barrier(w)
    dist.combine_dose(dose, w)
    t = dist.max_over_ranks(1.0 + rank, w)
    np.save(os.path.join(out_dir, "rank%d.npy" % rank), np.stack([own.numpy(), dose.numpy()]))
    assert t == float(world)
    td.destroy_process_group()


def test_rank_seeds_are_disjoint_keys():
    seeds = {dist.rank_seed(7, r) for r in range(8)}
    assert len(seeds) == 8 and dist.rank_seed(7, 0) == 7
    assert all((s & 0xFFFFFFFF) == 7 for s in seeds)          # the rank enters the high word of the Philox key
    assert dist.rank_seed((3 << 32) | 9, 2) == ((5 << 32) | 9)


def test_single_process_helpers_are_no_ops():
    d = torch.ones(4)
    assert dist.combine_dose(d, 1) is d and float(d.sum()) == 4.0
    assert dist.max_over_ranks(2.5, 1) == 2.5
    dist.barrier(1)


def test_two_ranks_gloo_combine(tmp_path):
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    a = np.load(tmp_path / "rank0.npy")
    b = np.load(tmp_path / "rank1.npy")
    assert np.array_equal(a[1], b[1])                          # both ranks hold the same combined grid
    assert np.allclose(a[1], 0.5 * (a[0] + b[0]), rtol=1e-12, atol=0)
    assert np.abs(a[0] - b[0]).max() > 0                       # different keys -> different samples
    # the two estimates agree statistically: integral dose within 2 %
    assert abs(a[0].sum() - b[0].sum()) < 0.02 * a[0].sum()
