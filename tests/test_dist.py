"""Multi-GPU host logic on CPU: world size 2, gloo backend.

The N > 1 path has no exchange inside the transport: rank r transports shard r of every spot's history-id range of the SAME
run, one all-reduce(SUM) gives the dose; influence matrices are sharded by rows (spots) and concatenated after an all-gather
of the per-rank nnz.  What can be wrong on the host side is the integer shard rule, the reduction, the row_ptr offsets and
the max-over-ranks timing.  The per-rank engine here is a stand-in with the library's interface (set_shard + dose) backed by
the CPU oracle on the shard's ids, driven through dist.sharded_dose -- the same function bench.py calls under torchrun -- so
the test also checks the claim the sharding rests on: the summed shards ARE the one-process run of the same ids."""
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


class OracleEngine:
    """The binding.Engine calls dist.py uses, computed by the oracle (test stand-in; there is no CPU product path)."""

    def __init__(self, case):
        from oracle import vpmc_oracle as orc
        from tests.helpers import oracle_problem
        self.orc, self.pb = orc, oracle_problem(case)
        self.index, self.count = 0, 1

    def set_shard(self, index, count):
        self.index, self.count = index, count

    def dose(self, n_total, seed, out=None, stream=None):
        orc, pb = self.orc, self.pb
        cnt = orc.spot_counts(pb, n_total).astype(np.int64)
        start = np.concatenate([[0], np.cumsum(cnt)])
        e = np.zeros(pb.nvox)
        for g in range(pb.n_spots):               # shard of every spot's id range, the library's integer rule
            lo, hi = dist.shard_range(int(start[g]), int(start[g + 1]), self.index, self.count)
            if hi > lo:
                orc.dose_edep(pb, n_total, seed, hid_begin=lo, hid_end=hi, edep=e)
        d = torch.from_numpy(orc.dose_from_edep(pb, e, pb.total_weight / float(n_total)))
        if out is not None:
            out.copy_(d)
            return out
        return d

    def influence_rows(self, hps, thr, seed):
        lo, hi = dist.shard_range(0, self.pb.n_spots, self.index, self.count)
        rp, col, val = self.orc.influence_csr(self.pb, hps, thr, seed, spots=range(lo, hi))
        full = np.zeros(self.pb.n_spots + 1, dtype=np.int64)
        full[lo:hi + 1] = rp
        full[hi + 1:] = rp[-1]
        return full, col, val


def _case():
    return wl.small_water(n=(10, 10, 30), energy=70.0, sigma=2.0, n_spots=5)


def _worker(rank, world, port, out_dir):
    os.environ.update({"RANK": str(rank), "LOCAL_RANK": str(rank), "WORLD_SIZE": str(world),
                       "MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port)})
    r, lr, w = dist.init(backend="gloo")
    assert (r, lr, w) == (rank, rank, world) and td.is_initialized()
    eng = OracleEngine(_case())
    N, seed = 3001, 5                              # an odd count: the shards of a spot differ in size
    eng.set_shard(rank, world)
    own = eng.dose(N, seed).clone()
    dist.barrier(w)
    full = dist.sharded_dose(eng, N, seed, rank, world)
    t = dist.max_over_ranks(1.0 + rank, w)
    # influence rows
    eng.set_shard(rank, world)
    rp, col, val = eng.influence_rows(300, 1e-3, seed)
    off, total, nnz = dist.csr_offsets(col.size, rank, world)
    grp = dist.global_row_ptr(torch.from_numpy(rp), eng.pb.n_spots, rank, world)
    np.savez(os.path.join(out_dir, "rank%d.npz" % rank), own=own.numpy(), full=full.numpy(), rp=rp, col=col, val=val,
             off=off, total=total, nnz=np.asarray(nnz), grp=grp.numpy())
    assert t == float(world)
    td.destroy_process_group()


def test_shard_ranges_partition_every_range():
    for lo, hi in ((0, 0), (5, 6), (10, 1011), (7, 7 + 2 ** 40 + 3)):
        for count in (1, 2, 3, 8):
            parts = [dist.shard_range(lo, hi, k, count) for k in range(count)]
            assert parts[0][0] == lo and parts[-1][1] == hi
            assert all(parts[k][1] == parts[k + 1][0] for k in range(count - 1))
            sizes = [b - a for a, b in parts]
            assert max(sizes) - min(sizes) <= 1


def test_single_process_helpers_are_no_ops():
    d = torch.ones(4)
    assert dist.combine_dose(d, 1) is d and float(d.sum()) == 4.0
    assert dist.max_over_ranks(2.5, 1) == 2.5
    assert dist.csr_offsets(7, 0, 1) == (0, 7, [7])
    rp = torch.tensor([0, 2, 5], dtype=torch.int64)
    assert torch.equal(dist.global_row_ptr(rp, 2, 0, 1), rp)
    dist.barrier(1)


def test_two_ranks_gloo_sum_of_shards_is_the_full_run(tmp_path):
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    a = np.load(tmp_path / "rank0.npz")
    b = np.load(tmp_path / "rank1.npz")
    from oracle import vpmc_oracle as orc
    from tests.helpers import oracle_problem
    pb = oracle_problem(_case())
    ref, _ = orc.dose(pb, 3001, 5)
    # dose: both ranks hold the same combined grid = the sum of the shards = the one-process run of the same ids
    assert np.array_equal(a["full"], b["full"])
    assert np.allclose(a["full"], a["own"] + b["own"], rtol=1e-14, atol=0)
    assert np.allclose(a["full"], ref, rtol=1e-12, atol=1e-300)
    assert a["own"].sum() > 0 and b["own"].sum() > 0 and np.abs(a["own"] - b["own"]).max() > 0
    assert abs(a["own"].sum() - b["own"].sum()) < 0.1 * a["own"].sum()      # every shard holds the same mix of spots
    # influence: concatenated pieces + offsets from the all-gathered nnz = the one-process CSR
    rp, col, val = orc.influence_csr(pb, 300, 1e-3, 5)
    assert int(a["off"]) == 0 and int(b["off"]) == a["col"].size and int(a["total"]) == int(b["total"]) == col.size
    assert list(a["nnz"]) == list(b["nnz"]) == [a["col"].size, b["col"].size]
    assert np.array_equal(a["grp"], rp) and np.array_equal(b["grp"], rp)
    assert np.array_equal(np.concatenate([a["col"], b["col"]]), col)
    assert np.array_equal(np.concatenate([a["val"], b["val"]]), val)
