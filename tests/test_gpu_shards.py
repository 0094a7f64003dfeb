"""SURVEY.md 8(e) on one device: two handles, each computing one shard (vpmc_set_shard), reproduce the full run -- dose as
the sum of the shards (same history ids, so equal up to the order of the fp32 additions; integer tallies exactly), influence
matrices as the concatenation of the shards' rows with row_ptr offsets from the shards' nnz."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

COUNT_FIELDS = ("n_stopped_ct", "n_stopped_rs", "n_stopped_brass", "n_nuclear", "n_escaped", "n_steps_ct", "n_steps_dev", "n_steps_slab")


def _case():
    from paper_2307_01416_b200 import workloads as wl
    return wl.small_water(n=(24, 24, 40), energy=90.0, sigma=3.0, with_aperture=True, opening_radius=4.0, n_spots=7, rs_wet=10.0)


@pytest.mark.parametrize("count", [2, 3])
def test_sum_of_dose_shards_is_the_full_run(count):
    from paper_2307_01416_b200 import binding, dist
    from oracle import vpmc_oracle as orc
    from tests.helpers import oracle_problem
    w = _case()
    N, seed = 200_003, 9
    full_eng = binding.Engine(w)
    full = full_eng.dose(N, seed).clone()
    tf = full_eng.tallies().as_dict()
    acc = torch.zeros_like(full)
    ts = {k: 0 for k in COUNT_FIELDS}
    inc = 0.0
    for k in range(count):
        e = binding.Engine(w)
        e.set_shard(k, count)
        acc += e.dose(N, seed)                               # the shard's own partial grid (already scaled by W / N)
        t = e.tallies().as_dict()
        for f in COUNT_FIELDS:
            ts[f] += t[f]
        inc += t["incident"]
        e.close()
    for f in COUNT_FIELDS:
        assert ts[f] == tf[f], f                             # the shards transport exactly the ids of the full run
    assert abs(inc - tf["incident"]) <= 1e-9 * tf["incident"]
    mx = float(full.max())
    assert mx > 0 and float((acc - full).abs().max()) <= 2e-6 * mx
    # and the full run is the oracle's (so the sharded result is checked against the oracle too)
    d_orc, _ = orc.dose(oracle_problem(w), N, seed)
    assert np.abs(acc.cpu().numpy().astype(np.float64) - d_orc).max() <= 1e-3 * d_orc.max()
    full_eng.close()


def test_concatenated_influence_shards_are_the_full_matrix():
    from paper_2307_01416_b200 import binding, dist
    w = _case()
    sc = [binding.scenario(), binding.scenario((0.0, 2.0, 0.0), 1.035)]
    hps, thr, seed = 4000, 1e-4, 4
    eng = binding.Engine(w)
    ref = eng.influence(sc, hps, thr, seed)
    count = 3
    parts = []
    for k in range(count):
        e = binding.Engine(w)
        e.set_shard(k, count)
        parts.append(e.influence(sc, hps, thr, seed))
        e.close()
    ns = eng.n_spots
    for s in range(len(sc)):
        rp_ref, col_ref, val_ref = ref[s]
        nnz = [int(parts[k][s][1].numel()) for k in range(count)]
        offs = np.concatenate([[0], np.cumsum(nnz)])
        rp = torch.zeros(ns + 1, dtype=torch.int64, device="cuda")
        for k in range(count):
            lo, hi = dist.shard_range(0, ns, k, count)
            rpk = parts[k][s][0]
            assert int(rpk[lo]) == 0 and int(rpk[hi]) == nnz[k] and bool((rpk[hi:] == nnz[k]).all())     # other rows are empty
            rp[lo:hi] = rpk[lo:hi] + int(offs[k])
        rp[ns] = int(offs[-1])
        col = torch.cat([parts[k][s][1] for k in range(count)])
        val = torch.cat([parts[k][s][2] for k in range(count)])
        # same histories per column; only the order of the fp32 additions differs, which can move an entry across the
        # threshold when it sits within rounding of it: compare structure exactly where the values are clear of it
        if torch.equal(rp, rp_ref) and torch.equal(col, col_ref):
            assert float((val - val_ref).abs().max()) <= 1e-5 * float(val_ref.max())
        else:
            a = torch.sparse_csr_tensor(rp, col.long(), val, size=(ns, eng.nvox)).to_dense()
            b = torch.sparse_csr_tensor(rp_ref, col_ref.long(), val_ref, size=(ns, eng.nvox)).to_dense()
            differ = (a != 0) != (b != 0)
            thr_row = thr * b.max(dim=1, keepdim=True).values
            assert int(differ.sum()) <= 3 and bool((torch.maximum(a, b)[differ] <= 1.001 * thr_row.expand_as(a)[differ]).all())
            both = (a != 0) & (b != 0)
            assert float((a - b)[both].abs().max()) <= 1e-5 * float(b.max())
    eng.close()
