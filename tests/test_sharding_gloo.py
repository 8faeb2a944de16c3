"""world_size-2 gloo test of the N>1 host path (column shards, max-over-ranks timing, summed units) and,
on the CPU oracle, of the property the sharding relies on: filtering column shards separately equals
filtering the whole block (Algorithm 3 is column-separable)."""
import os
import sys

import numpy as np
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out_dir):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from paper_2503_22652_b200.sharding import column_shard, reduce_job
    from oracle import chfsi_oracle as orc
    import workloads
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    prob = workloads.config1_dense_standard(m=120, n_wanted=8, block=11, degree=7, seed=5)
    A, B, Dinv = orc.operators_from_workload(prob)
    ritz, X, AX, BX = orc.rayleigh_ritz(A.apply, B.apply, prob["X0"])
    G = orc.residual_block(AX, BX, ritz)
    lo, hi = column_shard(11, rank, world)
    b = (prob["lam_min"], prob["lam_T"], prob["lam_max"])
    Y = orc.filter_rchfsi(A.apply, Dinv.apply, X[:, lo:hi], ritz[lo:hi], G[:, lo:hi], 7, *b)
    np.save(os.path.join(out_dir, "shard%d.npy" % rank), Y)
    ms, units = reduce_job(10.0 + 5.0 * rank, (hi - lo) * 120 * 7)
    np.save(os.path.join(out_dir, "red%d.npy" % rank), np.array([ms, units, lo, hi]))
    dist.barrier()
    dist.destroy_process_group()


def test_column_shards_cover_and_reduce_over_gloo(tmp_path):
    from paper_2503_22652_b200.sharding import column_shard
    for n in (0, 1, 7, 240, 1201):
        for w in (1, 2, 3, 8):
            spans = [column_shard(n, r, w) for r in range(w)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            assert all(spans[i][1] == spans[i + 1][0] for i in range(w - 1))
            assert max(h - l for l, h in spans) - min(h - l for l, h in spans) <= 1
    port = 29500 + os.getpid() % 2000
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    red = [np.load(tmp_path / ("red%d.npy" % r)) for r in range(2)]
    for r in red:
        assert r[0] == 15.0                      # max over ranks
        assert r[1] == 11 * 120 * 7              # summed units
    # column-separability on the oracle: shards stitched together equal the whole-block filter
    sys.path.insert(0, ROOT)
    from oracle import chfsi_oracle as orc
    import workloads
    prob = workloads.config1_dense_standard(m=120, n_wanted=8, block=11, degree=7, seed=5)
    A, B, Dinv = orc.operators_from_workload(prob)
    ritz, X, AX, BX = orc.rayleigh_ritz(A.apply, B.apply, prob["X0"])
    G = orc.residual_block(AX, BX, ritz)
    Y = orc.filter_rchfsi(A.apply, Dinv.apply, X, ritz, G, 7, prob["lam_min"], prob["lam_T"], prob["lam_max"])
    stitched = np.concatenate([np.load(tmp_path / ("shard%d.npy" % r)) for r in range(2)], axis=1)
    np.testing.assert_allclose(stitched, Y, rtol=1e-12, atol=1e-14)
