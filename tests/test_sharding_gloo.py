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


# ------------------------------------------------------------------------------------------------ row slabs
def _row_worker(rank, world, port, out_dir):
    """One rank of the row-sharded filter on the CPU: the partition and the neighbour exchange are the product's
    (sharding.slab_partition_fe, neighbor_exchange over gloo); the per-step arithmetic is the ORACLE's Algorithm 3
    restricted to the slab, with the interface rule of rchfsi_interface_pack / _apply restated in numpy:
    rows on the plane between two slabs get  base + (delta_own + delta_nbr),  delta = a T_local."""
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    from paper_2503_22652_b200.sharding import slab_partition_fe, neighbor_exchange
    from oracle import chfsi_oracle as orc
    import workloads
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    prob, X, ritz, G, p, b = _row_case()
    loc = slab_partition_fe(prob, rank, world)
    A = orc.FeOperator(loc["A_cells"], loc["conn"], loc["m"])
    Dinv = orc.DiagonalInverse(loc["dinv"])
    r0, r1 = loc["row0"], loc["row1"]
    Gl = G[r0:r1]
    rows = np.concatenate([loc["if_lower"], loc["if_upper"]]).astype(np.int64)
    n_lo, n_hi = len(loc["if_lower"]), len(loc["if_upper"])
    e, c, sigma, gamma = orc.cheb_scalars(*b)
    RX = np.zeros_like(Gl)
    RY = (sigma / e) * Gl
    LY = (sigma / e) * (ritz - c)
    LX = np.ones_like(ritz)
    send = torch.zeros((len(rows), X.shape[1]), dtype=torch.float64)
    recv = torch.zeros_like(send)
    for _k in range(2, p + 1):
        sigma2 = 1.0 / (gamma - sigma)
        a = 2.0 * sigma2 / e
        base = -a * c * RY - sigma * sigma2 * RX + a * Gl * LY[None, :]
        delta = a * A.apply(Dinv.apply(RY))                 # this slab's share of the product
        send.copy_(torch.from_numpy(delta[rows]))
        neighbor_exchange(send, recv, n_lo, n_hi, rank)
        new = base + delta
        new[rows] = base[rows] + (send.numpy() + recv.numpy())
        LXn = a * LY * ritz - a * c * LY - sigma * sigma2 * LX
        RX, RY, LX, LY, sigma = RY, new, LY, LXn, sigma2
    Y = Dinv.apply(RY) + X[r0:r1] * LY[None, :]
    np.save(os.path.join(out_dir, "rows%d.npy" % rank), Y)
    np.save(os.path.join(out_dir, "span%d.npy" % rank), np.array([r0, r1]))
    dist.barrier()
    dist.destroy_process_group()


def _row_case():
    import workloads
    from oracle import chfsi_oracle as orc
    prob = workloads.fe_problem(4, q=2, seed=9)
    A, B, Dinv = orc.operators_from_workload(prob)
    X0 = np.random.default_rng(1).standard_normal((prob["m"], 5))
    ritz, X, AX, BX = orc.rayleigh_ritz(A.apply, B.apply, X0)
    G = orc.residual_block(AX, BX, ritz)
    lam_max = workloads.fe.fe_lam_max_bound(prob["A_cells"], prob["B_cell"]) * 1.01
    return prob, X, ritz, G, 7, (ritz[0] - 1.0, ritz[-1] + 1.0, lam_max)


def test_row_slabs_partition_and_neighbour_exchange_over_gloo(tmp_path):
    """Row-sharded filter: (i) the slabs cover the mesh, neighbouring slabs share
    exactly one node plane, and the slab operators sum to the global operator; (ii) two gloo ranks that exchange one
    buffer per neighbour and step reproduce the oracle's global Algorithm 3 on their rows."""
    sys.path.insert(0, ROOT)
    from paper_2503_22652_b200.sharding import slab_partition_fe
    from oracle import chfsi_oracle as orc
    prob, X, ritz, G, p, b = _row_case()
    A, B, Dinv = orc.operators_from_workload(prob)
    for world in (1, 2, 3, 4):
        parts = [slab_partition_fe(prob, r, world) for r in range(world)]
        assert parts[0]["row0"] == 0 and parts[-1]["row1"] == prob["m"]
        assert sorted(np.concatenate([q["cells"] for q in parts]).tolist()) == list(range(prob["n_cells"]))
        V = np.random.default_rng(world).standard_normal((prob["m"], 3))
        acc = np.zeros_like(V)
        for r, q in enumerate(parts):
            acc[q["row0"]:q["row1"]] += orc.FeOperator(q["A_cells"], q["conn"], q["m"]).apply(V[q["row0"]:q["row1"]])
            if r + 1 < world:    # the shared plane: same global rows on both sides
                np.testing.assert_array_equal(q["row0"] + q["if_upper"], parts[r + 1]["row0"] + parts[r + 1]["if_lower"])
        np.testing.assert_allclose(acc, A.apply(V), rtol=1e-12, atol=1e-12)
    port = 31500 + os.getpid() % 2000
    mp.spawn(_row_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    Y = orc.filter_rchfsi(A.apply, Dinv.apply, X, ritz, G, p, *b)
    for r in range(2):
        r0, r1 = np.load(tmp_path / ("span%d.npy" % r))
        np.testing.assert_allclose(np.load(tmp_path / ("rows%d.npy" % r)), Y[r0:r1], rtol=1e-11, atol=1e-13)
