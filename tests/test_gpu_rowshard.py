"""Row-sharded R-ChFSI filter ("nearest-neighbour MPI communication ... in BF16
precision; we term this method TF32B"): several slabs of one FE mesh, each with its own library handle,
driven in lockstep in ONE process on one GPU (one kernel stream, no kernels waiting on each other); the buffers a real
run sends over NVLink are swapped by device copies.  Checked against the oracle's GLOBAL Algorithm 3."""
import numpy as np
import pytest

import workloads
from oracle import chfsi_oracle as orc
from tests.helpers import oracle_ops

pytestmark = pytest.mark.gpu


def _case(nc, q, N, seed):
    prob = workloads.fe_problem(nc, q=q, seed=seed)
    A, B, Dinv = oracle_ops(prob)
    X0 = np.random.default_rng(seed).standard_normal((prob["m"], N))
    ritz, X, AX, BX = orc.rayleigh_ritz(A.apply, B.apply, X0)
    G = orc.residual_block(AX, BX, ritz)
    lam_max = workloads.fe.fe_lam_max_bound(prob["A_cells"], prob["B_cell"]) * 1.01
    return prob, (A, B, Dinv), X, ritz, G, (ritz[0] - 1.0, ritz[-1] + 1.0, lam_max)


def _run_sharded(prob, X, ritz, G, p, b, world, wire, **opts):
    import torch
    import paper_2503_22652_b200 as P
    from paper_2503_22652_b200.sharding import slab_partition_fe, RowShardedFilter, filter_in_process
    shards, blocks, parts, solvers = [], [], [], []
    rd = torch.as_tensor(ritz).cuda()
    for r in range(world):
        loc = slab_partition_fe(prob, r, world)
        As, Bs, dinv = P.upload_problem(loc)
        s = P.Rchfsi(As, Bs, dinv, block_N=X.shape[1], **opts)
        shards.append(RowShardedFilter(s, loc["if_lower"], loc["if_upper"], wire=wire))
        blocks.append((torch.as_tensor(X[loc["row0"]:loc["row1"]].copy()).cuda(), rd,
                       torch.as_tensor(G[loc["row0"]:loc["row1"]].copy()).cuda()))
        parts.append(loc)
        solvers.append(s)
    out = filter_in_process(shards, blocks, p, *b)
    Y = np.zeros_like(X)
    replicas_equal = True
    for r, (loc, Yr) in enumerate(zip(parts, out)):
        Yh = Yr.cpu().numpy()
        if r > 0:      # the plane shared with the previous slab must hold the same bits on both ranks
            replicas_equal &= np.array_equal(Yh[loc["if_lower"]], Y[loc["row0"] + loc["if_lower"]])
        Y[loc["row0"]:loc["row1"]] = Yh
    per_step = [sh.bytes_per_step for sh in shards]
    for s in solvers:
        s.close()
    return Y, replicas_equal, per_step


@pytest.mark.parametrize("world", [2, 3])
def test_row_sharded_filter_fp64_equals_the_global_oracle_filter(world):
    """All-FP64 mode, FP64 on the wire: the stitched slabs equal the oracle's global filter to 1e-10 (north_star's
    bar for filtered blocks); a middle slab (world = 3) has two interfaces."""
    prob, (A, B, Dinv), X, ritz, G, b = _case(3, 3, 12, 5)
    p = 9
    Yo = orc.filter_rchfsi(A.apply, Dinv.apply, X, ritz, G, p, *b)
    Y, same, _ = _run_sharded(prob, X, ritz, G, p, b, world, "fp64")
    err = np.linalg.norm(Y - Yo, axis=0) / np.linalg.norm(Yo, axis=0)
    assert err.max() <= 1e-10, err.max()
    assert same


@pytest.mark.parametrize("apply_prec,store,wire,tol", [("bf16", "fp32", "bf16", 3e-2), ("bf16", "fp32", "fp32", 3e-2),
                                                       ("tf32", "fp32", "bf16", 1.2e-2), ("tf32", "fp64", "fp32", 6e-3)])
def test_row_sharded_tensor_core_filter_with_reduced_precision_wire(apply_prec, store, wire, tol):
    """The fused tcgen05 FE step on every slab (pipelined BF16 kernel / TF32 kernel, panel layout, in-place shadow) with
    BF16 or FP32 interface exchange: the residual part D^-1 R_p of the stitched block equals the oracle's within the
    operand-rounding bound (+ 2^-9 per step on interface rows for the BF16 wire), the replicated interface rows are
    bit-identical on both ranks, and the BF16 wire moves a quarter of the FP64 bytes."""
    prob, (A, B, Dinv), X, ritz, G, b = _case(3, 3, 136, 7)
    p = 3
    Yo = orc.filter_rchfsi(A.apply, Dinv.apply, X, ritz, G, p, *b)
    XL = X * orc.lambda_recurrence(ritz, p, *b)[p][None, :]
    Y, same, per_step = _run_sharded(prob, X, ritz, G, p, b, 3, wire, apply_prec=apply_prec, store_prec=store)
    err = np.linalg.norm((Y - XL) - (Yo - XL)) / np.linalg.norm(Yo - XL)
    assert 1e-9 < err < tol, err
    assert same
    plane = (prob["q"] * prob["nc"] + 1) ** 2
    assert per_step[1] == 2 * plane * 136 * (2 if wire == "bf16" else 4)      # middle slab: two interfaces
    assert per_step[0] == plane * 136 * (2 if wire == "bf16" else 4)


def test_row_sharded_solve_like_iteration_converges_with_bf16_wire():
    """Several outer iterations (sharded filter with BF16 exchange + the oracle's Rayleigh-Ritz on the stitched block,
    which is exact arithmetic outside the filter as in PAPER.md:253): the residual falls below 1e-8, i.e. the BF16
    interface error is tolerated by the residual recurrence."""
    prob, (A, B, Dinv), X, ritz, G, b = _case(2, 4, 16, 3)
    import scipy.linalg as sla
    m = prob["m"]
    ev = sla.eigh(A.apply(np.eye(m)), B.apply(np.eye(m)), eigvals_only=True)
    nw, p = 8, 30
    lam_max = b[2]
    for it in range(60):
        Y, same, _ = _run_sharded(prob, X, ritz, G, p, (ritz[0], ritz[-1], lam_max), 2, "bf16",
                                  apply_prec="tf32", store_prec="fp32")
        assert same
        ritz, X, AX, BX = orc.rayleigh_ritz(A.apply, B.apply, Y)
        G = orc.residual_block(AX, BX, ritz)
        res = np.linalg.norm(G, axis=0)[:nw].max()
        if res < 1e-8:
            break
    assert res < 1e-8, res
    np.testing.assert_allclose(ritz[:nw], ev[:nw], rtol=1e-8, atol=1e-9)
