"""Reduced-precision criteria of north_star at the BASELINE.json sizes ("match converged eigenvalues to a relative error
<= 1e-8 and reach residual norms <= 1e-8 ... on all five configs"), each checked against something the CUDA library
did not compute:

  configs[0]  prescribed spectrum lam of A = Q diag(lam) Q^T (pin P3), with the 1e-4 column-noise hook;
              ChFSI with the same hook must floor
  configs[1]  scipy.linalg.eigh(A, B) (LAPACK, "computed independently via LAPACK's dsygv")
  configs[2]  the ORACLE's CsrOperator residual of every returned pair (||A x - eps x||_2 <= tau
              certifies an eigenvalue within tau of eps) + the Weyl window around the closed-form Laplacian
              eigenvalues as the count check (pin P3)
  configs[3]  a degree-3 filter at full mesh size within the per-step operand-rounding bound, TF32 and BF16, FP32 and
              FP64 storage; and P8 with the ORACLE's FeOperator on sampled wanted pairs of the converged solves
configs[4] is certified the same way inside bench.py (its `solve` record): a 172 GB problem does not belong in pytest.
"""
import functools

import numpy as np
import pytest

import workloads
from oracle import chfsi_oracle as orc
from tests.helpers import oracle_ops

pytestmark = pytest.mark.gpu

TAU = 1e-8      # PAPER.md:341 "max_j r_j < 1e-8"


def _rel(ev, ref):
    return np.max(np.abs(ev - ref) / np.maximum(1.0, np.abs(ref)))


def test_config1_full_size_noisy_solve_eigenvalues_and_chfsi_floor():
    import torch
    import paper_2503_22652_b200 as P
    prob = workloads.config1_dense_standard()
    nw, N, p = prob["n_wanted"], prob["block"], prob["degree"]
    b = (prob["lam_min"], prob["lam_T"], prob["lam_max"])
    As, Bs, dinv = P.upload_problem(prob)
    out = {}
    for meth in (P.METHOD_RCHFSI, P.METHOD_CHFSI):
        s = P.Rchfsi(As, Bs, dinv, block_N=N, noise_eps=prob["noise_eps"], noise_seed=99)
        out[meth] = s.solve(meth, torch.as_tensor(prob["X0"]).cuda(), nw, p, *b, tol=TAU, max_iter=40)
        s.close()
    r = out[P.METHOD_RCHFSI]
    assert r["converged"] and r["iters"] <= 12, r["history"]
    assert _rel(r["evals"][:nw], prob["lam"][:nw]) <= 1e-8
    assert r["resnorm"][:nw].max() <= TAU
    c = out[P.METHOD_CHFSI]          # same inexact products in Algorithm 2: the residual floors at O(eps)
    assert not c["converged"] and min(c["history"]) > 1e-7, c["history"][-5:]


@functools.lru_cache(maxsize=1)
def _c2():
    import scipy.linalg as sla
    prob = workloads.config2_dense_generalized()
    ev = sla.eigh(prob["A"], prob["B"], eigvals_only=True)
    return prob, ev


@pytest.mark.parametrize("apply_prec", ["tf32", "bf16"])
def test_config2_full_size_reduced_precision_solve_matches_lapack(apply_prec):
    import torch
    import paper_2503_22652_b200 as P
    prob, ev = _c2()
    nw, N, p = prob["n_wanted"], prob["block"], prob["degree"]
    As, Bs, dinv = P.upload_problem(prob)
    s = P.Rchfsi(As, Bs, dinv, block_N=N, apply_prec=apply_prec, adaptive_bounds=True)
    r = s.solve(P.METHOD_RCHFSI, torch.as_tensor(prob["X0"]).cuda(), nw, p, -100.0, 0.0, 16.0, tol=TAU, max_iter=60)
    s.close()
    assert r["converged"], r["history"][-5:]
    assert r["resnorm"][:nw].max() <= TAU
    assert _rel(r["evals"][:nw], ev[:nw]) <= 1e-8


def test_config3_full_size_fp32_spmm_solve_certified_by_the_oracle_operator():
    import torch
    import paper_2503_22652_b200 as P
    prob = workloads.config3_sparse_laplacian()
    nw, N, p, n = prob["n_wanted"], prob["block"], prob["degree"], prob["n_grid"]
    As, Bs, dinv = P.upload_problem(prob)
    s = P.Rchfsi(As, Bs, dinv, block_N=N, apply_prec="fp32", adaptive_bounds=True)
    X = torch.as_tensor(workloads.start_block(prob["m"], N, prob["x0_seed"])).cuda()
    r = s.solve(P.METHOD_RCHFSI, X, nw, p, -100.0, 0.0, prob["lam_max"], tol=TAU, max_iter=60)
    s.close()
    assert r["converged"], r["history"][-5:]
    Xh = X[:, :nw].cpu().numpy()
    ev = r["evals"][:nw]
    A, _, _ = oracle_ops(prob)
    res = np.linalg.norm(A.apply(Xh) - Xh * ev[None, :], axis=0)        # the oracle's operator, B = I
    assert res.max() <= TAU * 1.01, res.max()                             # => an eigenvalue within 1e-8 of every eps_j
    assert np.abs(Xh.T @ Xh - np.eye(nw)).max() <= 1e-8                   # distinct pairs (B-orthonormal)
    assert np.all(np.diff(ev) >= -1e-12)
    # count check (no eigenvalue skipped): Weyl with -5 <= V <= 0 gives lam_k(L) - 5 <= lam_k(L + V) <= lam_k(L)
    lap = workloads.laplacian3d_exact_eigs(n)[:nw]
    assert np.all(ev <= lap + 1e-8) and np.all(ev >= lap - 5.0 - 1e-8)


@functools.lru_cache(maxsize=1)
def _c4():
    prob = workloads.config4_fe()
    lam_max = 1.02 * workloads.fe.fe_lam_max_bound(prob["A_cells"], prob["B_cell"], list(range(0, prob["n_cells"], 256)))
    return prob, lam_max


@pytest.mark.parametrize("apply_prec,tol", [("tf32", 6e-3), ("bf16", 3e-2)])
def test_config4_full_size_degree3_filter_within_the_operand_rounding_bound(apply_prec, tol):
    """Two operator applies at full mesh size (4096 cells, 10 column tiles, ragged last tile): the residual part
    D^-1 R_p = Y_p - X Lambda_p of the tcgen05 path against the oracle's on sampled columns, within the per-apply
    operand-rounding bound times the number of applies -- a tight bound where the 39-apply full-degree
    test can only catch O(1) mistakes."""
    import torch
    import paper_2503_22652_b200 as P
    prob, lam_max = _c4()
    m, N, p = prob["m"], prob["block"], 3
    A, B, Dinv = oracle_ops(prob)
    rng = np.random.default_rng(31)
    X = rng.standard_normal((m, N)) / np.sqrt(m)
    G = rng.standard_normal((m, N)) * 1e-2
    ritz = np.linspace(-9.0, 3.0, N)
    bounds = (-10.0, 3.5, lam_max)
    cols = np.array([0, 127, 128, 640, 1151, 1152, 1199])     # tile edges, a middle tile, the ragged tenth tile
    Yo = orc.filter_rchfsi(A.apply, Dinv.apply, X[:, cols].copy(), ritz[cols], G[:, cols].copy(), p, *bounds)
    XL = X[:, cols] * orc.lambda_recurrence(ritz[cols], p, *bounds)[p][None, :]
    As, Bs, dinv = P.upload_problem(prob)
    Gd, rd = torch.as_tensor(G).cuda(), torch.as_tensor(ritz).cuda()
    cd = torch.as_tensor(cols).cuda()
    for store in ("fp32", "fp64"):
        s = P.Rchfsi(As, None, dinv, block_N=N, apply_prec=apply_prec, store_prec=store)
        Xd = torch.as_tensor(X).cuda()
        s.filter(P.METHOD_RCHFSI, Xd, rd, Gd, p, *bounds)
        Yg = Xd[:, cd].cpu().numpy()
        s.close()
        del Xd
        torch.cuda.empty_cache()
        err = np.linalg.norm((Yg - XL) - (Yo - XL), axis=0) / np.linalg.norm(Yo - XL, axis=0)
        assert 1e-9 < err.max() < tol, (store, err)


@pytest.mark.parametrize("apply_prec", ["tf32", "bf16"])
def test_config4_full_size_solve_certified_by_the_oracle_operator(apply_prec):
    """The configs[3] solve (1000 lowest pairs of the 912,673-dof pencil, cell GEMMs in TF32 / BF16, FP32 recurrence):
    P8 with the oracle's FeOperator on 32 sampled wanted pairs."""
    import torch
    import paper_2503_22652_b200 as P
    prob, lam_max = _c4()
    m, N, nw, p = prob["m"], prob["block"], prob["n_wanted"], prob["degree"]
    As, Bs, dinv = P.upload_problem(prob)
    s = P.Rchfsi(As, Bs, dinv, block_N=N, apply_prec=apply_prec, store_prec="fp32", adaptive_bounds=True)
    X = torch.as_tensor(workloads.start_block(m, N, prob["x0_seed"])).cuda()
    r = s.solve(P.METHOD_RCHFSI, X, nw, p, -100.0, 0.0, lam_max, tol=TAU, max_iter=80)
    s.close()
    assert r["converged"], r["history"][-5:]
    cols = np.unique(np.concatenate(([0, nw - 1], np.random.default_rng(5).integers(0, nw, 30))))
    Xh = X[:, torch.as_tensor(cols).cuda()].cpu().numpy()
    del X
    torch.cuda.empty_cache()
    ev = r["evals"][cols]
    A, B, _ = oracle_ops(prob)
    BX = B.apply(Xh)
    res = np.linalg.norm(A.apply(Xh) - BX * ev[None, :], axis=0)
    assert res.max() <= TAU * 1.01, res.max()
    assert np.abs(Xh.T @ BX - np.eye(len(cols))).max() <= 1e-8
    assert np.all(np.diff(r["evals"][:nw]) >= -1e-12) and r["evals"][0] > -10.0 * 8 and r["evals"][nw - 1] < lam_max
