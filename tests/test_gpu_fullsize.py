"""Parity at BASELINE.json's FULL sizes, in the launch configurations bench.py times: the filter runs on the
whole block on the GPU and the oracle recomputes a sample of columns one by one (Algorithm 3 is column-separable,
PAPER.md:255-263, so a column of the block filter equals the filter of that column).  The filter is defined for any
X, Lambda, G (the derivation uses only the scalar recurrence), so the inputs are plain seeded blocks.
FP64 mode: <= 1e-10 column-wise (north_star).  Tensor-core mode at full size: a loose bound that only catches
structural mistakes (tile / ragged-edge / colouring errors); the tight reduced-precision criteria are the solves."""
import numpy as np
import pytest

import workloads
from oracle import chfsi_oracle as orc
from tests.helpers import oracle_ops

pytestmark = pytest.mark.gpu


def _inputs(m, N, seed):
    rng = np.random.default_rng(seed)
    X = rng.standard_normal((m, N)) / np.sqrt(m)
    G = rng.standard_normal((m, N)) * 1e-2
    return X, G


def _check_columns(Yg, X, ritz, G, A, Dinv, p, bounds, cols, tol):
    Yo = orc.filter_rchfsi(A.apply, Dinv.apply, X[:, cols].copy(), ritz[cols], G[:, cols].copy(), p, *bounds)
    err = np.linalg.norm(Yg[:, cols] - Yo, axis=0) / np.linalg.norm(Yo, axis=0)
    assert err.max() <= tol, err
    return Yo


def test_config2_full_size_fp64_all_columns():
    import torch
    import paper_2503_22652_b200 as P
    prob = workloads.config2_dense_generalized()
    m, N, p = prob["m"], prob["block"], prob["degree"]
    A, B, Dinv = oracle_ops(prob)
    X, G = _inputs(m, N, 1)
    ritz = np.linspace(-1.5, 0.6, N)
    bounds = (-2.5, 0.7, 16.0)
    As, Bs, dinv = P.upload_problem(prob)
    s = P.Rchfsi(As, Bs, dinv, block_N=N)
    Xd = torch.as_tensor(X).cuda()
    s.filter(P.METHOD_RCHFSI, Xd, torch.as_tensor(ritz).cuda(), torch.as_tensor(G).cuda(), p, *bounds)
    _check_columns(Xd.cpu().numpy(), X, ritz, G, A, Dinv, p, bounds, np.arange(N), 1e-10)
    s.close()


def test_config3_full_size_fp64_sampled_columns_and_fused_fp32_path():
    import torch
    import paper_2503_22652_b200 as P
    prob = workloads.config3_sparse_laplacian()
    m, N, p = prob["m"], prob["block"], prob["degree"]
    A, B, Dinv = oracle_ops(prob)
    X, G = _inputs(m, N, 2)
    ritz = np.linspace(-3.3, -2.8, N)
    bounds = (-3.4, -2.7, 12.0)
    cols = np.array([0, 131, 298, 299])          # first, middle, and the ragged last 128-bit vector
    As, Bs, dinv = P.upload_problem(prob)
    s = P.Rchfsi(As, Bs, dinv, block_N=N)
    Xd = torch.as_tensor(X).cuda()
    s.filter(P.METHOD_RCHFSI, Xd, torch.as_tensor(ritz).cuda(), torch.as_tensor(G).cuda(), p, *bounds)
    Yo = _check_columns(Xd.cpu().numpy(), X, ritz, G, A, Dinv, p, bounds, cols, 1e-10)
    s.close()
    # the configuration bench.py times: fused FP32 SpMM + FP64 recurrence.  FP32 products, 29 applies: the
    # error stays at the FP32 rounding level relative to the filtered column
    s = P.Rchfsi(As, Bs, dinv, block_N=N, apply_prec="fp32")
    Xd = torch.as_tensor(X).cuda()
    s.filter(P.METHOD_RCHFSI, Xd, torch.as_tensor(ritz).cuda(), torch.as_tensor(G).cuda(), p, *bounds)
    err = np.linalg.norm(Xd.cpu().numpy()[:, cols] - Yo, axis=0) / np.linalg.norm(Yo, axis=0)
    assert err.max() < 1e-4, err
    # the same call through the host entry point: at this size the block goes through the column-chunked pipeline
    # (128 + 128 + 44 columns, three streams); columns are independent, so the result is bit for bit the same
    Xh = torch.as_tensor(X.copy()).pin_memory()
    s.filter_host(P.METHOD_RCHFSI, Xh, ritz, G, p, *bounds)
    np.testing.assert_array_equal(Xh.numpy(), Xd.cpu().numpy())
    s.close()


def test_config4_full_size_fp64_and_tensor_core_sampled_columns():
    import torch
    import paper_2503_22652_b200 as P
    prob = workloads.config4_fe()
    m, N, p = prob["m"], prob["block"], prob["degree"]
    A, B, Dinv = oracle_ops(prob)
    X, G = _inputs(m, N, 3)
    ritz = np.linspace(-9.0, 3.0, N)
    lam_max = 1.02 * workloads.fe.fe_lam_max_bound(prob["A_cells"], prob["B_cell"], list(range(0, prob["n_cells"], 256)))
    bounds = (-10.0, 3.5, lam_max)
    cols = np.array([5, 1199])                   # 1199: last column of the ragged tenth 128-column tile
    As, Bs, dinv = P.upload_problem(prob)
    s = P.Rchfsi(As, None, dinv, block_N=N)
    Xd = torch.as_tensor(X).cuda()
    Gd = torch.as_tensor(G).cuda()
    rd = torch.as_tensor(ritz).cuda()
    s.filter(P.METHOD_RCHFSI, Xd, rd, Gd, p, *bounds)
    Yg = Xd[:, torch.as_tensor(cols).cuda()].cpu().numpy()
    Yo = orc.filter_rchfsi(A.apply, Dinv.apply, X[:, cols].copy(), ritz[cols], G[:, cols].copy(), p, *bounds)
    err = np.linalg.norm(Yg - Yo, axis=0) / np.linalg.norm(Yo, axis=0)
    assert err.max() <= 1e-10, err
    s.close()
    del Xd
    torch.cuda.empty_cache()
    # the configurations bench.py times: fused tcgen05 step, TF32 operands, FP64 and FP32 recurrence storage
    for store in ("fp64", "fp32"):
        s = P.Rchfsi(As, None, dinv, block_N=N, apply_prec="tf32", store_prec=store)
        Xd = torch.as_tensor(X).cuda()
        s.filter(P.METHOD_RCHFSI, Xd, rd, Gd, p, *bounds)
        Yt = Xd[:, torch.as_tensor(cols).cuda()].cpu().numpy()
        assert np.isfinite(Yt).all()
        err = np.linalg.norm(Yt - Yo, axis=0) / np.linalg.norm(Yo, axis=0)
        assert err.max() < 5e-2, (store, err)     # 39 TF32 applies; structural mistakes give O(1)
        s.close()
        del Xd
        torch.cuda.empty_cache()
