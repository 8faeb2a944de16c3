"""GPU parity: the CUDA library (through the C ABI binding) against the FP64 CPU oracle on the
same seeded inputs.  All-FP64 mode: filtered blocks to <= 1e-10 relative (north_star).  Reduced
precision modes: converged eigenvalues <= 1e-8 relative and residuals <= 1e-8."""
import numpy as np
import pytest

import workloads
from oracle import chfsi_oracle as orc
from tests.helpers import oracle_ops, rel_fro, small_dense_generalized

pytestmark = pytest.mark.gpu

TOL_FP64 = 1e-10   # north_star: "relative error <= 1e-10 on filtered blocks in an all-FP64 mode"


def _torch():
    import torch
    assert torch.cuda.is_available()
    return torch


def _setup(prob, N, seed, **opts):
    """Upload the problem, build X (B-orthonormal via the oracle RR), ritz, G on the host."""
    torch = _torch()
    import paper_2503_22652_b200 as P
    A, B, Dinv = oracle_ops(prob)
    X0 = np.random.default_rng(seed).standard_normal((prob["m"], N))
    ritz, X, AX, BX = orc.rayleigh_ritz(A.apply, B.apply, X0)
    G = orc.residual_block(AX, BX, ritz)
    As, Bs, dinv = P.upload_problem(prob)
    solver = P.Rchfsi(As, Bs, dinv, block_N=N, **opts)
    return solver, (A, B, Dinv), X, ritz, G


def _bounds(prob, A, B):
    """Spectral bounds from a library eigensolver on the (small) dense pencil."""
    import scipy.linalg as sla
    m = prob["m"]
    Ad = A.apply(np.eye(m))
    Bd = B.apply(np.eye(m))
    ev = sla.eigh(Ad, Bd, eigvals_only=True)
    dinv = prob.get("dinv")
    top = ev[-1]
    if dinv is not None:   # lam_max must also bound lam(D^-1 A) (reading S7)
        s = np.sqrt(dinv)
        top = max(top, np.linalg.eigvalsh(s[:, None] * Ad * s[None, :])[-1])
    return ev, top


def _run_filter_parity(prob, N, p, n_inside, method, seed=11):
    torch = _torch()
    import paper_2503_22652_b200 as P
    solver, (A, B, Dinv), X, ritz, G = _setup(prob, N, seed)
    ev, top = _bounds(prob, A, B)
    lam_min, lam_T, lam_max = ev[0] - 1e-3, ev[n_inside], top * 1.01 + 1e-6
    if method == "rchfsi":
        Yo = orc.filter_rchfsi(A.apply, Dinv.apply, X, ritz, G, p, lam_min, lam_T, lam_max)
    else:
        Yo = orc.filter_chfsi(A.apply, Dinv.apply, X, p, lam_min, lam_T, lam_max)
    Xd = torch.as_tensor(X).cuda()
    meth = P.METHOD_RCHFSI if method == "rchfsi" else P.METHOD_CHFSI
    solver.filter(meth, Xd, torch.as_tensor(ritz).cuda(), torch.as_tensor(G).cuda(), p, lam_min, lam_T, lam_max)
    Yg = Xd.cpu().numpy()
    # column-wise: every column must match, not only the Frobenius norm
    err = np.linalg.norm(Yg - Yo, axis=0) / np.linalg.norm(Yo, axis=0)
    assert err.max() <= TOL_FP64, err.max()
    assert solver.launch_count() > 0
    if method == "rchfsi":   # G = NULL => the library forms A X - B X Lambda itself
        Xd2 = torch.as_tensor(X).cuda()
        solver.filter(meth, Xd2, torch.as_tensor(ritz).cuda(), None, p, lam_min, lam_T, lam_max)
        # the library's own G differs from the oracle's by rounding of a cancelling difference;
        # the filter amplifies it by at most C_p'(eps) -- compare loosely
        assert rel_fro(Xd2.cpu().numpy(), Yo) <= 1e-6
    solver.close()


@pytest.mark.parametrize("method", ["rchfsi", "chfsi"])
@pytest.mark.parametrize("m,N,p", [(200, 12, 9), (333, 20, 16), (130, 7, 5), (64, 4, 1)])
def test_dense_generalized_filter_fp64(m, N, p, method):
    # sizes span several 64-row tiles with ragged tails, N not a multiple of 4, degree 1
    _run_filter_parity(small_dense_generalized(m, seed=m), N, p, N, method)


@pytest.mark.parametrize("method", ["rchfsi", "chfsi"])
def test_config1_dense_standard_filter_fp64_full_size(method):
    prob = workloads.config1_dense_standard()
    torch = _torch()
    import paper_2503_22652_b200 as P
    N, p = prob["block"], prob["degree"]
    solver, (A, B, Dinv), X, ritz, G = _setup(prob, N, 5)
    b = (prob["lam_min"], prob["lam_T"], prob["lam_max"])
    if method == "rchfsi":
        Yo = orc.filter_rchfsi(A.apply, Dinv.apply, X, ritz, G, p, *b)
    else:
        Yo = orc.filter_chfsi(A.apply, Dinv.apply, X, p, *b)
    Xd = torch.as_tensor(X).cuda()
    solver.filter(P.METHOD_RCHFSI if method == "rchfsi" else P.METHOD_CHFSI, Xd, torch.as_tensor(ritz).cuda(),
                  torch.as_tensor(G).cuda(), p, *b)
    err = np.linalg.norm(Xd.cpu().numpy() - Yo, axis=0) / np.linalg.norm(Yo, axis=0)
    assert err.max() <= TOL_FP64, err.max()
    solver.close()


@pytest.mark.parametrize("method", ["rchfsi", "chfsi"])
@pytest.mark.parametrize("n,N,p", [(6, 8, 12), (7, 10, 7), (9, 12, 20)])
def test_csr_laplacian_filter_fp64(n, N, p, method):
    prob = workloads.config3_sparse_laplacian(n=n, n_wanted=N - 2, block=N, degree=p, seed=n)
    _run_filter_parity(prob, N, p, N, method)


@pytest.mark.parametrize("method", ["rchfsi", "chfsi"])
@pytest.mark.parametrize("nc,q,N,p", [(2, 3, 8, 10), (3, 2, 13, 6), (2, 6, 16, 8)])
def test_fe_generalized_filter_fp64(nc, q, N, p, method):
    # q=6 is the paper-shaped element (343 nodes per cell); q=2,3 give ragged n_loc = 27, 64
    prob = workloads.fe_problem(nc, q=q, seed=nc + q)
    _run_filter_parity(prob, N, p, N, method)


def test_rayleigh_ritz_matches_oracle():
    torch = _torch()
    import paper_2503_22652_b200 as P
    prob = small_dense_generalized(300, seed=3)
    N = 24
    A, B, Dinv = oracle_ops(prob)
    Y = np.random.default_rng(8).standard_normal((300, N)) * np.logspace(0, 6, N)[None, :]
    ritz_o, X_o, AX, BX = orc.rayleigh_ritz(A.apply, B.apply, Y)
    res_o = orc.residual_norms(AX, BX, ritz_o)
    As, Bs, dinv = P.upload_problem(prob)
    s = P.Rchfsi(As, Bs, dinv, block_N=N)
    ritz, X, G, res = s.rayleigh_ritz(torch.as_tensor(Y).cuda())
    np.testing.assert_allclose(ritz.cpu().numpy(), ritz_o, rtol=1e-11, atol=1e-12)
    Xg = X.cpu().numpy()
    # eigenvector signs are free (S12): compare |x_j^T B x_j^oracle| = 1 and B-orthonormality
    Bd = prob["B"]
    np.testing.assert_allclose(np.abs(np.sum(Xg * (Bd @ X_o), axis=0)), 1.0, rtol=0, atol=1e-8)
    np.testing.assert_allclose(Xg.T @ Bd @ Xg, np.eye(N), rtol=0, atol=1e-10)
    np.testing.assert_allclose(res.cpu().numpy(), res_o, rtol=1e-6, atol=1e-11)
    Gg = G.cpu().numpy()
    np.testing.assert_allclose(Gg, prob["A"] @ Xg - (Bd @ Xg) * ritz.cpu().numpy()[None, :], rtol=0, atol=1e-10)
    # exact operator apply
    V = torch.as_tensor(Y).cuda()
    np.testing.assert_allclose(s.apply(0, V).cpu().numpy(), prob["A"] @ Y, rtol=1e-12, atol=1e-6)
    np.testing.assert_allclose(s.apply(1, V).cpu().numpy(), Bd @ Y, rtol=1e-12, atol=1e-6)
    s.close()


def test_solve_fp64_matches_oracle_solve_iterates_and_eigs():
    torch = _torch()
    import paper_2503_22652_b200 as P
    prob = workloads.config1_dense_standard(m=400, n_wanted=20, block=24, degree=12, seed=9)
    A, B, Dinv = oracle_ops(prob)
    b = (prob["lam_min"], prob["lam_T"], prob["lam_max"])
    ref = orc.solve(A, B, A, Dinv, prob["X0"], 20, 12, *b, tol=1e-8, max_iter=40)
    As, Bs, dinv = P.upload_problem(prob)
    s = P.Rchfsi(As, Bs, dinv, block_N=24)
    Xd = torch.as_tensor(prob["X0"]).cuda()
    out = s.solve(P.METHOD_RCHFSI, Xd, 20, 12, *b, tol=1e-8, max_iter=40)
    assert out["converged"] and out["iters"] == ref["iters"]
    np.testing.assert_allclose(out["evals"][:20], prob["lam"][:20], rtol=1e-10)
    np.testing.assert_allclose(out["evals"][:20], ref["evals"][:20], rtol=1e-10)
    assert out["resnorm"][:20].max() < 1e-8
    s.close()


@pytest.mark.parametrize("apply_prec,store_prec", [("fp32", "fp64"), ("fp32", "fp32"), ("tf32", "fp64"),
                                                   ("bf16", "fp64"), ("bf16", "fp32")])
def test_dense_generalized_reduced_precision_solve(apply_prec, store_prec):
    """Reduced-precision operator apply: converged eigenvalues <= 1e-8 relative to the exact ones,
    residual <= 1e-8 (north_star); ChFSI with the same inexact apply must not get there."""
    torch = _torch()
    import scipy.linalg as sla
    import paper_2503_22652_b200 as P
    prob = small_dense_generalized(600, seed=21)
    N, nw, p = 40, 30, 16
    ev = sla.eigh(prob["A"], prob["B"], eigvals_only=True)
    s = np.sqrt(prob["dinv"])
    top = max(ev[-1], np.linalg.eigvalsh(s[:, None] * prob["A"] * s[None, :])[-1])
    b = (ev[0] - 1e-2, ev[N], top * 1.02)
    As, Bs, dinv = P.upload_problem(prob)
    X0 = np.random.default_rng(1).standard_normal((600, N))
    sol = P.Rchfsi(As, Bs, dinv, block_N=N, apply_prec=apply_prec, store_prec=store_prec)
    out = sol.solve(P.METHOD_RCHFSI, torch.as_tensor(X0).cuda(), nw, p, *b, tol=1e-8, max_iter=60)
    assert out["converged"], out["history"]
    np.testing.assert_allclose(out["evals"][:nw], ev[:nw], rtol=1e-8)
    assert out["resnorm"][:nw].max() <= 1e-8
    sol.close()


def test_csr_fp32_fused_solve_matches_oracle_eigs_and_chfsi_stagnates():
    torch = _torch()
    import paper_2503_22652_b200 as P
    prob = workloads.config3_sparse_laplacian(n=12, n_wanted=24, block=32, degree=20, seed=3)
    A, B, Dinv = oracle_ops(prob)
    ev = np.linalg.eigvalsh(A.apply(np.eye(prob["m"])))
    b = (ev[0] - 1e-2, ev[32], 12.0)
    As, Bs, dinv = P.upload_problem(prob)
    X0 = workloads.start_block(prob["m"], 32, prob["x0_seed"])
    for store in ("fp64", "fp32"):
        sol = P.Rchfsi(As, Bs, dinv, block_N=32, apply_prec="fp32", store_prec=store)
        out = sol.solve(P.METHOD_RCHFSI, torch.as_tensor(X0).cuda(), 24, 20, *b, tol=1e-8, max_iter=60)
        assert out["converged"], (store, out["history"])
        np.testing.assert_allclose(out["evals"][:24], ev[:24], rtol=1e-8)
        assert out["resnorm"][:24].max() <= 1e-8
        sol.close()
    sol = P.Rchfsi(As, Bs, dinv, block_N=32, apply_prec="fp32", store_prec="fp64")
    out = sol.solve(P.METHOD_CHFSI, torch.as_tensor(X0).cuda(), 24, 20, *b, tol=1e-8, max_iter=30)
    assert not out["converged"] and out["history"][-1] > 1e-8    # FP32 ChFSI floors
    sol.close()


def test_csr_fused_step_matches_oracle_within_fp32_error():
    """One filter in FP32-apply mode is the oracle's filter up to FP32 rounding of the products
    (Thm 3.4: error proportional to the residual), far below the FP32 error of ChFSI."""
    torch = _torch()
    import paper_2503_22652_b200 as P
    prob = workloads.config3_sparse_laplacian(n=10, n_wanted=20, block=24, degree=15, seed=4)
    solver, (A, B, Dinv), X, ritz, G = _setup(prob, 24, 6, apply_prec="fp32")
    ev = np.linalg.eigvalsh(A.apply(np.eye(prob["m"])))
    b = (ev[0] - 1e-2, ev[24], 12.0)
    Yo = orc.filter_rchfsi(A.apply, Dinv.apply, X, ritz, G, 15, *b)
    Xd = torch.as_tensor(X).cuda()
    solver.filter(P.METHOD_RCHFSI, Xd, torch.as_tensor(ritz).cuda(), torch.as_tensor(G).cuda(), 15, *b)
    assert rel_fro(Xd.cpu().numpy(), Yo) < 1e-5
    solver.close()


def test_filter_host_entry_point_equals_device_entry_point():
    torch = _torch()
    import paper_2503_22652_b200 as P
    prob = small_dense_generalized(150, seed=2)
    solver, (A, B, Dinv), X, ritz, G = _setup(prob, 8, 3)
    ev, top = _bounds(prob, A, B)
    b = (ev[0] - 1e-3, ev[8], top * 1.01)
    Xd = torch.as_tensor(X).cuda()
    solver.filter(P.METHOD_RCHFSI, Xd, torch.as_tensor(ritz).cuda(), torch.as_tensor(G).cuda(), 7, *b)
    Xh = X.copy()
    solver.filter_host(P.METHOD_RCHFSI, Xh, ritz, G, 7, *b)
    np.testing.assert_array_equal(Xh, Xd.cpu().numpy())
    solver.close()


@pytest.mark.parametrize("kind,apply_prec,store", [("fe", "bf16", "fp32"), ("fe", "tf32", "fp64"), ("csr", "fp32", "fp64"),
                                                   ("dense", "fp64", "fp64")])
def test_filter_host_column_chunks_equal_the_device_entry_point_bitwise(monkeypatch, kind, apply_prec, store):
    """rchfsi_filter_host cuts the block into column chunks (three streams: upload chunk i+1, filter chunk i, download
    chunk i-1); the columns are independent through the whole filter, so the result must be
    bit for bit the device entry point's.  RCHFSI_HOST_CHUNK=128 forces three chunks (128 + 128 + 8 columns)."""
    torch = _torch()
    import paper_2503_22652_b200 as P
    monkeypatch.setenv("RCHFSI_HOST_CHUNK", "128")
    N, p = 264, 6
    if kind == "fe":
        prob = workloads.fe_problem(2, q=3, seed=51)
        lam_max = workloads.fe.fe_lam_max_bound(prob["A_cells"], prob["B_cell"]) * 1.01
    elif kind == "csr":
        prob = workloads.config3_sparse_laplacian(n=9, n_wanted=10, block=N, degree=p, seed=6)
        lam_max = 12.0
    else:
        prob = small_dense_generalized(300, seed=9)
        lam_max = 16.0
    solver, _, X, ritz, G = _setup(prob, N, 23, apply_prec=apply_prec, store_prec=store)
    b = (ritz[0] - 1.0, ritz[-1] + 1.0, lam_max)
    for method in (P.METHOD_RCHFSI, P.METHOD_CHFSI):
        Xd = torch.as_tensor(X).cuda()
        solver.filter(method, Xd, torch.as_tensor(ritz).cuda(), torch.as_tensor(G).cuda(), p, *b)
        Xh = torch.as_tensor(X.copy()).pin_memory()
        solver.filter_host(method, Xh, ritz, G, p, *b)
        np.testing.assert_array_equal(Xh.numpy(), Xd.cpu().numpy())
    with pytest.raises(TypeError):      # the binding validates host arrays (dtype / shape / contiguity)
        solver.filter_host(P.METHOD_RCHFSI, X.astype(np.float32), ritz, G, p, *b)
    solver.close()


def test_filter_host_takes_an_fp32_residual_block_with_g_input_f32():
    torch = _torch()
    import paper_2503_22652_b200 as P
    prob = workloads.fe_problem(2, q=3, seed=52)
    lam_max = workloads.fe.fe_lam_max_bound(prob["A_cells"], prob["B_cell"]) * 1.01
    N, p = 136, 5
    solver, _, X, ritz, G = _setup(prob, N, 24, apply_prec="bf16", store_prec="fp32", g_input_f32=True)
    b = (ritz[0] - 1.0, ritz[-1] + 1.0, lam_max)
    G32 = G.astype(np.float32)
    Xd = torch.as_tensor(X).cuda()
    solver.filter(P.METHOD_RCHFSI, Xd, torch.as_tensor(ritz).cuda(), torch.as_tensor(G32).cuda(), p, *b)
    Xh = X.copy()
    solver.filter_host(P.METHOD_RCHFSI, Xh, ritz, G32, p, *b)
    np.testing.assert_array_equal(Xh, Xd.cpu().numpy())
    with pytest.raises(TypeError):      # an FP64 host G would be misread as FP32
        solver.filter_host(P.METHOD_RCHFSI, Xh, ritz, G, p, *b)
    solver.close()


def test_fe_mesh_with_a_row_no_cell_touches_is_rejected_at_create():
    """A global row referenced by no cell has no first toucher in the coloured scatter (it would keep stale data):
    rchfsi_create returns EINVAL instead."""
    torch = _torch()
    import paper_2503_22652_b200 as P
    prob = dict(workloads.fe_problem(2, q=2, seed=3))
    prob["m"] = prob["m"] + 1                      # one extra, uncovered row
    prob["dinv"] = np.concatenate((prob["dinv"], [1.0]))
    As, Bs, dinv = P.upload_problem(prob)
    with pytest.raises(P.RchfsiError) as ei:
        P.Rchfsi(As, Bs, dinv, block_N=8)
    assert ei.value.status == P.EINVAL and "belongs to no cell" in str(ei.value)


def test_operator_changed_drops_the_reduced_precision_copies():
    """The filter keeps a reduced-precision copy of A with D^-1 folded in; after the caller rewrites A in place,
    rchfsi_operator_changed makes the next filter see the new operator."""
    torch = _torch()
    import paper_2503_22652_b200 as P
    prob = small_dense_generalized(256, seed=12)
    N, p = 16, 4
    A, B, Dinv = oracle_ops(prob)
    X0 = np.random.default_rng(1).standard_normal((prob["m"], N))
    ritz, X, AX, BX = orc.rayleigh_ritz(A.apply, B.apply, X0)
    G = orc.residual_block(AX, BX, ritz)
    As, Bs, dinv = P.upload_problem(prob)
    s = P.Rchfsi(As, Bs, dinv, block_N=N, apply_prec="tf32")
    b = (ritz[0] - 1.0, ritz[-1] + 1.0, 16.0)
    rd, Gd = torch.as_tensor(ritz).cuda(), torch.as_tensor(G).cuda()
    X1 = torch.as_tensor(X).cuda()
    s.filter(P.METHOD_RCHFSI, X1, rd, Gd, p, *b)
    As["A"].mul_(0.5)                               # the caller's operator evolves in place
    X2 = torch.as_tensor(X).cuda()
    s.filter(P.METHOD_RCHFSI, X2, rd, Gd, p, *b)    # stale copy: same result as before
    assert torch.equal(X1, X2)
    s.operator_changed()
    X3 = torch.as_tensor(X).cuda()
    s.filter(P.METHOD_RCHFSI, X3, rd, Gd, p, *b)
    Yo = orc.filter_rchfsi(orc.DenseOperator(0.5 * prob["A"]).apply, Dinv.apply, X, ritz, G, p, *b)
    XL = X * orc.lambda_recurrence(ritz, p, *b)[p][None, :]
    assert rel_fro(X3.cpu().numpy() - XL, Yo - XL) < 6e-3
    assert not torch.equal(X1, X3)
    s.close()


def test_caller_provided_workspace_single_buffer_and_exhaustion():
    """the caller (torch) allocates the workspace.  One uint8 tensor of rchfsi_workspace_bytes() bytes
    carries Rayleigh-Ritz, filter and solve; the plan is tight (most of it is used); a buffer that is too small makes
    the call fail with ENOMEM before X is touched.  (The library holds no cudaMalloc call; cuBLAS / cuSOLVER handles keep
    their own internal scratch.)"""
    torch = _torch()
    import paper_2503_22652_b200 as P
    prob = small_dense_generalized(500, seed=21)
    N, p = 24, 9
    A, B, Dinv = oracle_ops(prob)
    ev, top = _bounds(prob, A, B)
    b = (ev[0] - 1e-3, ev[N], top * 1.01)
    As, Bs, dinv = P.upload_problem(prob)
    uses = P.USE_FILTER | P.USE_RAYLEIGH_RITZ | P.USE_SOLVE
    need = P.Rchfsi.workspace_bytes(As, Bs, N, uses=uses, max_degree=p, apply_prec="tf32")
    ws = torch.empty(need, dtype=torch.uint8, device="cuda")
    s = P.Rchfsi(As, Bs, dinv, block_N=N, apply_prec="tf32", workspace=ws)
    X0 = np.random.default_rng(3).standard_normal((prob["m"], N))
    ritz, X, G, res = s.rayleigh_ritz(torch.as_tensor(X0).cuda())
    s.filter(P.METHOD_RCHFSI, X.clone(), ritz, G, p, *b)
    s.filter(P.METHOD_CHFSI, X.clone(), None, None, p, *b)
    out = s.solve(P.METHOD_RCHFSI, torch.as_tensor(X0).cuda(), 12, p, *b, tol=1e-8, max_iter=60)
    assert out["converged"]
    used = s.workspace_used()
    assert used <= need <= 1.5 * used + (16 << 20), (used, need)     # sufficient, and not a loose guess
    s.close()
    small = torch.empty(used // 3, dtype=torch.uint8, device="cuda")
    s = P.Rchfsi(As, Bs, dinv, block_N=N, apply_prec="tf32", workspace=small)
    Xd = torch.as_tensor(X0).cuda()
    with pytest.raises(P.RchfsiError) as ei:
        s.rayleigh_ritz(Xd)
    assert ei.value.status == P.ENOMEM and "workspace" in str(ei.value)
    np.testing.assert_array_equal(Xd.cpu().numpy(), X0)
    s.close()


def test_filter_rejects_bad_arguments_without_touching_X():
    torch = _torch()
    import paper_2503_22652_b200 as P
    prob = small_dense_generalized(64, seed=1)
    solver, _, X, ritz, G = _setup(prob, 4, 3)
    Xd = torch.as_tensor(X).cuda()
    rz, Gd = torch.as_tensor(ritz).cuda(), torch.as_tensor(G).cuda()
    for args in [(0, 0.0, 1.0, 2.0), (3, 1.0, 1.0, 2.0), (3, 0.0, 2.0, 2.0), (3, 0.0, float("nan"), 2.0)]:
        with pytest.raises(P.RchfsiError) as ei:
            solver.filter(P.METHOD_RCHFSI, Xd, rz, Gd, *args)
        assert ei.value.status == P.EINVAL
    with pytest.raises(P.RchfsiError):
        solver.filter(P.METHOD_RCHFSI, Xd, None, Gd, 3, 0.0, 1.0, 2.0)
    with pytest.raises(P.RchfsiError):
        solver.filter(7, Xd, rz, Gd, 3, 0.0, 1.0, 2.0)
    np.testing.assert_array_equal(Xd.cpu().numpy(), X)
    solver.close()


def test_noise_hook_matches_oracle_column_noise():
    """The library's counter-based generator and column scaling equal workloads.noise +
    oracle.ColumnNoise, so a noisy FP64 filter is reproduced to rounding."""
    torch = _torch()
    import paper_2503_22652_b200 as P
    prob = workloads.config1_dense_standard(m=256, n_wanted=10, block=12, degree=8, seed=3)
    solver, (A, B, Dinv), X, ritz, G = _setup(prob, 12, 4, noise_eps=1e-4, noise_seed=77)
    b = (prob["lam_min"], prob["lam_T"], prob["lam_max"])
    noisy = orc.ColumnNoise(A, 1e-4, lambda k, mm, nn: workloads.counter_gaussian(77, k, mm, nn))
    Yo = orc.filter_rchfsi(noisy.apply, Dinv.apply, X, ritz, G, 8, *b)
    Xd = torch.as_tensor(X).cuda()
    solver.filter(P.METHOD_RCHFSI, Xd, torch.as_tensor(ritz).cuda(), torch.as_tensor(G).cuda(), 8, *b)
    assert rel_fro(Xd.cpu().numpy(), Yo) <= 1e-9
    solver.close()


@pytest.mark.parametrize("apply_prec,tol", [("tf32", 6e-3), ("bf16", 3e-2)])
@pytest.mark.parametrize("m,N,p", [(600, 40, 3), (1000, 264, 4), (333, 16, 2)])
def test_dense_tensor_core_step_is_the_oracle_step_up_to_operand_rounding(apply_prec, tol, m, N, p):
    """tcgen05 path: the residual part D^-1 R_p of the filtered block (Y_p - X Lambda_p) equals the
    oracle's up to the operand rounding of p-1 <= 3 applies.  Tolerance: per apply the block is
    truncated to TF32 when it aliases the FP32 R_Y (2^-10) and the operator copy is rounded (2^-11),
    i.e. <= 1.5e-3 relative; BF16 2^-8 + 2^-9 = 5.9e-3; times 3 applies, rounded up: 6e-3 / 3e-2.
    Sizes: several 128-column and BN-row tiles, ragged K tail (m not a multiple of 32 / 64)."""
    torch = _torch()
    import paper_2503_22652_b200 as P
    prob = small_dense_generalized(m, seed=m + N)
    for store in ("fp64", "fp32"):
        solver, (A, B, Dinv), X, ritz, G = _setup(prob, N, 13, apply_prec=apply_prec, store_prec=store)
        ev, top = _bounds(prob, A, B)
        b = (ev[0] - 1e-3, ev[N], top * 1.01)
        Yo = orc.filter_rchfsi(A.apply, Dinv.apply, X, ritz, G, p, *b)
        XL = X * orc.lambda_recurrence(ritz, p, *b)[p][None, :]
        Xd = torch.as_tensor(X).cuda()
        solver.filter(P.METHOD_RCHFSI, Xd, torch.as_tensor(ritz).cuda(), torch.as_tensor(G).cuda(), p, *b)
        Yg = Xd.cpu().numpy()
        err = np.linalg.norm((Yg - XL) - (Yo - XL), axis=0) / np.linalg.norm(Yo - XL, axis=0)
        assert err.max() < tol, (store, err.max())
        assert err.max() > 1e-9, "suspiciously exact: the reduced-precision path did not run"
        # CHFSI through the same kernel (dinv applied to the output rows)
        Yc = orc.filter_chfsi(A.apply, Dinv.apply, X, p, *b)
        Xd = torch.as_tensor(X).cuda()
        solver.filter(P.METHOD_CHFSI, Xd, None, None, p, *b)
        assert rel_fro(Xd.cpu().numpy(), Yc) < tol
        solver.close()


@pytest.mark.parametrize("apply_prec,tol", [("tf32", 6e-3), ("bf16", 3e-2)])
@pytest.mark.parametrize("nc,q,N,p", [(2, 6, 136, 3), (3, 3, 16, 4), (3, 2, 264, 3)])
def test_fe_tensor_core_step_is_the_oracle_step_up_to_operand_rounding(apply_prec, tol, nc, q, N, p):
    """FE tcgen05 path (cp.async gather into the swizzled UMMA layout, coloured atomic-free scatter fused with the update):
    the residual part of the filtered block equals the oracle's up to operand rounding (tolerances
    as for the dense kernel).  q=6: 343 nodes per cell, two 176-wide accumulator halves, ragged K
    tail; q=2,3: single accumulator; N=136/264: a ragged second/third 128-column tile."""
    torch = _torch()
    import paper_2503_22652_b200 as P
    prob = workloads.fe_problem(nc, q=q, seed=nc * 10 + q)
    A, B, Dinv = oracle_ops(prob)
    lam_max = workloads.fe.fe_lam_max_bound(prob["A_cells"], prob["B_cell"]) * 1.01
    for store in ("fp64", "fp32"):
        solver, _, X, ritz, G = _setup(prob, N, 17, apply_prec=apply_prec, store_prec=store)
        b = (ritz[0] - 1.0, ritz[-1] + 1.0, lam_max)
        Yo = orc.filter_rchfsi(A.apply, Dinv.apply, X, ritz, G, p, *b)
        XL = X * orc.lambda_recurrence(ritz, p, *b)[p][None, :]
        Xd = torch.as_tensor(X).cuda()
        solver.filter(P.METHOD_RCHFSI, Xd, torch.as_tensor(ritz).cuda(), torch.as_tensor(G).cuda(), p, *b)
        Yg = Xd.cpu().numpy()
        err = np.linalg.norm((Yg - XL) - (Yo - XL), axis=0) / np.linalg.norm(Yo - XL, axis=0)
        assert err.max() < tol, (store, err.max())
        assert err.max() > 1e-9, "suspiciously exact: the reduced-precision path did not run"
        Yc = orc.filter_chfsi(A.apply, Dinv.apply, X, p, *b)
        Xd = torch.as_tensor(X).cuda()
        solver.filter(P.METHOD_CHFSI, Xd, None, None, p, *b)
        assert rel_fro(Xd.cpu().numpy(), Yc) < tol
        solver.close()


@pytest.mark.parametrize("apply_prec,store", [("bf16", "fp32"), ("bf16", "fp64"), ("tf32", "fp64")])
def test_fe_shadow_block_updated_in_place_equals_the_two_buffer_scheme(monkeypatch, apply_prec, store):
    """The FE step keeps ONE operand-precision shadow of R_Y and lets the last toucher of a node overwrite
    its row in place (filter.cu make_plan: every reader of that row belongs to an earlier colour launch or is
    the writer itself).  Bit-for-bit the same filtered block as the two-buffer scheme, over several steps,
    three column tiles (ragged last) and a 3^3-cell mesh where interior nodes have 8 touchers."""
    torch = _torch()
    import paper_2503_22652_b200 as P
    prob = workloads.fe_problem(3, q=3, seed=41)
    lam_max = workloads.fe.fe_lam_max_bound(prob["A_cells"], prob["B_cell"]) * 1.01
    N, p = 264, 7
    out = {}
    for pair in ("1", None):
        if pair:
            monkeypatch.setenv("RCHFSI_FE_SHADOW_PAIR", pair)
        else:
            monkeypatch.delenv("RCHFSI_FE_SHADOW_PAIR", raising=False)
        solver, _, X, ritz, G = _setup(prob, N, 29, apply_prec=apply_prec, store_prec=store)
        b = (ritz[0] - 1.0, ritz[-1] + 1.0, lam_max)
        for method in (P.METHOD_RCHFSI, P.METHOD_CHFSI):
            Xd = torch.as_tensor(X).cuda()
            solver.filter(method, Xd, torch.as_tensor(ritz).cuda(), torch.as_tensor(G).cuda(), p, *b)
            out[(pair, method)] = Xd.cpu().numpy()
        solver.close()
    for method in (P.METHOD_RCHFSI, P.METHOD_CHFSI):
        assert np.isfinite(out[(None, method)]).all()
        assert np.array_equal(out[("1", method)], out[(None, method)])


@pytest.mark.parametrize("kind", ["dense", "fe"])
@pytest.mark.parametrize("apply_prec", ["tf32", "bf16"])
def test_tensor_core_paths_edge_shapes(kind, apply_prec):
    """Degenerate shapes through the tcgen05 kernels: a problem smaller than one tile (m < 64 rows,
    N = 8 columns < 128), degree 1 (no step launch at all) and degree 2 (a single step)."""
    torch = _torch()
    import paper_2503_22652_b200 as P
    if kind == "dense":
        prob = small_dense_generalized(40, seed=5)
        lam_max_extra = None
    else:
        prob = workloads.fe_problem(1, q=2, seed=3)      # one cell, 27 nodes
        lam_max_extra = workloads.fe.fe_lam_max_bound(prob["A_cells"], prob["B_cell"]) * 1.01
    A, B, Dinv = oracle_ops(prob)
    N = 8
    tol = 6e-3 if apply_prec == "tf32" else 3e-2
    for p in (1, 2):
        solver, _, X, ritz, G = _setup(prob, N, 23, apply_prec=apply_prec)
        if lam_max_extra is None:
            ev, top = _bounds(prob, A, B)
            b = (ev[0] - 1e-3, ev[N], top * 1.01)
        else:
            b = (ritz[0] - 1.0, ritz[-1] + 1.0, lam_max_extra)
        Yo = orc.filter_rchfsi(A.apply, Dinv.apply, X, ritz, G, p, *b)
        Xd = torch.as_tensor(X).cuda()
        solver.filter(P.METHOD_RCHFSI, Xd, torch.as_tensor(ritz).cuda(), torch.as_tensor(G).cuda(), p, *b)
        err = rel_fro(Xd.cpu().numpy(), Yo)
        assert err < (1e-12 if p == 1 else tol), (p, err)      # degree 1 has no operator apply: exact
        solver.close()


def test_fe_tensor_core_solve_converges_to_exact_eigenvalues():
    """Whole R-ChFSI solve through the fused FE tcgen05 step (TF32 and BF16 operands, FP32 storage = the
    paper's scheme): eigenvalues <= 1e-8 relative, residual <= 1e-8 (north_star)."""
    torch = _torch()
    import scipy.linalg as sla
    import paper_2503_22652_b200 as P
    prob = workloads.fe_problem(2, q=4, seed=11)           # 8 cells, 125 nodes per cell, 729 nodes
    A, B, Dinv = oracle_ops(prob)
    m = prob["m"]
    ev = sla.eigh(A.apply(np.eye(m)), B.apply(np.eye(m)), eigvals_only=True)
    lam_max = workloads.fe.fe_lam_max_bound(prob["A_cells"], prob["B_cell"]) * 1.01
    N, nw, p = 16, 8, 30
    X0 = np.random.default_rng(2).standard_normal((m, N))
    As, Bs, dinv = P.upload_problem(prob)
    for apply_prec in ("tf32", "bf16"):
        sol = P.Rchfsi(As, Bs, dinv, block_N=N, apply_prec=apply_prec, store_prec="fp32", adaptive_bounds=True)
        out = sol.solve(P.METHOD_RCHFSI, torch.as_tensor(X0).cuda(), nw, p, ev[0] - 1.0, ev[N] , lam_max, tol=1e-8, max_iter=80)
        assert out["converged"], (apply_prec, out["history"][-5:])
        np.testing.assert_allclose(out["evals"][:nw], ev[:nw], rtol=1e-8, atol=1e-9)
        assert out["resnorm"][:nw].max() <= 1e-8
        sol.close()


@pytest.mark.parametrize("bn,ks", [(256, 4), (128, 2)])
def test_dense_split_k_cluster_fixup_matches_unsplit(monkeypatch, bn, ks):
    """The optional split-K variant of the dense tcgen05 step (K splits = one thread-block cluster, partial
    tiles summed over distributed shared memory in fixed rank order) gives the same filtered block as the
    default unsplit kernel up to FP32 summation order."""
    torch = _torch()
    import paper_2503_22652_b200 as P
    prob = small_dense_generalized(1000, seed=77)
    N, p = 264, 4
    outs = []
    for env in ({}, {"RCHFSI_DENSE_BN": str(bn), "RCHFSI_DENSE_KS": str(ks)}):
        for k in ("RCHFSI_DENSE_BN", "RCHFSI_DENSE_KS"):
            monkeypatch.delenv(k, raising=False)
        for k, v in env.items():
            monkeypatch.setenv(k, v)
        solver, (A, B, Dinv), X, ritz, G = _setup(prob, N, 13, apply_prec="tf32")
        ev, top = _bounds(prob, A, B)
        b = (ev[0] - 1e-3, ev[N], top * 1.01)
        Xd = torch.as_tensor(X).cuda()
        solver.filter(P.METHOD_RCHFSI, Xd, torch.as_tensor(ritz).cuda(), torch.as_tensor(G).cuda(), p, *b)
        outs.append(Xd.cpu().numpy())
        solver.close()
    # not bitwise: the FP32 partial sums are added in a different order, and the operand shadow of the next
    # step is rounded to TF32 (2^-11), so a last-bit difference can flip a rounding; bound: operand rounding
    assert rel_fro(outs[1], outs[0]) < 2.0 ** -11


@pytest.mark.parametrize("apply_prec", ["tf32", "bf16"])
@pytest.mark.parametrize("bn,ks", [(64, 1), (128, 2), (128, 1)])
def test_dense_operator_tile_multicast_is_bitwise_the_unicast_result(monkeypatch, apply_prec, bn, ks):
    """With an even number of column tiles the two column-tile CTAs of a cluster fetch half of the operator tile
    each and deliver it to both by TMA multicast (RCHFSI_DENSE_MC=0 switches it off).  Only the data path
    changes, not the arithmetic: the filtered blocks must be bitwise equal, with and without K splits, including
    a ragged last row tile (m = 1000) and a ragged second column tile (N = 200)."""
    torch = _torch()
    import paper_2503_22652_b200 as P
    prob = small_dense_generalized(1000, seed=78)
    N, p = 200, 4
    monkeypatch.setenv("RCHFSI_DENSE_BN", str(bn))
    monkeypatch.setenv("RCHFSI_DENSE_KS", str(ks))
    outs = []
    for mc in ("1", "0"):
        monkeypatch.setenv("RCHFSI_DENSE_MC", mc)
        solver, (A, B, Dinv), X, ritz, G = _setup(prob, N, 14, apply_prec=apply_prec)
        ev, top = _bounds(prob, A, B)
        b = (ev[0] - 1e-3, ev[N], top * 1.01)
        Xd = torch.as_tensor(X).cuda()
        solver.filter(P.METHOD_RCHFSI, Xd, torch.as_tensor(ritz).cuda(), torch.as_tensor(G).cuda(), p, *b)
        outs.append(Xd.cpu().numpy())
        solver.close()
    assert np.array_equal(outs[0], outs[1])
    # and it is the oracle's block up to operand rounding (same bound as the per-step test)
    Yo = orc.filter_rchfsi(A.apply, Dinv.apply, X, ritz, G, p, *b)
    assert rel_fro(outs[0], Yo) < (6e-3 if apply_prec == "tf32" else 3e-2)


@pytest.mark.parametrize("kind", ["fe", "csr"])
def test_fp32_residual_block_input_is_used_in_place(kind):
    """g_input_f32 (config-5 memory plan: an FP64 G does not fit): the filter with G given in FP32 equals the
    filter with the FP64 G up to the FP32 rounding of G, on the panel-layout FE path and a row-major path."""
    torch = _torch()
    import paper_2503_22652_b200 as P
    if kind == "fe":
        prob = workloads.fe_problem(2, q=3, seed=31)
        lam_max = workloads.fe.fe_lam_max_bound(prob["A_cells"], prob["B_cell"]) * 1.01
        N, prec = 136, "tf32"
    else:
        prob = workloads.config3_sparse_laplacian(n=9, n_wanted=10, block=12, degree=6, seed=5)
        lam_max, N, prec = 12.0, 12, "fp32"
    solver, (A, B, Dinv), X, ritz, G = _setup(prob, N, 19, apply_prec=prec, store_prec="fp32")
    b = (ritz[0] - 1.0, ritz[-1] + 1.0, lam_max)
    Xa = torch.as_tensor(X).cuda()
    solver.filter(P.METHOD_RCHFSI, Xa, torch.as_tensor(ritz).cuda(), torch.as_tensor(G).cuda(), 5, *b)
    solver.close()
    As, Bs, dinv = P.upload_problem(prob)
    s2 = P.Rchfsi(As, Bs, dinv, block_N=N, apply_prec=prec, store_prec="fp32", g_input_f32=True)
    Xb = torch.as_tensor(X).cuda()
    s2.filter(P.METHOD_RCHFSI, Xb, torch.as_tensor(ritz).cuda(), torch.as_tensor(G.astype(np.float32)).cuda(), 5, *b)
    assert rel_fro(Xb.cpu().numpy(), Xa.cpu().numpy()) < 1e-5
    with pytest.raises(P.RchfsiError):      # G is mandatory in this mode
        s2.filter(P.METHOD_RCHFSI, Xb, torch.as_tensor(ritz).cuda(), None, 5, *b)
    s2.close()
    with pytest.raises(P.RchfsiError):      # and needs FP32 storage
        P.Rchfsi(As, Bs, dinv, block_N=N, apply_prec=prec, store_prec="fp64", g_input_f32=True)


def test_chunked_rayleigh_ritz_matches_oracle_and_full_variant(monkeypatch):
    """Memory-light Rayleigh-Ritz (Gram matrices over column chunks, in-place row-panel rotation, residual block
    recomputed per chunk; SURVEY 8(d) config-5 plan), forced with RCHFSI_RR_CHUNKED=1: same Ritz values,
    B-orthonormal X, G and residual norms as the oracle."""
    torch = _torch()
    import paper_2503_22652_b200 as P
    monkeypatch.setenv("RCHFSI_RR_CHUNKED", "1")
    for prob, N in ((small_dense_generalized(300, seed=3), 24), (workloads.fe_problem(2, q=3, seed=8), 20)):
        A, B, Dinv = oracle_ops(prob)
        m = prob["m"]
        Y = np.random.default_rng(8).standard_normal((m, N)) * np.logspace(0, 4, N)[None, :]
        ritz_o, X_o, AX, BX = orc.rayleigh_ritz(A.apply, B.apply, Y)
        res_o = orc.residual_norms(AX, BX, ritz_o)
        As, Bs, dinv = P.upload_problem(prob)
        s = P.Rchfsi(As, Bs, dinv, block_N=N)
        ritz, X, G, res = s.rayleigh_ritz(torch.as_tensor(Y).cuda())
        np.testing.assert_allclose(ritz.cpu().numpy(), ritz_o, rtol=1e-10, atol=1e-10)
        Xg = X.cpu().numpy()
        BXg = B.apply(Xg)
        np.testing.assert_allclose(Xg.T @ BXg, np.eye(N), rtol=0, atol=1e-9)
        Gref = A.apply(Xg) - BXg * ritz.cpu().numpy()[None, :]
        np.testing.assert_allclose(G.cpu().numpy(), Gref, rtol=0, atol=1e-9 * max(1.0, np.abs(Gref).max()))
        np.testing.assert_allclose(res.cpu().numpy(), res_o, rtol=1e-5, atol=1e-9)
        s.close()


@pytest.mark.parametrize("apply_prec", ["tf32", "bf16"])
def test_memory_light_solve_keeps_fp32_residual_block(monkeypatch, apply_prec):
    """rchfsi_solve in the memory-light mode (chunked Rayleigh-Ritz + FP32 G read in place by the fused steps):
    still converges to the exact eigenvalues with residual <= 1e-8.  bf16 is the config-5 scheme as
    BASELINE.json states it: BF16 cell-GEMM operands through the one shadow block updated in place."""
    torch = _torch()
    import scipy.linalg as sla
    import paper_2503_22652_b200 as P
    monkeypatch.setenv("RCHFSI_RR_CHUNKED", "1")
    prob = workloads.fe_problem(2, q=4, seed=11)
    A, B, Dinv = oracle_ops(prob)
    m = prob["m"]
    ev = sla.eigh(A.apply(np.eye(m)), B.apply(np.eye(m)), eigvals_only=True)
    lam_max = workloads.fe.fe_lam_max_bound(prob["A_cells"], prob["B_cell"]) * 1.01
    N, nw, p = 16, 8, 30
    X0 = np.random.default_rng(2).standard_normal((m, N))
    As, Bs, dinv = P.upload_problem(prob)
    sol = P.Rchfsi(As, Bs, dinv, block_N=N, apply_prec=apply_prec, store_prec="fp32", adaptive_bounds=True)
    out = sol.solve(P.METHOD_RCHFSI, torch.as_tensor(X0).cuda(), nw, p, ev[0] - 1.0, ev[N], lam_max, tol=1e-8, max_iter=80)
    assert out["converged"], out["history"][-5:]
    np.testing.assert_allclose(out["evals"][:nw], ev[:nw], rtol=1e-8, atol=1e-9)
    assert out["resnorm"][:nw].max() <= 1e-8
    sol.close()


@pytest.mark.parametrize("i8", ["0", "1"])
def test_memory_light_solve_with_fp32_only_cells_borrows_the_filter_blocks(monkeypatch, i8):
    """configs[4] storage: FP32-only cell matrices, chunked Rayleigh-Ritz.  Inside rchfsi_solve the Rayleigh-Ritz parks
    an FP64 copy of the cell matrices (and, with the INT8 Gram products forced at this size, the transposed digit planes
    of Y) in the filter's blocks R_X / R_Y / shadow, which the next filter re-initialises.  Converges to the eigenvalues
    of the FP32-rounded operator (the operator the library was given), residual <= 1e-8."""
    torch = _torch()
    import scipy.linalg as sla
    import paper_2503_22652_b200 as P
    monkeypatch.setenv("RCHFSI_RR_CHUNKED", "1")
    monkeypatch.setenv("RCHFSI_RR_GRAM_I8", i8)
    monkeypatch.setenv("RCHFSI_RR_SPLIT", i8)
    # 27 cells of 64 nodes, m = 1000: the FP64 cell copy (885 KB) fits the 1 MB block R_Y of the FP64-storage filter
    prob = dict(workloads.fe_problem(3, q=3, seed=11))
    prob["A_cells"] = prob["A_cells"].astype(np.float32).astype(np.float64)
    A, B, Dinv = oracle_ops(prob)
    m = prob["m"]
    ev = sla.eigh(A.apply(np.eye(m)), B.apply(np.eye(m)), eigvals_only=True)
    lam_max = workloads.fe.fe_lam_max_bound(prob["A_cells"], prob["B_cell"]) * 1.01
    N, nw, p = 16, 8, 30
    assert prob["n_cells"] * prob["n_loc"] ** 2 * 8 <= m * 128 * 8
    X0 = np.random.default_rng(2).standard_normal((m, N))
    As, Bs, dinv = P.upload_problem(prob, fe_cells_f32_only=True)
    sol = P.Rchfsi(As, Bs, dinv, block_N=N, apply_prec="tf32", store_prec="fp64", adaptive_bounds=True)
    X = torch.as_tensor(X0).cuda()
    out = sol.solve(P.METHOD_RCHFSI, X, nw, p, ev[0] - 1.0, ev[N], lam_max, tol=1e-8, max_iter=80)
    assert out["converged"], out["history"][-5:]
    np.testing.assert_allclose(out["evals"][:nw], ev[:nw], rtol=1e-8, atol=1e-9)
    assert out["resnorm"][:nw].max() <= 1e-8
    # certified by the oracle's operators on the returned pairs
    Xh = X[:, :nw].cpu().numpy()
    BX = B.apply(Xh)
    assert np.linalg.norm(A.apply(Xh) - BX * out["evals"][:nw][None, :], axis=0).max() <= 1.01e-8
    assert np.abs(Xh.T @ BX - np.eye(nw)).max() <= 1e-9
    sol.close()


@pytest.mark.parametrize("f32_cells", [False, True])
@pytest.mark.parametrize("chunked", ["0", "1"])
def test_fe_rayleigh_ritz_batched_gemm_apply_equals_handwritten_apply(monkeypatch, f32_cells, chunked):
    """The Rayleigh-Ritz applies FE operators through gather -> batched DGEMM -> coloured scatter (fe_rr.cu);
    RCHFSI_RR_FE_SIMT=1 keeps the hand-written FP64 kernel.  Both must give the oracle's Ritz values, a
    B-orthonormal X and the exact residual block, with FP64 or FP32-only cell matrices (config-5 storage), in the
    full and in the chunked variant (lower-triangle Gram matrices in both)."""
    torch = _torch()
    import paper_2503_22652_b200 as P
    monkeypatch.setenv("RCHFSI_RR_CHUNKED", chunked)
    prob = dict(workloads.fe_problem(3, q=3, seed=5))
    if f32_cells:   # the operator IS the FP32-rounded one: give the oracle the same numbers
        prob["A_cells"] = prob["A_cells"].astype(np.float32).astype(np.float64)
    N = 28
    A, B, Dinv = oracle_ops(prob)
    m = prob["m"]
    Y = np.random.default_rng(21).standard_normal((m, N)) * np.logspace(0, 3, N)[None, :]
    ritz_o, X_o, AX, BX = orc.rayleigh_ritz(A.apply, B.apply, Y)
    res_o = orc.residual_norms(AX, BX, ritz_o)
    out = {}
    for simt in (False, True):
        if simt:
            monkeypatch.setenv("RCHFSI_RR_FE_SIMT", "1")
        else:
            monkeypatch.delenv("RCHFSI_RR_FE_SIMT", raising=False)
        As, Bs, dinv = P.upload_problem(prob, fe_cells_f32_only=f32_cells)
        s = P.Rchfsi(As, Bs, dinv, block_N=N)
        ritz, X, G, res = s.rayleigh_ritz(torch.as_tensor(Y).cuda())
        out[simt] = (ritz.cpu().numpy(), X.cpu().numpy(), G.cpu().numpy(), res.cpu().numpy())
        s.close()
        np.testing.assert_allclose(out[simt][0], ritz_o, rtol=1e-10, atol=1e-10)
        Xg = out[simt][1]
        BXg = B.apply(Xg)
        np.testing.assert_allclose(Xg.T @ BXg, np.eye(N), rtol=0, atol=1e-9)
        Gref = A.apply(Xg) - BXg * out[simt][0][None, :]
        np.testing.assert_allclose(out[simt][2], Gref, rtol=0, atol=1e-9 * max(1.0, np.abs(Gref).max()))
        np.testing.assert_allclose(out[simt][3], res_o, rtol=1e-5, atol=1e-9)
    np.testing.assert_allclose(out[False][0], out[True][0], rtol=1e-12, atol=1e-12)
