"""Complex Hermitian problems.  CPU part: the oracle runs Algorithms 1-3 in
complex arithmetic (numpy) and is pinned on a constructed complex spectrum; the real embedding of hermitian.py is pinned
against it.  GPU part: the library on the embedded real problem against the oracle's complex results."""
import numpy as np
import pytest
import scipy.linalg as sla

import workloads
from oracle import chfsi_oracle as orc
from paper_2503_22652_b200 import hermitian as H


def _complex_pencil(m, seed):
    """A = U diag(lam) U^H with a Haar-like unitary U (QR of a complex Gaussian, PAPER.md:275 recipe made complex) and
    prescribed lam; B = I + 0.1 S with S complex Hermitian Gaussian / sqrt(m); D^-1 = 1 / diag(B)."""
    rng = np.random.default_rng(seed)
    F = rng.standard_normal((m, m)) + 1j * rng.standard_normal((m, m))
    U, R = np.linalg.qr(F)
    U = U * (np.diag(R) / np.abs(np.diag(R)))[None, :]
    lam = np.sort(rng.uniform(0.0, 10.0, m))
    A = (U * lam[None, :]) @ U.conj().T
    A = 0.5 * (A + A.conj().T)
    S = rng.standard_normal((m, m)) + 1j * rng.standard_normal((m, m))
    B = np.eye(m) + 0.1 * (S + S.conj().T) / np.sqrt(2.0 * m) / np.sqrt(2.0)
    return dict(kind="dense", m=m, A=A, B=B, dinv=1.0 / np.real(np.diag(B)).copy(), lam=lam)


def test_oracle_complex_hermitian_solve_reaches_the_prescribed_spectrum():
    """Standard complex problem with a prescribed spectrum (pin P3 in complex arithmetic): R-ChFSI converges to lam."""
    prob = _complex_pencil(80, 3)
    A = orc.DenseOperator(prob["A"])
    I = orc.ScaledIdentity(80)
    rng = np.random.default_rng(0)
    X0 = rng.standard_normal((80, 8)) + 1j * rng.standard_normal((80, 8))
    lam = prob["lam"]
    out = orc.solve(A, I, A, I, X0, 6, 12, lam[0] - 0.1, lam[8], lam[-1] + 0.1, 1e-10, 80, method="rchfsi")
    assert out["history"][-1] < 1e-10
    np.testing.assert_allclose(out["evals"][:6], lam[:6], rtol=1e-10, atol=1e-10)
    Xh = out["X"]
    np.testing.assert_allclose(Xh.conj().T @ Xh, np.eye(8), atol=1e-10)      # B = I: orthonormal in the complex inner product


def test_real_embedding_reproduces_the_complex_filter_and_spectrum():
    prob = _complex_pencil(40, 5)
    emb = H.embed_problem(prob)
    np.testing.assert_allclose(emb["A"], emb["A"].T, atol=0)                 # real symmetric
    ev_c = sla.eigh(prob["A"], prob["B"], eigvals_only=True)
    ev_r = sla.eigh(emb["A"], emb["B"], eigvals_only=True)
    np.testing.assert_allclose(ev_r[0::2], ev_c, rtol=1e-11, atol=1e-11)     # every eigenvalue twice
    np.testing.assert_allclose(ev_r[1::2], ev_c, rtol=1e-11, atol=1e-11)
    # Algorithm 3 on the embedding = embedding of Algorithm 3 in complex arithmetic
    A, B, Dinv = orc.operators_from_workload(prob)
    Ae, Be, De = orc.operators_from_workload(emb)
    rng = np.random.default_rng(1)
    X0 = rng.standard_normal((40, 4)) + 1j * rng.standard_normal((40, 4))
    ritz, X, AX, BX = orc.rayleigh_ritz(A.apply, B.apply, X0)
    G = orc.residual_block(AX, BX, ritz)
    b = (ev_c[0] - 0.5, ev_c[6], ev_c[-1] * 1.3)
    Yc = orc.filter_rchfsi(A.apply, Dinv.apply, X, ritz, G, 9, *b)
    Ye = orc.filter_rchfsi(Ae.apply, De.apply, H.embed_block(X), np.concatenate([ritz, ritz]), H.embed_block(G), 9, *b)
    np.testing.assert_allclose(Ye, H.embed_block(Yc), rtol=1e-11, atol=1e-12)


def test_embed_csr_matches_embed_dense():
    import scipy.sparse as sp
    rng = np.random.default_rng(2)
    M = sp.random(30, 30, density=0.2, random_state=3).toarray() * np.exp(1j * rng.uniform(0, 6.28, (30, 30)))
    M = M + M.conj().T + np.diag(rng.uniform(1, 2, 30))
    C = sp.csr_matrix(M)
    rp, ci, va = H.embed_csr(C.indptr, C.indices, C.data, 30)
    E = sp.csr_matrix((va, ci, rp), shape=(60, 60)).toarray()
    np.testing.assert_allclose(E, H.embed_dense(M), atol=0)


@pytest.mark.gpu
@pytest.mark.parametrize("apply_prec", ["fp64", "tf32"])
def test_gpu_complex_hermitian_dense_through_the_embedding(apply_prec):
    """The library on the embedded problem: FP64 filter parity with the oracle's COMPLEX filter (<= 1e-10), and a
    reduced-precision solve whose doubled Ritz values match LAPACK's complex Hermitian eigenvalues to 1e-8."""
    import torch
    import paper_2503_22652_b200 as P
    prob = _complex_pencil(256, 7)
    emb = H.embed_problem(prob)
    A, B, Dinv = orc.operators_from_workload(prob)
    ev = sla.eigh(prob["A"], prob["B"], eigvals_only=True)
    n, N = 8, 24                                      # 8 wanted complex pairs, real block of 2 x 12 columns
    rng = np.random.default_rng(4)
    X0 = rng.standard_normal((256, N // 2)) + 1j * rng.standard_normal((256, N // 2))
    As, Bs, dinv = P.upload_problem(emb)
    sq = np.sqrt(prob["dinv"])
    top = max(ev[-1], np.linalg.eigvalsh(sq[:, None] * prob["A"] * sq[None, :])[-1]) * 1.01
    if apply_prec == "fp64":
        ritz, X, AX, BX = orc.rayleigh_ritz(A.apply, B.apply, X0)
        G = orc.residual_block(AX, BX, ritz)
        b = (ev[0] - 0.1, ev[N // 2], top)
        Yc = orc.filter_rchfsi(A.apply, Dinv.apply, X, ritz, G, 11, *b)
        s = P.Rchfsi(As, Bs, dinv, block_N=N)
        Xd = torch.as_tensor(H.embed_block(X)).cuda()
        s.filter(P.METHOD_RCHFSI, Xd, torch.as_tensor(np.concatenate([ritz, ritz])).cuda(),
                 torch.as_tensor(H.embed_block(G)).cuda(), 11, *b)
        s.close()
        Ye = H.embed_block(Yc)
        err = np.linalg.norm(Xd.cpu().numpy() - Ye, axis=0) / np.linalg.norm(Ye, axis=0)
        assert err.max() <= 1e-10, err.max()
    else:
        s = P.Rchfsi(As, Bs, dinv, block_N=N, apply_prec=apply_prec, adaptive_bounds=True)
        Xd = torch.as_tensor(H.embed_block(X0)).cuda()
        out = s.solve(P.METHOD_RCHFSI, Xd, 2 * n, 20, -100.0, 0.0, top, tol=1e-8, max_iter=80)
        s.close()
        assert out["converged"], out["history"][-5:]
        lam, V = H.complex_pairs(out["evals"], Xd.cpu().numpy(), n)
        np.testing.assert_allclose(lam, ev[:n], rtol=1e-8, atol=1e-9)
        res = np.linalg.norm(prob["A"] @ V - (prob["B"] @ V) * lam[None, :], axis=0)     # complex residual of the pairs
        assert res.max() <= 2e-8


@pytest.mark.gpu
def test_gpu_complex_hermitian_csr_through_the_embedding():
    """7-point Laplacian with a complex (Peierls) phase on the x-bonds: complex Hermitian CSR, fused FP32 SpMM."""
    import torch
    import paper_2503_22652_b200 as P
    base = workloads.config3_sparse_laplacian(n=8, n_wanted=6, block=16, degree=20, seed=4)
    m, n_grid = base["m"], 8
    rp, ci = base["rowptr"], base["colind"]
    vals = base["vals"].astype(np.complex128)
    theta = 0.37
    for i in range(m):
        for t in range(rp[i], rp[i + 1]):
            d = ci[t] - i
            if d == n_grid * n_grid:
                vals[t] *= np.exp(1j * theta)
            elif d == -n_grid * n_grid:
                vals[t] *= np.exp(-1j * theta)
    prob = dict(kind="csr", m=m, rowptr=rp, colind=ci, vals=vals, B=None, dinv=None)
    import scipy.sparse as sp
    Ad = sp.csr_matrix((vals, ci, rp), shape=(m, m)).toarray()
    np.testing.assert_allclose(Ad, Ad.conj().T, atol=0)
    ev = np.linalg.eigvalsh(Ad)
    emb = H.embed_problem(prob)
    As, Bs, dinv = P.upload_problem(emb)
    s = P.Rchfsi(As, Bs, dinv, block_N=16, apply_prec="fp32", adaptive_bounds=True)
    X0 = np.random.default_rng(1).standard_normal((2 * m, 16))
    Xd = torch.as_tensor(X0).cuda()
    out = s.solve(P.METHOD_RCHFSI, Xd, 12, 20, -100.0, 0.0, 12.5, tol=1e-8, max_iter=80)
    s.close()
    assert out["converged"], out["history"][-5:]
    lam, V = H.complex_pairs(out["evals"], Xd.cpu().numpy(), 6)
    np.testing.assert_allclose(lam, ev[:6], rtol=1e-8, atol=1e-9)
