"""Rotation X = Y E of the Rayleigh-Ritz on the INT8 tensor pipe (rr_i8.cu): the
digit-split product must be as good as the FP64 dgemm it replaces.  Checked against the oracle's Rayleigh-Ritz at the
tolerances of test_rayleigh_ritz_matches_oracle, against the dgemm path of the same library, and on blocks whose rows
span many orders of magnitude (the split is fixed-point relative to the ROW maximum)."""
import numpy as np
import pytest

from oracle import chfsi_oracle as orc
from tests.helpers import oracle_ops, small_dense_generalized

pytestmark = pytest.mark.gpu


def _rr(prob, Y, monkeypatch, split, chunked="0", rows=None, gram="0", prefilter=False, bn="128"):
    import torch
    import paper_2503_22652_b200 as P
    monkeypatch.setenv("RCHFSI_RR_I8_BN", bn)
    monkeypatch.setenv("RCHFSI_RR_SPLIT", split)
    monkeypatch.setenv("RCHFSI_RR_GRAM_I8", gram)
    monkeypatch.setenv("RCHFSI_RR_CHUNKED", chunked)
    if rows:
        monkeypatch.setenv("RCHFSI_RR_I8_ROWS", str(rows))
    else:
        monkeypatch.delenv("RCHFSI_RR_I8_ROWS", raising=False)
    As, Bs, dinv = P.upload_problem(prob)
    s = P.Rchfsi(As, Bs, dinv, block_N=Y.shape[1])
    if prefilter:   # the column-slab Gram products borrow the filter's blocks: they exist once a filter has run
        N = Y.shape[1]
        Xf = torch.as_tensor(Y / np.linalg.norm(Y, axis=0)).cuda()
        s.filter(P.METHOD_RCHFSI, Xf, torch.linspace(0.0, 1.0, N, dtype=torch.float64, device="cuda"),
                 torch.zeros_like(Xf), 2, -1.0, 2.0, 40.0)
    ritz, X, G, res = s.rayleigh_ritz(torch.as_tensor(Y).cuda())
    out = ritz.cpu().numpy(), X.cpu().numpy(), G.cpu().numpy(), res.cpu().numpy()
    launches = s.launch_count()
    s.close()
    return out + (launches,)


@pytest.mark.parametrize("bn", ["128", "64"])
@pytest.mark.parametrize("m,N,chunked,rows", [(700, 300, "0", None), (700, 300, "1", 256), (1000, 137, "0", 384),
                                              (333, 64, "1", None)])
def test_int8_rotation_matches_oracle_and_dgemm_path(monkeypatch, m, N, chunked, rows, bn):
    prob = small_dense_generalized(m, seed=3)
    A, B, _ = oracle_ops(prob)
    Y = np.random.default_rng(8).standard_normal((m, N)) * np.logspace(0, 6, N)[None, :]
    ritz_o, X_o, AX, BX = orc.rayleigh_ritz(A.apply, B.apply, Y)
    res_o = orc.residual_norms(AX, BX, ritz_o)
    ritz, X, G, res, _ = _rr(prob, Y, monkeypatch, "1", chunked, rows, bn=bn)
    ritz_d, X_d, G_d, res_d, _ = _rr(prob, Y, monkeypatch, "0", chunked)
    Bd = prob["B"]
    np.testing.assert_allclose(ritz, ritz_o, rtol=1e-11, atol=1e-12)
    np.testing.assert_allclose(np.abs(np.sum(X * (Bd @ X_o), axis=0)), 1.0, rtol=0, atol=1e-8)
    np.testing.assert_allclose(X.T @ Bd @ X, np.eye(N), rtol=0, atol=1e-10)
    np.testing.assert_allclose(res, res_o, rtol=1e-6, atol=1e-11)
    np.testing.assert_allclose(G, prob["A"] @ X - (Bd @ X) * ritz[None, :], rtol=0, atol=1e-10)
    # against the dgemm path of the same library (the column normalisation in front of the Gram products reduces with
    # atomics, so the two runs see eigenvector matrices that differ in the last bits: compare up to sign, S12)
    np.testing.assert_allclose(ritz, ritz_d, rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(np.abs(np.sum(X * (Bd @ X_d), axis=0)), 1.0, rtol=0, atol=1e-8)
    np.testing.assert_allclose(res, res_d, rtol=1e-6, atol=1e-11)


def _rotate(Y, E, monkeypatch, split, rows=None, bn="128"):
    """rchfsi_rotate on a handle of a throw-away operator (the rotation does not touch the operator)."""
    import torch
    import paper_2503_22652_b200 as P
    monkeypatch.setenv("RCHFSI_RR_I8_BN", bn)
    monkeypatch.setenv("RCHFSI_RR_SPLIT", split)
    if rows:
        monkeypatch.setenv("RCHFSI_RR_I8_ROWS", str(rows))
    else:
        monkeypatch.delenv("RCHFSI_RR_I8_ROWS", raising=False)
    m, N = Y.shape
    rp = torch.arange(m + 1, dtype=torch.int64, device="cuda")
    A = dict(kind="csr", rowptr=rp, colind=torch.arange(m, dtype=torch.int32, device="cuda"),
             vals=torch.ones(m, dtype=torch.float64, device="cuda"))
    s = P.Rchfsi(A, None, None, block_N=N)
    Yd = torch.as_tensor(Y).cuda()
    s.rotate(Yd, torch.as_tensor(np.ascontiguousarray(E.T)).cuda())
    out = Yd.cpu().numpy()
    s.close()
    return out


@pytest.mark.parametrize("m,N,rows,bn", [(900, 260, None, "128"), (1500, 129, 512, "128"), (2500, 2400, 1024, "128"),
                                         (130, 16, None, "128"), (900, 260, None, "64"), (2500, 2400, 1024, "64")])
def test_int8_rotation_error_is_at_the_fp64_level_for_badly_scaled_operands(monkeypatch, m, N, rows, bn):
    """Entries spanning 12 orders of magnitude inside a row of Y, rows of Y and columns of E differing by 2^+-100 in
    scale, an all-zero row: against a longdouble product (sampled rows) the INT8 result is within 8 sqrt(K) FP64 ulps of
    (row max of Y)(column max of E) per element -- the norm the fixed-point split is exact in; the dgemm path's own
    error in that norm is about a third of it (printed on failure).  A dropped digit pair would cost 256 x that."""
    rng = np.random.default_rng(12 + N)
    Y = rng.standard_normal((m, N)) * 10.0 ** rng.uniform(-12, 0, (m, N))
    Y *= 2.0 ** rng.integers(-100, 100, (m, 1))
    Y[5, :] = 0.0
    E = np.linalg.qr(rng.standard_normal((N, N)))[0] * 10.0 ** rng.uniform(-3, 0, (N, N))
    E *= 2.0 ** rng.integers(-100, 100, (1, N))
    X1 = _rotate(Y, E, monkeypatch, "1", rows, bn)
    X0 = _rotate(Y, E, monkeypatch, "0")
    rs = np.unique(np.concatenate(([0, 5, 127, 128, m - 1], rng.integers(0, m, 59))))
    ref = Y[rs].astype(np.longdouble) @ E.astype(np.longdouble)
    scale = (np.abs(Y[rs]).max(axis=1, keepdims=True) * np.abs(E).max(axis=0, keepdims=True)).astype(np.longdouble)
    scale[scale == 0] = 1.0
    e1 = float((np.abs(X1[rs] - ref) / scale).max()) * 2.0 ** 53
    e0 = float((np.abs(X0[rs] - ref) / scale).max()) * 2.0 ** 53
    assert e1 <= 8.0 * np.sqrt(N), (e1, e0)
    full = np.abs(Y).max(axis=1, keepdims=True) * np.abs(E).max(axis=0, keepdims=True)
    assert np.all(np.abs(X1 - X0) <= 1e-12 * full)                        # every element, against the dgemm path
    assert np.all(X1[5] == 0.0)
    # power-of-two row scaling commutes with the product exactly (row exponents)
    X2 = _rotate(Y * 2.0 ** 37, E, monkeypatch, "1", rows, bn)
    assert np.array_equal(X2, X1 * 2.0 ** 37)


def test_int8_rotation_propagates_non_finite_rows(monkeypatch):
    rng = np.random.default_rng(2)
    Y = rng.standard_normal((300, 64))
    Y[7, 3] = np.nan
    Y[9, 60] = np.inf
    E = np.linalg.qr(rng.standard_normal((64, 64)))[0]
    X = _rotate(Y, E, monkeypatch, "1")
    assert np.isnan(X[7]).all() and np.isnan(X[9]).all()
    ok = np.ones(300, bool)
    ok[[7, 9]] = False
    np.testing.assert_allclose(X[ok], Y[ok] @ E, rtol=0, atol=1e-13)


@pytest.mark.parametrize("bn", ["128", "64"])
@pytest.mark.parametrize("m,N,chunked,rows,generalized", [(700, 300, "0", None, True), (1000, 137, "0", 384, True),
                                                          (700, 300, "1", None, True), (900, 200, "1", None, False),
                                                          (640, 96, "0", 128, False)])
def test_int8_gram_products_match_oracle_and_dgemm_path(monkeypatch, m, N, chunked, rows, generalized, bn):
    """H_a = Y^T A Y and H_b = Y^T B Y (lower triangles) through transposed digit planes and K-split INT32 accumulators
    flushed into FP64: same Ritz values / vectors / residuals as the oracle at the tolerances of
    test_rayleigh_ritz_matches_oracle, full-block and column-slab variants, several row chunks, B = I included."""
    prob = small_dense_generalized(m, seed=4)
    if not generalized:
        prob = dict(prob, B=None, dinv=None)
    A, B, _ = oracle_ops(prob)
    Y = np.random.default_rng(9).standard_normal((m, N)) * np.logspace(0, 5, N)[None, :]
    ritz_o, X_o, AX, BX = orc.rayleigh_ritz(A.apply, B.apply, Y)
    res_o = orc.residual_norms(AX, BX, ritz_o)
    pre = chunked == "1"
    ritz, X, G, res, n1 = _rr(prob, Y, monkeypatch, "1", chunked, rows, gram="1", prefilter=pre, bn=bn)
    ritz_d, X_d, G_d, res_d, n0 = _rr(prob, Y, monkeypatch, "0", chunked, rows, gram="0", prefilter=pre)
    assert n1 != n0                                                    # the INT8 kernels really ran
    Bd = prob["B"] if prob.get("B") is not None else np.eye(m)
    np.testing.assert_allclose(ritz, ritz_o, rtol=1e-11, atol=1e-12)
    np.testing.assert_allclose(ritz, ritz_d, rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(np.abs(np.sum(X * (Bd @ X_o), axis=0)), 1.0, rtol=0, atol=1e-8)
    np.testing.assert_allclose(X.T @ Bd @ X, np.eye(N), rtol=0, atol=1e-10)
    np.testing.assert_allclose(res, res_o, rtol=1e-6, atol=1e-11)
    np.testing.assert_allclose(G, prob["A"] @ X - (Bd @ X) * ritz[None, :], rtol=0, atol=1e-10)
