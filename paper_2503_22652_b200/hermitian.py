"""Complex Hermitian problems (k-point sampling) through the real symmetric embedding.

A complex Hermitian pencil  A x = lambda B x,  A = A_r + i A_i (A_r symmetric, A_i antisymmetric), B likewise,
is the real symmetric pencil of twice the size

    [ A_r  -A_i ] [x_r]            [ B_r  -B_i ] [x_r]
    [ A_i   A_r ] [x_i]  = lambda  [ B_i   B_r ] [x_i]

whose operator apply performs exactly the four real products of a complex matvec, so the library's real kernels
(tcgen05 dense step, fused CSR step, FP64 Rayleigh-Ritz) run unchanged: "the theoretical guarantees of section 3
hold without modification for the complex Hermitian setting".  Every eigenvalue of the complex pencil
appears TWICE in the embedding, with eigenvectors [x_r; x_i] and [-x_i; x_r] (x and i x): a real block of 2 n vectors
converges to n complex pairs.  This module only arranges data (index bookkeeping and sign flips); all arithmetic on
blocks stays in the library.  FE operators are not embedded: 2 x 343 local nodes exceed the 512-node limit of the
FE tensor-core step (next steps).
"""
import numpy as np


def embed_dense(A):
    """[[A_r, -A_i], [A_i, A_r]] for a complex Hermitian dense matrix (float64, symmetric)."""
    A = np.asarray(A)
    Ar, Ai = np.ascontiguousarray(A.real, dtype=np.float64), np.ascontiguousarray(A.imag, dtype=np.float64)
    return np.block([[Ar, -Ai], [Ai, Ar]])


def embed_csr(rowptr, colind, vals, m):
    """CSR triplet of the embedding of a complex Hermitian CSR matrix (rows 0..m-1: [A_r, -A_i], rows m..2m-1:
    [A_i, A_r]); zero imaginary parts are kept so that the pattern is the same for every row block."""
    rowptr = np.asarray(rowptr, dtype=np.int64)
    colind = np.asarray(colind, dtype=np.int64)
    vals = np.asarray(vals)
    nnz_row = np.diff(rowptr)
    rp = np.zeros(2 * m + 1, dtype=np.int64)
    rp[1:m + 1] = np.cumsum(2 * nnz_row)
    rp[m + 1:] = rp[m] + np.cumsum(2 * nnz_row)
    ci = np.empty(4 * len(vals), dtype=np.int32)
    va = np.empty(4 * len(vals), dtype=np.float64)
    for i in range(m):
        t0, t1 = rowptr[i], rowptr[i + 1]
        n = t1 - t0
        o = rp[i]
        ci[o:o + n], va[o:o + n] = colind[t0:t1], vals[t0:t1].real
        ci[o + n:o + 2 * n], va[o + n:o + 2 * n] = colind[t0:t1] + m, -vals[t0:t1].imag
        o = rp[m + i]
        ci[o:o + n], va[o:o + n] = colind[t0:t1], vals[t0:t1].imag
        ci[o + n:o + 2 * n], va[o + n:o + 2 * n] = colind[t0:t1] + m, vals[t0:t1].real
    return rp, ci, va


def embed_problem(prob):
    """Workload dict of the embedded real problem for a dense or CSR complex Hermitian workload dict
    (keys as in `workloads`: kind, m, A / (rowptr, colind, vals), optional B (dense), dinv)."""
    m = prob["m"]
    out = dict(prob)
    out["m"] = 2 * m
    if prob["kind"] == "dense":
        out["A"] = embed_dense(prob["A"])
        out["B"] = embed_dense(prob["B"]) if prob.get("B") is not None else None
    elif prob["kind"] == "csr":
        out["rowptr"], out["colind"], out["vals"] = embed_csr(prob["rowptr"], prob["colind"], prob["vals"], m)
    else:
        raise ValueError("only dense and CSR operators are embedded")
    if prob.get("dinv") is not None:
        out["dinv"] = np.concatenate([prob["dinv"], prob["dinv"]])
    return out


def embed_block(X):
    """Complex block [m][n] -> real block [2m][2n]: columns [x_r; x_i] and their partners [-x_i; x_r] (= i x)."""
    X = np.asarray(X)
    top = np.concatenate([X.real, -X.imag], axis=1)
    bot = np.concatenate([X.imag, X.real], axis=1)
    return np.ascontiguousarray(np.concatenate([top, bot], axis=0), dtype=np.float64)


def complex_pairs(evals, X, n):
    """From the 2n lowest real pairs of the embedding (doubled spectrum) the n complex pairs: eigenvalue k is the mean
    of the k-th doublet; its eigenvector is x_r + i x_i of the first vector of the doublet."""
    evals = np.asarray(evals)
    m = X.shape[0] // 2
    lam = 0.5 * (evals[0:2 * n:2] + evals[1:2 * n:2])
    V = X[:m, 0:2 * n:2] + 1j * X[m:, 0:2 * n:2]
    return lam, V
