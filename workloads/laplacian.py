"""Sparse seeded problem: BASELINE.json configs[2] (3D 7-point finite-difference
Laplacian with Dirichlet boundaries plus a seeded diagonal potential), CSR."""
import numpy as np


def laplacian3d_csr(n, potential=None):
    """Unscaled 7-point stencil on an n^3 grid, Dirichlet by truncation
    (SURVEY.md S15): diagonal 6 (+ potential), six -1 neighbours.  Row index
    i = (ix*n + iy)*n + iz.  Returns (rowptr int64 [m+1], colind int32 [nnz],
    vals float64 [nnz]) with column indices ascending inside each row."""
    m = n * n * n
    idx = np.arange(m, dtype=np.int64)
    ix, iy, iz = idx // (n * n), (idx // n) % n, idx % n
    cols = np.full((m, 7), -1, dtype=np.int64)
    vals = np.zeros((m, 7))
    # ascending column order: -n^2, -n, -1, 0, +1, +n, +n^2
    for slot, (ok, off) in enumerate([(ix > 0, -n * n), (iy > 0, -n), (iz > 0, -1),
                                      (np.ones(m, bool), 0),
                                      (iz < n - 1, 1), (iy < n - 1, n), (ix < n - 1, n * n)]):
        cols[ok, slot] = idx[ok] + off
        vals[ok, slot] = 6.0 if off == 0 else -1.0
    if potential is not None:
        vals[:, 3] += potential
    mask = cols >= 0
    counts = mask.sum(axis=1)
    rowptr = np.zeros(m + 1, dtype=np.int64)
    np.cumsum(counts, out=rowptr[1:])
    return rowptr, cols[mask].astype(np.int32), vals[mask]


def laplacian3d_exact_eigs(n):
    """Textbook closed form for the potential-free stencil:
    lam_ijk = 4[sin^2(i pi/2(n+1)) + sin^2(j pi/2(n+1)) + sin^2(k pi/2(n+1))]."""
    s = 4.0 * np.sin(np.arange(1, n + 1) * np.pi / (2.0 * (n + 1))) ** 2
    return np.sort((s[:, None, None] + s[None, :, None] + s[None, None, :]).ravel())


def config3_sparse_laplacian(n=64, n_wanted=256, block=300, degree=30, seed=3,
                             with_potential=True):
    """BASELINE.json configs[2]: 64^3 grid (262,144 rows), potential V_i ~ U[-5,0]
    at a fixed seed, FP32-representable values.  Bounds: Gershgorin lam_max = 12;
    lam_T / lam_min are NOT known a priori (adaptive or supplied by the caller)."""
    m = n ** 3
    V = None
    if with_potential:
        V = np.random.default_rng(seed).uniform(-5.0, 0.0, m)
        V = V.astype(np.float32).astype(np.float64)   # single-rounded in FP32 (S15)
    rowptr, colind, vals = laplacian3d_csr(n, V)
    return dict(kind="csr", m=m, n_grid=n, rowptr=rowptr, colind=colind, vals=vals,
                potential=V, B=None, dinv=None, n_wanted=n_wanted, block=block,
                degree=degree, lam_max=12.0, lam_lower=-5.0, x0_seed=seed + 2000, tol=1e-8)
