"""FE-style seeded generalized problem: BASELINE.json configs[3], configs[4].

Uniform hexahedral cells (h = 1), degree-q Lagrange elements on Gauss-Lobatto-
Legendre (GLL) points, all nodes are DoFs (natural boundary conditions), cell
matrices A_c = 0.5 K_c + M_c[V] with a smooth seeded potential V (sum of
Gaussians), consistent Gauss-quadrature mass B_c (identical for every cell),
approximate inverse D^-1 = inverse of the assembled GLL (lumped) diagonal mass.
Constants are the reading SURVEY.md S16.  They stand in for the DFT-FE matrices
of PAPER.md:327-339 (Table 1), which are not available.

Local node l = (ix*(q+1) + iy)*(q+1) + iz; global node
g = ((cx*q+ix)*ng + (cy*q+iy))*ng + (cz*q+iz), ng = q*nc + 1; cell index
c = (cx*nc + cy)*nc + cz.
"""
import numpy as np
from numpy.polynomial import legendre as npleg


def gll_nodes_weights(q):
    """q+1 Gauss-Lobatto-Legendre points on [-1,1] and weights 2/(q(q+1)P_q(x)^2)."""
    Pq = npleg.Legendre.basis(q)
    interior = np.sort(np.real(Pq.deriv().roots()))
    x = np.concatenate(([-1.0], interior, [1.0]))
    for _ in range(3):                      # Newton polish on (1-x^2) P_q'(x)
        xi = x[1:-1]
        d1 = Pq.deriv()(xi)
        d2 = Pq.deriv(2)(xi)
        x[1:-1] = xi - d1 / d2
    w = 2.0 / (q * (q + 1) * Pq(x) ** 2)
    return x, w


def _lagrange_at(nodes, pts):
    """L[i, a] = a-th Lagrange polynomial on `nodes` at pts[i]; dL its derivative."""
    n = len(nodes)
    L = np.ones((len(pts), n))
    dL = np.zeros((len(pts), n))
    for a in range(n):
        others = [b for b in range(n) if b != a]
        den = np.prod([nodes[a] - nodes[b] for b in others])
        for i, xp in enumerate(pts):
            L[i, a] = np.prod([xp - nodes[b] for b in others]) / den
            s = 0.0
            for b in others:
                s += np.prod([xp - nodes[d] for d in others if d != b])
            dL[i, a] = s / den
    return L, dL


def fe_reference_matrices(q=6, n_quad=8):
    """1D reference matrices on [-1,1] with n_quad-point Gauss-Legendre (exact for
    2q <= 2 n_quad - 1): M1 = int phi_a phi_b, K1 = int phi_a' phi_b'.  Also the
    basis at the quadrature points (Phi, n_quad x (q+1)), quadrature (xq, wq) and
    the GLL rule (xg, wg)."""
    xg, wg = gll_nodes_weights(q)
    xq, wq = npleg.leggauss(n_quad)
    Phi, dPhi = _lagrange_at(xg, xq)
    M1 = Phi.T @ (wq[:, None] * Phi)
    K1 = dPhi.T @ (wq[:, None] * dPhi)
    return dict(xg=xg, wg=wg, xq=xq, wq=wq, Phi=Phi, dPhi=dPhi, M1=M1, K1=K1)


def _kron3(a, b, c):
    return np.kron(np.kron(a, b), c)


def fe_connectivity(nc, q=6):
    nl = q + 1
    ng = q * nc + 1
    cx, cy, cz = np.meshgrid(np.arange(nc), np.arange(nc), np.arange(nc), indexing="ij")
    ix, iy, iz = np.meshgrid(np.arange(nl), np.arange(nl), np.arange(nl), indexing="ij")
    gx = cx.reshape(-1, 1) * q + ix.reshape(1, -1)
    gy = cy.reshape(-1, 1) * q + iy.reshape(1, -1)
    gz = cz.reshape(-1, 1) * q + iz.reshape(1, -1)
    return ((gx * ng + gy) * ng + gz).astype(np.int32)


def fe_potential_centres(nc, seed, n_gauss=8):
    L = float(nc)
    return np.random.default_rng(seed).uniform(0.2 * L, 0.8 * L, (n_gauss, 3))


def fe_potential(x, y, z, centres, depth=-10.0, width=1.5):
    """V(x) = sum_g depth * exp(-|x - x_g|^2 / (2 width^2))."""
    V = np.zeros(np.broadcast(x, y, z).shape)
    for cg in centres:
        V += depth * np.exp(-((x - cg[0]) ** 2 + (y - cg[1]) ** 2 + (z - cg[2]) ** 2)
                            / (2.0 * width * width))
    return V


def fe_problem(nc, q=6, seed=4, n_quad=8, h=1.0, cell_dtype=np.float64, cell_chunk=64):
    """Build the FE generalized problem on nc^3 cells.

    Returns dict with: m, n_cells, n_loc, conn [n_cells][n_loc] int32,
    A_cells [n_cells][n_loc][n_loc] (cell_dtype), B_cell [n_loc][n_loc] float64 (one
    matrix shared by every cell), dinv [m] = 1 / assembled GLL weights, lam_max_bound
    (= max_c lam_max(A_c, B_c) >= lam_max(A, B)), centres.
    """
    ref = fe_reference_matrices(q, n_quad)
    nl = q + 1
    n_loc = nl ** 3
    ng = q * nc + 1
    m = ng ** 3
    s = h / 2.0
    M1, K1 = ref["M1"], ref["K1"]
    # K_c = (h/2)(K1 x M1 x M1 + M1 x K1 x M1 + M1 x M1 x K1); B_c = (h/2)^3 M1 x M1 x M1
    K_c = s * (_kron3(K1, M1, M1) + _kron3(M1, K1, M1) + _kron3(M1, M1, K1))
    B_c = s ** 3 * _kron3(M1, M1, M1)
    Phi3 = _kron3(ref["Phi"], ref["Phi"], ref["Phi"])           # [n_quad^3][n_loc]
    w3 = s ** 3 * _kron3(ref["wq"][:, None], ref["wq"][:, None], ref["wq"][:, None]).ravel()
    xq = ref["xq"]
    qx, qy, qz = np.meshgrid(xq, xq, xq, indexing="ij")
    qx, qy, qz = qx.ravel(), qy.ravel(), qz.ravel()
    centres = fe_potential_centres(nc, seed)
    conn = fe_connectivity(nc, q)
    n_cells = nc ** 3
    A_cells = np.empty((n_cells, n_loc, n_loc), dtype=cell_dtype)
    cidx = np.arange(n_cells)
    ccx, ccy, ccz = cidx // (nc * nc), (cidx // nc) % nc, cidx % nc
    for c0 in range(0, n_cells, cell_chunk):
        c1 = min(n_cells, c0 + cell_chunk)
        X = (ccx[c0:c1, None] + 0.5) * h + s * qx[None, :]
        Y = (ccy[c0:c1, None] + 0.5) * h + s * qy[None, :]
        Z = (ccz[c0:c1, None] + 0.5) * h + s * qz[None, :]
        wV = w3[None, :] * fe_potential(X, Y, Z, centres)        # [chunk][nq3]
        MV = np.matmul(Phi3.T[None, :, :] * wV[:, None, :], Phi3[None, :, :])
        Ac = 0.5 * K_c[None, :, :] + MV
        A_cells[c0:c1] = (0.5 * (Ac + Ac.transpose(0, 2, 1))).astype(cell_dtype)
    # lumped (GLL) diagonal mass, assembled
    wg3 = s ** 3 * _kron3(ref["wg"][:, None], ref["wg"][:, None], ref["wg"][:, None]).ravel()
    D = np.zeros(m)
    np.add.at(D, conn.ravel(), np.tile(wg3, n_cells))
    return dict(kind="fe", m=m, n_cells=n_cells, n_loc=n_loc, nc=nc, q=q, conn=conn,
                A_cells=A_cells, B_cell=B_c, K_cell=K_c, dinv=1.0 / D, lumped=D,
                centres=centres, ref=ref)


def fe_lam_max_bound(A_cells, B_cell, sample=None):
    """max over (a sample of) cells of lam_max(A_c, B_c): an upper bound on
    lam_max(A, B).  Library eigensolver; test/bench helper only."""
    import scipy.linalg as sla
    cells = range(A_cells.shape[0]) if sample is None else sample
    best = -np.inf
    for c in cells:
        best = max(best, sla.eigh(np.asarray(A_cells[c], dtype=np.float64), B_cell,
                                  eigvals_only=True, subset_by_index=[B_cell.shape[0] - 1,
                                                                      B_cell.shape[0] - 1])[0])
    return best


def config4_fe(seed=4, **kw):
    """BASELINE.json configs[3]: 16^3 cells, degree 6 (343 nodes/cell, 97^3 nodes);
    1000 lowest eigenpairs, block of 1200, degree 40."""
    p = fe_problem(16, 6, seed, **kw)
    p.update(n_wanted=1000, block=1200, degree=40, tol=1e-8, x0_seed=seed + 2000)
    return p


def config5_fe(seed=5, **kw):
    """BASELINE.json configs[4]: 24^3 cells, degree 6 (145^3 nodes); 2048 eigenpairs,
    block of 2400, degree 50."""
    kw.setdefault("cell_dtype", np.float32)
    p = fe_problem(24, 6, seed, **kw)
    p.update(n_wanted=2048, block=2400, degree=50, tol=1e-8, x0_seed=seed + 2000)
    return p
