"""FP64 CPU oracle for ChFSI and R-ChFSI (arxiv 2503.22652).

THIS IS TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl
reference`` legs may import it.  It shares no code with the CUDA library in
``paper_2503_22652_b200/`` and imports nothing from it; the only shared modules
are the seeded input generators in ``workloads/``.

Everything is plain numpy in float64, written in the paper's order and notation
so that it can be checked against PAPER.md by eye:

  cheb_scalars        Alg. 2 / Alg. 3 first line
  cheb_coefficients   a_k, b_k, c_k of eq. (7)
  filter_chfsi        Algorithm 2 / eq. (2), eq. (7)
  filter_rchfsi       Algorithm 3 / eqs. (11)-(13)
  rayleigh_ritz       Step 2-3 of Algorithm 1
                      (Y^dagger = conjugate transpose: complex Hermitian pencils of PAPER.md:373-401 included)
  residual_norms      r_j = ||A x_j - eps_j B x_j||_2
  solve               Algorithm 1 (do-while reading S1)
  tan_max_angle       Definition 2.1
  lanczos_upper_bound estimate of lam_max ("estimates lam_min, lam_max, lam_T"):
                      k-step Lanczos on D^-1/2 A D^-1/2, theta_max + its residual beta_k |s_k|
  gershgorin_upper    max_i d_i sum_j |a_ij| >= lam_max(D^-1 A)   (rigorous)
  fe_cellwise_upper   max_c lam_max(A_c, B_c) >= lam_max(A, B)     (rigorous; SURVEY reading S7)

Operators are objects with ``apply(V) -> A V`` on an [m][N] float64 block:
DenseOperator (a matmul), CsrOperator (library SpMM of the CSR triplet),
FeOperator (gather / cell matrix product / scatter-add),
ScaledIdentity.  Approximate inverses: DiagonalInverse (PAPER.md:325 mass lumping),
DenseInverse (D^-1 = B^-1 + zeta E of PAPER.md:283).  ColumnNoise wraps an
operator with the per-matvec noise model (reading S11 in DESIGN.md).

Readings of silent / ambiguous points (S1..S16) are listed in DESIGN.md.
Pins: tests/test_oracle_pins.py.  Unpinned by design: bitwise iterates of
reduced-precision runs and iteration counts ("parity unpinned" for those only;
the criteria there are eigenvalues and residuals).
"""
import numpy as np
import scipy.linalg as sla


# --------------------------------------------------------------------------- operators
class DenseOperator:
    def __init__(self, A):
        A = np.asarray(A)
        self.A = A.astype(np.complex128 if np.iscomplexobj(A) else np.float64)
        self.m = self.A.shape[0]

    def apply(self, V):
        return self.A @ V


class ScaledIdentity:
    """B = I (standard problem) or D = I."""

    def __init__(self, m, s=1.0):
        self.m, self.s = m, s

    def apply(self, V):
        return self.s * V


class CsrOperator:
    """(A V)_i = sum_{t in [rowptr_i, rowptr_{i+1})} vals_t V_{colind_t}.  The
    sparse-times-dense product is scipy.sparse's library SpMM (a library primitive
    used as one step); tests pin it against the row-by-row definition above."""

    def __init__(self, rowptr, colind, vals, m):
        import scipy.sparse as sp
        self.m = m
        self.M = sp.csr_matrix((np.asarray(vals, dtype=np.float64),
                                np.asarray(colind, dtype=np.int64),
                                np.asarray(rowptr, dtype=np.int64)), shape=(m, m))

    def apply(self, V):
        return np.asarray(self.M @ V)


class FeOperator:
    """A V = sum_c P_c^T A_c P_c V: for each cell gather the n_loc node rows, multiply
    by the cell matrix, scatter-add into the global rows (Remark 4.1).
    ``cell_mats`` is [n_cells][n_loc][n_loc], or one [n_loc][n_loc] matrix shared by
    every cell."""

    def __init__(self, cell_mats, conn, m):
        self.cell_mats = cell_mats
        self.conn = np.asarray(conn, dtype=np.int64)
        self.m = m
        self.shared = (np.ndim(cell_mats) == 2)

    def apply(self, V):
        out = np.zeros((self.m, V.shape[1]))
        for c in range(self.conn.shape[0]):
            Ac = self.cell_mats if self.shared else self.cell_mats[c]
            rows = self.conn[c]
            # rows of one cell are distinct, so fancy-index += is a true scatter-add
            out[rows] += np.asarray(Ac, dtype=np.float64) @ V[rows]
        return out


class DiagonalInverse:
    """D^-1 = diag(dinv): lumped / diagonal approximate inverse."""

    def __init__(self, dinv):
        self.dinv = np.asarray(dinv, dtype=np.float64)

    def apply(self, V):
        return self.dinv[:, None] * V


class DenseInverse:
    """D^-1 given as a dense matrix (controlled experiment)."""

    def __init__(self, Dinv):
        self.Dinv = np.asarray(Dinv, dtype=np.float64)

    def apply(self, V):
        return self.Dinv @ V


class ColumnNoise:
    """Inexact product A (x) V, per-matvec model (reading S11):
    T_j <- T_j + eps ||T_j||_2 g_j / ||g_j||_2 for every column j, with g drawn by
    the caller-supplied ``gauss(apply_index, m, n)`` (an input, see workloads.noise)."""

    def __init__(self, op, eps, gauss):
        self.op, self.eps, self.gauss = op, eps, gauss
        self.m = op.m
        self.count = 0

    def apply(self, V):
        T = self.op.apply(V)
        g = self.gauss(self.count, T.shape[0], T.shape[1])
        self.count += 1
        tn = np.sqrt(np.sum(T * T, axis=0))
        gn = np.sqrt(np.sum(g * g, axis=0))
        return T + (self.eps * tn / gn)[None, :] * g


def operators_from_workload(prob):
    """(A, B, Dinv) operator objects for a dict made by the `workloads` generators."""
    kind = prob["kind"]
    m = prob["m"]
    if kind == "dense":
        A = DenseOperator(prob["A"])
        B = DenseOperator(prob["B"]) if prob.get("B") is not None else ScaledIdentity(m)
    elif kind == "csr":
        A = CsrOperator(prob["rowptr"], prob["colind"], prob["vals"], m)
        B = ScaledIdentity(m)
    elif kind == "fe":
        A = FeOperator(prob["A_cells"], prob["conn"], m)
        B = FeOperator(prob["B_cell"], prob["conn"], m)
    else:
        raise ValueError(kind)
    Dinv = DiagonalInverse(prob["dinv"]) if prob.get("dinv") is not None else ScaledIdentity(m)
    return A, B, Dinv


# --------------------------------------------------------------------------- scalars
def cheb_scalars(lam_min, lam_T, lam_max):
    """e, c, sigma_1, gamma (first line of Alg. 2 and Alg. 3)."""
    e = (lam_max - lam_T) / 2.0
    c = (lam_max + lam_T) / 2.0
    sigma1 = e / (lam_min - c)
    gamma = 2.0 / sigma1
    return e, c, sigma1, gamma


def cheb_coefficients(p, lam_min, lam_T, lam_max):
    """[(a_k, b_k, c_k)] for k = 1..p-1 with sigma_{k+1} = 1/(gamma - sigma_k),
    a_k = 2 sigma_{k+1}/e, b_k = -2 sigma_{k+1} c/e, c_k = -sigma_k sigma_{k+1}
    (PAPER.md:53, 174-177).  Returned with the sigma sequence sigma_1..sigma_p."""
    e, c, sigma1, gamma = cheb_scalars(lam_min, lam_T, lam_max)
    sig = [sigma1]
    coef = []
    for _ in range(2, p + 1):
        s2 = 1.0 / (gamma - sig[-1])
        coef.append((2.0 * s2 / e, -2.0 * s2 * c / e, -sig[-1] * s2))
        sig.append(s2)
    return coef, sig


# --------------------------------------------------------------------------- Algorithm 2
def filter_chfsi(apply_A, apply_Dinv, X, p, lam_min, lam_T, lam_max):
    """Algorithm 2 with H V := D^-1 (A (x) V)  (eq. (7))."""
    e, c, sigma, gamma = cheb_scalars(lam_min, lam_T, lam_max)
    sigma1 = sigma

    def H(V):
        return apply_Dinv(apply_A(V))

    Xk = X.copy()
    Y = (sigma1 / e) * (H(X) - c * X)
    for _k in range(2, p + 1):
        sigma2 = 1.0 / (gamma - sigma)
        Xn = (2.0 * sigma2 / e) * H(Y) - (2.0 * sigma2 / e) * c * Y - sigma * sigma2 * Xk
        Xk, Y = Y, Xn                      # swap(X, Y)
        sigma = sigma2
    return Y


# --------------------------------------------------------------------------- Algorithm 3
def filter_rchfsi(apply_A, apply_Dinv, X, ritz, G, p, lam_min, lam_T, lam_max):
    """Algorithm 3.  ``ritz`` = eps_1..eps_N (diagonal of
    Lambda^(i)), ``G`` = A X - B X Lambda (the paper's temporary "Y"; exact A and B,
    reading S5).  Returns Y_p = D^-1 R_Y + X Lambda_Y."""
    e, c, sigma, gamma = cheb_scalars(lam_min, lam_T, lam_max)
    sigma1 = sigma
    ritz = np.asarray(ritz, dtype=np.float64)
    RX = np.zeros_like(G)
    RY = (sigma1 / e) * G
    LX = np.ones_like(ritz)
    LY = (sigma1 / e) * (ritz - c)
    for _k in range(2, p + 1):
        sigma2 = 1.0 / (gamma - sigma)
        a = 2.0 * sigma2 / e
        RXn = a * apply_A(apply_Dinv(RY)) - a * c * RY - sigma * sigma2 * RX + a * G * LY[None, :]
        LXn = a * LY * ritz - a * c * LY - sigma * sigma2 * LX
        RX, RY = RY, RXn                   # swap(R_X, R_Y)
        LX, LY = LY, LXn                   # swap(Lambda_X, Lambda_Y)
        sigma = sigma2
    return apply_Dinv(RY) + X * LY[None, :]


def lambda_recurrence(ritz, p, lam_min, lam_T, lam_max):
    """Lambda_k = C_k(Lambda), k = 0..p, by eq. (12); rows k."""
    e, c, sigma, gamma = cheb_scalars(lam_min, lam_T, lam_max)
    ritz = np.asarray(ritz, dtype=np.float64)
    table = [np.ones_like(ritz), (sigma / e) * (ritz - c)]
    for _k in range(2, p + 1):
        sigma2 = 1.0 / (gamma - sigma)
        a = 2.0 * sigma2 / e
        table.append(a * table[-1] * ritz - a * c * table[-1] - sigma * sigma2 * table[-2])
        sigma = sigma2
    return np.array(table[:p + 1])


# --------------------------------------------------------------------------- Rayleigh-Ritz
def rayleigh_ritz(apply_A, apply_B, Y, normalize_columns=True):
    """Steps 2-3 of Algorithm 1 on a non-orthogonal basis Y:
    solve (Y^T A Y) E = (Y^T B Y) E Lambda with E^T (Y^T B Y) E = I, eigenvalues
    ascending, X = Y E.  Columns of Y are first scaled to unit 2-norm (reading S6;
    it changes neither the subspace nor the Ritz pairs).  Returns (ritz, X, AX, BX)."""
    # "Y^dagger" of PAPER.md:55 is the conjugate transpose: complex Hermitian problems go through
    # the same lines; for real blocks conj() is the identity
    if normalize_columns:
        Y = Y / np.sqrt(np.sum(np.abs(Y) ** 2, axis=0))[None, :]
    AY = apply_A(Y)
    BY = apply_B(Y)
    Ha = Y.conj().T @ AY
    Hb = Y.conj().T @ BY
    Ha = 0.5 * (Ha + Ha.conj().T)
    Hb = 0.5 * (Hb + Hb.conj().T)
    ritz, E = sla.eigh(Ha, Hb)             # LAPACK dsygv-type: E^T Hb E = I, ascending
    return ritz, Y @ E, AY @ E, BY @ E


def residual_block(AX, BX, ritz):
    """G = A X - B X Lambda."""
    return AX - BX * np.asarray(ritz)[None, :]


def residual_norms(AX, BX, ritz):
    """r_j = ||A x_j - eps_j B x_j||_2, absolute (reading S8)."""
    G = residual_block(AX, BX, ritz)
    return np.sqrt(np.sum(np.abs(G) ** 2, axis=0))


# --------------------------------------------------------------------------- Algorithm 1
def solve(A_exact, B_exact, A_filter, Dinv, X0, n_wanted, p, lam_min, lam_T, lam_max,
          tol, max_iter, method="rchfsi", adaptive_bounds=False, early_stop=True,
          callback=None):
    """Algorithm 1 with the filter of Algorithm 2 ("chfsi") or
    Algorithm 3 ("rchfsi").  A_exact / B_exact are used in Rayleigh-Ritz and
    residuals, A_filter (possibly inexact) and Dinv only inside the filter
    (PAPER.md:253, 279).  Readings: S1 do-while, S2 one RR on X0 before the loop,
    S3 block N >= n_wanted with the test on the n_wanted lowest pairs, S7 optional
    adaptive lam_T / lam_min from the Ritz values.
    Returns dict(evals, X, resnorm, iters, history=[max wanted residual per iter])."""
    ritz, X, AX, BX = rayleigh_ritz(A_exact.apply, B_exact.apply, X0)
    history = []
    it = 0
    for it in range(1, max_iter + 1):
        if adaptive_bounds:
            lam_T, lam_min = float(ritz[-1]), float(ritz[0])
        if method == "rchfsi":
            G = residual_block(AX, BX, ritz)
            Y = filter_rchfsi(A_filter.apply, Dinv.apply, X, ritz, G, p, lam_min, lam_T, lam_max)
        elif method == "chfsi":
            Y = filter_chfsi(A_filter.apply, Dinv.apply, X, p, lam_min, lam_T, lam_max)
        else:
            raise ValueError(method)
        ritz, X, AX, BX = rayleigh_ritz(A_exact.apply, B_exact.apply, Y)
        r = residual_norms(AX, BX, ritz)
        history.append(float(np.max(r[:n_wanted])))
        if callback is not None:
            callback(it, ritz, X, r)
        if early_stop and history[-1] < tol:
            break
    return dict(evals=ritz, X=X, resnorm=r, iters=it, history=history)


# --------------------------------------------------------------------------- spectral bounds
def lanczos_upper_bound(apply_A, dinv, v0, k):
    """The filter is "parameterised by estimates lam_min, lam_max, lam_T" and
    lam_max must bound lam(D^-1 A) (the operator the recurrence applies, eq. (7) / Alg. 3).
    k-step Lanczos (no reorthogonalisation) on the symmetric S = D^-1/2 A D^-1/2, which has
    the spectrum of D^-1 A, from the start vector v0:
        v_1 = v0/||v0||;  w = S v_j - beta_{j-1} v_{j-1};  alpha_j = w.v_j;
        w -= alpha_j v_j;  beta_j = ||w||;  v_{j+1} = w / beta_j.
    (theta, s) = eigenpairs of tridiag(alpha, beta).  Every Ritz value lies inside the
    spectrum and the residual norm of the Ritz pair (theta_max, V s) is beta_k |s_k| (s_k =
    last component of s): an eigenvalue lies within that distance of theta_max, and
    `upper` = theta_max + beta_k |s_k| is the usual safeguarded ESTIMATE of lam_max (not a
    theorem: callers add a margin, the CUDA library 1 %); `upper_loose` = theta_max + beta_k.
    Returns dict(theta_min, theta_max, beta_k, s_k, upper, upper_loose, steps)."""
    from scipy.linalg import eigh_tridiagonal
    ds = np.sqrt(np.asarray(dinv, dtype=np.float64)) if dinv is not None else None

    def S(v):
        t = v if ds is None else ds * v
        t = apply_A(t[:, None])[:, 0]
        return t if ds is None else ds * t

    v = np.asarray(v0, dtype=np.float64).copy()
    v /= np.linalg.norm(v)
    v_prev = np.zeros_like(v)
    alpha, beta = [], []
    b = 0.0
    for _j in range(k):
        w = S(v) - b * v_prev
        a = float(w @ v)
        w = w - a * v
        b = float(np.linalg.norm(w))
        alpha.append(a)
        beta.append(b)
        if b <= 1e-300:
            break
        v_prev, v = v, w / b
    if len(alpha) > 1:
        theta, Sv = eigh_tridiagonal(np.array(alpha), np.array(beta[:-1]))
    else:
        theta, Sv = np.array(alpha), np.ones((1, 1))
    s_k = float(abs(Sv[-1, -1]))
    return dict(theta_min=float(theta[0]), theta_max=float(theta[-1]), beta_k=beta[-1], s_k=s_k,
                upper=float(theta[-1]) + beta[-1] * s_k, upper_loose=float(theta[-1]) + beta[-1],
                steps=len(alpha))


def gershgorin_upper(A_dense, dinv=None):
    """max_i d_i sum_j |a_ij| = ||D^-1 A||_inf >= every |eigenvalue| of D^-1 A."""
    r = np.sum(np.abs(np.asarray(A_dense, dtype=np.float64)), axis=1)
    return float(np.max(r if dinv is None else np.asarray(dinv) * r))


def fe_cellwise_upper(A_cells, B_cell, cells=None):
    """max over cells of lam_max(A_c, B_c) >= lam_max(A, B): x^T A x = sum_c x_c^T A_c x_c
    <= max_c lam_max(A_c, B_c) sum_c x_c^T B_c x_c (mediant inequality; SURVEY reading S7).
    `cells` = iterable of cell indices (all cells: rigorous; a sample: an estimate)."""
    cells = range(A_cells.shape[0]) if cells is None else cells
    n = B_cell.shape[0]
    return max(float(sla.eigh(np.asarray(A_cells[c], dtype=np.float64), B_cell, eigvals_only=True,
                              subset_by_index=[n - 1, n - 1])[0]) for c in cells)


# --------------------------------------------------------------------------- diagnostics
def tan_max_angle(U1, U2, Y):
    """Definition 2.1 with X = U1 (orthonormal, spans the wanted
    space) and X_perp = U2: tan angle = || U2^T Y (U1^T Y)^+ ||_2  (reading S13: never
    arccos of cosines)."""
    Z1 = U1.T @ Y
    Z2 = U2.T @ Y
    if np.linalg.matrix_rank(Z1) < Y.shape[1]:
        return np.inf
    return np.linalg.norm(Z2 @ np.linalg.pinv(Z1), 2)


def cheb_C(p, x, lam_min, lam_T, lam_max):
    """C_p(x) = T_p(L(x)) / T_p(L(lam_min)), L(x) = (x-c)/e, evaluated from the
    cos / cosh closed forms of T_p.  Used by pins only."""
    e, c, _, _ = cheb_scalars(lam_min, lam_T, lam_max)

    def T(t):
        t = np.asarray(t, dtype=np.float64)
        out = np.empty_like(t)
        inside = np.abs(t) <= 1.0
        out[inside] = np.cos(p * np.arccos(t[inside]))
        big = ~inside
        out[big] = np.sign(t[big]) ** p * np.cosh(p * np.arccosh(np.abs(t[big])))
        return out

    return T((np.asarray(x, dtype=np.float64) - c) / e) / T(np.array([(lam_min - c) / e]))[0]
