"""Dense seeded problems: BASELINE.json configs[0], configs[1] and the paper's
controlled experiment family E1 (section 4.1.1)."""
import numpy as np


def haar_orthogonal(m, seed):
    """Random orthogonal Q = QR factor of an m x m N(0,1) matrix (PAPER.md:275:
    "QR factorization (via Householder reflections ...) of an m x m matrix whose
    entries are drawn i.i.d. from N(0,1) with a fixed random seed").  The sign fix
    R_ii > 0 makes Q Haar distributed; it does not change any spectrum."""
    rng = np.random.default_rng(seed)
    F = rng.standard_normal((m, m))
    Q, R = np.linalg.qr(F)
    Q = Q * np.sign(np.diag(R))[None, :]
    return Q


def _sym_gaussian(m, rng):
    """S = (F + F^T)/sqrt(2 m), F_ij ~ N(0,1): spectrum ~ [-2, 2]."""
    F = rng.standard_normal((m, m))
    return (F + F.T) / np.sqrt(2.0 * m)


def config1_dense_standard(m=1000, n_wanted=50, block=60, degree=20, seed=1):
    """BASELINE.json configs[0]: A = Q diag(lam) Q^T, lam_i ~ U[0,1] sorted with a
    gap of 0.01 inserted after the 50th value; B = I.  Bounds from the known
    spectrum as in SURVEY.md 8(d) C1: lam_T = lam_{N+1} (first eigenvalue outside
    the block), lam_min = lam_1 - 1e-3, lam_max = lam_m + 1e-2."""
    rng = np.random.default_rng(seed + 1000)
    lam = np.sort(rng.uniform(0.0, 1.0, m))
    lam[n_wanted:] += 0.01
    Q = haar_orthogonal(m, seed)
    A = (Q * lam[None, :]) @ Q.T
    A = 0.5 * (A + A.T)
    X0 = np.random.default_rng(seed + 2000).standard_normal((m, block))
    return dict(kind="dense", m=m, A=A, B=None, dinv=None, Q=Q, lam=lam,
                n_wanted=n_wanted, block=block, degree=degree,
                lam_min=lam[0] - 1e-3, lam_T=lam[block], lam_max=lam[-1] + 1e-2,
                X0=X0, noise_eps=1e-4, tol=1e-8)


def config2_dense_generalized(m=4000, n_wanted=200, block=240, degree=25, seed=2):
    """BASELINE.json configs[1]: A = S_A + diag(linspace(0,10)), B = I + 0.1 S_B,
    S symmetric Gaussian / sqrt(m), approximate inverse
    D^-1 = diag(B)^-1.  Spectral bounds are NOT computed here (they need an
    eigensolve; tests obtain them from a library eigensolver, the bench from
    Gershgorin-style norms)."""
    rng = np.random.default_rng(seed)
    A = _sym_gaussian(m, rng) + np.diag(np.linspace(0.0, 10.0, m))
    B = np.eye(m) + 0.1 * _sym_gaussian(m, rng)
    dinv = 1.0 / np.diag(B).copy()
    X0 = np.random.default_rng(seed + 2000).standard_normal((m, block))
    return dict(kind="dense", m=m, A=A, B=B, dinv=dinv, n_wanted=n_wanted,
                block=block, degree=degree, X0=X0, tol=1e-8)


def _e1_spectrum(m, n):
    """wanted lam_j = 1 + 3(j-1)/(n-1), j=1..n; unwanted
    lam_j = 5 + 0.2 (j-n-1), j=n+1..m  (lam_m ~ 202.8 for m=1000, n=10)."""
    lam = np.empty(m)
    lam[:n] = 1.0 + 3.0 * np.arange(n) / (n - 1)
    lam[n:] = 5.0 + 0.2 * np.arange(m - n)
    return lam


def _unit_sym_perturbation(m, seed):
    """E = (F + F^T)/2 normalised to ||E||_2 = 1."""
    F = np.random.default_rng(seed).standard_normal((m, m))
    E = 0.5 * (F + F.T)
    return E / np.linalg.norm(E, 2)


def e1_standard(eps, m=1000, n=10, degree=8, seed=7):
    """standard problem, filter uses A~ = A + eps E, RR uses A."""
    lam = _e1_spectrum(m, n)
    Q = haar_orthogonal(m, seed)
    A = (Q * lam[None, :]) @ Q.T
    A = 0.5 * (A + A.T)
    A_filter = A + eps * _unit_sym_perturbation(m, seed + 1) if eps > 0 else A
    X0 = np.random.default_rng(seed + 2).standard_normal((m, n))
    return dict(m=m, n=n, degree=degree, A=A, A_filter=A_filter, Q=Q, lam=lam,
                lam_min=lam[0] - 0.05, lam_T=0.5 * (lam[n - 1] + lam[n]),
                lam_max=lam[-1] + 0.1, X0=X0)


def e1_generalized(zeta, m=1000, n=10, degree=8, seed=7):
    """B = Q diag(b) Q^T with the SAME eigenbasis as A,
    b_j = 1 + 4(j-1)/(m-1); D^-1 = B^-1 + zeta E, ||E||_2 = 1; generalized
    eigenvalues lam_j / b_j.  Bounds: the numbers of PAPER.md:277 taken literally
    (lam_min = 0.95, lam_T = 4.5, lam_max = lam_m(A) + 0.1), the paper states them once
    for the whole of section 4.1; they enclose the generalized spectrum [1, 40.6] and
    lam(D^-1 A) too (reading S18)."""
    a = _e1_spectrum(m, n)
    b = 1.0 + 4.0 * np.arange(m) / (m - 1)
    Q = haar_orthogonal(m, seed)
    A = (Q * a[None, :]) @ Q.T
    A = 0.5 * (A + A.T)
    B = (Q * b[None, :]) @ Q.T
    B = 0.5 * (B + B.T)
    Binv = (Q * (1.0 / b)[None, :]) @ Q.T
    Binv = 0.5 * (Binv + Binv.T)
    Dinv = Binv + zeta * _unit_sym_perturbation(m, seed + 1) if zeta > 0 else Binv
    gen = a / b
    order = np.argsort(gen)
    gen_sorted = gen[order]
    X0 = np.random.default_rng(seed + 2).standard_normal((m, n))
    return dict(m=m, n=n, degree=degree, A=A, B=B, Binv=Binv, Dinv=Dinv, Q=Q,
                gen_eigs=gen_sorted, eig_order=order,
                lam_min=a[0] - 0.05, lam_T=0.5 * (a[n - 1] + a[n]), lam_max=a[-1] + 0.1,
                X0=X0)
