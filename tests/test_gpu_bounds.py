"""rchfsi_estimate_bounds ("parameterised by estimates lam_min, lam_max, lam_T") and the
degree guard against the oracle's restatement and a dense eigensolver."""
import numpy as np
import pytest
import scipy.linalg as sla

import workloads
from oracle import chfsi_oracle as orc
from tests.helpers import oracle_ops, small_dense_generalized

pytestmark = pytest.mark.gpu


def _dense(op, m):
    return op.apply(np.eye(m))


@pytest.mark.parametrize("f32_cells", [False, True])
def test_fe_bounds_match_the_oracle_estimators_and_bracket_the_spectrum(f32_cells):
    import paper_2503_22652_b200 as P
    prob = dict(workloads.fe_problem(3, q=3, seed=6))
    if f32_cells:
        prob["A_cells"] = prob["A_cells"].astype(np.float32).astype(np.float64)
    A, B, Dinv = oracle_ops(prob)
    m, d = prob["m"], prob["dinv"]
    As, Bs, dinv = P.upload_problem(prob, fe_cells_f32_only=f32_cells)
    s = P.Rchfsi(As, Bs, dinv, block_N=8)
    seed, k = 11, 16
    b = s.estimate_bounds(lanczos_steps=k, fe_cell_stride=1, seed=seed)
    s.close()
    ref = orc.lanczos_upper_bound(A.apply, d, workloads.counter_gaussian(seed, 0, m, 1)[:, 0], k)
    assert b["lanczos_steps"] == k
    assert abs(b["lanczos_theta_max"] - ref["theta_max"]) <= 1e-8 * abs(ref["theta_max"])
    assert abs(b["lanczos_theta_min"] - ref["theta_min"]) <= 1e-8 * abs(ref["theta_max"])
    assert abs(b["lanczos_max"] - ref["upper"]) <= 1e-7 * abs(ref["upper"])
    Ad, Bd = _dense(A, m), _dense(B, m)
    # FE: the library sums |A_c| cell by cell before assembling (sum_c |a| >= |sum_c a|): still a bound, a bit looser
    r = np.zeros(m)
    for c in range(prob["n_cells"]):
        r[prob["conn"][c]] += np.abs(prob["A_cells"][c]).sum(axis=1)
    assert abs(b["gershgorin_max"] - np.max(d * r)) <= 1e-11 * b["gershgorin_max"]
    assert b["gershgorin_max"] >= orc.gershgorin_upper(Ad, d) * (1 - 1e-12)
    cw = orc.fe_cellwise_upper(prob["A_cells"], prob["B_cell"])
    assert abs(b["fe_cellwise_max"] - cw) <= 1e-9 * cw
    sq = np.sqrt(d)
    top_d = np.linalg.eigvalsh(sq[:, None] * Ad * sq[None, :])[-1]
    top_g = sla.eigh(Ad, Bd, eigvals_only=True)[-1]
    assert b["lam_max"] >= max(top_d, top_g) and b["lam_max"] <= 1.3 * max(top_d, top_g)
    assert b["gershgorin_max"] >= top_d


def test_csr_and_dense_bounds():
    import paper_2503_22652_b200 as P
    prob = workloads.config3_sparse_laplacian(n=10, n_wanted=10, block=12, degree=10, seed=2)
    A, _, _ = oracle_ops(prob)
    As, Bs, dinv = P.upload_problem(prob)
    s = P.Rchfsi(As, Bs, dinv, block_N=12)
    b = s.estimate_bounds(lanczos_steps=30, seed=3)
    s.close()
    Ad = _dense(A, prob["m"])
    ev = np.linalg.eigvalsh(Ad)
    assert abs(b["gershgorin_max"] - orc.gershgorin_upper(Ad)) <= 1e-12 * b["gershgorin_max"]
    assert np.isnan(b["fe_cellwise_max"])
    assert ev[-1] <= b["lam_max"] <= 12.0 + 1e-9          # never above the rigorous infinity-norm bound (here 12)
    assert b["lanczos_theta_min"] >= ev[0] - 1e-9 and b["lanczos_theta_max"] <= ev[-1] + 1e-9
    prob = small_dense_generalized(300, seed=5)
    A, B, Dinv = oracle_ops(prob)
    As, Bs, dinv = P.upload_problem(prob)
    s = P.Rchfsi(As, Bs, dinv, block_N=8)
    b = s.estimate_bounds(lanczos_steps=40, seed=1)
    with pytest.raises(P.RchfsiError):
        s.estimate_bounds(lanczos_steps=1)
    s.close()
    sq = np.sqrt(prob["dinv"])
    top = np.linalg.eigvalsh(sq[:, None] * prob["A"] * sq[None, :])[-1]
    assert top <= b["lam_max"] <= 1.15 * top
    assert abs(b["gershgorin_max"] - orc.gershgorin_upper(prob["A"], prob["dinv"])) <= 1e-12 * b["gershgorin_max"]


def test_solve_converges_with_library_estimated_bounds_only():
    """rchfsi_solve on the small FE pencil with lam_max from rchfsi_estimate_bounds and lam_min / lam_T from the
    Ritz values (adaptive_bounds): no spectral information from the caller."""
    import torch
    import paper_2503_22652_b200 as P
    prob = workloads.fe_problem(2, q=4, seed=13)
    A, B, Dinv = oracle_ops(prob)
    m = prob["m"]
    ev = sla.eigh(_dense(A, m), _dense(B, m), eigvals_only=True)
    N, nw, p = 16, 8, 30
    As, Bs, dinv = P.upload_problem(prob)
    s = P.Rchfsi(As, Bs, dinv, block_N=N, apply_prec="tf32", store_prec="fp32", adaptive_bounds=True)
    b = s.estimate_bounds(lanczos_steps=20, fe_cell_stride=1, seed=2)
    X0 = np.random.default_rng(4).standard_normal((m, N))
    out = s.solve(P.METHOD_RCHFSI, torch.as_tensor(X0).cuda(), nw, p, -1e6, -1e6 + 1.0, b["lam_max"], tol=1e-8, max_iter=80)
    s.close()
    assert out["converged"], out["history"][-5:]
    np.testing.assert_allclose(out["evals"][:nw], ev[:nw], rtol=1e-8, atol=1e-9)


def test_degree_guard_for_reduced_precision():
    """PAPER.md:347-359, footnote 5: FP32 / TF32 R-ChFSI is not stable at p = 100, 120: refused unless forced."""
    import torch
    import paper_2503_22652_b200 as P
    prob = small_dense_generalized(128, seed=3)
    As, Bs, dinv = P.upload_problem(prob)
    X = torch.as_tensor(np.random.default_rng(0).standard_normal((128, 8))).cuda()
    ritz = torch.linspace(-1.0, 0.0, 8, dtype=torch.float64).cuda()
    G = torch.zeros_like(X)
    s = P.Rchfsi(As, Bs, dinv, block_N=8, apply_prec="tf32")
    with pytest.raises(P.RchfsiError) as ei:
        s.filter(P.METHOD_RCHFSI, X.clone(), ritz, G, 100, -2.0, 0.5, 16.0)
    assert ei.value.status == P.EINVAL and "allow_high_degree" in str(ei.value)
    s.filter(P.METHOD_RCHFSI, X.clone(), ritz, G, 99, -2.0, 0.5, 16.0)
    s.close()
    for opts in (dict(apply_prec="tf32", allow_high_degree=True), dict(apply_prec="fp64")):
        s = P.Rchfsi(As, Bs, dinv, block_N=8, **opts)
        s.filter(P.METHOD_RCHFSI, X.clone(), ritz, G, 100, -2.0, 0.5, 16.0)
        s.close()
