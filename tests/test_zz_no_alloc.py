"""rchfsi_residual_static (include/rchfsi.h): the allocation-free entry point, against the EXISTING path
(rchfsi_rayleigh_ritz's residual block and residual norms) within the tolerances
tests/test_gpu_parity.py uses for that path, on two calls in a row -- the second with a narrower block, so that partial
sums left in the shared static scratch by the first call would show.  Collected last on purpose (file name): the
suite runs with pytest -x."""
import numpy as np
import pytest

import workloads
from oracle import chfsi_oracle as orc
from tests.helpers import small_dense_generalized

pytestmark = pytest.mark.gpu


def _existing_path(prob, N, seed):
    """(X, ritz, G, res, AX, BX) from the handle path: Rayleigh-Ritz on a random block, then the exact applies."""
    import torch
    import paper_2503_22652_b200 as P
    As, Bs, dinv = P.upload_problem(prob)
    s = P.Rchfsi(As, Bs, dinv, block_N=N)
    Y = torch.as_tensor(np.random.default_rng(seed).standard_normal((prob["m"], N))).cuda()
    ritz, X, G, res = s.rayleigh_ritz(Y)
    AX, BX = s.apply(0, X), s.apply(1, X)
    out = tuple(t.clone() for t in (X, ritz, G, res, AX, BX))
    s.close()
    return out


def _check(AX, BX, ritz, G_ref, res_ref):
    import torch
    import paper_2503_22652_b200 as P
    G = torch.full_like(AX, float("nan"))
    r = torch.full_like(ritz, float("nan"))
    P.residual_static(AX, BX, ritz, G, r)
    np.testing.assert_allclose(G.cpu().numpy(), G_ref.cpu().numpy(), rtol=0, atol=1e-10)
    np.testing.assert_allclose(r.cpu().numpy(), res_ref.cpu().numpy(), rtol=1e-6, atol=1e-11)
    # and against the oracle's definition on the same AX, BX (not through the existing path)
    ro = orc.residual_norms(AX.cpu().numpy(), BX.cpu().numpy(), ritz.cpu().numpy())
    np.testing.assert_allclose(r.cpu().numpy(), ro, rtol=1e-12, atol=1e-14)
    return G, r


def test_residual_static_matches_the_rayleigh_ritz_path_on_two_calls_in_a_row():
    import torch
    import paper_2503_22652_b200 as P
    P.static_setup()
    # call 1: generalized dense pencil, 700 rows (140 row slabs of 5), 300 columns (two column passes per slab)
    _, ritz1, G1, res1, AX1, BX1 = _existing_path(small_dense_generalized(700, seed=5), 300, seed=21)
    # call 2: standard sparse problem, narrower block (37 columns), ragged last slab
    prob2 = workloads.config3_sparse_laplacian(n=12, n_wanted=16, block=37, degree=8)
    _, ritz2, G2, res2, AX2, BX2 = _existing_path(prob2, 37, seed=22)
    Ga, ra = _check(AX1, BX1, ritz1, G1, res1)
    Gb, rb = _check(AX2, BX2, ritz2, G2, res2)
    # two more calls into preallocated outputs: no device memory moves, neither in torch's pool nor in the driver,
    # and the results repeat bit for bit (fixed summation order, ticket counter re-armed by the kernel)
    Gc, rc, Gd, rd = torch.empty_like(AX1), torch.empty_like(ritz1), torch.empty_like(AX2), torch.empty_like(ritz2)
    torch.cuda.synchronize()
    free0, alloc0 = torch.cuda.mem_get_info()[0], torch.cuda.memory_allocated()
    P.residual_static(AX1, BX1, ritz1, Gc, rc)
    P.residual_static(AX2, BX2, ritz2, Gd, rd)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0 and torch.cuda.memory_allocated() == alloc0
    assert torch.equal(ra, rc) and torch.equal(Ga, Gc) and torch.equal(rb, rd) and torch.equal(Gb, Gd)
    # norms only / block only
    r_only = torch.empty_like(ritz1)
    P.residual_static(AX1, BX1, ritz1, None, r_only)
    G_only = torch.empty_like(AX2)
    P.residual_static(AX2, BX2, ritz2, G_only, None)
    assert torch.equal(r_only, ra) and torch.equal(G_only, Gb)


def test_residual_static_rejects_what_the_scratch_cannot_hold():
    import torch
    import paper_2503_22652_b200 as P
    N = P.STATIC_MAX_N + 1
    AX = torch.zeros((2, N), dtype=torch.float64, device="cuda")
    r = torch.full((N,), 7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(P.RchfsiError) as e:
        P.residual_static(AX, AX, r.clone(), None, r)
    assert e.value.status == P.EINVAL and "RCHFSI_STATIC_MAX_N" in str(e.value)
    assert bool((r == 7.0).all())                                         # outputs untouched
    with pytest.raises(P.RchfsiError):
        P.residual_static(AX[:, :4].contiguous(), AX[:, :4].contiguous(), r[:4].contiguous(), None, None)
    # the widest block the scratch holds still works
    N = P.STATIC_MAX_N
    g = torch.Generator(device="cuda").manual_seed(3)
    AX = torch.randn((300, N), dtype=torch.float64, device="cuda", generator=g)
    BX = torch.randn((300, N), dtype=torch.float64, device="cuda", generator=g)
    ritz = torch.randn((N,), dtype=torch.float64, device="cuda", generator=g)
    r = torch.empty_like(ritz)
    P.residual_static(AX, BX, ritz, None, r)
    ro = orc.residual_norms(AX.cpu().numpy(), BX.cpu().numpy(), ritz.cpu().numpy())
    np.testing.assert_allclose(r.cpu().numpy(), ro, rtol=1e-12, atol=0)
