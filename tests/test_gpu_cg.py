"""GPU parity of the CG solver (next row f2) and of Q = gamma_5 Mhat_tm against the oracle."""
import numpy as np
import pytest
import torch

import lattice_inputs as li
import oracle
from oracle import cg_oracle

pytestmark = pytest.mark.gpu

APBC = (1, 1, 1, -1)
G5 = np.array([1, 1, -1, -1])[:, None]


def _solve_gpu(H, g, b_half, kappa, mu, tol, maxiter):
    x = g.buf()
    ws = torch.empty(g.ctx.cg_workspace_bytes(), dtype=torch.uint8, device=g.dev)
    it, res = g.ctx.cg_solve_tm(x, g.gauge, g.to_native(b_half, 0), kappa, mu, tol, maxiter, ws)
    return g.from_native(x, 0), it, res


@pytest.mark.parametrize("precision,recon,tol", [(64, 18, 1e-10), (64, 12, 1e-10), (32, 12, 1e-5)])
def test_cg_against_oracle(precision, recon, tol):
    import gpu_harness as H
    dims, kappa, mu = (8, 8, 8, 16), 0.15, 0.1
    U = li.links_for_config(2).astype(H.cdtype(precision))
    even = li.parity_mask(dims, 0)[..., None, None]
    b = (li.gaussian_spinor(dims, seed=41) * even).astype(H.cdtype(precision))
    g = H.Gpu(dims, precision, recon, APBC, U)

    # Q(mu) = gamma_5 Mhat(mu)
    q = g.buf()
    g.ctx.apply_Q_tm(q, g.gauge, g.to_native(H.half_of(b, dims, 0), 0), kappa, mu, g.buf())
    refq = H.half_of(G5 * oracle.apply_M_tm(U, b, dims, APBC, kappa, mu, 1), dims, 0)
    assert H.rel_l2(g.from_native(q, 0), refq) <= (1e-12 if precision == 64 else 1e-5)

    x_ref, it_ref, _ = cg_oracle.cg_solve_tm(U, b, dims, APBC, kappa, mu, tol, 500)
    x, it, res = _solve_gpu(H, g, H.half_of(b, dims, 0), kappa, mu, tol, 500)
    assert res <= tol and abs(it - it_ref) <= 1, (it, it_ref, res)
    # same solution up to the stopping tolerance (amplified by the condition number of A, O(10) here)
    assert H.rel_l2(x, H.half_of(x_ref, dims, 0)) <= 50 * tol
    # the equation itself, with the oracle's operator: |b - A x_gpu| <= a few tol |b|
    xf = H.scatter_half(x.astype(np.complex128), dims, 0)
    Ax = G5 * oracle.apply_M_tm(U, G5 * oracle.apply_M_tm(U, xf, dims, APBC, kappa, mu, 1), dims, APBC, kappa, -mu, 1)
    assert np.linalg.norm(b - Ax) <= 4 * tol * np.linalg.norm(b)


def test_cg_edge_cases():
    import gpu_harness as H
    dims, kappa, mu = (4, 6, 6, 6), 0.12, 0.2   # Vh = 432: ragged last tile and last reduction block
    U = li.random_su3_links(dims, seed=51)
    even = li.parity_mask(dims, 0)[..., None, None]
    b = li.gaussian_spinor(dims, seed=52) * even
    g = H.Gpu(dims, 64, 12, APBC, U)
    # zero right-hand side: zero iterations, zero solution
    x, it, res = _solve_gpu(H, g, np.zeros_like(H.half_of(b, dims, 0)), kappa, mu, 1e-10, 50)
    assert it == 0 and res == 0.0 and not x.any()
    # maxiter cut-off is honoured exactly and reports the residual reached so far
    x3, it3, res3 = _solve_gpu(H, g, H.half_of(b, dims, 0), kappa, mu, 1e-14, 3)
    x_ref3, it_ref3, res_ref3 = cg_oracle.cg_solve_tm(U, b, dims, APBC, kappa, mu, 1e-14, 3)
    assert it3 == it_ref3 == 3 and abs(res3 - res_ref3) <= 1e-9 * res_ref3
    assert H.rel_l2(x3, H.half_of(x_ref3, dims, 0)) <= 1e-12
    # converged run on the ragged lattice; deterministic reductions: two runs agree bit for bit
    xa, ita, resa = _solve_gpu(H, g, H.half_of(b, dims, 0), kappa, mu, 1e-11, 500)
    xb, itb, resb = _solve_gpu(H, g, H.half_of(b, dims, 0), kappa, mu, 1e-11, 500)
    x_ref, it_ref, _ = cg_oracle.cg_solve_tm(U, b, dims, APBC, kappa, mu, 1e-11, 500)
    assert ita == itb and resa == resb and np.array_equal(xa, xb)
    assert abs(ita - it_ref) <= 1 and H.rel_l2(xa, H.half_of(x_ref, dims, 0)) <= 1e-9
    # error codes
    import paper_1112_5280_b200 as L
    ws = torch.empty(g.ctx.cg_workspace_bytes(), dtype=torch.uint8, device=g.dev)
    xb_ = g.buf()
    with pytest.raises(L.LqcdError) as e:
        g.ctx.cg_solve_tm(xb_, g.gauge, xb_, kappa, mu, 1e-8, 10, ws)
    assert e.value.status == L.LQCD_EALIAS
    with pytest.raises(L.LqcdError) as e:
        g.ctx.cg_solve_tm(xb_, g.gauge, g.buf(), kappa, mu, -1.0, 10, ws)
    assert e.value.status == L.LQCD_EINVAL


@pytest.mark.parametrize("recon64,recon32,link32", [(18, 12, 0), (12, 12, 0), (12, 12, 16)])
def test_mixed_precision_cg(recon64, recon32, link32):
    """lqcd_cg_solve_tm_mixed: fp64-accurate solution from fp32 iterations; compared with the fp64 oracle CG
    and with the mixed-precision oracle (outer correction count)."""
    import gpu_harness as H
    dims, kappa, mu, tol = (8, 8, 8, 16), 0.15, 0.1, 1e-11
    U = li.links_for_config(2)
    even = li.parity_mask(dims, 0)[..., None, None]
    b = li.gaussian_spinor(dims, seed=41) * even
    g64 = H.Gpu(dims, 64, recon64, APBC, U)
    g32 = H.Gpu(dims, 32, recon32, APBC, U.astype(np.complex64), link_precision=link32)  # 16: inner operator with half links
    x = g64.buf()
    ws = torch.empty(g64.ctx.cg_mixed_workspace_bytes(g32.ctx), dtype=torch.uint8, device=g64.dev)
    it, outer, res = g64.ctx.cg_solve_tm_mixed(g32.ctx, x, g64.gauge, g32.gauge, g64.to_native(H.half_of(b, dims, 0), 0),
                                               kappa, mu, tol, 1e-4, 2000, ws)
    xg = H.scatter_half(g64.from_native(x, 0), dims, 0)
    Ax = G5 * oracle.apply_M_tm(U, G5 * oracle.apply_M_tm(U, xg, dims, APBC, kappa, mu, 1), dims, APBC, kappa, -mu, 1)
    assert res <= tol and np.linalg.norm(b - Ax) <= 1.5 * tol * np.linalg.norm(b)
    x_ref, it_ref, _ = cg_oracle.cg_solve_tm(U, b, dims, APBC, kappa, mu, tol, 500)
    assert np.linalg.norm(xg - x_ref) <= 100 * tol * np.linalg.norm(x_ref)
    _, it_mix, outer_mix, _ = cg_oracle.cg_mixed_solve_tm(U, b, dims, APBC, kappa, mu, tol, 1e-4, 2000)
    if link32 == 0:
        assert abs(outer - outer_mix) <= 1 and abs(it - it_mix) <= max(3, it_mix // 10), (it, it_mix, outer, outer_mix)
    else:  # a slightly different inner operator: a few more corrections are allowed, the answer is the same
        assert outer <= outer_mix + 3 and it <= 2 * it_mix
    # mismatched contexts are rejected
    import paper_1112_5280_b200 as L
    with pytest.raises(L.LqcdError):
        g32.ctx.cg_solve_tm_mixed(g64.ctx, x, g64.gauge, g32.gauge, g64.buf(), kappa, mu, tol, 1e-4, 10, ws)


def test_mixed_precision_cg_16bit_inner():
    """lqcd_cg_solve_tm_mixed with a precision-16 inner context (16-bit solver, next row f4): the inner CG keeps x and r
    in fp32 and p, Q p, A p in 16-bit storage; the fp64 defect correction restores full accuracy.  Checked like the fp32
    inner solver: true residual with the oracle's operator, solution against the fp64 oracle CG; the iteration count
    may exceed the fp32-inner model of the oracle (a 2^-11 perturbed operator and search direction), bounded at 2x."""
    import gpu_harness as H
    dims, kappa, mu, tol = (8, 8, 8, 16), 0.15, 0.1, 1e-11
    U = li.links_for_config(2)
    even = li.parity_mask(dims, 0)[..., None, None]
    b = li.gaussian_spinor(dims, seed=41) * even
    g64 = H.Gpu(dims, 64, 12, APBC, U)
    g16 = H.Gpu(dims, 16, 12, APBC, U.astype(np.complex64))
    x = g64.buf()
    ws = torch.empty(g64.ctx.cg_mixed_workspace_bytes(g16.ctx), dtype=torch.uint8, device=g64.dev)
    it, outer, res = g64.ctx.cg_solve_tm_mixed(g16.ctx, x, g64.gauge, g16.gauge, g64.to_native(H.half_of(b, dims, 0), 0),
                                               kappa, mu, tol, 1e-3, 4000, ws)
    xg = H.scatter_half(g64.from_native(x, 0), dims, 0)
    Ax = G5 * oracle.apply_M_tm(U, G5 * oracle.apply_M_tm(U, xg, dims, APBC, kappa, mu, 1), dims, APBC, kappa, -mu, 1)
    assert res <= tol and np.linalg.norm(b - Ax) <= 1.5 * tol * np.linalg.norm(b)
    x_ref, it_ref, _ = cg_oracle.cg_solve_tm(U, b, dims, APBC, kappa, mu, tol, 500)
    assert np.linalg.norm(xg - x_ref) <= 100 * tol * np.linalg.norm(x_ref)
    _, it_mix, outer_mix, _ = cg_oracle.cg_mixed_solve_tm(U, b, dims, APBC, kappa, mu, tol, 1e-3, 4000)
    assert it <= 2 * it_mix + 10 and outer <= 2 * outer_mix + 4, (it, it_mix, outer, outer_mix)


def test_cg_16bit_context():
    """lqcd_cg_solve_tm on a precision-16 context: 16-bit b in, 16-bit x out, fp32 iterate inside.  The operator it
    inverts is the one on the stored (rounded) links; against the oracle on those links the solution is good to the
    storage rounding of x (2^-11 per site) plus cond(A) times the 16-bit noise of the recurrences."""
    import gpu_harness as H
    import test_gpu_parity as T
    dims, kappa, mu, tol = (8, 8, 8, 16), 0.15, 0.1, 2e-3
    U = li.links_for_config(2).astype(np.complex64)
    even = li.parity_mask(dims, 0)[..., None, None]
    b = (li.gaussian_spinor(dims, seed=43) * even).astype(np.complex64)
    g = H.Gpu(dims, 16, 12, APBC, U)
    ws = torch.empty(g.ctx.cg_workspace_bytes(), dtype=torch.uint8, device=g.dev)
    x = g.buf()
    it, res = g.ctx.cg_solve_tm(x, g.gauge, g.to_native(H.half_of(b, dims, 0), 0), kappa, mu, tol, 500, ws)
    assert 0 < it < 100 and res <= tol
    Uq, bq = T._quantise_links(U), T._quantise_spinor(b)
    xg = H.scatter_half(g.from_native(x, 0), dims, 0)
    Ax = G5 * oracle.apply_M_tm(Uq, G5 * oracle.apply_M_tm(Uq, xg, dims, APBC, kappa, mu, 1), dims, APBC, kappa, -mu, 1)
    assert np.linalg.norm(bq - Ax) <= 5 * tol * np.linalg.norm(bq)
    # zero source, and the iteration cut-off
    it0, res0 = g.ctx.cg_solve_tm(x, g.gauge, g.to_native(np.zeros_like(H.half_of(b, dims, 0)), 0), kappa, mu, tol, 50, ws)
    assert it0 == 0 and res0 == 0.0 and not g.from_native(x, 0).any()
    it3, _ = g.ctx.cg_solve_tm(x, g.gauge, g.to_native(H.half_of(b, dims, 0), 0), kappa, mu, 1e-9, 3, ws)
    assert it3 == 3
