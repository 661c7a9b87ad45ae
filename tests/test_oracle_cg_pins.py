"""Pins of the CG oracle (next row f2): none of the expected values comes from oracle.cg_oracle itself."""
import numpy as np

import lattice_inputs as li
import oracle
from oracle import cg_oracle

APBC = (1, 1, 1, -1)


def test_C1_dense_spd_system_against_lapack():
    rng = np.random.default_rng(1)
    B = rng.standard_normal((60, 60)) + 1j * rng.standard_normal((60, 60))
    A = B.conj().T @ B + 5.0 * np.eye(60)
    b = rng.standard_normal(60) + 1j * rng.standard_normal(60)
    x, it, res = cg_oracle.cg(lambda v: A @ v, b, 1e-12, 500)
    assert it <= 2 * 60 and res <= 1e-12  # finite precision: a few more than n steps
    assert np.linalg.norm(x - np.linalg.solve(A, b)) <= 1e-10 * np.linalg.norm(x)


def test_C2_exact_termination_in_n_distinct_eigenvalues():
    """CG terminates (in exact arithmetic) after as many steps as A has distinct eigenvalues."""
    d = np.array([1.0] * 10 + [2.5] * 10 + [7.0] * 10)
    b = np.random.default_rng(2).standard_normal(30) + 0j
    x, it, res = cg_oracle.cg(lambda v: d * v, b, 1e-13, 50)
    assert it == 3 and np.allclose(x, b / d, rtol=1e-12)


def test_C3_free_field_constant_source_closed_form():
    """U = 1, all-periodic, constant even source: H_eo H_oe const = 64 const (pin P6 twice), so
    Mhat = (1 + i th g5) - 64 kappa^2 (1 + i th g5)^-1 is a number per chirality, lam_+- = (1 +- i th) - 64 k^2/(1 +- i th),
    and x = b / |lam_+-|^2; two distinct eigenvalues of A => at most 2 iterations."""
    dims, kappa, mu = (4, 4, 4, 4), 0.1, 0.3
    th = 2 * kappa * mu
    U = li.unit_links(dims)
    even = li.parity_mask(dims, 0)[..., None, None]
    chi = np.random.default_rng(3).standard_normal((4, 3)) + 1j * np.random.default_rng(4).standard_normal((4, 3))
    b = np.broadcast_to(chi, (*dims[::-1], 4, 3)) * even
    x, it, res = cg_oracle.cg_solve_tm(U, b, dims, (1, 1, 1, 1), kappa, mu, 1e-13, 20)
    lam = np.array([(1 + 1j * th) - 64 * kappa ** 2 / (1 + 1j * th), (1 - 1j * th) - 64 * kappa ** 2 / (1 - 1j * th)])
    scale = np.repeat(1.0 / np.abs(lam) ** 2, 2)[:, None]  # spins 0,1: lam_+, spins 2,3: lam_-
    assert it <= 2
    assert np.abs(x - b * scale).max() <= 1e-12 * np.abs(x).max()


def test_C4_lattice_solution_satisfies_the_equation():
    """Random SU(3) links, antiperiodic t: the returned x has true residual ||b - A x|| <= 2 tol ||b||, with A
    applied here from oracle.apply_M_tm and an explicit gamma_5 (not through cg_oracle's operator)."""
    dims, kappa, mu, tol = (4, 4, 4, 8), 0.15, 0.1, 1e-10
    U = li.random_su3_links(dims, seed=31)
    even = li.parity_mask(dims, 0)[..., None, None]
    b = li.gaussian_spinor(dims, seed=32) * even
    x, it, res = cg_oracle.cg_solve_tm(U, b, dims, APBC, kappa, mu, tol, 500)
    g5 = np.array([1, 1, -1, -1])[:, None]
    t = oracle.apply_M_tm(U, x, dims, APBC, kappa, mu, 1)
    Ax = g5 * oracle.apply_M_tm(U, g5 * t, dims, APBC, kappa, -mu, 1)
    assert 1 < it < 500 and res <= tol
    assert np.linalg.norm(b - Ax) <= 2 * tol * np.linalg.norm(b)
    assert np.abs(x * (~even)).max() == 0.0


def test_C5_mixed_precision_reaches_fp64_accuracy():
    """Defect correction with an fp32 inner CG: the TRUE fp64 residual (operator composed here) reaches a tolerance
    far below fp32 epsilon in a few corrections, and the solution is the fp64 CG's."""
    dims, kappa, mu, tol = (4, 4, 4, 8), 0.15, 0.1, 1e-11
    U = li.random_su3_links(dims, seed=31)
    even = li.parity_mask(dims, 0)[..., None, None]
    b = li.gaussian_spinor(dims, seed=32) * even
    x, total, outer, res = cg_oracle.cg_mixed_solve_tm(U, b, dims, APBC, kappa, mu, tol, 1e-4, 2000)
    g5 = np.array([1, 1, -1, -1])[:, None]
    Ax = g5 * oracle.apply_M_tm(U, g5 * oracle.apply_M_tm(U, x, dims, APBC, kappa, mu, 1), dims, APBC, kappa, -mu, 1)
    assert np.linalg.norm(b - Ax) <= tol * np.linalg.norm(b) and res <= tol
    assert 2 <= outer <= 6
    x64, it64, _ = cg_oracle.cg_solve_tm(U, b, dims, APBC, kappa, mu, tol, 500)
    assert np.linalg.norm(x - x64) <= 100 * tol * np.linalg.norm(x64)
    # a single fp32 solve cannot do this: its true residual stalls near fp32 epsilon
    x32, _, _ = cg_oracle._cg32(lambda v: cg_oracle.normal_operator_tm(U.astype(np.complex64), dims, APBC, kappa, mu)(v).astype(np.complex64),
                                b.astype(np.complex64), 1e-11, 300)
    Ax32 = g5 * oracle.apply_M_tm(U, g5 * oracle.apply_M_tm(U, x32.astype(np.complex128), dims, APBC, kappa, mu, 1), dims, APBC, kappa, -mu, 1)
    assert np.linalg.norm(b - Ax32) > 1e3 * tol * np.linalg.norm(b)
