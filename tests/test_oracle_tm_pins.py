"""Pins of the twisted-mass operator of the oracle (next row f1; "N_f = 2 twisted-mass Wilson
fermions", "even-odd preconditioning"; the formula is DESIGN.md reading F1):

    M_tm(mu)    = (1 + 2 i kappa mu g5) - kappa H
    Mhat_tm(mu) = (1 + 2 i kappa mu g5) - kappa^2 H_eo (1 + 2 i kappa mu g5)^-1 H_oe      (even sites)

None of the expected values below comes from oracle.apply_M_tm itself.
"""
import itertools

import numpy as np
import pytest

import lattice_inputs as li
import oracle

APBC = (1, 1, 1, -1)
G5 = np.diag([1.0, 1.0, -1.0, -1.0]).astype(np.complex128)  # chiral basis, SURVEY.md Appendix A.2


def _pauli_gamma(mu):
    """gamma_mu = [[0, A], [A^dagger, 0]], A_x,y,z = -i sigma_1,2,3, A_t = -1 (retyped from Appendix A.2)."""
    s = [np.array([[0, 1], [1, 0]]), np.array([[0, -1j], [1j, 0]]), np.array([[1, 0], [0, -1]])]
    A = -1j * s[mu] if mu < 3 else -np.eye(2)
    g = np.zeros((4, 4), dtype=np.complex128)
    g[:2, 2:] = A
    g[2:, :2] = A.conj().T
    return g


def _g5(psi):
    return np.einsum("st,...ta->...sa", G5, psi)


def _inner(a, b):
    return np.vdot(a.ravel(), b.ravel())


def test_T1_mu_zero_reduces_to_wilson():
    dims, kappa = (4, 4, 6, 8), 0.15
    U = li.random_su3_links(dims, seed=5)
    psi = li.gaussian_spinor(dims, seed=6)
    for eo in (0, 1):
        assert np.array_equal(oracle.apply_M_tm(U, psi, dims, APBC, kappa, 0.0, eo), oracle.apply_M(U, psi, dims, APBC, kappa, eo))


@pytest.mark.parametrize("mu", [0.05, -0.3])
def test_T2_free_field_plane_waves(mu):
    """U = 1: M_tm psi = [(1 - 2 kappa sum cos p) + 2 i kappa mu g5 + 2 i kappa sum gamma sin p] psi sitewise,
    and (M_tm - a)^2 psi = -((2 kappa mu)^2 + 4 kappa^2 sum sin^2 p) psi  (g5 anticommutes with every gamma_mu)."""
    dims, kappa = (4, 4, 4, 4), 0.125
    U = li.unit_links(dims)
    rng = np.random.default_rng(11)
    worst = worst2 = 0.0
    for n in itertools.product(range(4), repeat=4):
        chi = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
        psi, p = li.plane_wave(dims, n, APBC, chi)
        a = 1 - 2 * kappa * np.cos(p).sum()
        mat = a * np.eye(4) + 2j * kappa * mu * G5
        for d in range(4):
            mat = mat + 2j * kappa * np.sin(p[d]) * _pauli_gamma(d)
        out = oracle.apply_M_tm(U, psi, dims, APBC, kappa, mu, 0)
        worst = max(worst, np.abs(out - np.einsum("st,...ta->...sa", mat, psi)).max())
        once = out - a * psi
        twice = oracle.apply_M_tm(U, once, dims, APBC, kappa, mu, 0) - a * once
        lam2 = (2 * kappa * mu) ** 2 + 4 * kappa ** 2 * (np.sin(p) ** 2).sum()
        worst2 = max(worst2, np.abs(twice + lam2 * psi).max())
    assert worst < 5e-14 and worst2 < 5e-14


@pytest.mark.parametrize("bc", [APBC, tuple(np.exp(1j * np.array([0.4, 0.0, -2.2, 1.3])))])
def test_T3_gamma5_hermiticity_flips_the_twist(bc):
    """g5 M_tm(mu) g5 = M_tm(-mu)^dagger, full and even-odd:  <phi, M(mu) psi> = <g5 M(-mu) g5 phi, psi>."""
    dims, kappa, mu = (4, 6, 4, 8), 0.14, 0.21
    U = li.random_su3_links(dims, seed=7)
    psi = li.gaussian_spinor(dims, seed=8)
    phi = li.gaussian_spinor(dims, seed=9)
    even = li.parity_mask(dims, 0)[..., None, None]
    for eo in (0, 1):
        a, b = (psi, phi) if eo == 0 else (psi * even, phi * even)
        lhs = _inner(b, oracle.apply_M_tm(U, a, dims, bc, kappa, mu, eo))
        rhs = _inner(_g5(oracle.apply_M_tm(U, _g5(b), dims, bc, kappa, -mu, eo)), a)
        assert abs(lhs - rhs) <= 1e-13 * abs(lhs)
        wrong = _inner(_g5(oracle.apply_M_tm(U, _g5(b), dims, bc, kappa, +mu, eo)), a)
        assert abs(lhs - wrong) > 1e-4 * abs(lhs)  # the sign of mu matters


def test_T4_even_odd_form_is_the_schur_complement():
    """Take psi_e at random and psi_o = kappa (1 + 2 i kappa mu g5)^-1 H_oe psi_e.  Then the full operator gives
    (M_tm psi)_o = 0 and (M_tm psi)_e = Mhat_tm psi_e.  The inverse is typed here in closed form,
    (1 - i theta g5) / (1 + theta^2), which the oracle does not use."""
    dims, kappa, mu = (4, 4, 6, 8), 0.16, 0.35
    theta = 2 * kappa * mu
    U = li.random_su3_links(dims, seed=12)
    even = li.parity_mask(dims, 0)[..., None, None]
    psi_e = li.gaussian_spinor(dims, seed=13) * even
    h = oracle.dslash_eo(U, psi_e, dims, APBC, 1)                      # H_oe psi_e on odd sites
    psi_o = kappa * (h - 1j * theta * _g5(h)) / (1 + theta ** 2)
    full = oracle.apply_M_tm(U, psi_e + psi_o, dims, APBC, kappa, mu, 0)
    hat = oracle.apply_M_tm(U, psi_e, dims, APBC, kappa, mu, 1)
    scale = np.abs(hat).max()
    assert np.abs(full * (~even)).max() <= 1e-14 * scale
    assert np.abs(full * even - hat).max() <= 1e-14 * scale
    assert np.abs(hat * (~even)).max() == 0.0
