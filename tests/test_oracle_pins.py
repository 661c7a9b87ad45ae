"""Pins for the CPU oracle.  CPU only (-m "not gpu").

The paper prints no worked example for the dslash (PAPER.md:89 names it, gives no formula),
so every pin is something the mathematics fixes: closed forms, invariants, brute force,
special cases written out by hand, and a second independently written formulation.
Each pin is chosen so that a plausible slip in oracle/wilson_oracle.c (dropped term, wrong
sign, wrong neighbour, U vs U^T vs U^+, wrong bc conjugate) fails at least one of them.
"""
import itertools
import os

import numpy as np
import pytest

import lattice_inputs as li
import oracle
from oracle.roll_formulation import dslash_roll, gamma_from_pauli

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
APBC = (1, 1, 1, -1)


def rel_l2(a, b):
    return np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel())


# ------------------------------------------------------------------ P8: gamma algebra
def test_P8_gamma_table_is_hermitian_clifford_chiral():
    g = [oracle.gamma(mu) for mu in range(4)]
    one = np.eye(4)
    for mu in range(4):
        assert np.array_equal(g[mu], g[mu].conj().T)
        for nu in range(4):
            anti = g[mu] @ g[nu] + g[nu] @ g[mu]
            assert np.array_equal(anti, 2 * one * (mu == nu))
    g5 = g[3] @ g[0] @ g[1] @ g[2]
    assert np.array_equal(g5, np.diag([1, 1, -1, -1]))
    assert np.array_equal(oracle.gamma(4), g5)
    # typed-in table == table built from Pauli matrices (independent construction)
    for mu in range(4):
        assert np.array_equal(g[mu], gamma_from_pauli(mu))


def test_P8_projectors():
    for mu in range(4):
        g = oracle.gamma(mu)
        pm, pp = np.eye(4) - g, np.eye(4) + g
        assert np.array_equal(pm @ pm, 2 * pm)
        assert np.array_equal(pp @ pp, 2 * pp)
        assert np.array_equal(pm @ pp, np.zeros((4, 4)))
        assert np.linalg.matrix_rank(pm) == 2 and np.linalg.matrix_rank(pp) == 2


# ------------------------------------------------------------------ P6: constant field
def test_P6_constant_field_gives_8psi():
    dims = (4, 6, 4, 8)
    U = li.unit_links(dims)
    chi = np.arange(1, 13).reshape(4, 3) * (1 + 0.5j)
    psi = np.broadcast_to(chi, (dims[3], dims[2], dims[1], dims[0], 4, 3)).copy()
    out = oracle.dslash_full(U, psi, dims, (1, 1, 1, 1))
    assert np.array_equal(out, 8 * psi)
    # antiperiodic t: the two t-hops of the first/last timeslice flip sign -> (1-g_t) and (1+g_t)
    # pieces no longer add to 2; interior slices still give 8 psi.
    out = oracle.dslash_full(U, psi, dims, APBC)
    assert np.array_equal(out[1:-1], 8 * psi[1:-1])
    assert not np.allclose(out[0], 8 * psi[0])


# ------------------------------------------------------------------ P7: point source by hand
@pytest.mark.parametrize("bc", [(1, 1, 1, 1), APBC, tuple(np.exp(1j * np.array([0.3, -1.1, 2.0, 0.7])))])
def test_P7_point_source_hits_exactly_8_neighbours(bc):
    dims = (4, 4, 6, 4)
    X, Y, Z, T = dims
    L = np.array(dims)
    U = li.random_su3_links(dims, seed=11)
    bcv = li.bc_phases(bc)
    for x0, s0, c0 in [((0, 0, 0, 0), 0, 0), ((3, 1, 5, 3), 2, 1), ((2, 3, 0, 3), 3, 2), ((1, 0, 5, 0), 1, 0)]:
        psi = np.zeros((T, Z, Y, X, 4, 3), dtype=np.complex128)
        psi[x0[3], x0[2], x0[1], x0[0], s0, c0] = 1.0
        out = oracle.dslash_full(U, psi, dims, bc)
        expect = np.zeros_like(out)
        for mu in range(4):
            g = gamma_from_pauli(mu)
            e = np.zeros(4, dtype=int)
            e[mu] = 1
            # site y = x0 + mu^ sees x0 through its BACKWARD hop: (1+g_mu) U_mu(x0)^+ psi(x0),
            # times conj(bc_mu) if y_mu = 0 (the hop y -> y-mu^ crosses the boundary).
            y = (np.array(x0) + e) % L
            ph = np.conj(bcv[mu]) if y[mu] == 0 else 1.0
            Ux0 = U[mu, x0[3], x0[2], x0[1], x0[0]]
            spin = (np.eye(4) + g)[:, s0]
            col = np.conj(Ux0[c0, :])          # (U^+)[a][c0] = conj(U[c0][a])
            expect[y[3], y[2], y[1], y[0]] += ph * np.outer(spin, col)
            # site y = x0 - mu^ sees x0 through its FORWARD hop: (1-g_mu) U_mu(y) psi(x0),
            # times bc_mu if y_mu = L_mu - 1.
            y = (np.array(x0) - e) % L
            ph = bcv[mu] if y[mu] == L[mu] - 1 else 1.0
            Uy = U[mu, y[3], y[2], y[1], y[0]]
            spin = (np.eye(4) - g)[:, s0]
            col = Uy[:, c0]
            expect[y[3], y[2], y[1], y[0]] += ph * np.outer(spin, col)
        assert np.allclose(out, expect, rtol=0, atol=1e-15)
        nz = np.argwhere(np.abs(out).sum(axis=(-1, -2)) > 0)
        assert len(nz) == 8


def test_P7_one_entry_fully_by_hand():
    # psi = delta at x0=(1,1,1,1), spin 0, colour 0; look at y = x0 - x^ = (0,1,1,1):
    # out(y) = (1 - gamma_x)[:,0] (x) U_x(y)[:,0];  gamma_x[:,0] = (0,0,0,i)  ->  spin vector (1,0,0,-i)
    dims = (4, 4, 4, 4)
    U = li.random_su3_links(dims, seed=5)
    psi = np.zeros((4, 4, 4, 4, 4, 3), dtype=np.complex128)
    psi[1, 1, 1, 1, 0, 0] = 1.0
    out = oracle.dslash_full(U, psi, dims, APBC)
    col = U[0, 1, 1, 1, 0][:, 0]
    assert np.allclose(out[1, 1, 1, 0, 0], col, atol=1e-15)
    assert np.allclose(out[1, 1, 1, 0, 1], 0, atol=1e-15)
    assert np.allclose(out[1, 1, 1, 0, 2], 0, atol=1e-15)
    assert np.allclose(out[1, 1, 1, 0, 3], -1j * col, atol=1e-15)
    # and y = x0 + t^ = (1,1,1,2): (1 + gamma_t)[:,0] = (1,0,-1,0), colour vector conj(U_t(x0)[0,:])
    row = np.conj(U[3, 1, 1, 1, 1][0, :])
    assert np.allclose(out[2, 1, 1, 1, 0], row, atol=1e-15)
    assert np.allclose(out[2, 1, 1, 1, 2], -row, atol=1e-15)
    assert np.allclose(out[2, 1, 1, 1, 1], 0, atol=1e-15)
    assert np.allclose(out[2, 1, 1, 1, 3], 0, atol=1e-15)


# ------------------------------------------------------------------ P1: plane waves
@pytest.mark.parametrize("bc", [APBC, (1, 1, 1, 1), tuple(np.exp(1j * np.array([0.4, 0.0, -2.2, 1.3])))])
def test_P1_free_field_plane_waves(bc):
    dims = (4, 4, 4, 4)
    kappa = 0.125
    U = li.unit_links(dims)
    rng = np.random.default_rng(3)
    worst = 0.0
    for n in itertools.product(range(4), repeat=4):
        chi = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
        psi, p = li.plane_wave(dims, n, bc, chi)
        out = oracle.apply_M(U, psi, dims, bc, kappa, 0)
        mat = (1 - 2 * kappa * np.cos(p).sum()) * np.eye(4, dtype=np.complex128)
        for mu in range(4):
            mat = mat + 2j * kappa * np.sin(p[mu]) * gamma_from_pauli(mu)
        expect = np.einsum("st,...ta->...sa", mat, psi)
        worst = max(worst, np.abs(out - expect).max())
    assert worst < 5e-14


# ------------------------------------------------------------------ P2: spectrum, brute force
def _free_spectrum(dims, kappa, bc):
    theta = np.angle(li.bc_phases(bc))
    lam = []
    for n in itertools.product(*[range(L) for L in dims]):
        p = (2 * np.pi * np.array(n) + theta) / np.array(dims)
        re = 1 - 2 * kappa * np.cos(p).sum()
        im = 2 * kappa * np.sqrt((np.sin(p) ** 2).sum())
        lam += [re + 1j * im] * 6 + [re - 1j * im] * 6
    return np.array(lam)


def _dense_matrix(U, dims, bc, kappa):
    X, Y, Z, T = dims
    n = X * Y * Z * T * 12
    M = np.empty((n, n), dtype=np.complex128)
    e = np.zeros(n, dtype=np.complex128)
    for k in range(n):
        e[k] = 1.0
        M[:, k] = oracle.apply_M(U, e.reshape(T, Z, Y, X, 4, 3), dims, bc, kappa, 0).ravel()
        e[k] = 0.0
    return M


def _sorted_multiset(v, decimals=9):
    v = np.round(v, decimals) + 0.0
    return v[np.lexsort((v.imag, v.real))]


def test_P2_free_field_spectrum_dense_4444():
    dims = (4, 4, 4, 4)
    kappa = 0.125
    M = _dense_matrix(li.unit_links(dims), dims, APBC, kappa)
    ev = np.linalg.eigvals(M)
    closed = _free_spectrum(dims, kappa, APBC)
    a, b = _sorted_multiset(ev, 8), _sorted_multiset(closed, 8)
    assert np.abs(a.real - b.real).max() < 1e-7
    # degenerate eigenvalues may swap order within a rounding bin; compare sorted moduli and real parts,
    # then every closed-form value must have a partner
    assert np.abs(np.sort(np.abs(ev)) - np.sort(np.abs(closed))).max() < 1e-8
    for lam in np.unique(np.round(closed, 9)):
        assert np.sum(np.abs(ev - lam) < 1e-7) == np.sum(np.abs(closed - lam) < 1e-7)
    # worked values quoted in SURVEY.md §8(c) P2 (tests/golden/free_field_eigs_4444.txt)
    rows = [l.split() for l in open(os.path.join(GOLDEN, "free_field_eigs_4444.txt")) if l[0] != "#"]
    for r in rows:
        re, im = float(r[4]), float(r[5])
        for sgn in (+1, -1):
            assert np.sum(np.abs(ev - (re + sgn * 1j * im)) < 5e-9) >= 6
    assert abs(np.abs(ev).min() - 0.1913417162) < 5e-9


def test_P2_dense_matrix_random_links_matches_roll_formulation_columns():
    # brute force on a tiny lattice with random links: every column of the dense matrix
    dims = (2, 2, 4, 2)
    U = li.random_su3_links(dims, seed=9)
    bc = tuple(np.exp(1j * np.array([0.2, 1.0, -0.7, np.pi])))
    M = _dense_matrix(U, dims, bc, 0.13)
    X, Y, Z, T = dims
    n = X * Y * Z * T * 12
    for k in range(0, n, 7):
        e = np.zeros(n, dtype=np.complex128)
        e[k] = 1
        psi = e.reshape(T, Z, Y, X, 4, 3)
        col = (psi - 0.13 * dslash_roll(U, psi, dims, bc)).ravel()
        assert np.abs(M[:, k] - col).max() < 1e-14


# ------------------------------------------------------------------ P3: gamma5-hermiticity
@pytest.mark.parametrize("bc", [APBC, tuple(np.exp(1j * np.array([0.9, -0.4, 0.1, 2.5])))])
def test_P3_gamma5_hermiticity(bc):
    dims = (4, 4, 6, 8)
    U = li.random_su3_links(dims, seed=1)
    phi = li.gaussian_spinor(dims, seed=21)
    psi = li.gaussian_spinor(dims, seed=22)
    g5 = np.array([1, 1, -1, -1])[:, None]
    lhs = np.vdot(phi, oracle.dslash_full(U, psi, dims, bc))
    rhs = np.vdot(g5 * oracle.dslash_full(U, g5 * phi, dims, bc), psi)
    assert abs(lhs - rhs) / abs(lhs) < 1e-13
    # even-odd form: <phi_e, H_eo psi_o> = <g5 H_oe g5 phi_e, psi_o>
    even = li.parity_mask(dims, 0)[..., None, None]
    phi_e, psi_o = phi * even, psi * ~even
    lhs = np.vdot(phi_e, oracle.dslash_eo(U, psi_o, dims, bc, 0))
    rhs = np.vdot(g5 * oracle.dslash_eo(U, g5 * phi_e, dims, bc, 1), psi_o)
    assert abs(lhs - rhs) / abs(lhs) < 1e-13


# ------------------------------------------------------------------ P4: even-odd == full
def test_P4_even_odd_decomposition_reproduces_full():
    dims = (8, 8, 8, 16)  # config 2 shape
    U = li.random_su3_links(dims, seed=1)
    psi = li.gaussian_spinor(dims, seed=2)
    even = li.parity_mask(dims, 0)[..., None, None]
    full = oracle.dslash_full(U, psi, dims, APBC)
    h_eo = oracle.dslash_eo(U, psi, dims, APBC, 0)   # reads odd sites only
    h_oe = oracle.dslash_eo(U, psi, dims, APBC, 1)
    assert np.array_equal(h_eo * ~even, np.zeros_like(h_eo))
    assert np.array_equal(h_oe * even, np.zeros_like(h_oe))
    assert np.array_equal(h_eo + h_oe, full)
    # H on an odd-supported field lives on even sites only and equals H_eo there
    odd_only = oracle.dslash_full(U, psi * ~even, dims, APBC)
    assert np.array_equal(odd_only, h_eo)
    # dslash_eo must not read the same-parity sites: poison them
    poisoned = np.where(even, np.nan, psi)
    assert np.array_equal(oracle.dslash_eo(U, poisoned, dims, APBC, 0), h_eo)
    # M_eo = 1 - kappa^2 H_eo H_oe assembled from the pieces
    kappa = 0.15
    m = oracle.apply_M(U, psi, dims, APBC, kappa, 1)
    tmp = oracle.dslash_eo(U, psi, dims, APBC, 1)
    ref = (psi - kappa ** 2 * oracle.dslash_eo(U, tmp, dims, APBC, 0)) * even
    assert np.allclose(m, ref, rtol=0, atol=1e-13)
    assert np.array_equal(m * ~even, np.zeros_like(m))


# ------------------------------------------------------------------ P5: gauge covariance
def test_P5_gauge_covariance():
    dims = (8, 8, 8, 16)
    U = li.random_su3_links(dims, seed=1)
    psi = li.gaussian_spinor(dims, seed=2)
    g = li.random_su3_field(dims, seed=4)
    Ug = np.empty_like(U)
    for mu in range(4):
        g_fwd = np.roll(g, -1, axis=3 - mu)       # g(x + mu^), periodic
        Ug[mu] = g @ U[mu] @ np.conj(np.swapaxes(g_fwd, -1, -2))
    psig = np.einsum("...ab,...sb->...sa", g, psi)
    lhs = oracle.dslash_full(Ug, psig, dims, APBC)
    rhs = np.einsum("...ab,...sb->...sa", g, oracle.dslash_full(U, psi, dims, APBC))
    assert rel_l2(lhs, rhs) < 1e-14


# ------------------------------------------------------------------ P9: two-row reconstruction
def test_P9_two_row_reconstruction_and_the_minus_U_trap():
    dims = (4, 4, 4, 4)
    for U in (li.random_su3_links(dims, seed=1), li.near_unit_links(dims, seed=1, eps=0.3)):
        flat = U.reshape(-1, 3, 3)
        assert np.abs(np.linalg.det(flat) - 1).max() < 1e-13
        assert np.abs(flat @ np.conj(np.swapaxes(flat, -1, -2)) - np.eye(3)).max() < 1e-13
        worst = bad = 0.0
        for m in flat[::17]:
            worst = max(worst, np.abs(oracle.recon_row2(m[0], m[1]) - m[2]).max())
            bad = max(bad, np.abs(oracle.recon_row2(-m[0], -m[1]) - (-m[2])).max())
        assert worst < 1e-15
        assert bad > 1.0   # -U has det -1: folding the antiperiodic sign into stored links breaks recon-12
    # closed-form special cases of conj(r0 x r1)
    assert np.array_equal(oracle.recon_row2([1, 0, 0], [0, 1, 0]), [0, 0, 1])
    assert np.array_equal(oracle.recon_row2([0, 1j, 0], [0, 0, 1]), [-1j, 0, 0])


# ------------------------------------------------------------------ P10: second formulation
@pytest.mark.parametrize("cfg", [1, 2])
def test_P10_roll_formulation_agrees(cfg):
    c = li.CONFIGS[cfg]
    dims = c["dims"]
    U = li.links_for_config(cfg)
    psi = li.gaussian_spinor(dims)
    a = oracle.dslash_full(U, psi, dims, c["bc"])
    b = dslash_roll(U, psi, dims, c["bc"])
    assert rel_l2(a, b) < 1e-15
    bc = tuple(np.exp(1j * np.array([0.3, -1.1, 2.0, 0.7])))
    assert rel_l2(oracle.dslash_full(U, psi, dims, bc), dslash_roll(U, psi, dims, bc)) < 1e-15


def test_P10_non_cubic_extents_catch_axis_mixups():
    dims = (4, 6, 8, 10)
    U = li.near_unit_links(dims, seed=3, eps=0.3)
    psi = li.gaussian_spinor(dims, seed=8)
    assert rel_l2(oracle.dslash_full(U, psi, dims, APBC), dslash_roll(U, psi, dims, APBC)) < 1e-15


# ------------------------------------------------------------------ P11: linearity, translation
def test_P11_linearity_and_translation_invariance():
    dims = (4, 4, 4, 8)
    U = li.random_su3_links(dims, seed=1)
    psi, phi = li.gaussian_spinor(dims, seed=2), li.gaussian_spinor(dims, seed=3)
    a, b = 0.3 - 1.2j, -2.0 + 0.1j
    lhs = oracle.dslash_full(U, a * psi + b * phi, dims, APBC)
    rhs = a * oracle.dslash_full(U, psi, dims, APBC) + b * oracle.dslash_full(U, phi, dims, APBC)
    assert rel_l2(lhs, rhs) < 1e-14
    U1 = li.unit_links(dims)
    per = (1, 1, 1, 1)
    for ax, sh in [(3, 1), (2, 2), (1, 3), (0, 5)]:
        lhs = oracle.dslash_full(U1, np.roll(psi, sh, axis=ax), dims, per)
        rhs = np.roll(oracle.dslash_full(U1, psi, dims, per), sh, axis=ax)
        assert np.array_equal(lhs, rhs)


# ------------------------------------------------------------------ sampled-site entry points, fp32 inputs
def test_site_sampling_entry_points_match_field_versions():
    dims = (4, 6, 4, 8)
    U = li.near_unit_links(dims, seed=1, eps=0.3)
    psi = li.gaussian_spinor(dims, seed=2)
    bc = tuple(np.exp(1j * np.array([0.0, 0.5, 0.0, np.pi])))
    rng = np.random.default_rng(0)
    coords = np.stack([rng.integers(0, L, 64) for L in dims], axis=1)
    coords[:8] = [[0, 0, 0, 0], [3, 5, 3, 7], [0, 5, 0, 7], [3, 0, 3, 0], [1, 1, 1, 1], [2, 0, 0, 0], [0, 0, 0, 7],
                  [3, 5, 3, 6]]
    full = oracle.dslash_full(U, psi, dims, bc)
    got = oracle.dslash_sites(U, psi, dims, bc, coords)
    for k, (x, y, z, t) in enumerate(coords):
        assert np.array_equal(got[k], full[t, z, y, x])
    m0 = oracle.apply_M(U, psi, dims, bc, 0.16, 0)
    got = oracle.apply_M_sites(U, psi, dims, bc, 0.16, 0, coords)
    for k, (x, y, z, t) in enumerate(coords):
        assert np.array_equal(got[k], m0[t, z, y, x])
    ev = coords[coords.sum(axis=1) % 2 == 0]
    m1 = oracle.apply_M(U, psi, dims, bc, 0.16, 1)
    got = oracle.apply_M_sites(U, psi, dims, bc, 0.16, 1, ev)
    for k, (x, y, z, t) in enumerate(ev):
        assert np.allclose(got[k], m1[t, z, y, x], rtol=0, atol=1e-13)


def test_fp32_inputs_are_promoted_elementwise():
    dims = (4, 4, 4, 4)
    U32 = li.random_su3_links(dims, seed=1).astype(np.complex64)
    psi32 = li.gaussian_spinor(dims, seed=2).astype(np.complex64)
    a = oracle.dslash_full(U32, psi32, dims, APBC)
    b = oracle.dslash_full(U32.astype(np.complex128), psi32.astype(np.complex128), dims, APBC)
    assert a.dtype == np.complex128 and np.array_equal(a, b)


def test_input_generators_are_slice_reproducible():
    dims = (4, 4, 6, 8)
    U = li.near_unit_links(dims, seed=1, eps=0.3)
    u = li.link_at(dims, 1, "near_unit", 0.3, 2, (1, 3, 5, 7))
    assert np.array_equal(u, U[2, 7, 5, 3, 1])
    psi = li.gaussian_spinor(dims, seed=2)
    s = li.gaussian_spinor_sites(dims, 2, [(1, 3, 5, 7), (0, 0, 0, 0)])
    assert np.array_equal(s[0], psi[7, 5, 3, 1]) and np.array_equal(s[1], psi[0, 0, 0, 0])
    # A11 links are smooth: <Re tr U>/3 well above 0 (SURVEY.md A11 quotes ~0.885 on 8^4)
    plaq = np.trace(U, axis1=-2, axis2=-1).real.mean() / 3
    assert 0.8 < plaq < 0.95
