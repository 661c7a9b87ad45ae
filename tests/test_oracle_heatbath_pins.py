"""Pins of the heatbath oracle (oracle/heatbath_oracle.py; "SU(3) heatbath algorithm [20]") against what
the definitions and the mathematics fix, none of it computed by the oracle's own formulas:

  H1  staples: changing one link changes the action, evaluated from the plaquette definition, by
      -(beta/3) Re tr((U' - U) A); the plaquette of unit links and of a pure gauge is 1; one hand-built plaquette
  H2  Kennedy-Pendleton: mean and second moment of a0 against numerical quadrature of sqrt(1 - a0^2) exp(alpha a0);
      a step with no accepted attempt is the identity
  H3  a Cabibbo-Marinari step multiplies by an SU(3) matrix that is the identity outside its 2x2 block; updated links
      stay in SU(3); links of the other sublattices are untouched bit for bit
  H4  the SU(2) element the step produces: a = g V/k has the a0 of the sampler and a direction with <a_i> = 0, i.e.
      Re tr of the block of G W equals 2 k a0
  H5  physics at both ends of the coupling: strong coupling <P> = beta/18 + O(beta^2), weak coupling (equipartition of the
      24 non-gauge degrees of freedom per site over 6 plaquettes) <1 - P> = 2/beta + O(1/beta^2)
  H6  reunitarise: the result is in SU(3) for arbitrary input; an SU(3) matrix is a fixed point; a perturbed one moves by
      no more than the perturbation's order; rows 0 and 1 are what a library QR of U^+ gives (Gram-Schmidt on the rows
      of U is the QR factorisation of U^+ with a positive real diagonal of R); one hand-worked matrix
"""
import numpy as np
import pytest
from scipy import integrate

import lattice_inputs as li
from oracle import heatbath_oracle as hb

DIMS = (4, 4, 4, 4)


def _plaq_sum_bruteforce(U, dims):
    """sum over all plaquettes of Re tr U_p with explicit site loops and modulo indexing (no roll)."""
    X, Y, Z, T = dims
    L = (X, Y, Z, T)
    tot = 0.0
    for t in range(T):
        for z in range(Z):
            for y in range(Y):
                for x in range(X):
                    c = [x, y, z, t]
                    for mu in range(4):
                        for nu in range(mu + 1, 4):
                            cm, cn = list(c), list(c)
                            cm[mu] = (cm[mu] + 1) % L[mu]
                            cn[nu] = (cn[nu] + 1) % L[nu]
                            g = lambda d, s: U[d][s[3], s[2], s[1], s[0]]
                            P = g(mu, c) @ g(nu, cm) @ g(mu, cn).conj().T @ g(nu, c).conj().T
                            tot += np.trace(P).real
    return tot


def test_H1_staple_is_the_derivative_of_the_action():
    U = li.random_su3_links(DIMS, seed=7)
    beta = 5.7
    nplaq = 6 * 4 ** 4
    S0 = beta * (nplaq - _plaq_sum_bruteforce(U, DIMS) / 3.0)
    assert abs(hb.action(U, beta) - S0) <= 1e-9 * abs(S0)
    rng = np.random.default_rng(3)
    for mu, (x, y, z, t) in ((0, (1, 2, 3, 0)), (1, (0, 0, 0, 0)), (2, (3, 3, 3, 3)), (3, (2, 0, 1, 3))):
        new = li.random_su3_links((4, 4, 4, 4), seed=int(rng.integers(1 << 30)))[0][0, 0, 0, 0]
        V = U.copy()
        V[mu][t, z, y, x] = new
        S1 = beta * (nplaq - _plaq_sum_bruteforce(V, DIMS) / 3.0)
        A = hb.staple_sum(U, mu)[t, z, y, x]
        assert abs((S1 - S0) + beta / 3.0 * np.trace((new - U[mu][t, z, y, x]) @ A).real) <= 1e-10 * abs(S0)


def test_H1_plaquette_special_cases():
    unit = li.unit_links(DIMS)
    assert hb.plaquette(unit) == pytest.approx(1.0, abs=1e-15)
    # pure gauge: U_mu(x) = g(x) g(x+mu)^+ has every plaquette equal to 1
    g = li.random_su3_field(DIMS, seed=5)
    pure = np.stack([g @ np.conj(np.swapaxes(np.roll(g, -1, axis=3 - mu), -1, -2)) for mu in range(4)])
    assert hb.plaquette(pure) == pytest.approx(1.0, abs=1e-13)
    # one link of the unit field replaced by diag(e^{ia}, e^{-ia}, 1): its 6 plaquettes have Re tr = 2 cos a + 1
    a = 0.7
    V = unit.copy()
    V[2][1, 2, 3, 0] = np.diag([np.exp(1j * a), np.exp(-1j * a), 1.0])
    n = 6 * 4 ** 4
    assert hb.plaquette(V) == pytest.approx(((n - 6) + 6 * (2 * np.cos(a) + 1) / 3.0) / n, abs=1e-14)


@pytest.mark.parametrize("alpha", [0.7, 2.5, 9.0])
def test_H2_kennedy_pendleton_distribution(alpha):
    rng = np.random.default_rng(11)
    n = 400000
    r = 1.0 - rng.random((n, 4 * 40))
    a0, acc = hb.kennedy_pendleton(np.full(n, alpha), r)
    assert acc.mean() > 0.999
    a0 = a0[acc]
    w = lambda x: np.sqrt(1 - x * x) * np.exp(alpha * x)
    norm = integrate.quad(w, -1, 1)[0]
    m1 = integrate.quad(lambda x: x * w(x), -1, 1)[0] / norm
    m2 = integrate.quad(lambda x: x * x * w(x), -1, 1)[0] / norm
    assert abs(a0.mean() - m1) <= 5 * a0.std() / np.sqrt(len(a0))
    assert abs((a0 ** 2).mean() - m2) <= 5 * (a0 ** 2).std() / np.sqrt(len(a0))
    assert a0.min() >= -1.0 and a0.max() <= 1.0
    # uniforms that reject every attempt (r4 = 1, lambda^2 > 0): nothing accepted
    bad = np.ones((5, 8))
    bad[:, 0::4] = 0.5
    _, acc0 = hb.kennedy_pendleton(np.full(5, alpha), bad)
    assert not acc0.any()


def test_H3_steps_stay_in_the_group_and_touch_only_their_sublattice():
    U = li.random_su3_links(DIMS, seed=21)
    Vh = 4 ** 4 // 2
    rng = np.random.default_rng(2)
    u = 1.0 - rng.random((Vh, 3, 4 * 6 + 2))
    W = rng.standard_normal((50, 3, 3)) + 1j * rng.standard_normal((50, 3, 3))
    for (i, j) in hb.SUBGROUPS:
        G = hb.su2_update(W, i, j, 5.0, u[:50, 0])
        k = 3 - i - j
        assert np.allclose(G @ np.conj(np.swapaxes(G, -1, -2)), np.eye(3), atol=1e-14)
        assert np.allclose(np.linalg.det(G), 1.0, atol=1e-14)
        assert np.all(G[:, k, k] == 1.0) and np.all(G[:, k, i] == 0) and np.all(G[:, i, k] == 0) and np.all(G[:, k, j] == 0) and np.all(G[:, j, k] == 0)
    # rejected everywhere: the identity
    bad = np.ones((50, 4 * 6 + 2))
    bad[:, 0:24:4] = 0.5
    assert np.array_equal(hb.su2_update(W, 0, 1, 5.0, bad), np.broadcast_to(np.eye(3), W.shape))
    mu, parity = 2, 1
    V = hb.heatbath_sublattice(U, 5.7, mu, parity, u)
    mask = li.parity_mask(DIMS, parity)
    for nu in range(4):
        if nu != mu:
            assert np.array_equal(V[nu], U[nu])
    assert np.array_equal(V[mu][~mask], U[mu][~mask]) and not np.array_equal(V[mu][mask], U[mu][mask])
    new = V[mu][mask]
    assert np.allclose(new @ np.conj(np.swapaxes(new, -1, -2)), np.eye(3), atol=1e-13)
    assert np.allclose(np.linalg.det(new), 1.0, atol=1e-13)


def test_H4_the_step_draws_a_times_the_staple_direction():
    """For a fixed W the block of G W has Re tr = 2 k a0 with a0 from the sampler, and the direction of a is isotropic."""
    rng = np.random.default_rng(31)
    n = 200000
    W1 = rng.standard_normal((3, 3)) + 1j * rng.standard_normal((3, 3))
    W = np.broadcast_to(W1, (n, 3, 3))
    beta, (i, j) = 4.0, (0, 2)
    r = 1.0 - rng.random((n, 4 * 30 + 2))
    G = hb.su2_update(W, i, j, beta, r)
    GW = G @ W
    v = np.array([(W1[i, i] + W1[j, j]).real, (W1[i, j] + W1[j, i]).imag, (W1[i, j] - W1[j, i]).real, (W1[i, i] - W1[j, j]).imag]) / 2
    k = np.linalg.norm(v)
    a0_expected, acc = hb.kennedy_pendleton(np.full(n, 2 * beta * k / 3), r[:, :-2])
    a0 = (GW[:, i, i] + GW[:, j, j]).real / (2 * k)
    assert np.allclose(a0[acc], a0_expected[acc], atol=1e-12)
    a3 = (GW[:, i, i] - GW[:, j, j]).imag / (2 * k)
    a1 = (GW[:, i, j] + GW[:, j, i]).imag / (2 * k)
    a2 = (GW[:, i, j] - GW[:, j, i]).real / (2 * k)
    assert np.allclose(a0 ** 2 + a1 ** 2 + a2 ** 2 + a3 ** 2, 1.0, atol=1e-12)
    for a in (a1, a2, a3):
        assert abs(a[acc].mean()) <= 5 * a.std() / np.sqrt(n)
    # isotropy of the direction: <a_i^2> equal for i = 1, 2, 3
    m = [np.mean(a[acc] ** 2) for a in (a1, a2, a3)]
    assert max(m) - min(m) <= 0.01 * np.mean(m) + 5 * np.std(a1 ** 2) / np.sqrt(n)


def test_H5_strong_and_weak_coupling_plaquette():
    rng = np.random.default_rng(77)
    # strong coupling: <P> = beta/18 + O(beta^2)
    beta = 0.4
    U = li.random_su3_links(DIMS, seed=9)
    P = []
    for s in range(90):
        U = hb.sweep(U, beta, rng, ntries=8)
        if s >= 10:
            P.append(hb.plaquette(U))
    assert abs(np.mean(P) - beta / 18) <= 0.004, np.mean(P)
    # weak coupling: <1 - P> = 2/beta (24 quadratic modes per site, 6 plaquettes per site), up to O(1/beta^2) and the
    # zero modes of a 4^4 torus
    beta = 48.0
    U = li.unit_links(DIMS)
    P = []
    for s in range(60):
        U = hb.sweep(U, beta, rng, ntries=4)
        if s >= 20:
            P.append(hb.plaquette(U))
    assert abs((1 - np.mean(P)) * beta / 2 - 1.0) <= 0.08, (1 - np.mean(P)) * beta / 2


def test_H6_reunitarise_projects_to_su3():
    rng = np.random.default_rng(66)
    # (i) arbitrary complex matrices end up unitary with det = +1
    A = rng.standard_normal((500, 3, 3)) + 1j * rng.standard_normal((500, 3, 3))
    P = hb.reunitarise(A)
    assert np.abs(P @ np.conj(np.swapaxes(P, -1, -2)) - np.eye(3)).max() < 5e-15
    assert np.abs(np.linalg.det(P) - 1.0).max() < 5e-15
    # (ii) rows 0 and 1 against the library QR of A^+ : A^+ = Q R  =>  rows of A = R^+ Q^+, so with the phases of diag(R)
    # removed the rows of Q^+ are the Gram-Schmidt rows.  (Row 2 is fixed by det = +1, checked in (i).)
    for a, p in zip(A[:50], P[:50]):
        Q, R = np.linalg.qr(np.conj(a.T))
        ph = np.diag(R) / np.abs(np.diag(R))
        rows = np.conj((Q * ph).T)
        assert np.abs(rows[:2] - p[:2]).max() < 1e-13
    # (iii) SU(3) matrices are fixed points; a perturbation of size d moves the projection by O(d) and not more
    U = li.random_su3_links((4, 4, 4, 4), seed=9)
    assert np.abs(hb.reunitarise(U) - U).max() < 1e-15
    d = 1e-9
    noisy = U + d * (rng.standard_normal(U.shape) + 1j * rng.standard_normal(U.shape))
    back = hb.reunitarise(noisy)
    assert 0 < np.abs(back - U).max() < 20 * d
    assert np.abs(back @ np.conj(np.swapaxes(back, -1, -2)) - np.eye(3)).max() < 5e-15
    # (iv) by hand: rows (2, 0, 0), (1, 1, 0), anything -> e0, e1, and e0 x e1 = e2 (real, so conj changes nothing);
    # with a phase on row 0: row0 = i e0, row1 = e1  =>  row2 = conj(i e0 x e1) = conj(i e2) = -i e2, det = i * 1 * (-i) = 1
    M = np.array([[2, 0, 0], [1, 1, 0], [7, 7, 7]], dtype=complex)
    assert np.allclose(hb.reunitarise(M), np.eye(3), atol=1e-15)
    M = np.array([[3j, 0, 0], [5, 2, 0], [0, 0, 0]], dtype=complex)
    assert np.allclose(hb.reunitarise(M), np.diag([1j, 1, -1j]), atol=1e-15)

