"""Pure-gauge SU(3) heatbath oracle (next row f4, last clause) -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

"On the PGT side we need a SU(3) heatbath algorithm [20]" (the heatbath is the task the paper runs
beside the inverter).  Ref. [20] is Creutz's heatbath, the Cabibbo-Marinari sweep over
SU(2) subgroups and the Kennedy-Pendleton SU(2) sampler; the paper prints none of them.  This file follows those three
papers step by step in fp64 numpy (reading F7), vectorised over the links of one sublattice only:

  action     S = beta sum_plaquettes (1 - 1/3 Re tr U_p),   U_p = U_mu(x) U_nu(x+mu^) U_mu(x+nu^)^+ U_nu(x)^+
  staples    A_mu(x) = sum_{nu != mu} [ U_nu(x+mu^) U_mu(x+nu^)^+ U_nu(x)^+  +  U_nu(x+mu^-nu^)^+ U_mu(x-nu^)^+ U_nu(x-nu^) ]
             so that the part of S that contains U_mu(x) is  -(beta/3) Re tr( U_mu(x) A_mu(x) )
  sublattice the links U_mu(x) of one direction mu on the sites of one parity do not see each other through the action:
             they are updated together (8 sublattices make a sweep)
  subgroups  (Cabibbo-Marinari) for (i, j) in (0,1), (0,2), (1,2), in this order: W = U A; the 2x2 block of W in rows and
             columns i, j is v0 + i sigma.v plus a part that drops out of Re tr, with
                 v0 = Re(W_ii + W_jj)/2, v1 = Im(W_ij + W_ji)/2, v2 = Re(W_ij - W_ji)/2, v3 = Im(W_ii - W_jj)/2,
             k = |v|.  Left multiplication of U by an SU(2) element g embedded in that block changes the action by
             -(beta/3) 2 k a0, a = g (v0 + i sigma.v)/k, so a is drawn with density sqrt(1 - a0^2) exp(alpha a0),
             alpha = 2 beta k / 3, direction of (a1, a2, a3) uniform, and g = a (v0 - i sigma.v)/k;  U <- G U
  a0         (Kennedy-Pendleton) from uniforms r1..r4 in (0, 1]:  lambda^2 = -(ln r1 + cos^2(2 pi r2) ln r3) / (2 alpha);
             accept if r4^2 <= 1 - lambda^2, then a0 = 1 - 2 lambda^2.  At most `ntries` attempts; if none is accepted
             the subgroup is left alone (the acceptance probability depends on alpha only, not on U, so the step is a
             mixture of the heatbath and the identity and keeps the Boltzmann weight invariant)
  direction  cos(theta) = 2 u5 - 1, phi = 2 pi u6:  a1 = s sin(theta) cos(phi), a2 = s sin(theta) sin(phi),
             a3 = s cos(theta), s = sqrt(1 - a0^2)

Random numbers are INPUTS (the method's uniforms are passed in by the caller, the same array to the oracle and to the
CUDA path): uniforms[site cb of the sublattice][subgroup 3][4 ntries + 2], the 4 numbers of attempt t at [4 t, 4 t + 4),
the two direction numbers last.  Links are periodic and carry no boundary phase (reading A6).
Arrays: links [4][T][Z][Y][X][3][3] complex128 (canonical layout).  Imports nothing from paper_1112_5280_b200.

  reunitarise  every update multiplies a link by a rounded SU(2) element, so over many sweeps the links drift off the
             group by accumulated rounding.  The standard cure (reading F8; it is the "Gram-Schmidt
             reunitarised" construction BASELINE.json's configs name for the random links) projects a link back:
                 row0 <- row0 / |row0|;  row1 <- row1 - <row0, row1> row0, then / |row1|;  row2 <- conj(row0 x row1)
             which is unitary with det = +1 by construction and leaves an exact SU(3) matrix unchanged.
"""
from __future__ import annotations

import numpy as np

SUBGROUPS = ((0, 1), (0, 2), (1, 2))


def _shift(F: np.ndarray, mu: int, steps: int) -> np.ndarray:
    """F(x + steps mu^) as a field of x; site axes are [T][Z][Y][X], so direction mu is axis 3 - mu."""
    return np.roll(F, -steps, axis=3 - mu)


def _dag(M: np.ndarray) -> np.ndarray:
    return np.conj(np.swapaxes(M, -1, -2))


def staple_sum(U: np.ndarray, mu: int) -> np.ndarray:
    """A_mu(x) on all sites: the six staples written out as in the header."""
    A = np.zeros(U.shape[1:], dtype=np.complex128)
    for nu in range(4):
        if nu == mu:
            continue
        # upper staple: U_nu(x+mu) U_mu(x+nu)^+ U_nu(x)^+
        A += _shift(U[nu], mu, 1) @ _dag(_shift(U[mu], nu, 1)) @ _dag(U[nu])
        # lower staple: U_nu(x+mu-nu)^+ U_mu(x-nu)^+ U_nu(x-nu)
        Unu_dn = _shift(U[nu], nu, -1)
        A += _dag(_shift(Unu_dn, mu, 1)) @ _dag(_shift(U[mu], nu, -1)) @ Unu_dn
    return A


def plaquette(U: np.ndarray) -> float:
    """Average of 1/3 Re tr U_p over the 6 V plaquettes, from the definition."""
    total, n = 0.0, 0
    for mu in range(4):
        for nu in range(mu + 1, 4):
            P = U[mu] @ _shift(U[nu], mu, 1) @ _dag(_shift(U[mu], nu, 1)) @ _dag(U[nu])
            total += float(np.trace(P, axis1=-2, axis2=-1).real.sum())
            n += P.shape[0] * P.shape[1] * P.shape[2] * P.shape[3]
    return total / (3.0 * n)


def action(U: np.ndarray, beta: float) -> float:
    """S = beta sum_p (1 - 1/3 Re tr U_p)."""
    nplaq = 6 * U.shape[1] * U.shape[2] * U.shape[3] * U.shape[4]
    return beta * nplaq * (1.0 - plaquette(U))


def kennedy_pendleton(alpha: np.ndarray, r: np.ndarray):
    """a0 for every element of alpha from the uniforms r[..., 4 ntries]; returns (a0, accepted)."""
    ntries = r.shape[-1] // 4
    a0 = np.ones_like(alpha)
    accepted = np.zeros(alpha.shape, dtype=bool)
    for t in range(ntries):
        r1, r2, r3, r4 = (r[..., 4 * t + j] for j in range(4))
        c = np.cos(2.0 * np.pi * r2)
        lam2 = -(np.log(r1) + c * c * np.log(r3)) / (2.0 * alpha)
        ok = (~accepted) & (r4 * r4 <= 1.0 - lam2)
        a0 = np.where(ok, 1.0 - 2.0 * lam2, a0)
        accepted |= ok
    return a0, accepted


def su2_update(W: np.ndarray, i: int, j: int, beta: float, r: np.ndarray) -> np.ndarray:
    """The 3x3 matrices G (identity outside rows / columns i, j) of one Cabibbo-Marinari step for W = U A;
    r[..., 4 ntries + 2] are the step's uniforms."""
    v0 = 0.5 * (W[..., i, i] + W[..., j, j]).real
    v3 = 0.5 * (W[..., i, i] - W[..., j, j]).imag
    v1 = 0.5 * (W[..., i, j] + W[..., j, i]).imag
    v2 = 0.5 * (W[..., i, j] - W[..., j, i]).real
    k = np.sqrt(v0 * v0 + v1 * v1 + v2 * v2 + v3 * v3)
    alpha = 2.0 * beta * k / 3.0
    a0, accepted = kennedy_pendleton(alpha, r[..., :-2])
    s = np.sqrt(np.maximum(1.0 - a0 * a0, 0.0))
    ct = 2.0 * r[..., -2] - 1.0
    st = np.sqrt(np.maximum(1.0 - ct * ct, 0.0))
    phi = 2.0 * np.pi * r[..., -1]
    a1, a2, a3 = s * st * np.cos(phi), s * st * np.sin(phi), s * ct
    # g = a vbar / k with a = a0 + i sigma.a, vbar = v0 - i sigma.v  (quaternion product)
    b0, b1, b2, b3 = v0 / k, -v1 / k, -v2 / k, -v3 / k
    g0 = a0 * b0 - a1 * b1 - a2 * b2 - a3 * b3
    g1 = a0 * b1 + a1 * b0 - (a2 * b3 - a3 * b2)
    g2 = a0 * b2 + a2 * b0 - (a3 * b1 - a1 * b3)
    g3 = a0 * b3 + a3 * b0 - (a1 * b2 - a2 * b1)
    # not accepted: the identity
    g0 = np.where(accepted, g0, 1.0)
    g1, g2, g3 = (np.where(accepted, x, 0.0) for x in (g1, g2, g3))
    G = np.zeros(W.shape, dtype=np.complex128)
    for d in range(3):
        G[..., d, d] = 1.0
    # g0 + i sigma.g = [[g0 + i g3, g2 + i g1], [-g2 + i g1, g0 - i g3]]
    G[..., i, i] = g0 + 1j * g3
    G[..., i, j] = g2 + 1j * g1
    G[..., j, i] = -g2 + 1j * g1
    G[..., j, j] = g0 - 1j * g3
    return G


def heatbath_sublattice(U: np.ndarray, beta: float, mu: int, parity: int, uniforms: np.ndarray) -> np.ndarray:
    """One heatbath update of the links U_mu(x), x of the given parity; returns the new field (U is not modified).
    uniforms: [V/2][3][4 ntries + 2], sites of the sublattice in lexicographic order (cb = lex >> 1)."""
    U = np.array(U, dtype=np.complex128, copy=True)
    T, Z, Y, X = U.shape[1:5]
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(Z), np.arange(Y), np.arange(X), indexing="ij")
    mask = ((x + y + z + t) & 1) == parity
    A = staple_sum(U, mu)[mask]                    # [V/2][3][3], lexicographic order of the sites
    Ul = U[mu][mask]
    r = np.asarray(uniforms, dtype=np.float64).reshape(Ul.shape[0], 3, -1)
    for n, (i, j) in enumerate(SUBGROUPS):
        W = Ul @ A
        Ul = su2_update(W, i, j, beta, r[:, n]) @ Ul
    U[mu][mask] = Ul
    return U


def sweep(U: np.ndarray, beta: float, rng: np.random.Generator, ntries: int = 8) -> np.ndarray:
    """All 8 sublattices once (mu = 0..3, parity 0, 1), uniforms in (0, 1] drawn from rng in that order."""
    Vh = U.shape[1] * U.shape[2] * U.shape[3] * U.shape[4] // 2
    for mu in range(4):
        for parity in (0, 1):
            u = 1.0 - rng.random((Vh, 3, 4 * ntries + 2))
            U = heatbath_sublattice(U, beta, mu, parity, u)
    return U


def reunitarise(U: np.ndarray) -> np.ndarray:
    """Project every 3x3 matrix of U[..., 3, 3] back to SU(3): Gram-Schmidt on rows 0 and 1 in this order, with
    <a, b> = sum_k conj(a_k) b_k, then row 2 = conj(row 0 x row 1).  Returns a new array."""
    U = np.asarray(U, dtype=np.complex128)
    r0 = U[..., 0, :]
    r0 = r0 / np.sqrt(np.sum(np.abs(r0) ** 2, axis=-1, keepdims=True))
    r1 = U[..., 1, :]
    r1 = r1 - np.sum(np.conj(r0) * r1, axis=-1, keepdims=True) * r0
    r1 = r1 / np.sqrt(np.sum(np.abs(r1) ** 2, axis=-1, keepdims=True))
    r2 = np.conj(np.cross(r0, r1))
    return np.stack([r0, r1, r2], axis=-2)

