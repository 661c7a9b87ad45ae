"""Second, independently written CPU formulation of the Wilson hopping term (pin P10).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Whole-field numpy.roll shifts + einsum instead of
the C oracle's per-site loop, and gamma matrices BUILT from Pauli matrices
(gamma_mu = [[0, A_mu], [A_mu^dagger, 0]], A_x,y,z = -i sigma_1,2,3, A_t = -1; SURVEY.md
Appendix A.2) instead of typed in as a table -- so a typo in either shows up as a mismatch.

Same definition as oracle/wilson_oracle.c:
    (H psi)(x) = sum_mu [(1 - g_mu) U_mu(x) psi(x+mu^) + (1 + g_mu) U_mu(x-mu^)^+ psi(x-mu^)],
    psi(x + L_mu mu^) = bc_mu psi(x).
Canonical layout: psi [T][Z][Y][X][4][3], U [4][T][Z][Y][X][3][3], dims = (X,Y,Z,T).
"""
from __future__ import annotations

import numpy as np

_SIGMA = [
    np.array([[0, 1], [1, 0]], dtype=np.complex128),
    np.array([[0, -1j], [1j, 0]], dtype=np.complex128),
    np.array([[1, 0], [0, -1]], dtype=np.complex128),
]


def gamma_from_pauli(mu: int) -> np.ndarray:
    a = -1j * _SIGMA[mu] if mu < 3 else -np.eye(2, dtype=np.complex128)
    z = np.zeros((2, 2), dtype=np.complex128)
    return np.block([[z, a], [a.conj().T, z]])


def _axis(mu: int) -> int:
    # array axes are [T][Z][Y][X]: direction mu = 0(x) is axis 3, ..., mu = 3(t) is axis 0
    return 3 - mu


def dslash_roll(U: np.ndarray, psi: np.ndarray, dims, bc) -> np.ndarray:
    U = np.asarray(U, dtype=np.complex128)
    psi = np.asarray(psi, dtype=np.complex128)
    bc = np.asarray(bc, dtype=np.complex128)
    out = np.zeros_like(psi)
    one = np.eye(4, dtype=np.complex128)
    for mu in range(4):
        ax = _axis(mu)
        L = dims[mu]
        g = gamma_from_pauli(mu)

        # psi(x + mu^): shift the field down by one; the last slab wrapped around -> times bc
        fwd = np.roll(psi, -1, axis=ax)
        idx = [slice(None)] * 4
        idx[ax] = L - 1
        fwd[tuple(idx)] *= bc[mu]
        w = np.einsum("...ab,...sb->...sa", U[mu], fwd)
        out += np.einsum("st,...ta->...sa", one - g, w)

        # U_mu(x - mu^)^+ psi(x - mu^): multiply at the source site, then shift up by one
        w = np.einsum("...ba,...sb->...sa", U[mu].conj(), psi)
        bwd = np.roll(w, +1, axis=ax)
        idx[ax] = 0
        bwd[tuple(idx)] *= np.conj(bc[mu])
        out += np.einsum("st,...ta->...sa", one + g, bwd)
    return out
