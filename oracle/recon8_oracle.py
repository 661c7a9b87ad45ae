"""8-real SU(3) link encoding (next row f4) -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

The paper names link compression as the bandwidth lever of the dslash kernel ("RECONSTRUCT TWELVE [3]", PAPER.md:89;
ref. [3] at PAPER.md:139 also describes the minimal 8-parameter storage).  The paper prints no formula; this is the
parametrisation written out from the defining properties of SU(3) (rows orthonormal, det = 1), in plain fp64 numpy,
one link at a time in vectorised form, no blocking or reordering.

With the rows of U called a, b, c (U[0] = a, U[1] = b, U[2] = c), the 8 stored reals are

    r = ( Re a1, Im a1, Re a2, Im a2, Re b0, Im b0, arg(a0) / pi, arg(c0) / pi )

and U is rebuilt from them as follows (N2 = |a1|^2 + |a2|^2):

    |a0|^2 = 1 - N2                      (row a has unit norm)          a0 = |a0| exp(i pi r6)
    |c0|^2 = N2 - |b0|^2                 (column 0 has unit norm)       c0 = |c0| exp(i pi r7)
    b1 = -(a1 conj(a0) b0 + conj(a2) conj(c0)) / N2                     (a . conj(b) = 0  and  c0 = conj(a1 b2 - a2 b1),
    b2 =  (conj(a1) conj(c0) - a2 conj(a0) b0) / N2                      a 2 x 2 linear system for b1, b2 of determinant N2)
    c  = conj(a x b)                                                    (det U = 1; the same step as 12-real storage)

The encoding is singular for N2 = 0 (|U00| = 1, e.g. unit links): then b0 = c0 = 0 and the lower-right 2 x 2 block is
not determined by the 8 reals.  `min_N2` reports how close a field comes to that.
Imports nothing from paper_1112_5280_b200.
"""
from __future__ import annotations

import numpy as np


def pack8(U: np.ndarray) -> np.ndarray:
    """[..., 3, 3] complex -> [..., 8] float64."""
    U = np.asarray(U, dtype=np.complex128)
    a1, a2, b0 = U[..., 0, 1], U[..., 0, 2], U[..., 1, 0]
    return np.stack([a1.real, a1.imag, a2.real, a2.imag, b0.real, b0.imag,
                     np.angle(U[..., 0, 0]) / np.pi, np.angle(U[..., 2, 0]) / np.pi], axis=-1)


def unpack8(r: np.ndarray) -> np.ndarray:
    """[..., 8] real -> [..., 3, 3] complex128, by the formulas of the module header."""
    r = np.asarray(r, dtype=np.float64)
    a1 = r[..., 0] + 1j * r[..., 1]
    a2 = r[..., 2] + 1j * r[..., 3]
    b0 = r[..., 4] + 1j * r[..., 5]
    N2 = np.abs(a1) ** 2 + np.abs(a2) ** 2
    a0 = np.sqrt(np.maximum(1.0 - N2, 0.0)) * np.exp(1j * np.pi * r[..., 6])
    c0 = np.sqrt(np.maximum(N2 - np.abs(b0) ** 2, 0.0)) * np.exp(1j * np.pi * r[..., 7])
    with np.errstate(divide="ignore", invalid="ignore"):
        b1 = -(a1 * np.conj(a0) * b0 + np.conj(a2) * np.conj(c0)) / N2
        b2 = (np.conj(a1) * np.conj(c0) - a2 * np.conj(a0) * b0) / N2
    a = np.stack([a0, a1, a2], axis=-1)
    b = np.stack([b0, b1, b2], axis=-1)
    c = np.conj(np.cross(a, b))
    return np.stack([a, b, c], axis=-2)


def min_N2(U: np.ndarray) -> float:
    """Smallest |U01|^2 + |U02|^2 over the field: the distance from the singular set of the encoding."""
    U = np.asarray(U)
    return float((np.abs(U[..., 0, 1]) ** 2 + np.abs(U[..., 0, 2]) ** 2).min())
