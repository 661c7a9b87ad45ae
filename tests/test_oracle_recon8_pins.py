"""Pins of the 8-real link encoding oracle (oracle/recon8_oracle.py; next row f4, "RECONSTRUCT TWELVE [3]",
ref. [3] at :139).  The formulas are pinned against what SU(3) fixes, not against themselves:

R1  unpack8 of ANY admissible 8 reals is in SU(3): U U^+ = 1 and det U = 1 (LAPACK det), and reproduces the 8 reals.
R2  two links typed out by hand (a real rotation in the (0,1) plane; a complex matrix built from two phases and a
    (0,2)-plane rotation) come back entry by entry.
R3  unpack8(pack8(U)) = U for the A10 / A11 link ensembles of lattice_inputs, to fp64 rounding amplified by the
    conditioning of the encoding, eps / min(|a0|, sqrt(N2), |c0|).
R4  the singular set: N2 -> 0 loses digits like eps / sqrt(N2); N2 = 0 (unit links) does not decode (not finite).
R5  the accuracy a 32-bit store of the 8 reals gives (the bound DESIGN.md quotes for recon 8 in fp32).
"""
import numpy as np

import lattice_inputs as li
from oracle import recon8_oracle as r8

EPS64, EPS32 = 2.0 ** -53, 2.0 ** -24


def _admissible(n, seed):
    """Random admissible parameters: |a1|^2 + |a2|^2 = N2 in (0, 1), |b0|^2 <= N2, two phases in (-1, 1]."""
    rng = np.random.default_rng(seed)
    N2 = rng.uniform(0.02, 0.98, n)
    v = rng.standard_normal((n, 4))
    v *= np.sqrt(N2 / (v ** 2).sum(axis=1))[:, None]
    b = rng.standard_normal((n, 2))
    b *= (np.sqrt(N2 * rng.uniform(0.0, 1.0, n)) / np.linalg.norm(b, axis=1))[:, None]
    return np.concatenate([v, b, rng.uniform(-1, 1, (n, 2))], axis=1)


def test_R1_any_admissible_parameters_decode_to_su3():
    r = _admissible(2000, 1)
    U = r8.unpack8(r)
    eye = np.eye(3)
    assert np.abs(U @ np.conj(np.swapaxes(U, -1, -2)) - eye).max() < 1e-13
    assert np.abs(np.linalg.det(U) - 1.0).max() < 1e-13
    back = r8.pack8(U)
    # phases are defined modulo 2 (in units of pi)
    d = back - r
    d[:, 6:] = (d[:, 6:] + 1.0) % 2.0 - 1.0
    assert np.abs(d).max() < 1e-12


def test_R2_links_typed_out_by_hand():
    phi = 0.7
    c, s = np.cos(phi), np.sin(phi)
    U = np.array([[c, s, 0], [-s, c, 0], [0, 0, 1]], dtype=complex)
    r = np.array([s, 0, 0, 0, -s, 0, 0, 0.3])       # arg(c0) is arbitrary when c0 = 0
    assert np.abs(r8.unpack8(r) - U).max() < 1e-15
    # rows a = (e^{ia} cos t, 0, e^{ib} sin t), b = (0, e^{-i(a+b)}... chosen so that det = 1:
    al, be, t = 0.4, -1.1, 0.9
    ct, st = np.cos(t), np.sin(t)
    U = np.array([[np.exp(1j * al) * ct, 0, np.exp(1j * be) * st],
                  [0, 1, 0],
                  [-np.exp(-1j * be) * st, 0, np.exp(-1j * al) * ct]])
    assert abs(np.linalg.det(U) - 1) < 1e-15 and np.abs(U @ U.conj().T - np.eye(3)).max() < 1e-15
    r = np.array([0, 0, (np.exp(1j * be) * st).real, (np.exp(1j * be) * st).imag, 0, 0, al / np.pi, (np.pi - be) / np.pi - 2.0])   # arg(-e^{-i be}) = pi - be, taken in (-pi, pi]
    assert np.abs(r8.unpack8(r) - U).max() < 1e-15
    assert np.abs(r8.pack8(U) - r).max() < 1e-15


def _conditioning(U):
    """1 / min(|a0|, sqrt(N2), |c0|): the moduli the decoder gets from differences (1 - N2, N2 - |b0|^2) and divides by."""
    N2 = np.abs(U[..., 0, 1]) ** 2 + np.abs(U[..., 0, 2]) ** 2
    return 1.0 / np.maximum(np.minimum(np.minimum(np.abs(U[..., 0, 0]), np.sqrt(N2)), np.abs(U[..., 2, 0])), 1e-300)


def test_R3_ensembles_round_trip():
    for U in (li.random_su3_links((8, 8, 8, 16)), li.near_unit_links((8, 8, 8, 16), eps=0.3), li.links_for_config(1)):
        V = r8.unpack8(r8.pack8(U))
        err = np.abs(V - U).reshape(*U.shape[:-2], 9).max(axis=-1)
        assert (err <= 40 * EPS64 * _conditioning(U)).all()
        assert err.max() < 1e-12
        assert np.abs(np.linalg.det(V) - 1).max() < 1e-12


def test_R4_singular_set():
    base = li.random_su3_links((4, 4, 4, 4), seed=9)[0, 0, 0, 0]          # 4 links
    for N in (1e-2, 1e-4, 1e-6):
        # left-multiplying by a (0,1),(0,2)-plane rotation of small angle on a block-diagonal link gives N2 ~ N^2
        blk = np.zeros_like(base)
        blk[..., 0, 0] = np.exp(1j * 0.3)
        w = li.random_su3_field((4, 4, 4, 4), seed=11)[0, 0, 0]
        q, _ = np.linalg.qr(w[..., 1:, 1:])
        q = q * (np.exp(-1j * 0.3) / np.linalg.det(q))[..., None, None] ** 0.5
        blk[..., 1:, 1:] = q
        g = np.zeros_like(base)
        g[...] = np.eye(3)
        g[..., 0, 0] = g[..., 1, 1] = np.cos(N)
        g[..., 0, 1], g[..., 1, 0] = np.sin(N), -np.sin(N)
        U = blk @ g
        assert np.abs(np.linalg.det(U) - 1).max() < 1e-12
        N2 = r8.min_N2(U)
        assert 0.2 * N * N < N2 < 5 * N * N
        err = np.abs(r8.unpack8(r8.pack8(U)) - U).max()
        assert err <= 40 * EPS64 * _conditioning(U).max()
    unit = li.unit_links((4, 4, 4, 4))
    assert r8.min_N2(unit) == 0.0
    assert not np.isfinite(r8.unpack8(r8.pack8(unit))).all()


def test_R5_accuracy_of_a_32_bit_store():
    """fp32 runs (reading A14): the links are rounded to complex64 once; the 8 reals of the rounded link are stored as
    fp32.  Field-wide the decoded link differs from the rounded one by ~1e-7 (relative Frobenius norm); the worst
    link by eps32 x conditioning."""
    for U in (li.random_su3_links((8, 8, 8, 16)), li.near_unit_links((8, 8, 8, 16), eps=0.3)):
        U32 = U.astype(np.complex64).astype(np.complex128)
        V = r8.unpack8(r8.pack8(U32).astype(np.float32))
        rel = np.sqrt((np.abs(V - U32) ** 2).sum() / (np.abs(U32) ** 2).sum())
        assert rel < 3e-7
        err = np.abs(V - U32).reshape(*U.shape[:-2], 9).max(axis=-1)
        assert (err <= 8 * EPS32 * _conditioning(U)).all()
