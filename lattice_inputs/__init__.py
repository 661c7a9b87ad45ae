"""Seeded synthetic input generators shared by the tests, the oracle legs and bench.py.

This module holds NO arithmetic of the method (no hopping term, no gamma
matrices, no projection): it only draws random numbers and shapes them into
the canonical interchange layout of SURVEY.md Appendix A.4:

    spinor  [T][Z][Y][X][spin 4][colour 3]           complex
    links   [mu 4][T][Z][Y][X][row 3][col 3]          complex, (U psi)_a = sum_b U[a][b] psi_b

Both the CPU oracle and the CUDA path are always fed THE SAME arrays produced
here; neither generates its own.

Recipe (stated in DESIGN.md "Input recipe"):
  * every (mu, t) link slice and every t spinor slice has its own counter-based
    stream  numpy.random.default_rng([seed, mu, t])  /  default_rng([seed, t]),
    real parts drawn first, then imaginary parts, in C order [z][y][x][..];
    so any sub-volume can be regenerated independently and in parallel.
  * A10 "random SU(3)": A = G1 + i G2, Gram-Schmidt on rows 0,1, row2 = conj(row0 x row1)
    (det = +1 exactly, which 12-real link storage needs).
  * A11 "near a thermalised ensemble": H = (A + A^dagger)/2 - tr/3, U = exp(i eps H) (scaled Taylor series),
    then one A10 pass.
dims are always given as (X, Y, Z, T)  (mu = 0,1,2,3 = x,y,z,t).
"""
from __future__ import annotations

from concurrent.futures import ThreadPoolExecutor
import os

import numpy as np

__all__ = [
    "CONFIGS", "gaussian_spinor", "random_su3_links", "near_unit_links", "unit_links",
    "random_su3_field", "plane_wave", "parity_mask", "bc_phases", "gaussian_spinor_sites",
]

# BASELINE.json configs, restated in SURVEY.md §8(d).  bc = (+,+,+,-) for all.
CONFIGS = {
    1: dict(dims=(4, 4, 4, 4), kappa=0.125, links="su3", eps=None, bc=(1, 1, 1, -1)),
    2: dict(dims=(8, 8, 8, 16), kappa=0.15, links="su3", eps=None, bc=(1, 1, 1, -1)),
    3: dict(dims=(16, 16, 16, 32), kappa=0.16, links="near_unit", eps=0.3, bc=(1, 1, 1, -1)),
    4: dict(dims=(32, 32, 32, 64), kappa=0.16, links="su3", eps=None, bc=(1, 1, 1, -1)),
    5: dict(dims=(48, 48, 48, 96), kappa=0.1615, links="near_unit", eps=0.3, bc=(1, 1, 1, -1)),
}
LINK_SEED = 1
SPINOR_SEED = 2


def _nthreads() -> int:
    try:
        return max(1, len(os.sched_getaffinity(0)))
    except AttributeError:  # pragma: no cover
        return os.cpu_count() or 1


def _complex_normal(rng: np.random.Generator, shape) -> np.ndarray:
    re = rng.standard_normal(shape)
    im = rng.standard_normal(shape)
    return re + 1j * im


def _gram_schmidt_su3(a: np.ndarray) -> np.ndarray:
    """Rows 0,1 orthonormalised, row 2 = conj(row0 x row1)."""
    r0 = a[..., 0, :]
    r0 = r0 / np.linalg.norm(r0, axis=-1, keepdims=True)
    r1 = a[..., 1, :]
    r1 = r1 - np.sum(r0.conj() * r1, axis=-1, keepdims=True) * r0
    r1 = r1 / np.linalg.norm(r1, axis=-1, keepdims=True)
    r2 = np.conj(np.cross(r0, r1))
    return np.stack([r0, r1, r2], axis=-2)


def _mul3(a, b):
    """3x3 product of two component-major stacks [3][3][n], entry by entry on contiguous whole arrays (these
    operations release the GIL, so a thread pool generates the (mu, t) slices of a field in parallel; numpy's batched
    eigh / matmul on [n][3][3] do not)."""
    return [[a[i][0] * b[0][j] + a[i][1] * b[1][j] + a[i][2] * b[2][j] for j in range(3)] for i in range(3)]


def _near_unit(a: np.ndarray, eps: float) -> np.ndarray:
    """exp(i eps H), H traceless Hermitian part of a, then one A10 pass.  The exponential is the
    Taylor series of order 12 of exp(i eps H / 8) (|eps H / 8| < 0.3 for eps = 0.3: truncation below 1e-17), squared
    three times."""
    h = 0.5 * (a + np.conj(np.swapaxes(a, -1, -2)))
    tr = np.trace(h, axis1=-2, axis2=-1) / 3.0
    h = h - tr[..., None, None] * np.eye(3)
    shape = h.shape
    hc = np.ascontiguousarray(np.moveaxis(h.reshape(-1, 3, 3), 0, -1))       # [3][3][n]
    x = [[(0.125j * eps) * hc[i, j] for j in range(3)] for i in range(3)]
    one = lambda i, j: 1.0 if i == j else 0.0
    u = [[x[i][j] / 12.0 + one(i, j) for j in range(3)] for i in range(3)]
    for k in range(11, 0, -1):          # Horner: 1 + x/1 (1 + x/2 (1 + ... (1 + x/12)))
        xu = _mul3(x, u)
        u = [[xu[i][j] / k + one(i, j) for j in range(3)] for i in range(3)]
    for _ in range(3):
        u = _mul3(u, u)
    out = np.empty(shape, dtype=np.complex128).reshape(-1, 3, 3)
    for i in range(3):
        for j in range(3):
            out[:, i, j] = u[i][j]
    return _gram_schmidt_su3(out.reshape(shape))


def _link_slice(dims, seed, mu, t, kind, eps):
    X, Y, Z, _ = dims
    a = _complex_normal(np.random.default_rng([seed, mu, t]), (Z, Y, X, 3, 3))
    if kind == "su3":
        return _gram_schmidt_su3(a)
    if kind == "near_unit":
        return _near_unit(a, eps)
    raise ValueError(kind)


def _links(dims, seed, kind, eps, dtype):
    X, Y, Z, T = dims
    out = np.empty((4, T, Z, Y, X, 3, 3), dtype=dtype)

    def work(job):
        mu, t = job
        out[mu, t] = _link_slice(dims, seed, mu, t, kind, eps)

    jobs = [(mu, t) for mu in range(4) for t in range(T)]
    nthr = _nthreads()
    if nthr > 1 and len(jobs) > 8:
        with ThreadPoolExecutor(nthr) as ex:
            list(ex.map(work, jobs))
    else:
        for j in jobs:
            work(j)
    return out


def random_su3_links(dims, seed=LINK_SEED, dtype=np.complex128) -> np.ndarray:
    """A10: iid Gaussian complex 3x3 reunitarised by Gram-Schmidt, det = +1."""
    return _links(dims, seed, "su3", None, dtype)


def near_unit_links(dims, seed=LINK_SEED, eps=0.3, dtype=np.complex128) -> np.ndarray:
    """A11: exp(i eps H) with H random traceless Hermitian."""
    return _links(dims, seed, "near_unit", eps, dtype)


def unit_links(dims, dtype=np.complex128) -> np.ndarray:
    X, Y, Z, T = dims
    out = np.zeros((4, T, Z, Y, X, 3, 3), dtype=dtype)
    out[..., 0, 0] = out[..., 1, 1] = out[..., 2, 2] = 1.0
    return out


def links_for_config(cfg_id: int, dtype=np.complex128) -> np.ndarray:
    c = CONFIGS[cfg_id]
    if c["links"] == "su3":
        return random_su3_links(c["dims"], LINK_SEED, dtype)
    return near_unit_links(c["dims"], LINK_SEED, c["eps"], dtype)


def links_time_slices(cfg_id: int, t_list, dtype=np.complex128) -> np.ndarray:
    """The time slices `t_list` of links_for_config(cfg_id): [4][len(t_list)][Z][Y][X][3][3], without generating the rest
    (every (mu, t) slice has its own random stream) -- what one rank of a time-slab decomposition needs."""
    c = CONFIGS[cfg_id]
    X, Y, Z, _ = c["dims"]
    kind = "su3" if c["links"] == "su3" else "near_unit"
    out = np.empty((4, len(t_list), Z, Y, X, 3, 3), dtype=dtype)

    def work(job):
        mu, k = job
        out[mu, k] = _link_slice(c["dims"], LINK_SEED, mu, t_list[k], kind, c["eps"])

    with ThreadPoolExecutor(_nthreads()) as ex:
        list(ex.map(work, [(mu, k) for mu in range(4) for k in range(len(t_list))]))
    return out


def gaussian_spinor_time_slices(dims, t_list, seed=SPINOR_SEED, dtype=np.complex128) -> np.ndarray:
    """The time slices `t_list` of gaussian_spinor(dims, seed)."""
    X, Y, Z, T = dims
    out = np.empty((len(t_list), Z, Y, X, 4, 3), dtype=dtype)
    for k, t in enumerate(t_list):
        out[k] = _complex_normal(np.random.default_rng([seed, t]), (Z, Y, X, 4, 3))
    return out


def link_at(dims, seed, kind, eps, mu, coords) -> np.ndarray:
    """The single link U_mu(x) of the field `_links` would produce (regenerates one (mu,t) slice)."""
    x, y, z, t = coords
    return _link_slice(dims, seed, mu, t, kind, eps)[z, y, x]


def gaussian_spinor(dims, seed=SPINOR_SEED, dtype=np.complex128) -> np.ndarray:
    """iid complex Gaussian, 12 components per site."""
    X, Y, Z, T = dims
    out = np.empty((T, Z, Y, X, 4, 3), dtype=dtype)
    for t in range(T):
        out[t] = _complex_normal(np.random.default_rng([seed, t]), (Z, Y, X, 4, 3))
    return out


def gaussian_spinor_sites(dims, seed, coords_list) -> np.ndarray:
    """Spinor values at the listed (x,y,z,t) sites of gaussian_spinor(dims, seed)."""
    X, Y, Z, T = dims
    cache = {}
    out = np.empty((len(coords_list), 4, 3), dtype=np.complex128)
    for n, (x, y, z, t) in enumerate(coords_list):
        if t not in cache:
            cache[t] = _complex_normal(np.random.default_rng([seed, t]), (Z, Y, X, 4, 3))
        out[n] = cache[t][z, y, x]
    return out


def random_su3_field(dims, seed) -> np.ndarray:
    """g(x) in SU(3) per site, [T][Z][Y][X][3][3]; for the gauge-covariance pin P5."""
    X, Y, Z, T = dims
    a = _complex_normal(np.random.default_rng([seed, 777]), (T, Z, Y, X, 3, 3))
    return _gram_schmidt_su3(a)


def site_coords(dims):
    """Integer coordinate arrays x,y,z,t of shape [T][Z][Y][X]."""
    X, Y, Z, T = dims
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(Z), np.arange(Y), np.arange(X), indexing="ij")
    return x, y, z, t


def parity_mask(dims, parity: int) -> np.ndarray:
    """Boolean [T][Z][Y][X]: True where (x+y+z+t) mod 2 == parity."""
    x, y, z, t = site_coords(dims)
    return ((x + y + z + t) & 1) == parity


def bc_phases(bc) -> np.ndarray:
    """Complex boundary phases bc_mu (|bc| = 1) from a tuple of numbers."""
    b = np.asarray(bc, dtype=np.complex128)
    assert b.shape == (4,)
    return b


def plane_wave(dims, n, bc, chi) -> np.ndarray:
    """psi(x) = exp(i p.x) chi with p_mu = (2 pi n_mu + theta_mu)/L_mu, bc_mu = exp(i theta_mu).

    A pure input shape (a phase times a constant 4x3 spinor chi); returns (psi, p).
    """
    X, Y, Z, T = dims
    L = np.array([X, Y, Z, T], dtype=np.float64)
    theta = np.angle(bc_phases(bc))
    p = (2.0 * np.pi * np.asarray(n, dtype=np.float64) + theta) / L
    x, y, z, t = site_coords(dims)
    phase = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))
    return phase[..., None, None] * np.asarray(chi, dtype=np.complex128), p
