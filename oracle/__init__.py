"""CPU oracle for the Wilson dslash path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin ctypes wrapper around oracle/wilson_oracle.c (plain C99, fp64, OpenMP over
output sites).  See that file's header for the definition it implements and the
passages it follows.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It imports nothing from paper_1112_5280_b200.

All arrays use the canonical layout of SURVEY.md Appendix A.4 with dims = (X, Y, Z, T):
    spinor [T][Z][Y][X][4][3] complex,  links [4][T][Z][Y][X][3][3] complex.
Inputs may be complex128 or complex64 (promoted to fp64 element-wise, reading A14);
outputs are always complex128.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "wilson_oracle.c")
_LIB = os.path.join(_HERE, "libwilson_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the C oracle with gcc -O2 -fopenmp."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        c_int, c_long, c_dbl, c_void = ctypes.c_int, ctypes.c_long, ctypes.c_double, ctypes.c_void_p
        lib.oracle_gamma.argtypes = [c_int, c_void]
        lib.oracle_gamma.restype = None
        lib.oracle_num_threads.restype = c_int
        lib.oracle_set_num_threads.argtypes = [c_int]
        lib.oracle_set_num_threads.restype = None
        common = [c_void, c_void, c_int, c_void, c_int, c_void, c_void, c_void]
        lib.oracle_dslash_full.argtypes = common
        lib.oracle_dslash_eo.argtypes = common + [c_int]
        lib.oracle_apply_M.argtypes = common + [c_dbl, c_int]
        lib.oracle_apply_M_tm.argtypes = common + [c_dbl, c_dbl, c_int]
        lib.oracle_dslash_sites.argtypes = common + [c_void, c_long]
        lib.oracle_apply_M_sites.argtypes = common + [c_dbl, c_int, c_void, c_long]
        lib.oracle_recon_row2.argtypes = [c_void, c_void, c_void]
        lib.oracle_recon_row2.restype = None
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def set_num_threads(n: int) -> None:
    _load().oracle_set_num_threads(int(n))


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


def _prep(U, psi, dims, bc):
    X, Y, Z, T = (int(d) for d in dims)
    U = np.ascontiguousarray(U)
    psi = np.ascontiguousarray(psi)
    assert U.dtype in (np.complex64, np.complex128) and psi.dtype in (np.complex64, np.complex128)
    assert U.shape == (4, T, Z, Y, X, 3, 3), (U.shape, dims)
    assert psi.shape == (T, Z, Y, X, 4, 3), (psi.shape, dims)
    d = np.array([X, Y, Z, T], dtype=np.int32)
    b = np.asarray(bc, dtype=np.complex128).reshape(4)
    bre = np.ascontiguousarray(b.real)
    bim = np.ascontiguousarray(b.imag)
    return U, int(U.dtype == np.complex64), psi, int(psi.dtype == np.complex64), d, bre, bim


def _check(rc):
    if rc != 0:
        raise RuntimeError(f"oracle returned error {rc}")


def gamma(mu: int) -> np.ndarray:
    """Dense 4x4 gamma_mu (mu = 0..3 = x,y,z,t) or gamma_5 (mu = 4), Appendix A.2."""
    out = np.empty((4, 4), dtype=np.complex128)
    _load().oracle_gamma(int(mu), _ptr(out))
    return out


def dslash_full(U, psi, dims, bc) -> np.ndarray:
    """out = H psi on all sites."""
    U, uf, psi, pf, d, bre, bim = _prep(U, psi, dims, bc)
    out = np.empty(psi.shape, dtype=np.complex128)
    _check(_load().oracle_dslash_full(_ptr(out), _ptr(U), uf, _ptr(psi), pf, _ptr(d), _ptr(bre), _ptr(bim)))
    return out


def dslash_eo(U, psi, dims, bc, out_parity: int) -> np.ndarray:
    """out_p = H_{p,1-p} psi_{1-p}; full-lattice array, zero on the other parity."""
    U, uf, psi, pf, d, bre, bim = _prep(U, psi, dims, bc)
    out = np.empty(psi.shape, dtype=np.complex128)
    _check(_load().oracle_dslash_eo(_ptr(out), _ptr(U), uf, _ptr(psi), pf, _ptr(d), _ptr(bre), _ptr(bim),
                                    int(out_parity)))
    return out


def apply_M(U, psi, dims, bc, kappa: float, eo: int) -> np.ndarray:
    """eo=0: psi - kappa H psi.  eo=1: psi_e - kappa^2 H_eo H_oe psi_e on even sites, zero on odd."""
    U, uf, psi, pf, d, bre, bim = _prep(U, psi, dims, bc)
    out = np.empty(psi.shape, dtype=np.complex128)
    _check(_load().oracle_apply_M(_ptr(out), _ptr(U), uf, _ptr(psi), pf, _ptr(d), _ptr(bre), _ptr(bim),
                                  float(kappa), int(eo)))
    return out


def apply_M_tm(U, psi, dims, bc, kappa: float, mu: float, eo: int) -> np.ndarray:
    """Twisted-mass fermion matrix (next row f1).  eo=0: (1 + 2i kappa mu g5) psi - kappa H psi.
    eo=1: (1 + 2i kappa mu g5) psi_e - kappa^2 H_eo (1 + 2i kappa mu g5)^-1 H_oe psi_e on even sites, zero on odd."""
    U, uf, psi, pf, d, bre, bim = _prep(U, psi, dims, bc)
    out = np.empty(psi.shape, dtype=np.complex128)
    _check(_load().oracle_apply_M_tm(_ptr(out), _ptr(U), uf, _ptr(psi), pf, _ptr(d), _ptr(bre), _ptr(bim),
                                     float(kappa), float(mu), int(eo)))
    return out


def _coords(coords):
    c = np.ascontiguousarray(np.asarray(coords, dtype=np.int32).reshape(-1, 4))
    return c, c.shape[0]


def dslash_sites(U, psi, dims, bc, coords) -> np.ndarray:
    """(H psi)(x) at listed sites; coords [n][4] = (x,y,z,t); returns [n][4][3]."""
    U, uf, psi, pf, d, bre, bim = _prep(U, psi, dims, bc)
    c, n = _coords(coords)
    out = np.empty((n, 4, 3), dtype=np.complex128)
    _check(_load().oracle_dslash_sites(_ptr(out), _ptr(U), uf, _ptr(psi), pf, _ptr(d), _ptr(bre), _ptr(bim),
                                       _ptr(c), n))
    return out


def apply_M_sites(U, psi, dims, bc, kappa: float, eo: int, coords) -> np.ndarray:
    """(M psi)(x) at listed sites (for eo=1 the sites must be even)."""
    U, uf, psi, pf, d, bre, bim = _prep(U, psi, dims, bc)
    c, n = _coords(coords)
    if eo == 1:
        assert np.all(c.sum(axis=1) % 2 == 0), "eo=1 is defined on even sites"
    out = np.empty((n, 4, 3), dtype=np.complex128)
    _check(_load().oracle_apply_M_sites(_ptr(out), _ptr(U), uf, _ptr(psi), pf, _ptr(d), _ptr(bre), _ptr(bim),
                                        float(kappa), int(eo), _ptr(c), n))
    return out


def recon_row2(r0, r1) -> np.ndarray:
    """Appendix A.7: row2 = conj(row0 x row1) for one SU(3) matrix."""
    r0 = np.ascontiguousarray(r0, dtype=np.complex128)
    r1 = np.ascontiguousarray(r1, dtype=np.complex128)
    out = np.empty(3, dtype=np.complex128)
    _load().oracle_recon_row2(_ptr(r0), _ptr(r1), _ptr(out))
    return out
