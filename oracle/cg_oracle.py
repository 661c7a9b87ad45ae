"""CG oracle (next row f2) -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

"the inversion of the fermion matrix" is the cost the paper's solver kernels exist for (
the inverter is one of the physics modules of PAPER.md:73).  The paper prints no algorithm; this is the
textbook conjugate-gradient iteration (Hestenes-Stiefel) for a Hermitian positive-definite operator A,
written out step by step in fp64 numpy, x0 = 0, stopping on the recursive residual:

    r = b; p = r; rr = <r, r>
    repeat:  s = A p;  alpha = rr / <p, s>;  x += alpha p;  r -= alpha s;  rr' = <r, r>
             stop if rr' <= tol^2 <b, b>;  beta = rr' / rr;  p = r + beta p;  rr = rr'

For the fermion matrix, A = Mhat(mu)^dagger Mhat(mu) on the even sites with Mhat = oracle.apply_M_tm(eo=1)
and Mhat(mu)^dagger = g5 Mhat(-mu) g5 (pin T3 of tests/test_oracle_tm_pins.py), reading F2.
Imports nothing from paper_1112_5280_b200.
"""
from __future__ import annotations

import numpy as np

from . import apply_M_tm


def cg(apply_A, b: np.ndarray, tol: float, maxiter: int):
    """Solve A x = b.  Returns (x, iterations, sqrt(rr / <b,b>) of the recursive residual)."""
    b = np.asarray(b, dtype=np.complex128)
    x = np.zeros_like(b)
    r = b.copy()
    p = r.copy()
    bb = float(np.vdot(b, b).real)
    rr = bb
    if bb == 0.0:
        return x, 0, 0.0
    it = 0
    while it < maxiter:
        s = apply_A(p)
        alpha = rr / float(np.vdot(p, s).real)
        x += alpha * p
        r -= alpha * s
        rr_new = float(np.vdot(r, r).real)
        it += 1
        if rr_new <= tol * tol * bb:
            rr = rr_new
            break
        p = r + (rr_new / rr) * p
        rr = rr_new
    return x, it, float(np.sqrt(rr / bb))


def _g5(v):
    out = v.copy()
    out[..., 2:, :] *= -1.0  # gamma_5 = diag(1, 1, -1, -1), spin is the second-to-last axis
    return out


def normal_operator_tm(U, dims, bc, kappa: float, mu: float):
    """A = Mhat(mu)^dagger Mhat(mu) acting on full-lattice arrays supported on even sites."""
    def A(v):
        t = apply_M_tm(U, v, dims, bc, kappa, mu, 1)
        return _g5(apply_M_tm(U, _g5(t), dims, bc, kappa, -mu, 1))
    return A


def cg_solve_tm(U, b, dims, bc, kappa: float, mu: float, tol: float, maxiter: int):
    """Solve Mhat(mu)^dagger Mhat(mu) x = b on the even sites (b zero on odd sites)."""
    return cg(normal_operator_tm(U, dims, bc, kappa, mu), b, tol, maxiter)


def cg_mixed(apply_A64, apply_A32, b: np.ndarray, tol: float, inner_tol: float, maxiter: int):
    """Mixed-precision defect correction (reading F2), step by step:
        x = 0, r = b
        while |r| > tol |b|:  e = CG_fp32(A32, (complex64) r, max(inner_tol, tol |b| / (2 |r|)));  x += e;  r = b - A64 x
    The inner CG is `cg` above with every vector held in complex64 (apply_A32 must return complex64).
    Returns (x, total inner iterations, outer corrections, |b - A x| / |b|)."""
    b = np.asarray(b, dtype=np.complex128)
    x = np.zeros_like(b)
    r = b.copy()
    bb = float(np.vdot(b, b).real)
    rr, total, outer = bb, 0, 0
    while bb > 0.0 and rr > tol * tol * bb and total < maxiter and outer < 50:
        need = tol * np.sqrt(bb / rr)
        e, it, _ = _cg32(apply_A32, r.astype(np.complex64), max(inner_tol, 0.5 * need), maxiter - total)
        total += it
        outer += 1
        x += e.astype(np.complex128)
        r = b - apply_A64(x)
        rr_old, rr = rr, float(np.vdot(r, r).real)
        if it == 0 or not rr < rr_old:
            break
    return x, total, outer, float(np.sqrt(rr / bb)) if bb > 0 else 0.0


def _cg32(apply_A, b, tol, maxiter):
    """`cg` with complex64 vectors and float32 alpha / beta; the scalar products are accumulated in fp64."""
    x = np.zeros_like(b)
    r = b.copy()
    p = r.copy()
    bb = float(np.vdot(b.astype(np.complex128), b.astype(np.complex128)).real)
    rr = bb
    if bb == 0.0:
        return x, 0, 0.0
    it = 0
    while it < maxiter:
        s = apply_A(p)
        assert s.dtype == np.complex64
        pap = float(np.vdot(p.astype(np.complex128), s.astype(np.complex128)).real)
        alpha = np.float32(rr / pap)
        x = x + alpha * p
        r = r - alpha * s
        rr_new = float(np.vdot(r.astype(np.complex128), r.astype(np.complex128)).real)
        it += 1
        if rr_new <= tol * tol * bb:
            rr = rr_new
            break
        p = r + np.float32(rr_new / rr) * p
        rr = rr_new
    return x, it, float(np.sqrt(rr / bb))


def cg_mixed_solve_tm(U, b, dims, bc, kappa: float, mu: float, tol: float, inner_tol: float, maxiter: int):
    """Mixed-precision solve of Mhat(mu)^dagger Mhat(mu) x = b: the fp32 operator sees links and vectors rounded to
    complex64 and returns its result rounded to complex64 (its internal arithmetic is the fp64 oracle's)."""
    A64 = normal_operator_tm(U, dims, bc, kappa, mu)
    A32_ = normal_operator_tm(U.astype(np.complex64), dims, bc, kappa, mu)
    return cg_mixed(A64, lambda v: A32_(v).astype(np.complex64), b, tol, inner_tol, maxiter)
