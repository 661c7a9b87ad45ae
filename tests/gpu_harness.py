"""Test-side glue: canonical numpy arrays -> device -> C-ABI call -> canonical numpy result.

Holds no arithmetic of the method: it only moves data through lqcd_pack_* / lqcd_unpack_*
and the hot-path entry points of paper_1112_5280_b200.
"""
from __future__ import annotations

import os

import numpy as np
import torch

import paper_1112_5280_b200 as L
from lattice_inputs import parity_mask


def cdtype(precision):
    return np.complex128 if precision == 64 else np.complex64  # precision 16 exchanges complex64


def half_of(psi_full: np.ndarray, dims, parity: int) -> np.ndarray:
    """Canonical half spinor [Vh][4][3]: the sites of one parity in lexicographic order."""
    return np.ascontiguousarray(psi_full.reshape(-1, 4, 3)[parity_mask(dims, parity).ravel()])


def scatter_half(half: np.ndarray, dims, parity: int) -> np.ndarray:
    """Inverse of half_of; the other parity is zero."""
    X, Y, Z, T = dims
    out = np.zeros((T * Z * Y * X, 4, 3), dtype=half.dtype)
    out[parity_mask(dims, parity).ravel()] = half
    return out.reshape(T, Z, Y, X, 4, 3)


class Gpu:
    """One context plus the packed gauge field on cuda:0."""

    def __init__(self, dims, precision, recon, bc, U: np.ndarray, link_precision=0, kernel=None):
        self.ctx = L.Context(dims, precision, recon, bc, link_precision)
        # kernel: "gather" / "pipe" (lqcd_set_kernel); None: $LQCD_TEST_KERNEL where the ctx supports it (lets the whole
        # suite be re-run on the pipelined kernel), else the library default
        if kernel is None and precision != 16 and not link_precision:
            kernel = os.environ.get("LQCD_TEST_KERNEL")
        if kernel is not None:
            self.ctx.set_kernel({"gather": L.KERNEL_GATHER, "pipe": L.KERNEL_PIPE, "blocked": L.KERNEL_BLOCKED, "lstage": L.KERNEL_LSTAGE}[kernel])
        self.dims, self.precision = tuple(dims), precision
        self.cd = cdtype(precision)
        self.dev = torch.device("cuda:0")
        self.gauge = torch.empty(self.ctx.gauge_bytes(), dtype=torch.uint8, device=self.dev)
        Uc = torch.from_numpy(np.ascontiguousarray(U.astype(self.cd))).to(self.dev)
        self.ctx.pack_gauge(self.gauge, Uc)
        torch.cuda.synchronize()

    def buf(self, half=True):
        return torch.empty(self.ctx.spinor_bytes(half), dtype=torch.uint8, device=self.dev)

    def to_native(self, canonical: np.ndarray, parity: int):
        """canonical half [Vh][4][3] (parity 0/1) or full [T][Z][Y][X][4][3] (parity -1) -> native buffer."""
        c = torch.from_numpy(np.ascontiguousarray(canonical.astype(self.cd))).to(self.dev)
        n = self.buf(half=parity >= 0)
        self.ctx.pack_spinor(n, c, parity)
        torch.cuda.synchronize()
        return n

    def from_native(self, native, parity: int) -> np.ndarray:
        X, Y, Z, T = self.dims
        shape = (self.ctx.Vh, 4, 3) if parity >= 0 else (T, Z, Y, X, 4, 3)
        c = torch.empty(shape, dtype=L.complex_dtype(self.precision), device=self.dev)
        self.ctx.unpack_spinor(c, native, parity)
        torch.cuda.synchronize()
        return c.cpu().numpy()

    # --- hot path wrappers returning canonical numpy (complex of the run's precision)
    def dslash_full(self, psi_full):
        out = self.buf(half=False)
        self.ctx.dslash_full(out, self.gauge, self.to_native(psi_full, -1))
        return self.from_native(out, -1)

    def dslash_eo(self, psi_half, out_parity):
        out = self.buf()
        self.ctx.dslash_eo(out, self.gauge, self.to_native(psi_half, 1 - out_parity), out_parity)
        return self.from_native(out, out_parity)

    def apply_M(self, psi, kappa, eo, mu=None):
        """mu = None: lqcd_apply_M; otherwise lqcd_apply_M_tm with twisted mass mu."""
        def call(out, inp, ws):
            if mu is None:
                self.ctx.apply_M(out, self.gauge, inp, kappa, eo, ws)
            else:
                self.ctx.apply_M_tm(out, self.gauge, inp, kappa, mu, eo, ws)
        if eo:
            out, ws = self.buf(), self.buf()
            call(out, self.to_native(psi, 0), ws)
            return self.from_native(out, 0)
        out = self.buf(half=False)
        call(out, self.to_native(psi, -1), None)
        return self.from_native(out, -1)


def rel_l2(a: np.ndarray, ref: np.ndarray) -> float:
    """||a - ref||_2 / ||ref||_2 over all complex components, in fp64."""
    a = np.asarray(a, dtype=np.complex128).ravel()
    ref = np.asarray(ref, dtype=np.complex128).ravel()
    return float(np.linalg.norm(a - ref) / np.linalg.norm(ref))


# Per-site comparator (beside the global rel-L2 north_star defines): max over sites x of |a(x) - ref(x)| / |ref(x)|,
# the 2-norm over the 12 complex components of the site.  A defect confined to a few boundary or corner sites moves
# it by O(1) while it moves the global norm only by sqrt(#bad sites / #sites).  Bars: each output
# component is a sum over 8 hops of about 170 rounded operations on O(|psi|) operands, and sum |terms| / |out(x)| stays
# below ~10 for Gaussian data, so the worst case is 170 x 10 x eps / 2: 1e-4 (fp32), 1e-11 (fp64, with margin);
# observed values are ~1e-6 / ~1e-15.  Sites whose reference norm is below 1 % of the rms site norm (exact zeros of
# structured test fields) are measured against that floor instead.
SITE_TOL = {64: 1e-11, 32: 1e-4}


def max_site_rel(a: np.ndarray, ref: np.ndarray):
    """(max over sites of the relative 2-norm error, flat index of the worst site); a, ref: [..., 4, 3] complex."""
    a = np.asarray(a, dtype=np.complex128).reshape(-1, 12)
    ref = np.asarray(ref, dtype=np.complex128).reshape(-1, 12)
    num = np.linalg.norm(a - ref, axis=1)
    den = np.linalg.norm(ref, axis=1)
    floor = 1e-2 * np.sqrt(np.mean(den ** 2))
    r = num / np.maximum(den, floor if floor > 0 else 1.0)
    k = int(np.argmax(r))
    return float(r[k]), k


def assert_parity(a, ref, precision, l2_tol=None, site_tol=None, what=""):
    """Both comparators at once; on failure names the worst site (flat site index in the order of `ref`)."""
    l2_tol = {64: 1e-12, 32: 1e-5}[precision] if l2_tol is None else l2_tol
    site_tol = SITE_TOL[precision] if site_tol is None else site_tol
    e2 = rel_l2(a, ref)
    es, k = max_site_rel(a, ref)
    assert e2 <= l2_tol, f"{what}: rel-L2 {e2:.3e} > {l2_tol:g} (worst site {k}: {es:.3e})"
    assert es <= site_tol, f"{what}: per-site relative error {es:.3e} > {site_tol:g} at site {k} (rel-L2 {e2:.3e})"
    return e2, es


def site_tol_for(U, precision, recon):
    """Per-site bar of a run with `recon`-real links.  12 / 18: the common bar.  8: the worst link is decoded to about
    8 eps / min(|U00|, sqrt(1 - |U00|^2), |U20|) (pins R3 / R5 of tests/test_oracle_recon8_pins.py), so the bar follows
    the conditioning of the worst link of the field; never below the common bar."""
    if recon != 8:
        return SITE_TOL[precision]
    m = np.minimum(np.minimum(np.abs(U[..., 0, 0]), np.sqrt(np.abs(U[..., 0, 1]) ** 2 + np.abs(U[..., 0, 2]) ** 2)),
                   np.abs(U[..., 2, 0])).min()
    eps = 2.0 ** -53 if precision == 64 else 2.0 ** -24
    return max(SITE_TOL[precision], 16 * eps / float(m))


def recon8_margin(U):
    return float(np.minimum(np.minimum(np.abs(U[..., 0, 0]), np.sqrt(np.abs(U[..., 0, 1]) ** 2 + np.abs(U[..., 0, 2]) ** 2)),
                            np.abs(U[..., 2, 0])).min())
