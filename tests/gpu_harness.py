"""Test-side glue: canonical numpy arrays -> device -> C-ABI call -> canonical numpy result.

Holds no arithmetic of the method: it only moves data through lqcd_pack_* / lqcd_unpack_*
and the hot-path entry points of paper_1112_5280_b200.
"""
from __future__ import annotations

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

    def __init__(self, dims, precision, recon, bc, U: np.ndarray, link_precision=0):
        self.ctx = L.Context(dims, precision, recon, bc, link_precision)
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
