"""paper_1112_5280_b200 -- B200-native Wilson dslash (arXiv:1112.5280 hot path).

Thin ctypes binding of the C ABI in include/lqcd.h (same names, argument marshalling only:
every step of the path runs in the CUDA kernels of csrc/).  PyTorch supplies device memory
and streams.  There is no CPU fallback: if liblqcd.so cannot be loaded the import of any
entry point raises.
"""
from __future__ import annotations

import ctypes
import os

from . import _build

LQCD_OK, LQCD_EINVAL, LQCD_EALIGN, LQCD_EALIAS, LQCD_EUNSUPPORTED, LQCD_ECUDA, LQCD_ETOOBIG = range(7)
PARITY_EVEN, PARITY_ODD, PARITY_BOTH = 0, 1, -1
KERNEL_GATHER, KERNEL_PIPE, KERNEL_BLOCKED, KERNEL_LSTAGE = 0, 1, 2, 3
HAS_RECON8 = True

EXPORTS = [
    "lqcd_create", "lqcd_destroy", "lqcd_spinor_bytes", "lqcd_gauge_bytes", "lqcd_workspace_bytes",
    "lqcd_host_workspace_bytes", "lqcd_pack_gauge", "lqcd_pack_spinor", "lqcd_unpack_spinor",
    "lqcd_dslash_full", "lqcd_dslash_eo", "lqcd_apply_M", "lqcd_set_time_slab", "lqcd_dslash_eo_range", "lqcd_pack_gauge_slab", "lqcd_halo_bytes", "lqcd_slab_push_faces", "lqcd_dslash_eo_slab", "lqcd_apply_M_tm", "lqcd_apply_Q_tm", "lqcd_cg_workspace_bytes", "lqcd_cg_solve_tm", "lqcd_cg_mixed_workspace_bytes", "lqcd_cg_solve_tm_mixed", "lqcd_dslash_eo_host", "lqcd_dslash_eo_host_batch", "lqcd_launch_count",
    "lqcd_gauge_recon8_margin", "lqcd_set_kernel", "lqcd_selftest_fastdiv", "lqcd_update_links_bytes", "lqcd_pack_update_links", "lqcd_unpack_update_links",
    "lqcd_heatbath_uniforms", "lqcd_heatbath_sublattice",
    "lqcd_plaquette_workspace_bytes", "lqcd_plaquette", "lqcd_status_string", "lqcd_last_cuda_error",
    "lqcd_static_scratch_bytes", "lqcd_apply_M_eo_static", "lqcd_reunitarise_links",
]


class lqcd_params(ctypes.Structure):
    _fields_ = [("dims", ctypes.c_int * 4), ("precision", ctypes.c_int), ("recon", ctypes.c_int),
                ("bc_re", ctypes.c_double * 4), ("bc_im", ctypes.c_double * 4), ("link_precision", ctypes.c_int)]


class LqcdError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = _lib().lqcd_status_string(status).decode()
        if status == LQCD_ECUDA:
            msg += ": " + _lib().lqcd_last_cuda_error().decode()
        super().__init__(f"{where}: {msg} (status {status})")


_LIB = None


def _lib():
    global _LIB
    if _LIB is None:
        path = _build.LIB
        if not os.path.exists(path):
            raise RuntimeError(f"{path} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                               "(the CUDA library is the only implementation; there is no fallback)")
        lib = ctypes.CDLL(path)
        vp, ci, cd, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
        lib.lqcd_create.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(lqcd_params)]
        lib.lqcd_destroy.argtypes = [vp]
        for n in ("lqcd_gauge_bytes", "lqcd_workspace_bytes", "lqcd_host_workspace_bytes", "lqcd_cg_workspace_bytes"):
            getattr(lib, n).argtypes = [vp]
            getattr(lib, n).restype = sz
        lib.lqcd_spinor_bytes.argtypes = [vp, ci]
        lib.lqcd_spinor_bytes.restype = sz
        lib.lqcd_pack_gauge.argtypes = [vp, vp, vp, vp]
        lib.lqcd_pack_spinor.argtypes = [vp, vp, vp, ci, vp]
        lib.lqcd_unpack_spinor.argtypes = [vp, vp, vp, ci, vp]
        lib.lqcd_dslash_full.argtypes = [vp, vp, vp, vp, vp]
        lib.lqcd_dslash_eo.argtypes = [vp, vp, vp, vp, ci, vp]
        lib.lqcd_apply_M.argtypes = [vp, vp, vp, vp, cd, ci, vp, vp]
        lib.lqcd_apply_M_eo_static.argtypes = [vp, vp, vp, vp, cd, vp]
        lib.lqcd_static_scratch_bytes.argtypes = []
        lib.lqcd_static_scratch_bytes.restype = sz
        lib.lqcd_set_time_slab.argtypes = [vp, ci, ci]
        lib.lqcd_set_kernel.argtypes = [vp, ci]
        lib.lqcd_selftest_fastdiv.argtypes = [ctypes.c_uint, ctypes.c_uint]
        lib.lqcd_selftest_fastdiv.restype = ctypes.c_uint
        lib.lqcd_update_links_bytes.argtypes = [vp]
        lib.lqcd_update_links_bytes.restype = sz
        lib.lqcd_pack_update_links.argtypes = [vp, vp, vp, vp]
        lib.lqcd_unpack_update_links.argtypes = [vp, vp, vp, vp]
        lib.lqcd_heatbath_uniforms.argtypes = [vp, ci]
        lib.lqcd_heatbath_uniforms.restype = sz
        lib.lqcd_heatbath_sublattice.argtypes = [vp, vp, cd, ci, ci, vp, ci, vp]
        lib.lqcd_reunitarise_links.argtypes = [vp, vp, vp]
        lib.lqcd_plaquette_workspace_bytes.argtypes = [vp]
        lib.lqcd_plaquette_workspace_bytes.restype = sz
        lib.lqcd_plaquette.argtypes = [vp, vp, vp, ctypes.POINTER(cd), vp]
        lib.lqcd_dslash_eo_range.argtypes = [vp, vp, vp, vp, ci, ci, ci, vp]
        lib.lqcd_halo_bytes.argtypes = [vp]
        lib.lqcd_halo_bytes.restype = sz
        lib.lqcd_pack_gauge_slab.argtypes = [vp, vp, vp, vp, vp]
        lib.lqcd_slab_push_faces.argtypes = [vp, vp, vp, vp, vp, vp, ctypes.c_ulonglong, vp]
        lib.lqcd_dslash_eo_slab.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, ctypes.c_ulonglong, ci, ci, ci, vp]
        lib.lqcd_apply_M_tm.argtypes = [vp, vp, vp, vp, cd, cd, ci, vp, vp]
        lib.lqcd_apply_Q_tm.argtypes = [vp, vp, vp, vp, cd, cd, vp, vp]
        lib.lqcd_cg_mixed_workspace_bytes.argtypes = [vp, vp]
        lib.lqcd_cg_mixed_workspace_bytes.restype = sz
        lib.lqcd_cg_solve_tm_mixed.argtypes = [vp, vp, vp, vp, vp, vp, cd, cd, cd, cd, ci, vp, ctypes.POINTER(ci),
                                               ctypes.POINTER(ci), ctypes.POINTER(cd), vp]
        lib.lqcd_cg_solve_tm.argtypes = [vp, vp, vp, vp, cd, cd, cd, ci, vp, ctypes.POINTER(ci), ctypes.POINTER(cd), vp]
        lib.lqcd_dslash_eo_host.argtypes = [vp, vp, vp, vp, ci, vp, vp]
        lib.lqcd_dslash_eo_host_batch.argtypes = [vp, ci, ctypes.POINTER(vp), vp, ctypes.POINTER(vp), ctypes.POINTER(ci), vp, vp]
        lib.lqcd_gauge_recon8_margin.argtypes = [vp, vp, vp, ctypes.POINTER(cd), vp]
        lib.lqcd_launch_count.argtypes = []
        lib.lqcd_launch_count.restype = ctypes.c_ulonglong
        lib.lqcd_status_string.argtypes = [ci]
        lib.lqcd_status_string.restype = ctypes.c_char_p
        lib.lqcd_last_cuda_error.argtypes = []
        lib.lqcd_last_cuda_error.restype = ctypes.c_char_p
        _LIB = lib
    return _LIB


def _ptr(t):
    """Device/host address of a torch tensor, a numpy array, an int, or None."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if hasattr(t, "data_ptr"):
        return t.data_ptr()
    return t.ctypes.data


def _stream(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return getattr(stream, "cuda_stream", stream)


def _chk(status: int, where: str):
    if status != LQCD_OK:
        raise LqcdError(status, where)


class Context:
    """Owns one lqcd_ctx.  Methods carry the names of the C entry points minus the prefix."""

    def __init__(self, dims, precision=64, recon=18, bc=(1, 1, 1, -1), link_precision=0):
        p = lqcd_params()
        p.dims[:] = [int(d) for d in dims]
        p.precision, p.recon, p.link_precision = int(precision), int(recon), int(link_precision)
        b = [complex(z) for z in bc]
        p.bc_re[:] = [z.real for z in b]
        p.bc_im[:] = [z.imag for z in b]
        self._h = ctypes.c_void_p()
        _chk(_lib().lqcd_create(ctypes.byref(self._h), ctypes.byref(p)), "lqcd_create")
        self.dims, self.precision, self.recon = tuple(p.dims), p.precision, p.recon
        self.Vh = self.dims[0] * self.dims[1] * self.dims[2] * self.dims[3] // 2

    def __del__(self):
        h, self._h = getattr(self, "_h", None), None
        if h and _LIB is not None:
            _LIB.lqcd_destroy(h)

    # sizes
    def spinor_bytes(self, half=True): return _lib().lqcd_spinor_bytes(self._h, int(half))
    def gauge_bytes(self): return _lib().lqcd_gauge_bytes(self._h)
    def workspace_bytes(self): return _lib().lqcd_workspace_bytes(self._h)
    def host_workspace_bytes(self): return _lib().lqcd_host_workspace_bytes(self._h)
    def cg_workspace_bytes(self): return _lib().lqcd_cg_workspace_bytes(self._h)

    # layout conversion
    def pack_gauge(self, native, canonical, stream=None):
        _chk(_lib().lqcd_pack_gauge(self._h, _ptr(native), _ptr(canonical), _stream(stream)), "lqcd_pack_gauge")

    def gauge_recon8_margin(self, canonical, scratch, stream=None):
        m = ctypes.c_double(0.0)
        _chk(_lib().lqcd_gauge_recon8_margin(self._h, _ptr(canonical), _ptr(scratch), ctypes.byref(m), _stream(stream)),
             "lqcd_gauge_recon8_margin")
        return m.value

    def pack_spinor(self, native, canonical, parity, stream=None):
        _chk(_lib().lqcd_pack_spinor(self._h, _ptr(native), _ptr(canonical), int(parity), _stream(stream)),
             "lqcd_pack_spinor")

    def unpack_spinor(self, canonical, native, parity, stream=None):
        _chk(_lib().lqcd_unpack_spinor(self._h, _ptr(canonical), _ptr(native), int(parity), _stream(stream)),
             "lqcd_unpack_spinor")

    # hot path
    def dslash_full(self, out, gauge, inp, stream=None):
        _chk(_lib().lqcd_dslash_full(self._h, _ptr(out), _ptr(gauge), _ptr(inp), _stream(stream)), "lqcd_dslash_full")

    def dslash_eo(self, out, gauge, inp, out_parity, stream=None):
        _chk(_lib().lqcd_dslash_eo(self._h, _ptr(out), _ptr(gauge), _ptr(inp), int(out_parity), _stream(stream)),
             "lqcd_dslash_eo")

    # pure-gauge heatbath (link field in the update layout, in place)
    def update_links_bytes(self): return _lib().lqcd_update_links_bytes(self._h)

    def pack_update_links(self, update, canonical, stream=None):
        _chk(_lib().lqcd_pack_update_links(self._h, _ptr(update), _ptr(canonical), _stream(stream)), "lqcd_pack_update_links")

    def unpack_update_links(self, canonical, update, stream=None):
        _chk(_lib().lqcd_unpack_update_links(self._h, _ptr(canonical), _ptr(update), _stream(stream)), "lqcd_unpack_update_links")

    def heatbath_uniforms(self, ntries): return _lib().lqcd_heatbath_uniforms(self._h, int(ntries))

    def heatbath_sublattice(self, links, beta, mu, parity, uniforms, ntries, stream=None):
        _chk(_lib().lqcd_heatbath_sublattice(self._h, _ptr(links), float(beta), int(mu), int(parity), _ptr(uniforms),
                                             int(ntries), _stream(stream)), "lqcd_heatbath_sublattice")

    def reunitarise_links(self, links, stream=None):
        _chk(_lib().lqcd_reunitarise_links(self._h, _ptr(links), _stream(stream)), "lqcd_reunitarise_links")

    def plaquette_workspace_bytes(self): return _lib().lqcd_plaquette_workspace_bytes(self._h)

    def plaquette(self, links, workspace, stream=None):
        p = ctypes.c_double(0.0)
        _chk(_lib().lqcd_plaquette(self._h, _ptr(links), _ptr(workspace), ctypes.byref(p), _stream(stream)), "lqcd_plaquette")
        return p.value

    def set_kernel(self, kernel):
        _chk(_lib().lqcd_set_kernel(self._h, int(kernel)), "lqcd_set_kernel")

    def set_time_slab(self, t_cross_fwd, t_cross_bwd):
        _chk(_lib().lqcd_set_time_slab(self._h, int(t_cross_fwd), int(t_cross_bwd)), "lqcd_set_time_slab")

    def dslash_eo_range(self, out, gauge, inp, out_parity, t_begin, t_end, stream=None):
        _chk(_lib().lqcd_dslash_eo_range(self._h, _ptr(out), _ptr(gauge), _ptr(inp), int(out_parity), int(t_begin),
                                         int(t_end), _stream(stream)), "lqcd_dslash_eo_range")

    def halo_bytes(self): return _lib().lqcd_halo_bytes(self._h)

    def pack_gauge_slab(self, native, canonical, tlinks_below, stream=None):
        _chk(_lib().lqcd_pack_gauge_slab(self._h, _ptr(native), _ptr(canonical), _ptr(tlinks_below), _stream(stream)),
             "lqcd_pack_gauge_slab")

    def slab_push_faces(self, inp, dst_up, dst_down, flag_up=None, flag_down=None, epoch=0, stream=None):
        _chk(_lib().lqcd_slab_push_faces(self._h, _ptr(inp), _ptr(dst_up), _ptr(dst_down), _ptr(flag_up), _ptr(flag_down),
                                         int(epoch), _stream(stream)), "lqcd_slab_push_faces")

    def dslash_eo_slab(self, out, gauge, inp, halo_from_up, halo_from_down, out_parity, t_begin, t_end, wait_up=None,
                       wait_down=None, epoch=0, stream=None):
        _chk(_lib().lqcd_dslash_eo_slab(self._h, _ptr(out), _ptr(gauge), _ptr(inp), _ptr(halo_from_up), _ptr(halo_from_down),
                                        _ptr(wait_up), _ptr(wait_down), int(epoch), int(out_parity), int(t_begin), int(t_end),
                                        _stream(stream)), "lqcd_dslash_eo_slab")

    def apply_M(self, out, gauge, inp, kappa, eo, workspace=None, stream=None):
        _chk(_lib().lqcd_apply_M(self._h, _ptr(out), _ptr(gauge), _ptr(inp), float(kappa), int(eo),
                                 _ptr(workspace), _stream(stream)), "lqcd_apply_M")

    def apply_M_eo_static(self, out, gauge, inp, kappa, stream=None):
        """lqcd_apply_M_eo_static: apply_M(eo=1) without a workspace argument, for callers that cannot allocate one (a
        driver that was only handed the three fields by an application whose pool owns the GPU).  The intermediate field
        lives in a 16 MiB array inside liblqcd.so, shared by every call on the GPU: larger lattices raise LQCD_ETOOBIG,
        overlapping calls race, and the first call on a device (which looks the array up) belongs outside stream capture."""
        _chk(_lib().lqcd_apply_M_eo_static(self._h, _ptr(out), _ptr(gauge), _ptr(inp), float(kappa), _stream(stream)),
             "lqcd_apply_M_eo_static")

    def apply_M_tm(self, out, gauge, inp, kappa, mu, eo, workspace=None, stream=None):
        _chk(_lib().lqcd_apply_M_tm(self._h, _ptr(out), _ptr(gauge), _ptr(inp), float(kappa), float(mu), int(eo),
                                    _ptr(workspace), _stream(stream)), "lqcd_apply_M_tm")

    def apply_Q_tm(self, out, gauge, inp, kappa, mu, workspace, stream=None):
        _chk(_lib().lqcd_apply_Q_tm(self._h, _ptr(out), _ptr(gauge), _ptr(inp), float(kappa), float(mu),
                                    _ptr(workspace), _stream(stream)), "lqcd_apply_Q_tm")

    def cg_solve_tm(self, x, gauge, b, kappa, mu, tol, maxiter, workspace, stream=None):
        """Returns (iterations, |r|/|b|); synchronises the stream."""
        it, res = ctypes.c_int(0), ctypes.c_double(0.0)
        _chk(_lib().lqcd_cg_solve_tm(self._h, _ptr(x), _ptr(gauge), _ptr(b), float(kappa), float(mu), float(tol),
                                     int(maxiter), _ptr(workspace), ctypes.byref(it), ctypes.byref(res),
                                     _stream(stream)), "lqcd_cg_solve_tm")
        return it.value, res.value

    def cg_mixed_workspace_bytes(self, ctx32):
        return _lib().lqcd_cg_mixed_workspace_bytes(self._h, ctx32._h)

    def cg_solve_tm_mixed(self, ctx32, x, gauge64, gauge32, b, kappa, mu, tol, inner_tol, maxiter, workspace, stream=None):
        """self is the fp64 context.  Returns (inner iterations, outer corrections, |b - A x| / |b|)."""
        it, outer, res = ctypes.c_int(0), ctypes.c_int(0), ctypes.c_double(0.0)
        _chk(_lib().lqcd_cg_solve_tm_mixed(self._h, ctx32._h, _ptr(x), _ptr(gauge64), _ptr(gauge32), _ptr(b), float(kappa),
                                           float(mu), float(tol), float(inner_tol), int(maxiter), _ptr(workspace),
                                           ctypes.byref(it), ctypes.byref(outer), ctypes.byref(res), _stream(stream)),
             "lqcd_cg_solve_tm_mixed")
        return it.value, outer.value, res.value

    def dslash_eo_host(self, out_host, gauge_host, in_host, out_parity, workspace, stream=None):
        _chk(_lib().lqcd_dslash_eo_host(self._h, _ptr(out_host), _ptr(gauge_host), _ptr(in_host), int(out_parity),
                                        _ptr(workspace), _stream(stream)), "lqcd_dslash_eo_host")

    def dslash_eo_host_batch(self, outs_host, gauge_host, ins_host, out_parities, workspace, stream=None):
        n = len(outs_host)
        assert len(ins_host) == n and len(out_parities) == n
        outs = (ctypes.c_void_p * n)(*[_ptr(t) for t in outs_host])
        ins = (ctypes.c_void_p * n)(*[_ptr(t) for t in ins_host])
        par = (ctypes.c_int * n)(*[int(p) for p in out_parities])
        _chk(_lib().lqcd_dslash_eo_host_batch(self._h, n, outs, _ptr(gauge_host), ins, par, _ptr(workspace),
                                              _stream(stream)), "lqcd_dslash_eo_host_batch")


def static_scratch_bytes() -> int:
    """Size of the built-in scratch array behind Context.apply_M_eo_static (held once per GPU for the life of the process)."""
    return int(_lib().lqcd_static_scratch_bytes())


def launch_count() -> int:
    return int(_lib().lqcd_launch_count())


def real_dtype(precision):
    """dtype of the canonical (interchange) buffers: precision 16 exchanges complex64 like precision 32."""
    import torch
    return torch.float64 if precision == 64 else torch.float32


def complex_dtype(precision):
    import torch
    return torch.complex128 if precision == 64 else torch.complex64
