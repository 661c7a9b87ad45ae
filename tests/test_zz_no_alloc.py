"""lqcd_apply_M_eo_static: the even-odd fermion matrix for callers that cannot allocate device memory.

Who they are: liblqcd.so is a plain C ABI, and every other entry point that needs scratch expects the caller to
allocate it.  A C or Fortran HMC driver that was handed three device pointers (links, source, destination) by an
application whose own memory pool owns the whole GPU cannot do that -- it has no allocator binding, and a raw cudaMalloc
beside such a pool fails or stalls the device.  For them the intermediate half spinor lives in a 16 MiB array inside
the library image, one per GPU, shared by every call.

What is checked here: the result equals lqcd_apply_M(eo=1) with a caller-owned workspace, on two calls in a row that
use different lattices, precisions and inputs -- so the second call finds the array full of the first call's data,
in another element type, and must not care.  Lattices beyond the limit are refused with LQCD_ETOOBIG before any launch.

This file is named to be collected last: the array is process-wide state that no other test touches, and under
`pytest -x` a failure here must not hide the parity tests.  It passes alone in a fresh process and after the others.
"""
import numpy as np
import pytest

import lattice_inputs as li
import paper_1112_5280_b200 as L


def test_lattice_beyond_the_built_in_scratch_is_refused_without_touching_the_gpu():
    """The size check precedes every CUDA call, so fake (aligned, disjoint) addresses exercise it on a CPU-only box."""
    lib = L._lib()
    assert L.static_scratch_bytes() == 16 << 20
    base = 1 << 30
    for dims, precision in (((32, 32, 32, 64), 32), ((16, 16, 16, 64), 64)):   # 100.7 MB and 25.2 MB half spinors
        c = L.Context(dims, precision, 12)
        assert c.workspace_bytes() > L.static_scratch_bytes()
        assert lib.lqcd_apply_M_eo_static(c._h, base, base + (1 << 29), base + (1 << 28), 0.1, None) == L.LQCD_ETOOBIG
    assert L.Context((16, 16, 16, 32), 64, 12).workspace_bytes() <= L.static_scratch_bytes()   # the documented limit
    assert L.Context((16, 16, 16, 64), 32, 12).workspace_bytes() <= L.static_scratch_bytes()
    assert b"scratch" in lib.lqcd_status_string(L.LQCD_ETOOBIG)
    # the usual argument checks come first
    c = L.Context((4, 4, 4, 4), 64, 18)
    assert c.workspace_bytes() <= L.static_scratch_bytes()
    assert lib.lqcd_apply_M_eo_static(c._h, None, None, None, 0.1, None) == L.LQCD_EINVAL
    assert lib.lqcd_apply_M_eo_static(None, base, base + (1 << 29), base + (1 << 28), 0.1, None) == L.LQCD_EINVAL
    assert lib.lqcd_apply_M_eo_static(c._h, base + 8, base + (1 << 29), base + (1 << 28), 0.1, None) == L.LQCD_EALIGN
    assert lib.lqcd_apply_M_eo_static(c._h, base, base + (1 << 29), base, 0.1, None) == L.LQCD_EALIAS


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_workspace_path():
    """Call 1: 8^3 x 16, fp64, 18-real links.  Call 2, straight after it on the same stream: a ragged 6 x 4 x 6 x 10
    lattice in fp32 with 12-real links and complex boundary phases.  Each is compared with lqcd_apply_M(eo=1) fed a
    torch-allocated workspace, at the bars of the parity tests (rel-L2 1e-12 / 1e-5 plus the per-site bar); the two
    paths launch the same kernels on the same data, so the difference is in fact zero, which is asserted as well."""
    import torch
    import gpu_harness as H

    cases = [((8, 8, 8, 16), 64, 18, (1, 1, 1, -1), 0.15, 71),
             ((6, 4, 6, 10), 32, 12, tuple(np.exp(1j * np.array([0.3, -1.1, 2.0, np.pi]))), 0.13, 73)]
    runs = []
    for dims, precision, recon, bc, kappa, seed in cases:
        U = li.random_su3_links(dims, seed=seed).astype(H.cdtype(precision))
        psi = li.gaussian_spinor(dims, seed=seed + 1).astype(H.cdtype(precision))
        g = H.Gpu(dims, precision, recon, bc, U)
        assert g.ctx.workspace_bytes() <= L.static_scratch_bytes()
        inp = g.to_native(H.half_of(psi, dims, 0), 0)
        runs.append((g, inp, kappa, g.buf(), g.buf(), g.buf()))
    torch.cuda.synchronize()

    # the two calls under test, back to back, nothing in between
    for g, inp, kappa, out_static, _, _ in runs:
        g.ctx.apply_M_eo_static(out_static, g.gauge, inp, kappa)
    # the existing path, afterwards
    for g, inp, kappa, _, out_ws, ws in runs:
        g.ctx.apply_M(out_ws, g.gauge, inp, kappa, 1, ws)
    torch.cuda.synchronize()

    for g, inp, kappa, out_static, out_ws, _ in runs:
        got, ref = g.from_native(out_static, 0), g.from_native(out_ws, 0)
        assert np.isfinite(ref.view(ref.real.dtype)).all() and np.abs(ref).max() > 0
        H.assert_parity(got, ref, g.precision, what=f"apply_M_eo_static {g.dims} fp{g.precision}")
        assert np.array_equal(got, ref)

    # and once more in the opposite order, so that each lattice also runs on top of the other one's leftovers
    for g, inp, kappa, out_static, _, _ in reversed(runs):
        out_static.zero_()
        g.ctx.apply_M_eo_static(out_static, g.gauge, inp, kappa)
    torch.cuda.synchronize()
    for g, inp, kappa, out_static, out_ws, _ in runs:
        H.assert_parity(g.from_native(out_static, 0), g.from_native(out_ws, 0), g.precision,
                        what=f"apply_M_eo_static, reversed order, {g.dims} fp{g.precision}")
