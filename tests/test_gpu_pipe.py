"""GPU parity of the pipelined kernel (lqcd_set_kernel(LQCD_KERNEL_PIPE): persistent CTAs, TMA bulk copies into a
shared-memory ring, csrc/pipe_kernel.cuh) against the CPU oracle, at north_star's tolerances, on lattices chosen to
hit every staging case: planes that are multiples of 32 sites (everything staged), rows that straddle tiles (X/2 = 6,
24), planes smaller than a tile (4^4), ragged last tiles, both parities in one launch, complex boundary phases,
every link format and every epilogue; and bit for bit against the gather kernel, which does the same arithmetic in the
same order.
"""
import numpy as np
import pytest

import lattice_inputs as li
import oracle

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def H():
    import gpu_harness
    return gpu_harness


LATTICES = [
    ((8, 8, 8, 16), (1, 1, 1, -1)),        # config 2: z planes of 32 sites, tiles of 8 rows
    ((4, 4, 4, 4), (1, 1, 1, -1)),         # minimum extent: a tile spans 4 z planes
    ((4, 6, 8, 10), "complex"),            # Vh = 960: 30 tiles, rows of 2 sites, complex phases
    ((12, 4, 6, 8), (1, -1, 1, -1)),       # X/2 = 6: rows straddle tiles, z planes of 24 sites
    ((48, 4, 4, 4), (-1, 1, 1, 1)),        # X/2 = 24 (config 5's row length): rows straddle tiles, x boundary phase
    ((32, 4, 4, 6), (1, 1, 1, -1)),        # X/2 = 16 (config 4's row length): two rows per tile
    ((6, 6, 6, 6), (1, 1, 1, -1)),         # Vh = 648: ragged last tile (8 sites)
]


def _bc(bc):
    return np.exp(1j * np.array([0.3, -1.1, 2.0, np.pi])) if isinstance(bc, str) else bc


@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("recon", [18, 12, 8])
@pytest.mark.parametrize("dims,bc", LATTICES)
@pytest.mark.parametrize("kernel", ["pipe", "lstage"])
def test_pipe_eo_full_and_matrix(H, dims, bc, precision, recon, kernel):
    bc = _bc(bc)
    cd = H.cdtype(precision)
    U = li.random_su3_links(dims, seed=31).astype(cd)
    psi = li.gaussian_spinor(dims, seed=32).astype(cd)
    g = H.Gpu(dims, precision, recon, bc, U, kernel=kernel)
    ref_g = H.Gpu(dims, precision, recon, bc, U, kernel="gather")
    st = H.site_tol_for(U, precision, recon)
    for op in (0, 1):
        ref = H.half_of(oracle.dslash_eo(U, psi, dims, bc, op), dims, op)
        got = g.dslash_eo(H.half_of(psi, dims, 1 - op), op)
        H.assert_parity(got, ref, precision, site_tol=st, what=f"pipe dslash_eo {op}")
        assert np.array_equal(got, ref_g.dslash_eo(H.half_of(psi, dims, 1 - op), op)), "pipe and gather kernels differ bitwise"
    full = g.dslash_full(psi)
    H.assert_parity(full, oracle.dslash_full(U, psi, dims, bc), precision, site_tol=st, what="pipe dslash_full")
    assert np.array_equal(full, ref_g.dslash_full(psi))
    kappa = 0.14
    refM = H.half_of(oracle.apply_M(U, psi, dims, bc, kappa, 1), dims, 0)
    H.assert_parity(g.apply_M(H.half_of(psi, dims, 0), kappa, 1), refM, precision, site_tol=st, what="pipe apply_M eo")
    refT = oracle.apply_M_tm(U, psi, dims, bc, kappa, -0.3, 0)
    H.assert_parity(g.apply_M(psi, kappa, 0, mu=-0.3), refT, precision, site_tol=st, what="pipe apply_M_tm full")
    refTe = H.half_of(oracle.apply_M_tm(U, psi, dims, bc, kappa, 0.2, 1), dims, 0)
    H.assert_parity(g.apply_M(H.half_of(psi, dims, 0), kappa, 1, mu=0.2), refTe, precision, site_tol=st, what="pipe apply_M_tm eo")


@pytest.mark.parametrize("precision,recon", [(64, 12), (32, 12), (32, 18), (64, 8)])
@pytest.mark.parametrize("kernel", ["pipe", "lstage"])
def test_pipe_many_tiles_per_cta(H, precision, recon, kernel):
    """Config 3 (16^3x32: 2048 tiles per parity, ~14 per CTA): every ring slot is reused several times, by different
    consumer warps in turn."""
    c = li.CONFIGS[3]
    dims, bc = c["dims"], c["bc"]
    cd = H.cdtype(precision)
    U = li.links_for_config(3).astype(cd)
    psi = li.gaussian_spinor(dims).astype(cd)
    g = H.Gpu(dims, precision, recon, bc, U, kernel=kernel)
    ref_g = H.Gpu(dims, precision, recon, bc, U, kernel="gather")
    st = H.site_tol_for(U, precision, recon)
    for op in (0, 1):
        got = g.dslash_eo(H.half_of(psi, dims, 1 - op), op)
        H.assert_parity(got, H.half_of(oracle.dslash_eo(U, psi, dims, bc, op), dims, op), precision, site_tol=st, what=f"pipe dslash_eo {op}")
        assert np.array_equal(got, ref_g.dslash_eo(H.half_of(psi, dims, 1 - op), op)), "pipe and gather kernels differ bitwise"
    refM = oracle.apply_M(U, psi, dims, bc, c["kappa"], 0)
    H.assert_parity(g.apply_M(psi, c["kappa"], 0), refM, precision, site_tol=st, what="pipe apply_M full")


@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("kernel", ["pipe", "lstage"])
def test_pipe_time_slice_ranges(H, precision, kernel):
    """lqcd_dslash_eo_range on the pipelined kernel: ranges that start and end inside tiles (z planes of 12 sites)."""
    import torch
    dims, bc = (4, 6, 4, 8), (1, 1, 1, -1)
    cd = H.cdtype(precision)
    U = li.random_su3_links(dims, seed=41).astype(cd)
    psi = li.gaussian_spinor(dims, seed=42).astype(cd)
    g = H.Gpu(dims, precision, 12, bc, U, kernel=kernel)
    ref = H.half_of(oracle.dslash_eo(U, psi, dims, bc, 0), dims, 0)
    inp = g.to_native(H.half_of(psi, dims, 1), 1)
    out = g.buf()
    out.zero_()
    for t0, t1 in ((0, 3), (3, 4), (4, 8)):
        g.ctx.dslash_eo_range(out, g.gauge, inp, 0, t0, t1)
    H.assert_parity(g.from_native(out, 0), ref, precision, what="pipe ranges")
    # a range writes nothing outside itself
    out.zero_()
    g.ctx.dslash_eo_range(out, g.gauge, inp, 0, 2, 5)
    got = g.from_native(out, 0)
    st = dims[0] // 2 * dims[1] * dims[2]
    assert np.array_equal(got[2 * st:5 * st], g.from_native(_full(g, inp), 0)[2 * st:5 * st])
    assert not got[:2 * st].any() and not got[5 * st:].any()
    torch.cuda.synchronize()


def _full(g, inp):
    out = g.buf()
    g.ctx.dslash_eo(out, g.gauge, inp, 0)
    return out


def test_pipe_unsupported_contexts(H):
    import paper_1112_5280_b200 as L
    for kw in (dict(precision=16, recon=12), dict(precision=32, recon=12, link_precision=16)):
        ctx = L.Context((8, 8, 8, 8), bc=(1, 1, 1, -1), **kw)
        with pytest.raises(L.LqcdError) as e:
            ctx.set_kernel(L.KERNEL_PIPE)
        assert e.value.status == L.LQCD_EUNSUPPORTED
    ctx = L.Context((8, 8, 8, 8), 32, 12)
    with pytest.raises(L.LqcdError) as e:
        ctx.set_kernel(7)
    assert e.value.status == L.LQCD_EINVAL
