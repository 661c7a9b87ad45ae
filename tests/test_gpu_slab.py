"""Time-slab decomposition (next row f3) emulated on one GPU: N ranks as N slab objects in one process, the projected
half-spinor faces pushed straight into the neighbouring slabs' halo buffers (the same kernels and pointers a multi-GPU
run uses over peer memory).  The assembled result must match the oracle at north_star's tolerances and the
undecomposed GPU result to rounding: the interior sites are bit-identical (same kernel), the two boundary slices differ
only in the order of the projection add, which is exact in both (one rounding of the same sum), so they are
bit-identical too.  Halos start as 0xFF bytes (NaN) so a missed push shows."""
import numpy as np
import pytest
import torch

import lattice_inputs as li
import oracle

pytestmark = pytest.mark.gpu


def _run_slabs(H, dims, precision, recon, bc, world, U, psi, gp, use_flags):
    from paper_1112_5280_b200.slab import TimeSlab, LocalRingTransport
    X, Y, Z, T = dims
    cd = H.cdtype(precision)
    dev = torch.device("cuda:0")
    slabs = [TimeSlab(dims, precision, recon, bc, r, world) for r in range(world)]
    ring = LocalRingTransport(slabs, dev, use_flags=use_flags)
    gauges, ins, outs = [], [], []
    for s in slabs:
        tl = s.time_indices()
        Ul = torch.from_numpy(np.ascontiguousarray(U[:, tl])).to(dev)
        Ub = torch.from_numpy(np.ascontiguousarray(U[3, s.t_below()])).to(dev)
        g = torch.empty(s.ctx.gauge_bytes(), dtype=torch.uint8, device=dev)
        s.pack_gauge(g, Ul, Ub)
        local = np.ascontiguousarray(psi[tl])
        f = torch.empty(s.ctx.spinor_bytes(True), dtype=torch.uint8, device=dev)
        s.ctx.pack_spinor(f, torch.from_numpy(H.half_of(local, s.local_dims, 1 - gp)).to(dev), 1 - gp)
        gauges.append(g); ins.append(f); outs.append(torch.zeros_like(f))
    for _rep in range(2):          # twice: the second application reuses the buffers with the next epoch
        ring.push_all(ins)
        for r, s in enumerate(slabs):
            s.dslash_eo(outs[r], gauges[r], ins[r], gp, ring)
    torch.cuda.synchronize()
    got = np.zeros((T, Z, Y, X, 4, 3), dtype=cd)
    for r, s in enumerate(slabs):
        c = torch.empty((s.ctx.Vh, 4, 3), dtype=torch.complex128 if precision == 64 else torch.complex64, device=dev)
        s.ctx.unpack_spinor(c, outs[r], gp)
        got[s.t0:s.t0 + s.Tl] = H.scatter_half(c.cpu().numpy(), s.local_dims, gp)
    return got


@pytest.mark.parametrize("world", [1, 2, 4])
@pytest.mark.parametrize("precision,recon,bc", [(64, 12, (1, 1, 1, -1)), (32, 18, tuple(np.exp(1j * np.array([0.3, 0.0, -0.7, 2.1])))),
                                                (64, 8, (1, 1, 1, -1))])
def test_time_slabs_reproduce_the_whole_lattice(world, precision, recon, bc):
    import gpu_harness as H
    dims = (8, 8, 8, 16)
    cd = H.cdtype(precision)
    U = li.links_for_config(2).astype(cd)
    psi = li.gaussian_spinor(dims, seed=101).astype(cd)
    whole = H.Gpu(dims, precision, recon, bc, U)
    for gp in (0, 1):   # global output parity
        ref_gpu = H.scatter_half(whole.dslash_eo(H.half_of(psi, dims, 1 - gp), gp), dims, gp)
        got = _run_slabs(H, dims, precision, recon, bc, world, U, psi, gp, use_flags=(world == 2))
        assert np.isfinite(got.view(np.float64 if precision == 64 else np.float32)).all()
        assert np.array_equal(got, ref_gpu), (world, gp)
        H.assert_parity(H.half_of(got, dims, gp), H.half_of(oracle.dslash_eo(U, psi, dims, bc, gp), dims, gp), precision,
                        site_tol=H.site_tol_for(U, precision, recon))


def test_ragged_faces_and_anisotropic_slabs():
    """A time slice of 4 x 6 x 6 / 2 = 72 sites per parity is not a whole number of 32-site tiles: the halo buffers pad
    their last tile and the slab range launches start in the middle of a tile."""
    import gpu_harness as H
    dims, bc, precision, recon = (4, 6, 6, 8), (1, -1, 1, np.exp(0.4j)), 32, 12
    U = li.random_su3_links(dims, seed=131).astype(np.complex64)
    psi = li.gaussian_spinor(dims, seed=132).astype(np.complex64)
    for gp in (0, 1):
        got = _run_slabs(H, dims, precision, recon, bc, 2, U, psi, gp, use_flags=True)
        H.assert_parity(H.half_of(got, dims, gp), H.half_of(oracle.dslash_eo(U, psi, dims, bc, gp), dims, gp), precision)


def test_slab_argument_checks():
    import paper_1112_5280_b200 as L
    from paper_1112_5280_b200.slab import TimeSlab
    with pytest.raises(ValueError):
        TimeSlab((8, 8, 8, 16), 64, 12, (1, 1, 1, -1), 0, 3)        # 16 / 3
    with pytest.raises(ValueError):
        TimeSlab((8, 8, 8, 12), 64, 12, (1, 1, 1, -1), 0, 4)        # 3 slices per rank: odd
    with pytest.raises(ValueError):
        TimeSlab((8, 8, 8, 16), 16, 12, (1, 1, 1, -1), 0, 2)        # 16-bit storage has no slab path
    s = TimeSlab((4, 4, 6, 8), 64, 12, (1, 1, 1, -1), 0, 2)         # ragged faces are fine: 48 sites -> 2 tiles
    assert s.halo_bytes == 2 * 32 * 12 * 8 and s.ctx.halo_bytes() == s.halo_bytes
    c = L.Context((8, 8, 8, 16), 64, 12)
    with pytest.raises(L.LqcdError):
        c.set_time_slab(16, 0)
    g = torch.empty(c.gauge_bytes(), dtype=torch.uint8, device="cuda:0")
    a, b = (torch.empty(c.spinor_bytes(True), dtype=torch.uint8, device="cuda:0") for _ in range(2))
    h = torch.empty(c.halo_bytes(), dtype=torch.uint8, device="cuda:0")
    with pytest.raises(L.LqcdError):
        c.dslash_eo_range(a, g, b, 0, 3, 17)
    with pytest.raises(L.LqcdError) as e:
        c.dslash_eo_slab(a, g, b, h, None, 0, 0, 1)
    assert e.value.status == L.LQCD_EINVAL
    with pytest.raises(L.LqcdError) as e:
        c.dslash_eo_slab(a, g, b, h.data_ptr() + 16, h, 0, 0, 1)
    assert e.value.status == L.LQCD_EALIGN
    with pytest.raises(L.LqcdError) as e:
        c.slab_push_faces(b, h, h, h.data_ptr() + 4, None, 1)
    assert e.value.status == L.LQCD_EALIGN
    torch.cuda.synchronize()
