"""Time-slab decomposition (next row f3) emulated on one GPU: N ranks as N slab objects in one process, ghost
exchange by device copies.  The assembled result must equal the undecomposed GPU result bit for bit (same
kernel, same arithmetic order) and the oracle within tolerance; ghosts start as NaN so a missed exchange shows."""
import numpy as np
import pytest
import torch

import lattice_inputs as li
import oracle

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("world", [1, 2, 4])
@pytest.mark.parametrize("precision,recon,bc", [(64, 12, (1, 1, 1, -1)), (32, 18, tuple(np.exp(1j * np.array([0.3, 0.0, -0.7, 2.1]))))])
def test_time_slabs_reproduce_the_whole_lattice(world, precision, recon, bc):
    import gpu_harness as H
    from paper_1112_5280_b200.slab import TimeSlab, exchange_emulated
    dims = (8, 8, 8, 16)
    X, Y, Z, T = dims
    cd = H.cdtype(precision)
    U = li.links_for_config(2).astype(cd)
    psi = li.gaussian_spinor(dims, seed=101).astype(cd)
    whole = H.Gpu(dims, precision, recon, bc, U)
    dev = torch.device("cuda:0")
    for gp in (0, 1):   # global output parity
        ref_gpu = H.scatter_half(whole.dslash_eo(H.half_of(psi, dims, 1 - gp), gp), dims, gp)
        slabs = [TimeSlab(dims, precision, recon, bc, r, world) for r in range(world)]
        gauges, ins, outs = [], [], []
        for s in slabs:
            tl = s.time_indices()
            Ul = torch.from_numpy(np.ascontiguousarray(U[:, tl])).to(dev)
            g = torch.empty(s.ctx.gauge_bytes(), dtype=torch.uint8, device=dev)
            s.ctx.pack_gauge(g, Ul)
            local = np.ascontiguousarray(psi[tl])
            local[0], local[-1] = np.nan, np.nan            # ghosts must come from the exchange
            lp_in = s.local_parity(1 - gp)
            f = torch.empty(s.ctx.spinor_bytes(True), dtype=torch.uint8, device=dev)
            s.ctx.pack_spinor(f, torch.from_numpy(H.half_of(local, s.local_dims, lp_in)).to(dev), lp_in)
            gauges.append(g); ins.append(f); outs.append(torch.zeros_like(f))
        torch.cuda.synchronize()
        done = []
        def exchange(_field):
            if not done:  # the emulation moves every rank's ghosts at once, at the first rank's request
                exchange_emulated(slabs, ins); done.append(1)
        for r, s in enumerate(slabs):
            s.dslash_eo(outs[r], gauges[r], ins[r], gp, exchange)
        torch.cuda.synchronize()
        got = np.zeros((T, Z, Y, X, 4, 3), dtype=cd)
        for r, s in enumerate(slabs):
            lp = s.local_parity(gp)
            c = torch.empty((s.ctx.Vh, 4, 3), dtype=torch.complex128 if precision == 64 else torch.complex64, device=dev)
            s.ctx.unpack_spinor(c, outs[r], lp)
            local = H.scatter_half(c.cpu().numpy(), s.local_dims, lp)
            got[s.t0:s.t0 + s.Tl] = local[1:s.Tl + 1]
        assert np.isfinite(got.view(np.float64 if precision == 64 else np.float32)).all()
        assert np.array_equal(got, ref_gpu), (world, gp)
        H.assert_parity(H.half_of(got, dims, gp), H.half_of(oracle.dslash_eo(U, psi, dims, bc, gp), dims, gp), precision)


def test_slab_argument_checks():
    import paper_1112_5280_b200 as L
    from paper_1112_5280_b200.slab import TimeSlab
    with pytest.raises(ValueError):
        TimeSlab((8, 8, 8, 16), 64, 12, (1, 1, 1, -1), 0, 3)        # 16 / 3
    with pytest.raises(ValueError):
        TimeSlab((8, 8, 8, 12), 64, 12, (1, 1, 1, -1), 0, 4)        # 3 slices per rank: odd
    with pytest.raises(ValueError):
        TimeSlab((4, 4, 6, 8), 64, 12, (1, 1, 1, -1), 0, 2)         # a slice is 48 sites: not whole tiles
    c = L.Context((8, 8, 8, 16), 64, 12)
    with pytest.raises(L.LqcdError):
        c.set_time_slab(16, 0)
    g = torch.empty(c.gauge_bytes(), dtype=torch.uint8, device="cuda:0")
    a, b = (torch.empty(c.spinor_bytes(True), dtype=torch.uint8, device="cuda:0") for _ in range(2))
    with pytest.raises(L.LqcdError):
        c.dslash_eo_range(a, g, b, 0, 3, 17)
