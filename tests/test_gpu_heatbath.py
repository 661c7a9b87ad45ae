"""GPU parity of the pure-gauge heatbath (lqcd_heatbath_sublattice, lqcd_plaquette, lqcd_pack/unpack_update_links; next row f4) against
oracle/heatbath_oracle.py on the same links and the same uniforms: every link of the field after each of the eight
sublattice updates, to fp64 rounding (the accept / reject decisions are taken in fp64 on both sides; a decision closer
to its threshold than the 1e-15 the two libms differ by has probability ~1e-15 per attempt)."""
import numpy as np
import pytest
import torch

import lattice_inputs as li
from oracle import heatbath_oracle as hb

pytestmark = pytest.mark.gpu


def _setup(dims, seed):
    import paper_1112_5280_b200 as L
    ctx = L.Context(dims, 64, 18, (1, 1, 1, 1))
    U = li.random_su3_links(dims, seed=seed)
    dev = torch.device("cuda:0")
    return L, ctx, U, dev


class _Links:
    """A link field on the device in the update layout, converted from / to canonical numpy arrays."""

    def __init__(self, ctx, U, dev):
        self.ctx, self.dev, self.shape = ctx, dev, U.shape
        self.buf = torch.empty(ctx.update_links_bytes(), dtype=torch.uint8, device=dev)
        self.put(U)

    def put(self, U):
        self.ctx.pack_update_links(self.buf, torch.from_numpy(np.ascontiguousarray(U)).to(self.dev))
        torch.cuda.synchronize()

    def get(self):
        c = torch.empty(self.shape, dtype=torch.complex128, device=self.dev)
        self.ctx.unpack_update_links(c, self.buf)
        torch.cuda.synchronize()
        return c.cpu().numpy()


@pytest.mark.parametrize("dims,beta,ntries", [((4, 4, 4, 4), 5.7, 6), ((4, 6, 8, 10), 2.0, 3), ((8, 8, 8, 16), 6.0, 4), ((6, 4, 4, 8), 0.8, 1)])
def test_heatbath_sweep_matches_oracle(dims, beta, ntries):
    L, ctx, U, dev = _setup(dims, 61)
    Vh = ctx.Vh
    assert ctx.heatbath_uniforms(ntries) == Vh * 3 * (4 * ntries + 2)
    Ud = _Links(ctx, U, dev)
    assert np.array_equal(Ud.get(), U)           # pack / unpack is a pure permutation
    ws = torch.empty(ctx.plaquette_workspace_bytes(), dtype=torch.uint8, device=dev)
    assert abs(ctx.plaquette(Ud.buf, ws) - hb.plaquette(U)) <= 1e-13
    rng = np.random.default_rng(5)
    changed_subgroups = 0
    for mu in range(4):
        for parity in (0, 1):
            u = 1.0 - rng.random((Vh, 3, 4 * ntries + 2))
            ref = hb.heatbath_sublattice(U, beta, mu, parity, u)
            ctx.heatbath_sublattice(Ud.buf, beta, mu, parity, torch.from_numpy(u).to(dev), ntries)
            got = Ud.get()
            assert np.abs(got - ref).max() <= 1e-12, (mu, parity, np.abs(got - ref).max())
            changed_subgroups += int((np.abs(ref[mu] - U[mu]).reshape(-1, 9).max(axis=1) > 0).sum())
            U = ref          # the oracle's field is the reference the next update starts from on both sides
            Ud.put(U)
    assert changed_subgroups > 0
    assert abs(ctx.plaquette(Ud.buf, ws) - hb.plaquette(U)) <= 1e-13
    # still SU(3)
    M = U.reshape(-1, 3, 3)
    assert np.allclose(M @ np.conj(np.swapaxes(M, -1, -2)), np.eye(3), atol=1e-12)


def test_heatbath_free_running_plaquette():
    """Eight sweeps without resynchronising with the oracle: the two fields stay together to rounding, and the
    plaquette moves from the random start (0) towards the beta = 6 value."""
    dims, beta, ntries = (4, 4, 4, 8), 6.0, 4
    L, ctx, U, dev = _setup(dims, 62)
    Ud = _Links(ctx, U, dev)
    ws = torch.empty(ctx.plaquette_workspace_bytes(), dtype=torch.uint8, device=dev)
    rng = np.random.default_rng(8)
    for sweep in range(8):
        for mu in range(4):
            for parity in (0, 1):
                u = 1.0 - rng.random((ctx.Vh, 3, 4 * ntries + 2))
                U = hb.heatbath_sublattice(U, beta, mu, parity, u)
                ctx.heatbath_sublattice(Ud.buf, beta, mu, parity, torch.from_numpy(u).to(dev), ntries)
    assert np.abs(Ud.get() - U).max() <= 1e-10
    p = ctx.plaquette(Ud.buf, ws)
    assert abs(p - hb.plaquette(U)) <= 1e-12 and 0.4 < p < 0.7


def test_heatbath_error_codes():
    import paper_1112_5280_b200 as L
    dims = (4, 4, 4, 4)
    _, ctx, U, dev = _setup(dims, 63)
    links = _Links(ctx, U, dev)
    Ud = links.buf
    u = torch.rand(ctx.heatbath_uniforms(2), dtype=torch.float64, device=dev)
    for kw, status in ((dict(mu=4), L.LQCD_EINVAL), (dict(parity=2), L.LQCD_EINVAL), (dict(ntries=0), L.LQCD_EINVAL),
                       (dict(beta=0.0), L.LQCD_EINVAL)):
        args = dict(beta=5.0, mu=0, parity=0, ntries=2)
        args.update(kw)
        with pytest.raises(L.LqcdError) as e:
            ctx.heatbath_sublattice(Ud, args["beta"], args["mu"], args["parity"], u, args["ntries"])
        assert e.value.status == status
    with pytest.raises(L.LqcdError) as e:
        ctx.heatbath_sublattice(Ud.data_ptr() + 8, 5.0, 0, 0, u, 2)
    assert e.value.status == L.LQCD_EALIGN
    c32 = L.Context(dims, 32, 12)
    with pytest.raises(L.LqcdError) as e:
        c32.heatbath_sublattice(Ud, 5.0, 0, 0, u, 2)
    assert e.value.status == L.LQCD_EUNSUPPORTED
    assert np.array_equal(links.get(), U)   # nothing was launched


def _group_defect(U):
    M = U.reshape(-1, 3, 3)
    return max(np.abs(M @ np.conj(np.swapaxes(M, -1, -2)) - np.eye(3)).max(), np.abs(np.linalg.det(M) - 1.0).max())


def test_reunitarise_links_matches_oracle_and_stops_the_drift():
    """lqcd_reunitarise_links against oracle.reunitarise (reading F8, pin H6): on links pushed off the group by a 1e-6
    perturbation (ragged lattice: the last tile is padded), and on the field 100 free-running GPU sweeps leave behind,
    whose rounding drift the projection removes.  12-real storage of the projected field then reproduces its third row."""
    dims = (6, 4, 6, 10)                     # V/2 = 720: not a multiple of the 32-site tile
    L, ctx, U, dev = _setup(dims, 63)
    rng = np.random.default_rng(11)
    noisy = U + 1e-6 * (rng.standard_normal(U.shape) + 1j * rng.standard_normal(U.shape))
    Ud = _Links(ctx, noisy, dev)
    ctx.reunitarise_links(Ud.buf)
    got, ref = Ud.get(), hb.reunitarise(noisy)
    assert np.abs(got - ref).max() <= 1e-14
    assert _group_defect(got) <= 1e-14 and _group_defect(noisy) > 1e-7
    # a field in SU(3) is a fixed point up to rounding
    Ud.put(U)
    ctx.reunitarise_links(Ud.buf)
    same = Ud.get()
    assert np.abs(same - hb.reunitarise(U)).max() <= 1e-14
    assert np.abs(same - U).max() <= 1e-13           # by as much as the generator's U is off the group, i.e. rounding

    # 100 sweeps on 4^4 at beta = 6 without any projection, then one
    dims, beta, ntries = (4, 4, 4, 4), 6.0, 4
    L, ctx, U, dev = _setup(dims, 64)
    Ud = _Links(ctx, U, dev)
    n = ctx.heatbath_uniforms(ntries)
    gen = torch.Generator(device=dev)
    gen.manual_seed(1234)
    for sweep in range(100):
        for mu in range(4):
            for parity in (0, 1):
                u = 1.0 - torch.rand(n, dtype=torch.float64, device=dev, generator=gen)
                ctx.heatbath_sublattice(Ud.buf, beta, mu, parity, u, ntries)
    drifted = Ud.get()
    d0 = _group_defect(drifted)
    assert np.isfinite(drifted.view(np.float64)).all() and d0 < 1e-10       # 2400 rounded SU(2) multiplications per link
    ctx.reunitarise_links(Ud.buf)
    fixed = Ud.get()
    assert _group_defect(fixed) <= 1e-14 and _group_defect(fixed) <= max(d0, 4e-15)
    assert np.abs(fixed - hb.reunitarise(drifted)).max() <= 1e-14
    assert np.abs(fixed - drifted).max() <= 4 * d0 + 1e-14                   # the projection moves a link by the drift, not more
    assert np.abs(np.conj(np.cross(fixed[..., 0, :], fixed[..., 1, :])) - fixed[..., 2, :]).max() <= 5e-15   # what recon 12 rebuilds
