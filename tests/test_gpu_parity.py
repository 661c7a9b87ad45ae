"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element,
on the same seeded inputs.  Tolerances are BASELINE.json north_star's: relative L2 error
<= 1e-12 (fp64), <= 1e-5 (fp32)  (error norm: SURVEY.md A15).
"""
import numpy as np
import pytest

import lattice_inputs as li
import oracle

pytestmark = pytest.mark.gpu

TOL = {64: 1e-12, 32: 1e-5}


def _inputs(cfg_id, precision):
    from gpu_harness import cdtype
    c = li.CONFIGS[cfg_id]
    cd = cdtype(precision)
    # fp32 runs: inputs rounded to fp32 once, the oracle promotes those values (reading A14)
    U = li.links_for_config(cfg_id).astype(cd)
    psi = li.gaussian_spinor(c["dims"]).astype(cd)
    return c, U, psi


@pytest.fixture(scope="module")
def H():
    import gpu_harness
    return gpu_harness


# ------------------------------------------------------------------ config 1: 4^4 fp64 full
@pytest.mark.parametrize("recon", [18, 12])
def test_config1_full_fp64(H, recon):
    c, U, psi = _inputs(1, 64)
    g = H.Gpu(c["dims"], 64, recon, c["bc"], U)
    ref = oracle.dslash_full(U, psi, c["dims"], c["bc"])
    H.assert_parity(g.dslash_full(psi), ref, 64)
    refM = oracle.apply_M(U, psi, c["dims"], c["bc"], c["kappa"], 0)
    H.assert_parity(g.apply_M(psi, c["kappa"], 0), refM, 64)


def test_config1_free_field_plane_wave(H):
    """Unit links: M psi = [(1 - 2k sum cos p) + 2ik sum gamma_mu sin p_mu] psi sitewise (pin P1 on the GPU)."""
    c = li.CONFIGS[1]
    dims, bc, kappa = c["dims"], c["bc"], c["kappa"]
    U = li.unit_links(dims)
    g = H.Gpu(dims, 64, 18, bc, U)
    rng = np.random.default_rng(5)
    for n in [(0, 0, 0, 0), (1, 0, 0, 0), (1, 2, 3, 1), (2, 2, 2, 2), (3, 1, 0, 2)]:
        chi = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
        psi, p = li.plane_wave(dims, n, bc, chi)
        m = (1 - 2 * kappa * np.cos(p).sum()) * np.eye(4, dtype=complex)
        for mu in range(4):
            m = m + 2j * kappa * np.sin(p[mu]) * oracle.gamma(mu)
        expect = np.einsum("st,...ta->...sa", m, psi)
        H.assert_parity(g.apply_M(psi, kappa, 0), expect, 64)


# ------------------------------------------------------------------ config 2: 8^3x16 fp64 eo
@pytest.mark.parametrize("recon", [18, 12, 8])
def test_config2_eo_fp64(H, recon):
    c, U, psi = _inputs(2, 64)
    dims, bc = c["dims"], c["bc"]
    g = H.Gpu(dims, 64, recon, bc, U)
    st = H.site_tol_for(U, 64, recon)
    for out_parity in (0, 1):
        ref = H.half_of(oracle.dslash_eo(U, psi, dims, bc, out_parity), dims, out_parity)
        got = g.dslash_eo(H.half_of(psi, dims, 1 - out_parity), out_parity)
        H.assert_parity(got, ref, 64, site_tol=st)
    # even-odd pieces reassemble the full operator (pin P4 on the GPU)
    full = g.dslash_full(psi)
    H.assert_parity(full, oracle.dslash_full(U, psi, dims, bc), 64, site_tol=st)
    refM = H.half_of(oracle.apply_M(U, psi, dims, bc, c["kappa"], 1), dims, 0)
    H.assert_parity(g.apply_M(H.half_of(psi, dims, 0), c["kappa"], 1), refM, 64, site_tol=st)


def test_config2_gamma5_hermiticity_and_covariance(H):
    """P3 and P5 evaluated on GPU outputs (properties that hold at any size)."""
    c, U, psi = _inputs(2, 64)
    dims, bc = c["dims"], c["bc"]
    g = H.Gpu(dims, 64, 12, bc, U)
    phi = li.gaussian_spinor(dims, seed=11)
    g5 = np.array([1, 1, -1, -1])[:, None]
    lhs = np.vdot(phi, g.dslash_full(psi))
    rhs = np.vdot(g5 * g.dslash_full(g5 * phi), psi)
    assert abs(lhs - rhs) / abs(lhs) <= 1e-12
    gx = li.random_su3_field(dims, seed=3)
    Ug = np.empty_like(U)
    for mu in range(4):
        gshift = np.roll(gx, -1, axis=3 - mu)
        Ug[mu] = gx @ U[mu] @ np.conj(np.swapaxes(gshift, -1, -2))
    g2 = H.Gpu(dims, 64, 12, bc, Ug)
    psig = np.einsum("...ab,...sb->...sa", gx, psi)
    expect = np.einsum("...ab,...sb->...sa", gx, g.dslash_full(psi))
    H.assert_parity(g2.dslash_full(psig), expect, 64)


# ------------------------------------------------------------------ config 3: 16^3x32 full, fp32 + fp64
@pytest.mark.parametrize("precision,recon", [(64, 18), (64, 12), (32, 18), (32, 12), (64, 8), (32, 8)])
def test_config3_full(H, precision, recon):
    c, U, psi = _inputs(3, precision)
    dims, bc = c["dims"], c["bc"]
    g = H.Gpu(dims, precision, recon, bc, U)
    st = H.site_tol_for(U, precision, recon)
    H.assert_parity(g.dslash_full(psi), oracle.dslash_full(U, psi, dims, bc), precision, site_tol=st)
    refM = oracle.apply_M(U, psi, dims, bc, c["kappa"], 0)
    H.assert_parity(g.apply_M(psi, c["kappa"], 0), refM, precision, site_tol=st)


# ------------------------------------------------------------------ edge cases
@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("recon", [18, 12, 8])
def test_ragged_anisotropic_complex_bc(H, precision, recon):
    """Vh = 960 is not a multiple of the block size; all extents differ; general U(1) phases."""
    from gpu_harness import cdtype
    dims = (4, 6, 8, 10)
    bc = np.exp(1j * np.array([0.3, -1.1, 2.0, np.pi]))
    U = li.random_su3_links(dims, seed=21).astype(cdtype(precision))
    psi = li.gaussian_spinor(dims, seed=22).astype(cdtype(precision))
    g = H.Gpu(dims, precision, recon, bc, U)
    st = H.site_tol_for(U, precision, recon)
    H.assert_parity(g.dslash_full(psi), oracle.dslash_full(U, psi, dims, bc), precision, site_tol=st)
    for op in (0, 1):
        ref = H.half_of(oracle.dslash_eo(U, psi, dims, bc, op), dims, op)
        H.assert_parity(g.dslash_eo(H.half_of(psi, dims, 1 - op), op), ref, precision, site_tol=st)
    refM = H.half_of(oracle.apply_M(U, psi, dims, bc, 0.13, 1), dims, 0)
    H.assert_parity(g.apply_M(H.half_of(psi, dims, 0), 0.13, 1), refM, precision, site_tol=st)


@pytest.mark.parametrize("dims", [(6, 6, 6, 6), (4, 6, 6, 6), (6, 4, 6, 10)])
@pytest.mark.parametrize("precision,recon", [(64, 12), (32, 18)])
def test_ragged_last_tile(H, dims, precision, recon):
    """V/2 = 648, 432, 720 are not multiples of the 32-site tile of the native layout (nor of the block
    size): the padded lanes of the last tile are never read or written and nothing is lost."""
    from gpu_harness import cdtype
    U = li.random_su3_links(dims, seed=61).astype(cdtype(precision))
    psi = li.gaussian_spinor(dims, seed=62).astype(cdtype(precision))
    bc = (1, 1, 1, -1)
    g = H.Gpu(dims, precision, recon, bc, U)
    assert np.prod(dims) // 2 % 32 != 0
    H.assert_parity(g.dslash_full(psi), oracle.dslash_full(U, psi, dims, bc), precision)
    for op in (0, 1):
        ref = H.half_of(oracle.dslash_eo(U, psi, dims, bc, op), dims, op)
        H.assert_parity(g.dslash_eo(H.half_of(psi, dims, 1 - op), op), ref, precision)
    refM = H.half_of(oracle.apply_M(U, psi, dims, bc, 0.14, 1), dims, 0)
    H.assert_parity(g.apply_M(H.half_of(psi, dims, 0), 0.14, 1), refM, precision)
    # pack -> unpack round trip is bit exact on the ragged layout too
    assert np.array_equal(g.from_native(g.to_native(psi, -1), -1), psi)


def test_minimum_extent_and_all_periodic(H):
    dims = (4, 4, 4, 4)
    U = li.random_su3_links(dims, seed=31)
    psi = li.gaussian_spinor(dims, seed=32)
    for bc in [(1, 1, 1, 1), (-1, -1, -1, -1)]:
        g = H.Gpu(dims, 64, 12, bc, U)
        H.assert_parity(g.dslash_full(psi), oracle.dslash_full(U, psi, dims, bc), 64)


def test_pack_unpack_roundtrip_bit_exact(H):
    dims = (4, 6, 8, 10)
    U = li.random_su3_links(dims, seed=21)
    psi = li.gaussian_spinor(dims, seed=22)
    for precision in (64, 32):
        g = H.Gpu(dims, precision, 18, (1, 1, 1, -1), U)
        p = psi.astype(H.cdtype(precision))
        assert np.array_equal(g.from_native(g.to_native(p, -1), -1), p)
        for par in (0, 1):
            h = H.half_of(p, dims, par)
            assert np.array_equal(g.from_native(g.to_native(h, par), par), h)


def test_error_codes(H):
    import torch
    import paper_1112_5280_b200 as L
    dims = (4, 4, 4, 4)
    g = H.Gpu(dims, 64, 18, (1, 1, 1, -1), li.unit_links(dims))
    a, b = g.buf(), g.buf()
    with pytest.raises(L.LqcdError) as e:
        g.ctx.dslash_eo(a, g.gauge, a, 0)
    assert e.value.status == L.LQCD_EALIAS
    with pytest.raises(L.LqcdError) as e:
        g.ctx.dslash_eo(a, g.gauge, b, 2)
    assert e.value.status == L.LQCD_EINVAL
    # native fields are read and written with 256-bit words: anything short of 32-byte alignment is refused with a
    # return code (never a misaligned-address fault); the context stays usable afterwards
    ws, full, full2 = g.buf(), g.buf(half=False), g.buf(half=False)
    c = torch.empty((g.ctx.Vh, 4, 3), dtype=torch.complex128, device="cuda:0")
    for off in (8, 16, 24):
        for call in (lambda: g.ctx.dslash_eo(a.data_ptr() + off, g.gauge, b, 0),
                     lambda: g.ctx.dslash_eo(a, g.gauge, b.data_ptr() + off, 0),
                     lambda: g.ctx.dslash_eo(a, g.gauge.data_ptr() + off, b, 0),
                     lambda: g.ctx.dslash_full(full.data_ptr() + off, g.gauge, full2),
                     lambda: g.ctx.dslash_full(full, g.gauge, full2.data_ptr() + off),
                     lambda: g.ctx.apply_M(a.data_ptr() + off, g.gauge, b, 0.1, 1, ws),
                     lambda: g.ctx.apply_M(a, g.gauge, b, 0.1, 1, ws.data_ptr() + off),
                     lambda: g.ctx.apply_M(full, g.gauge.data_ptr() + off, full2, 0.1, 0, None),
                     lambda: g.ctx.pack_spinor(a.data_ptr() + off, c, 0),
                     lambda: g.ctx.unpack_spinor(c, a.data_ptr() + off, 0)):
            with pytest.raises(L.LqcdError) as e:
                call()
            assert e.value.status == L.LQCD_EALIGN
    torch.cuda.synchronize()
    g.ctx.dslash_eo(a, g.gauge, b, 0)   # no sticky error was raised
    torch.cuda.synchronize()
    with pytest.raises(L.LqcdError) as e:
        g.ctx.apply_M(a, g.gauge, b, 0.1, 1, None)
    assert e.value.status == L.LQCD_EINVAL
    with pytest.raises(L.LqcdError) as e:
        g.ctx.apply_M(a, g.gauge, b, 0.1, 1, b)
    assert e.value.status == L.LQCD_EALIAS
    torch.cuda.synchronize()


# ------------------------------------------------------------------ next row f1: twisted-mass matrix
@pytest.mark.parametrize("precision,recon", [(64, 18), (64, 12), (32, 12), (32, 18), (64, 8), (32, 8)])
def test_twisted_mass_matrix(H, precision, recon):
    """lqcd_apply_M_tm against oracle.apply_M_tm: full and even-odd (Schur complement) form, both signs of mu,
    on configs 2 (random SU(3)) and the ragged anisotropic lattice with complex boundary phases."""
    from gpu_harness import cdtype
    cases = [(li.CONFIGS[2]["dims"], li.CONFIGS[2]["bc"], li.links_for_config(2), li.gaussian_spinor(li.CONFIGS[2]["dims"]), 0.15),
             ((4, 6, 8, 10), np.exp(1j * np.array([0.3, -1.1, 2.0, np.pi])), li.random_su3_links((4, 6, 8, 10), seed=21),
              li.gaussian_spinor((4, 6, 8, 10), seed=22), 0.13)]
    for dims, bc, U, psi, kappa in cases:
        U, psi = U.astype(cdtype(precision)), psi.astype(cdtype(precision))
        g = H.Gpu(dims, precision, recon, bc, U)
        st = H.site_tol_for(U, precision, recon)
        for mu in (0.25, -0.4):
            ref = oracle.apply_M_tm(U, psi, dims, bc, kappa, mu, 0)
            H.assert_parity(g.apply_M(psi, kappa, 0, mu=mu), ref, precision, site_tol=st)
            ref = H.half_of(oracle.apply_M_tm(U, psi, dims, bc, kappa, mu, 1), dims, 0)
            H.assert_parity(g.apply_M(H.half_of(psi, dims, 0), kappa, 1, mu=mu), ref, precision, site_tol=st)
        # mu = 0 is lqcd_apply_M bit for bit
        a = g.apply_M(H.half_of(psi, dims, 0), kappa, 1, mu=0.0)
        b = g.apply_M(H.half_of(psi, dims, 0), kappa, 1)
        assert H.rel_l2(a, b) <= 1e-15 if precision == 64 else H.rel_l2(a, b) <= 1e-7


@pytest.mark.parametrize("precision", [32, 16])
@pytest.mark.parametrize("dims", [(8, 8, 8, 16), (6, 6, 6, 6)])
def test_host_batch_pipeline_matches_device_path(H, dims, precision):
    """lqcd_dslash_eo_host_batch with more items than pipeline slots (3): every item equals the device-resident
    path bit for bit and the oracle within tolerance; also on a lattice whose last tile is ragged."""
    import torch
    U = li.random_su3_links(dims, seed=71).astype(np.complex64)
    g = H.Gpu(dims, precision, 12, (1, 1, 1, -1), U)
    n = 7
    psis = [li.gaussian_spinor(dims, seed=80 + i).astype(np.complex64) for i in range(n)]
    par = [i & 1 for i in range(n)]
    ins = [torch.from_numpy(H.half_of(psis[i], dims, 1 - par[i])).pin_memory() for i in range(n)]
    outs = [torch.empty_like(t).pin_memory() for t in ins]
    ws = torch.empty(g.ctx.host_workspace_bytes(), dtype=torch.uint8, device="cuda:0")
    g.ctx.dslash_eo_host_batch(outs, torch.from_numpy(U).pin_memory(), ins, par, ws)
    for i in range(n):
        dev = g.dslash_eo(ins[i].numpy(), par[i])
        assert np.array_equal(outs[i].numpy(), dev), i
        ref = H.half_of(oracle.dslash_eo(U, psis[i], dims, (1, 1, 1, -1), par[i]), dims, par[i])
        assert H.rel_l2(outs[i].numpy(), ref) <= (TOL[32] if precision == 32 else TOL16)
    # links stay packed in the workspace: a second call without them reproduces the result
    outs2 = [torch.zeros_like(t).pin_memory() for t in ins]
    g.ctx.dslash_eo_host_batch(outs2, None, ins, par, ws)
    assert all(np.array_equal(a.numpy(), b.numpy()) for a, b in zip(outs, outs2))
    g.ctx.dslash_eo_host_batch([], None, [], [], ws)  # empty batch is a no-op


# ------------------------------------------------------------------ next row f4: 16-bit storage
TOL16 = 2e-3   # 4 x 2^-11: DESIGN.md section 7 (inputs, links and output each rounded to an 11-bit significand)


def _quantise_spinor(psi):
    """What precision 16 stores: components / site max rounded to IEEE half, times the fp32 site max (numpy emulation
    of the storage format only; no arithmetic of the method)."""
    v = np.ascontiguousarray(psi.astype(np.complex64)).view(np.float32).reshape(*psi.shape[:-2], 24)
    n = np.abs(v).max(axis=-1, keepdims=True)
    inv = np.where(n > 0, np.float32(1) / np.where(n > 0, n, 1), 0).astype(np.float32)
    q = (v * inv).astype(np.float16).astype(np.float32) * n
    return q.reshape(*psi.shape[:-2], 4, 6).view(np.complex64).reshape(psi.shape)


def _quantise_links(U):
    """First two rows rounded to half; the third row is what conj(row0 x row1) rebuilds from them (fp64 here)."""
    r = np.ascontiguousarray(U.astype(np.complex64)).view(np.float32).astype(np.float16).astype(np.float32)
    Uq = r.view(np.complex64).reshape(U.shape).astype(np.complex128)
    Uq[..., 2, :] = np.conj(np.cross(Uq[..., 0, :], Uq[..., 1, :]))
    return Uq


@pytest.mark.parametrize("dims,bc", [((8, 8, 8, 16), (1, 1, 1, -1)), ((6, 6, 6, 6), tuple(np.exp(1j * np.array([0.3, -1.1, 2.0, np.pi]))))])
def test_half_precision_storage(H, dims, bc):
    U = li.random_su3_links(dims, seed=91).astype(np.complex64)
    psi = li.gaussian_spinor(dims, seed=92).astype(np.complex64)
    psi *= np.exp(np.random.default_rng(93).uniform(-6, 6, size=dims[::-1]))[..., None, None].astype(np.float32)  # site norms over 5 decades
    g = H.Gpu(dims, 16, 12, bc, U)
    # storage round trip is exactly the emulated quantisation
    assert np.array_equal(g.from_native(g.to_native(psi, -1), -1), _quantise_spinor(psi))
    Uq, psiq = _quantise_links(U), _quantise_spinor(psi)
    for op in (0, 1):
        got = g.dslash_eo(H.half_of(psi, dims, 1 - op), op)
        ref = H.half_of(oracle.dslash_eo(U, psi, dims, bc, op), dims, op)
        assert H.rel_l2(got, ref) <= TOL16
        # against the oracle fed the values actually stored (reading F4): left are the output rounding
        # (2^-11 of the site max: 1.8e-4) and the two f16 roundings per hop of the arithmetic on stored operands -- the
        # projected half spinor (rms 2^-11 x 0.42 = 2.0e-4 of each component) and the rebuilt third link row (the same on a
        # third of the link entries: 1.2e-4): 3.0e-4 in quadrature, bar at twice that
        refq = H.half_of(oracle.dslash_eo(Uq, psiq, dims, bc, op), dims, op)
        assert H.rel_l2(got, refq) <= 6e-4
        # both sides on the output grid: the arithmetic part alone (2.3e-4) plus grid points it flips; same bar
        assert H.rel_l2(got, _quantise_spinor(refq.astype(np.complex64))) <= 6e-4
    assert H.rel_l2(g.dslash_full(psi), oracle.dslash_full(U, psi, dims, bc)) <= TOL16
    refM = H.half_of(oracle.apply_M(U, psi, dims, bc, 0.15, 1), dims, 0)
    assert H.rel_l2(g.apply_M(H.half_of(psi, dims, 0), 0.15, 1), refM) <= TOL16
    refT = H.half_of(oracle.apply_M_tm(U, psi, dims, bc, 0.15, 0.3, 1), dims, 0)
    assert H.rel_l2(g.apply_M(H.half_of(psi, dims, 0), 0.15, 1, mu=0.3), refT) <= TOL16
    assert H.rel_l2(g.apply_M(psi, 0.15, 0, mu=-0.2), oracle.apply_M_tm(U, psi, dims, bc, 0.15, -0.2, 0)) <= TOL16
    # a zero site stays zero (norm 0)
    z = np.zeros_like(H.half_of(psi, dims, 1))
    assert not g.dslash_eo(z, 0).any()


@pytest.mark.parametrize("precision,kernel", [(16, "gather"), (32, "gather"), (64, "gather"), (32, "pipe"), (64, "pipe"),
                                              (32, "lstage"), (64, "lstage"), (32, "blocked")])
def test_no_writes_outside_the_declared_buffer_sizes(H, precision, kernel):
    """Every output / workspace buffer is carved out of a larger allocation filled with a canary byte; after the
    hot-path calls on a lattice with a ragged last tile, everything outside the declared sizes is untouched."""
    import torch
    dims, bc = (6, 6, 6, 6), (1, 1, 1, -1)
    U = li.random_su3_links(dims, seed=95).astype(H.cdtype(precision))
    psi = li.gaussian_spinor(dims, seed=96).astype(H.cdtype(precision))
    g = H.Gpu(dims, precision, 12, bc, U, kernel=kernel)
    G = 4096
    def guarded(nbytes):
        big = torch.full((nbytes + 2 * G,), 0xAB, dtype=torch.uint8, device="cuda:0")
        return big, big[G:G + nbytes]
    def intact(big, nbytes):
        return bool((big[:G] == 0xAB).all() and (big[G + nbytes:] == 0xAB).all())
    hb, fb = g.ctx.spinor_bytes(True), g.ctx.spinor_bytes(False)
    bo, out = guarded(hb); bw, ws = guarded(g.ctx.workspace_bytes()); bf, outf = guarded(fb)
    in_e, in_o, in_f = g.to_native(H.half_of(psi, dims, 0), 0), g.to_native(H.half_of(psi, dims, 1), 1), g.to_native(psi, -1)
    g.ctx.dslash_eo(out, g.gauge, in_o, 0)
    g.ctx.dslash_eo(out, g.gauge, in_e, 1)
    g.ctx.apply_M(out, g.gauge, in_e, 0.13, 1, ws)
    g.ctx.apply_M_tm(out, g.gauge, in_e, 0.13, 0.2, 1, ws)
    g.ctx.dslash_full(outf, g.gauge, in_f)
    g.ctx.apply_M_tm(outf, g.gauge, in_f, 0.13, 0.2, 0, None)
    torch.cuda.synchronize()
    assert intact(bo, hb) and intact(bw, g.ctx.workspace_bytes()) and intact(bf, fb)
    if precision != 16:
        bc_, cws = guarded(g.ctx.cg_workspace_bytes())
        g.ctx.cg_solve_tm(out, g.gauge, in_e, 0.13, 0.2, 1e-4, 50, cws)
        assert intact(bo, hb) and intact(bc_, g.ctx.cg_workspace_bytes())
    # pack / unpack stay inside their buffers too
    bp, nat = guarded(fb)
    g.ctx.pack_spinor(nat, torch.from_numpy(psi).to("cuda:0"), -1)
    bg, gn = guarded(g.ctx.gauge_bytes())
    g.ctx.pack_gauge(gn, torch.from_numpy(np.ascontiguousarray(U)).to("cuda:0"))
    torch.cuda.synchronize()
    assert intact(bp, fb) and intact(bg, g.ctx.gauge_bytes())


def test_fp32_spinors_with_half_links(H):
    """link_precision = 16: fp32 fields, links stored as 12 halfs.  Against the oracle fed the rounded links the
    result is an ordinary fp32 result (1e-5); against the exact links it is off by the 2^-11 link rounding."""
    dims, bc = (8, 8, 8, 16), (1, 1, 1, -1)
    U = li.random_su3_links(dims, seed=97).astype(np.complex64)
    psi = li.gaussian_spinor(dims, seed=98).astype(np.complex64)
    g = H.Gpu(dims, 32, 12, bc, U, link_precision=16)
    assert g.ctx.gauge_bytes() == 2 * 8 * 4096 * 24
    Uq = _quantise_links(U)
    for op in (0, 1):
        got = g.dslash_eo(H.half_of(psi, dims, 1 - op), op)
        H.assert_parity(got, H.half_of(oracle.dslash_eo(Uq, psi, dims, bc, op), dims, op), 32)
        err = H.rel_l2(got, H.half_of(oracle.dslash_eo(U, psi, dims, bc, op), dims, op))
        assert 1e-5 < err <= 1e-3
    refT = H.half_of(oracle.apply_M_tm(Uq, psi, dims, bc, 0.15, 0.3, 1), dims, 0)
    H.assert_parity(g.apply_M(H.half_of(psi, dims, 0), 0.15, 1, mu=0.3), refT, 32)
    import paper_1112_5280_b200 as L
    with pytest.raises(L.LqcdError) as e:
        L.Context(dims, 64, 12, bc, 16)
    assert e.value.status == L.LQCD_EUNSUPPORTED


# ------------------------------------------------------------------ next row f4: 8-real link storage
@pytest.mark.parametrize("precision", [64, 32])
def test_recon8_links(H, precision):
    """lqcd_pack_gauge with recon = 8: the stored reals are the oracle's pack8 (phases to rounding), the margin the
    library reports is the numpy one, and the operator matches the oracle fed the full 18-real links at north_star's
    rel-L2 tolerances; the per-site bar follows the conditioning of the worst link."""
    import torch
    from oracle import recon8_oracle as r8
    cd = H.cdtype(precision)
    for dims, U in (((8, 8, 8, 16), li.links_for_config(2)), ((6, 6, 6, 6), li.near_unit_links((6, 6, 6, 6), seed=5, eps=0.3))):
        U = U.astype(cd)
        bc = (1, 1, 1, -1)
        psi = li.gaussian_spinor(dims, seed=33).astype(cd)
        g = H.Gpu(dims, precision, 8, bc, U)
        assert g.ctx.gauge_bytes() == 2 * 8 * 8 * 32 * ((g.ctx.Vh + 31) // 32) * (precision // 8)
        site_tol, margin = H.site_tol_for(U, precision, 8), H.recon8_margin(U)
        scratch = torch.zeros(1, dtype=torch.float64, device="cuda:0")
        got_margin = g.ctx.gauge_recon8_margin(torch.from_numpy(np.ascontiguousarray(U)).to("cuda:0"), scratch)
        assert abs(got_margin - margin) <= 1e-6 * margin
        # the packed reals: forward link of the even site cb = 0 is hop 0 of tile 0, lane 0: words [hop][w 2][32][4]
        real = torch.float64 if precision == 64 else torch.float32
        nat = g.gauge.view(real).cpu().numpy().reshape(2, -1, 8, 2, 32, 4)
        for mu in range(4):
            stored = nat[0, 0, 2 * mu, :, 0, :].reshape(8)
            want = r8.pack8(U[mu, 0, 0, 0, 0])
            d = stored - want
            d[6:] = (d[6:] + 1.0) % 2.0 - 1.0
            assert np.abs(d).max() <= (1e-15 if precision == 64 else 1e-7)
        for op in (0, 1):
            ref = H.half_of(oracle.dslash_eo(U, psi, dims, bc, op), dims, op)
            H.assert_parity(g.dslash_eo(H.half_of(psi, dims, 1 - op), op), ref, precision, site_tol=site_tol)
        H.assert_parity(g.dslash_full(psi), oracle.dslash_full(U, psi, dims, bc), precision, site_tol=site_tol)
        refM = H.half_of(oracle.apply_M_tm(U, psi, dims, bc, 0.15, 0.3, 1), dims, 0)
        H.assert_parity(g.apply_M(H.half_of(psi, dims, 0), 0.15, 1, mu=0.3), refM, precision, site_tol=site_tol)
    # unit links are outside the encoding: the library says so (margin 0) and precision 16 has no 8-real variant
    dims = (4, 4, 4, 4)
    c = H.Gpu(dims, precision, 8, (1, 1, 1, -1), li.random_su3_links(dims, seed=3).astype(cd)).ctx
    assert c.gauge_recon8_margin(torch.from_numpy(li.unit_links(dims).astype(cd)).to("cuda:0"), scratch) == 0.0
    import paper_1112_5280_b200 as L
    # ... and lqcd_pack_gauge refuses them instead of packing something the dslash turns into NaN: the whole unit field,
    # a single unit link in an otherwise random field, one link with U00 = 0 (a cyclic permutation matrix), one NaN
    good = li.random_su3_links(dims, seed=3).astype(cd)
    one_unit, one_perm, one_nan = good.copy(), good.copy(), good.copy()
    one_unit[2, 1, 3, 0, 2] = np.eye(3)
    one_perm[1, 3, 2, 1, 0] = np.roll(np.eye(3), 1, axis=1)
    one_nan[0, 0, 0, 0, 0, 0, 1] = np.nan
    native = torch.empty(c.gauge_bytes(), dtype=torch.uint8, device="cuda:0")
    for what, bad in (("unit field", li.unit_links(dims).astype(cd)), ("one unit link", one_unit),
                      ("one permutation link", one_perm), ("one NaN", one_nan)):
        with pytest.raises(L.LqcdError) as e:
            c.pack_gauge(native, torch.from_numpy(np.ascontiguousarray(bad)).to("cuda:0"))
            pytest.fail(f"recon 8: {what} was packed without complaint")
        assert e.value.status == L.LQCD_EUNSUPPORTED, what
    c.pack_gauge(native, torch.from_numpy(np.ascontiguousarray(good)).to("cuda:0"))   # the flag does not stick
    # a cold start therefore goes through 12-real links and gives finite numbers (H psi = 8 psi for constant psi)
    g12 = H.Gpu(dims, precision, 12, (1, 1, 1, 1), li.unit_links(dims).astype(cd))
    const = np.ones(dims[::-1] + (4, 3), dtype=cd)
    assert np.allclose(g12.dslash_full(const), 8 * const)
    with pytest.raises(L.LqcdError) as e:
        L.Context(dims, 16, 8)
    assert e.value.status == L.LQCD_EUNSUPPORTED
