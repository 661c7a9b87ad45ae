"""GPU parity at BASELINE.json's full sizes (configs 4 and 5), in the launch configuration
bench.py times: the oracle computes sampled output sites one by one (oracle.dslash_sites /
apply_M_sites) and the CUDA result is compared there; plus properties that hold at any size.
"""
import numpy as np
import pytest

import lattice_inputs as li
import oracle

pytestmark = pytest.mark.gpu

TOL = {64: 1e-12, 32: 1e-5}


def sample_sites(dims, parity, n, seed):
    """n random sites of the given parity plus the corners/faces where the wrap logic lives."""
    X, Y, Z, T = dims
    rng = np.random.default_rng(seed)
    c = np.stack([rng.integers(0, L, size=4 * n) for L in dims], axis=1)
    edge = [[a, b, cc, d] for a in (0, 1, X - 2, X - 1) for b in (0, Y - 1) for cc in (0, Z - 1) for d in (0, 1, T - 1)]
    c = np.concatenate([np.array(edge), c])
    c = c[(c.sum(axis=1) & 1) == parity]
    return c[: n + len(edge)]


def cb_index(dims, coords):
    X, Y, Z, T = dims
    lex = coords[:, 0] + X * (coords[:, 1] + Y * (coords[:, 2] + Z * coords[:, 3]))
    return lex >> 1


@pytest.fixture(scope="module")
def cfg4():
    c = li.CONFIGS[4]
    U = li.links_for_config(4)
    psi = li.gaussian_spinor(c["dims"])
    return c, U, psi


@pytest.mark.parametrize("recon", [12, 8])
@pytest.mark.parametrize("precision", [32, 64])
def test_config4_eo_recon12_sampled(cfg4, precision, recon):
    import gpu_harness as H
    c, U64, psi64 = cfg4
    dims, bc = c["dims"], c["bc"]
    U = U64.astype(H.cdtype(precision))
    psi = psi64.astype(H.cdtype(precision))
    g = H.Gpu(dims, precision, recon, bc, U)
    site_tol = H.site_tol_for(U, precision, recon)   # recon 8: from the conditioning of the worst of the 8.4 M links
    for out_parity in (0, 1):
        got = g.dslash_eo(H.half_of(psi, dims, 1 - out_parity), out_parity)
        sites = sample_sites(dims, out_parity, 4096, seed=40 + out_parity)
        ref = oracle.dslash_sites(U, psi, dims, bc, sites)
        H.assert_parity(got[cb_index(dims, sites)], ref, precision, site_tol=site_tol)
        assert np.isfinite(got.view(np.float32 if precision == 32 else np.float64)).all()
    if recon != 12:
        return
    # host-buffer entry point (what bench.py's e2e leg times) gives the same result bit for bit
    import torch
    ws = torch.empty(g.ctx.host_workspace_bytes(), dtype=torch.uint8, device="cuda:0")
    in_h = torch.from_numpy(H.half_of(psi, dims, 1)).pin_memory()
    U_h = torch.from_numpy(np.ascontiguousarray(U)).pin_memory()
    out_h = torch.empty_like(in_h).pin_memory()
    g.ctx.dslash_eo_host(out_h, U_h, in_h, 0, ws)
    dev = g.dslash_eo(H.half_of(psi, dims, 1), 0)
    assert np.array_equal(out_h.numpy(), dev)


def test_config4_full_field_fp32_vs_oracle(cfg4):
    """Whole-field comparison at the headline size (the oracle needs a few seconds here)."""
    import gpu_harness as H
    c, U64, psi64 = cfg4
    dims, bc = c["dims"], c["bc"]
    U = U64.astype(np.complex64)
    psi = psi64.astype(np.complex64)
    g = H.Gpu(dims, 32, 12, bc, U)
    ref = H.half_of(oracle.dslash_eo(U, psi, dims, bc, 0), dims, 0)
    H.assert_parity(g.dslash_eo(H.half_of(psi, dims, 1), 0), ref, 32)


@pytest.fixture(scope="module")
def cfg5():
    """Config-5 inputs, generated once for both link-storage variants (the A11 link field takes minutes)."""
    c = li.CONFIGS[5]
    return c, li.links_for_config(5, dtype=np.complex64), li.gaussian_spinor(c["dims"], dtype=np.complex64)


@pytest.mark.parametrize("recon", [12, 18])
def test_config5_chain_per_step_parity(cfg5, recon):
    """Config 5 (reading A16): x_{k+1} = M x_k chained 100 times in fp32; per-step parity at
    k in {1, 50, 100}: the oracle is fed the GPU's own x_k and compared with x_{k+1} at sampled sites."""
    import torch
    import gpu_harness as H
    c, U, psi = cfg5
    dims, bc, kappa = c["dims"], c["bc"], c["kappa"]
    g = H.Gpu(dims, 32, recon, bc, U)
    x = g.to_native(H.half_of(psi, dims, 0), 0)
    y, ws = g.buf(), g.buf()
    sites = sample_sites(dims, 0, 1024, seed=50)
    idx = cb_index(dims, sites)
    for k in range(1, 101):
        g.ctx.apply_M(y, g.gauge, x, kappa, 1, ws)
        if k in (1, 50, 100):
            xk = H.scatter_half(g.from_native(x, 0), dims, 0)
            got = g.from_native(y, 0)
            assert np.isfinite(got.view(np.float32)).all()
            ref = oracle.apply_M_sites(U, xk, dims, bc, kappa, 1, sites)
            H.assert_parity(got[idx], ref, 32, what=str(k))
        x, y = y, x
    torch.cuda.synchronize()


@pytest.mark.parametrize("precision", [32, 64])
def test_config4_properties_at_full_size(cfg4, precision):
    """Properties that hold at any size, checked on the GPU at 32^3x64 with the bench's launch configuration:
    gamma5-hermiticity <phi_e, H_eo psi_o> = <g5 H_oe g5 phi_e, psi_o> (pin P3), linearity, and
    Q(mu)^dagger = Q(-mu) for the twisted-mass operator the solver iterates with."""
    import torch
    import gpu_harness as H
    c, U64, psi64 = cfg4
    dims, bc = c["dims"], c["bc"]
    cd = H.cdtype(precision)
    g = H.Gpu(dims, precision, 12, bc, U64.astype(cd))
    phi = li.gaussian_spinor(dims, seed=77).astype(cd)
    g5 = np.array([1, 1, -1, -1], dtype=np.float64)[:, None]
    psi_o, phi_e = H.half_of(psi64.astype(cd), dims, 1), H.half_of(phi, dims, 0)
    lhs = np.vdot(phi_e.astype(np.complex128), g.dslash_eo(psi_o, 0).astype(np.complex128))
    rhs = np.vdot((g5 * g.dslash_eo((g5 * phi_e).astype(cd), 1)).astype(np.complex128), psi_o.astype(np.complex128))
    tol = 1e-12 if precision == 64 else 2e-6
    assert abs(lhs - rhs) <= tol * abs(lhs)
    # linearity
    a, b = 0.7 - 0.2j, -1.3 + 0.4j
    psi2 = H.half_of(li.gaussian_spinor(dims, seed=78).astype(cd), dims, 1)
    comb = g.dslash_eo((a * psi_o + b * psi2).astype(cd), 0)
    H.assert_parity(comb, a * g.dslash_eo(psi_o, 0).astype(np.complex128) + b * g.dslash_eo(psi2, 0).astype(np.complex128), precision)
    # <phi, Q(mu) psi> = <Q(-mu) phi, psi> on even fields
    kappa, mu = c["kappa"], 0.05
    psi_e = H.half_of(psi64.astype(cd), dims, 0)
    def Q(v, m):
        out = g.buf()
        g.ctx.apply_Q_tm(out, g.gauge, g.to_native(v, 0), kappa, m, g.buf())
        return g.from_native(out, 0).astype(np.complex128)
    l2 = np.vdot(phi_e.astype(np.complex128), Q(psi_e, mu))
    r2 = np.vdot(Q(phi_e, -mu), psi_e.astype(np.complex128))
    assert abs(l2 - r2) <= tol * abs(l2)


def test_largest_lattice_index_headroom():
    """64^3x128 fp32 recon-12 (V/2 = 16.8 M sites; 12.9 GB of packed links, 9.7 GB canonical): checkerboard
    indices, tile offsets and byte offsets well past 2^32 bytes; sampled parity against the oracle incl. the corners."""
    import torch
    import gpu_harness as H
    dims, bc = (64, 64, 64, 128), (1, 1, 1, -1)
    free, _ = torch.cuda.mem_get_info()
    if free < 40e9:
        pytest.skip("needs 40 GB of free device memory")
    U = li.random_su3_links(dims, seed=111, dtype=np.complex64)
    psi = li.gaussian_spinor(dims, seed=112, dtype=np.complex64)
    g = H.Gpu(dims, 32, 12, bc, U)
    assert g.ctx.gauge_bytes() > 2 ** 33
    for out_parity in (0, 1):
        got = g.dslash_eo(H.half_of(psi, dims, 1 - out_parity), out_parity)
        sites = sample_sites(dims, out_parity, 2048, seed=120 + out_parity)
        ref = oracle.dslash_sites(U, psi, dims, bc, sites)
        H.assert_parity(got[cb_index(dims, sites)], ref, 32)
        assert np.isfinite(got.view(np.float32)).all()


@pytest.mark.parametrize("precision", [32, 64])
@pytest.mark.parametrize("kernel", ["pipe", "lstage", "blocked"])
def test_config4_kernel_variants_bitwise(cfg4, precision, kernel):
    """At the bench size (32^3 x 64: 32768 warp tiles per parity, ~220 per persistent CTA) the data-movement variants
    of lqcd_set_kernel give the gather kernel's result bit for bit, both parities; the gather kernel itself is checked
    against the oracle on sampled sites above."""
    import gpu_harness as H
    c, U64, psi64 = cfg4
    dims, bc = c["dims"], c["bc"]
    U = U64.astype(H.cdtype(precision))
    psi = psi64.astype(H.cdtype(precision))
    ref = H.Gpu(dims, precision, 12, bc, U, kernel="gather")
    g = H.Gpu(dims, precision, 12, bc, U, kernel=kernel)
    for out_parity in (0, 1):
        half = H.half_of(psi, dims, 1 - out_parity)
        assert np.array_equal(g.dslash_eo(half, out_parity), ref.dslash_eo(half, out_parity)), (kernel, precision, out_parity)
    e = H.half_of(psi, dims, 0)
    assert np.array_equal(g.apply_M(e, c["kappa"], 1, mu=0.1), ref.apply_M(e, c["kappa"], 1, mu=0.1))
