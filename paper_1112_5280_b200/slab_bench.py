"""bench.py's `slab` leg: the even-odd dslash of the bench workload decomposed into time slabs over the ranks of the
process group (next row f3; paper_1112_5280_b200/slab.py).  One rank = one GPU = T / world time slices.  With one rank
the ring closes on itself (the faces go through the halo buffers back into the same GPU): that measures what the
decomposition costs -- face projection, halo reads, three launches instead of one -- without any link in between.
Plumbing and timing only; the kernels are lqcd_slab_push_faces / lqcd_dslash_eo_range / lqcd_dslash_eo_slab."""
from __future__ import annotations

import numpy as np


def run(torch, dist, timer, dev, cfg_id, precision, recon, steps, warmup, peak, world, rank, flop_per_site, nbuf=4):
    import lattice_inputs as li
    from .slab import TimeSlab, make_transport, SendRecvTransport
    c = li.CONFIGS[cfg_id]
    dims, bc = c["dims"], c["bc"]
    cd = np.complex128 if precision == 64 else np.complex64
    s = TimeSlab(dims, precision, recon, bc, rank, world)
    if world > 1:
        transport, tname = make_transport(s, dist, dev, "auto")
    else:
        transport, tname = SendRecvTransport(s, None, dev), "ring of one: device copies of the own faces"
    tl = s.time_indices()
    U = li.links_time_slices(cfg_id, tl + [s.t_below()], dtype=cd)
    gauge = torch.empty(s.ctx.gauge_bytes(), dtype=torch.uint8, device=dev)
    s.pack_gauge(gauge, torch.from_numpy(np.ascontiguousarray(U[:, :-1])).to(dev), torch.from_numpy(np.ascontiguousarray(U[3, -1])).to(dev))
    del U
    mask = [li.parity_mask(s.local_dims, p).ravel() for p in (0, 1)]
    inp, out = [], []
    for b in range(nbuf):
        psi = li.gaussian_spinor_time_slices(dims, tl, seed=li.SPINOR_SEED + b, dtype=cd)
        half = np.ascontiguousarray(psi.reshape(-1, 4, 3)[mask[1 - (b & 1)]])
        n = torch.empty(s.ctx.spinor_bytes(True), dtype=torch.uint8, device=dev)
        s.ctx.pack_spinor(n, torch.from_numpy(half).to(dev), 1 - (b & 1))
        inp.append(n)
        out.append(torch.empty_like(n))
    torch.cuda.synchronize(dev)

    def step():
        for b in range(nbuf):
            s.dslash_eo(out[b], gauge, inp[b], b & 1, transport)

    m = timer.measure(step, steps, warmup, 4 * nbuf, nregions=3)
    ms = m["median"]["ms_per_step"]
    us = ms / nbuf * 1e3
    Vh_global = int(np.prod(dims)) // 2
    per_site = (48 + 8 * recon) * (precision // 8)
    halo = 2 * s.halo_bytes
    return {
        "workload": f"config {cfg_id}: {'x'.join(map(str, dims))} even-odd dslash on {world} time slab(s) of {s.Tl} slices, "
                    f"fp{precision} recon-{recon}",
        "transport": tname,
        "us_per_application": us,                                   # max over ranks (timer)
        "gflops_aggregate": Vh_global * flop_per_site / (us * 1e-6) / 1e9,
        "gbs_per_gpu": per_site * s.ctx.Vh / (us * 1e-6) / 1e9,
        "frac_of_hbm_peak_per_gpu": per_site * s.ctx.Vh / (us * 1e-6) / 1e9 / peak,
        "halo_bytes_sent_per_rank_per_application": halo,
        "halo": "projected half spinors, 12 reals per face site, one face up and one down",
        "launches_per_application": 4 + (1 if isinstance(transport, SendRecvTransport) and world > 1 else 0),
        "sm_mhz": m["median"]["clocks"]["sm_mhz"] if m["median"]["clocks"] else None,
        "regions_us": [r["ms_per_step"] / nbuf * 1e3 for r in m["regions"]],
    }
