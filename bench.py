#!/usr/bin/env python
"""bench.py -- Wilson dslash benchmark on B200 (BASELINE.json metric: dslash GFLOP/s at 1320 flop/site
and achieved HBM GB/s vs roofline at 32^3x64).

    python bench.py --gpus 1 --steps K --warmup W            # this repo's CUDA path (default)
    python bench.py --impl reference --steps K --warmup W    # the CPU oracle on the host cores

Workload (config.workload): BASELINE.json configs[3] = SURVEY.md sec. 8(d) config 4, the headline
bandwidth case: 32^3x64, even-odd dslash, 12-real links, random SU(3) links (seed 1), Gaussian
spinors (seed 2), antiperiodic in t.  Primary line fp32.  Further legs ride in the same JSON line (--legs):
"fp64" (the other precision), "matrix" (apply_M / apply_M_tm), "cg", "cg_fp64", "cg_mixed", "cg_mixed_half_links"
(the solver), "fp16_storage" and "fp32_half_links" (16-bit storage variants), "e2e" (host buffers), "cpu_baseline"
(the oracle), and with --chain the config-5 M-chain at 48^3x96.

A step = one pass of the hot path (K1..L6 of SURVEY.md sec. 8(a)) over one batch of NBUF = 4
half-lattice spinors: NBUF launches of lqcd_dslash_eo, alternating out_parity 0,1 (H_eo, H_oe),
each reading its own input buffer and writing its own output buffer.  Rotating buffers keeps the
spinor working set (NBUF x 2 x 100/201 MB) above the 126 MB L2 so no launch finds its input
resident from the previous one; the 403/805 MB link field is streamed once per launch.

Multi-GPU: the path does not shard in this build ("replicas only"): --gpus N runs N
independent replicas, one process per GPU, no data-path collective; value = N replicas' sites / max time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

FLOP_PER_SITE = 1320                  # BASELINE.json convention: 8 x (12 + 132) + 7 x 24
REALS_PER_SITE = {12: 144, 18: 192}   # compulsory eo model: 24 in + 24 out + 8 links
NBUF = 4
METRIC = "dslash GFLOP/s (1320 flop/site), 32^3x64 even-odd recon-12"
FALLBACK_HBM_GBS = 6650.0             # /opt/skills/guides/B200_PROFILING.md fallback
NOMINAL_HBM_GBS = 8000.0              # north_star's "~8 TB/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=500)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", type=int, default=4, help="lattice_inputs.CONFIGS id of the main workload")
    ap.add_argument("--precision", type=int, default=32, choices=[16, 32, 64], help="precision of the primary line (16: half storage, fp32 arithmetic)")
    ap.add_argument("--recon", type=int, default=12, choices=[12, 18])
    ap.add_argument("--block", type=int, default=0, help="dslash block size override (tuning)")
    ap.add_argument("--chain", action="store_true", help="also time config 5: apply_M(eo=1) x100 chained at 48^3x96")
    ap.add_argument("--no-extras", action="store_true", help="skip the fp64 / chain / e2e / cpu legs (profiling runs)")
    ap.add_argument("--legs", default="all", help="comma list of extra legs to run: matrix,cg,e2e,other,fp16,cgmixed,cpu (default all)")
    return ap.parse_args()


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, device copy)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(precision, recon):
    """dram bytes per launch of the dslash kernel from the committed ncu --set full summary, or None."""
    path = os.path.join(ROOT, "profiles", "dram_traffic.csv")
    try:
        with open(path) as f:
            for line in f:
                p = [x.strip() for x in line.split(",")]
                if len(p) >= 4 and p[0] == "config4" and p[1] == f"fp{precision}" and p[2] == f"recon{recon}":
                    return float(p[3])
    except OSError:
        pass
    return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 50 ms while the kernels run."""
    Q = ("clocks.sm,clocks.max.sm,utilization.gpu,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "50"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._read, daemon=True)
            self.thr.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.12)
        self.proc.terminate()
        self.thr.join(timeout=2)
        sm, smax, reasons, n = [], None, set(), 0
        for ts, line in self.rows:
            if not (t0 <= ts <= t1 + 0.06):
                continue
            p = [x.strip() for x in line.split(",")]
            try:
                clk, mx, util = float(p[0]), float(p[1]), float(p[2])
            except (ValueError, IndexError):
                continue
            n += 1
            smax = mx
            if util >= 50 or not sm:
                sm.append(clk)
            for name, v in zip(self.NAMES, p[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": smax, "reasons": sorted(reasons),
                "samples": n}


# ------------------------------------------------------------------------------------------------
# this repo's arm
# ------------------------------------------------------------------------------------------------
class Workload:
    """Seeded inputs of one config on the device in native layout, plus pinned host copies."""

    def __init__(self, cfg_id, precision, recon, dev, block=0, nbuf=NBUF, keep_host=True, in_parity=None, U=None, link_precision=0):
        import numpy as np
        import torch
        import lattice_inputs as li
        import paper_1112_5280_b200 as L
        self.L, self.torch = L, torch
        c = li.CONFIGS[cfg_id]
        self.cfg_id, self.dims, self.bc, self.kappa = cfg_id, c["dims"], c["bc"], c["kappa"]
        self.precision, self.recon, self.dev, self.nbuf = precision, recon, dev, nbuf
        cd = np.complex128 if precision == 64 else np.complex64  # precision 16 exchanges complex64
        self.ctx = L.Context(self.dims, precision, recon, self.bc, link_precision)
        if block:
            self.ctx.set_block_threads(block)
        self.Vh = self.ctx.Vh
        if U is None:
            U = li.links_for_config(cfg_id, dtype=cd)
        self.U_host = torch.from_numpy(U).pin_memory() if keep_host else None
        self.gauge = torch.empty(self.ctx.gauge_bytes(), dtype=torch.uint8, device=dev)
        Ud = torch.from_numpy(U).to(dev)
        self.ctx.pack_gauge(self.gauge, Ud)
        torch.cuda.synchronize(dev)
        del Ud, U
        mask = [li.parity_mask(self.dims, p).ravel() for p in (0, 1)]
        self.inp, self.out, self.in_host = [], [], []
        for b in range(nbuf):
            out_parity = (b & 1) if in_parity is None else 1 - in_parity
            psi = li.gaussian_spinor(self.dims, seed=li.SPINOR_SEED + b, dtype=cd)
            half = np.ascontiguousarray(psi.reshape(-1, 4, 3)[mask[1 - out_parity]])
            h = torch.from_numpy(half).pin_memory()
            n = torch.empty(self.ctx.spinor_bytes(True), dtype=torch.uint8, device=dev)
            self.ctx.pack_spinor(n, h.to(dev), 1 - out_parity)
            self.inp.append(n)
            self.out.append(torch.empty_like(n))
            if keep_host:
                self.in_host.append(h)
        torch.cuda.synchronize(dev)

    def step(self):
        for b in range(self.nbuf):
            self.ctx.dslash_eo(self.out[b], self.gauge, self.inp[b], b & 1)

    def sites_per_step(self):
        return self.nbuf * self.Vh

    def bytes_per_launch(self):
        # 16-bit storage: 24 halfs + one fp32 norm per spinor site (in and out), 12 halfs per link
        per_site = 2 * 52 + 8 * 24 if self.precision == 16 else REALS_PER_SITE[self.recon] * (self.precision // 8)
        return per_site * self.Vh


def timed_steps(torch, dist, fn, steps, warmup, reduce_device="cuda"):
    """W untimed steps, then K steps between two CUDA events on the launching (current) stream,
    barrier + synchronize on both sides; returns max-over-ranks milliseconds for the K steps."""
    for _ in range(warmup):
        fn()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    e0.record()
    for _ in range(steps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    return max_over_ranks(torch, dist, e0.elapsed_time(e1), reduce_device)


def max_over_ranks(torch, dist, ms, device):
    """Multi-GPU timing rule: the time of a replicated run is the slowest rank's device time."""
    if dist is None:
        return float(ms)
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_gflops(world, sites_per_step_per_rank, ms_per_step):
    """Whole-job throughput of `world` independent replicas (weak scaling, no data-path collective)."""
    return world * sites_per_step_per_rank * FLOP_PER_SITE / (ms_per_step * 1e-3) / 1e9


def kernel_leg(torch, dist, w, steps, warmup, world, reduce_device="cuda"):
    """Device-resident timing of one Workload: returns the numbers of one precision/recon case."""
    L = w.L
    n0 = L.launch_count()
    ms = timed_steps(torch, dist, w.step, steps, warmup, reduce_device)
    launches = (L.launch_count() - n0) - warmup * w.nbuf
    ms_step = ms / steps
    t_launch = ms_step / w.nbuf * 1e-3
    return {
        "ms_per_step": ms_step,
        "us_per_launch": t_launch * 1e6,
        "gflops": aggregate_gflops(world, w.sites_per_step(), ms_step),
        "gbs": w.bytes_per_launch() / t_launch / 1e9,
        "launches": launches,
    }


def e2e_leg(torch, w, steps, world):
    """Same metric through the host-buffer entry point lqcd_dslash_eo_host_batch: per item pinned canonical half
    spinor in (H2D), pack, dslash, unpack, canonical half spinor out (D2H), all inside the timed region; the
    library overlaps upload, kernels and download of consecutive items on three streams.
    The link field is uploaded once before (it is constant across applications, like weights)."""
    ctx = w.ctx
    ws = torch.empty(ctx.host_workspace_bytes(), dtype=torch.uint8, device=w.dev)
    out_h = [torch.empty_like(h).pin_memory() for h in w.in_host]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    # gauge upload + pack + one application, timed separately (3 repetitions, best)
    tg = []
    for _ in range(3):
        torch.cuda.synchronize()
        e0.record()
        ctx.dslash_eo_host(out_h[0], w.U_host, w.in_host[0], 0, ws)
        e1.record()
        torch.cuda.synchronize()
        tg.append(e0.elapsed_time(e1))
    par = [b & 1 for b in range(w.nbuf)]
    ctx.dslash_eo_host_batch(out_h, None, w.in_host, par, ws)  # warm-up
    torch.cuda.synchronize()
    regions = []
    for _ in range(2):  # the host link is shared with other tenants of the box: two regions, the quieter one counts
        t0 = time.perf_counter()
        e0.record()
        for _ in range(steps):
            ctx.dslash_eo_host_batch(out_h, None, w.in_host, par, ws)  # one step = the batch of NBUF half spinors
        e1.record()
        torch.cuda.synchronize()
        wall = (time.perf_counter() - t0) * 1e3
        regions.append(max(e0.elapsed_time(e1), wall) / steps)
    ms = min(regions)
    hb = w.in_host[0].numel() * w.in_host[0].element_size()
    return {
        "value": world * w.sites_per_step() * FLOP_PER_SITE / (ms * 1e-3) / 1e9,
        "unit": "GFLOP/s",
        "h2d_bytes_per_step": hb * w.nbuf,
        "d2h_bytes_per_step": hb * w.nbuf,
        "ms_per_step": ms,
        "ms_per_step_regions": regions,
        "steps": steps,
        "gauge": "resident (uploaded and packed once before the timed region)",
        "ms_one_application_with_gauge_upload": min(tg),
        "gauge_h2d_bytes": w.U_host.numel() * w.U_host.element_size(),
    }


def chain_leg(torch, cfg_id, precision, recon, dev, napply=100, reps=3, U=None):
    """Config 5 (reading A16): x_{k+1} = M x_k, M = 1 - kappa^2 H_eo H_oe, `napply` times back to back,
    ping-pong buffers, timed as one block."""
    w = Workload(cfg_id, precision, recon, dev, nbuf=1, keep_host=False, in_parity=0, U=U)  # even half spinor
    x, y = w.inp[0], w.out[0]
    ws = torch.empty_like(x)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    best = None
    for _ in range(reps + 1):
        a, b = x.clone(), y
        torch.cuda.synchronize()
        e0.record()
        for _k in range(napply):
            w.ctx.apply_M(b, w.gauge, a, w.kappa, 1, ws)
            a, b = b, a
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        best = ms if best is None else min(best, ms)
    reals = REALS_PER_SITE[recon] * 2 + 24  # pass 1 + pass 2 with the xpay read
    nbytes = reals * (precision // 8) * w.Vh
    finite = bool(torch.isfinite(a.view(torch.float32 if precision == 32 else torch.float64)).all().item())
    return {
        "workload": f"config {cfg_id}: {'x'.join(map(str, w.dims))} fp{precision} recon-{recon} apply_M(eo=1) x{napply} chained",
        "ms_per_chain": best, "ms_per_application": best / napply,
        "gflops": 2 * FLOP_PER_SITE * w.Vh * napply / (best * 1e-3) / 1e9,
        "gbs": nbytes * napply / (best * 1e-3) / 1e9,
        "bytes_per_application": nbytes, "finite": finite,
    }


def matrix_leg(torch, w, napply=50, reps=3):
    """Fermion-matrix applications on the primary workload's fields: lqcd_apply_M(eo=1) and the twisted-mass
    lqcd_apply_M_tm(eo=1) (next row f1), napply back-to-back applications alternating between two input
    buffers, best of `reps`.  2 launches, 2 x 1320 flop and (2 x (24 + 24 + 8 recon) + 24) reals per even site."""
    x, y, ws = w.inp[1], w.out[1], w.out[0]   # inp[1] holds an even half spinor (out_parity 1)
    x2, y2 = w.inp[3 % w.nbuf], w.out[3 % w.nbuf]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    res = {}
    for name, fn in (("apply_M", lambda o, i: w.ctx.apply_M(o, w.gauge, i, w.kappa, 1, ws)),
                     ("apply_M_tm", lambda o, i: w.ctx.apply_M_tm(o, w.gauge, i, w.kappa, 0.05, 1, ws))):
        best = None
        for _ in range(reps + 1):
            torch.cuda.synchronize()
            e0.record()
            for k in range(napply):
                fn(y, x) if k & 1 else fn(y2, x2)
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / napply
            best = ms if best is None else min(best, ms)
        nbytes = 2 * w.bytes_per_launch() + w.bytes_per_launch() * 24 // (2 * 24 + 8 * w.recon)  # two passes + the xpay read
        if w.precision == 16:
            nbytes = 2 * w.bytes_per_launch() + 52 * w.Vh
        res[name] = {"us_per_application": best * 1e3, "gflops": 2 * FLOP_PER_SITE * w.Vh / (best * 1e-3) / 1e9,
                     "gbs": nbytes / (best * 1e-3) / 1e9}
    return res


def cg_leg(torch, w, mu=0.05, tol=None, maxiter=400):
    """Next row f2: lqcd_cg_solve_tm on the primary workload (even source = inp[1]).  One iteration = two
    applications of Q = gamma_5 Mhat_tm (4 dslash launches) + 5 BLAS-1/scalar launches; flops counted by the dslash
    convention only (4 x 1320 per even site per iteration); bytes: 2 x (2 x (48 + 8 recon) + 24) + 240 reals."""
    tol = tol or (1e-5 if w.precision == 32 else 1e-10)
    x = torch.empty_like(w.inp[1])
    ws = torch.empty(w.ctx.cg_workspace_bytes(), dtype=torch.uint8, device=w.dev)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    best, it, res = None, 0, 0.0
    for _ in range(2):
        torch.cuda.synchronize()
        e0.record()
        it, res = w.ctx.cg_solve_tm(x, w.gauge, w.inp[1], w.kappa, mu, tol, maxiter, ws)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        best = ms if best is None else min(best, ms)
    enq = it   # the flag is read every iteration near convergence, so (almost) no iteration is enqueued in vain
    reals = 2 * (2 * REALS_PER_SITE[w.recon] + 24) + 240
    return {"iterations": it, "relres": res, "tol": tol, "kappa": w.kappa, "mu": mu, "ms": best,
            "us_per_iteration": best * 1e3 / max(enq, 1),
            "gflops": 4 * FLOP_PER_SITE * w.Vh * enq / (best * 1e-3) / 1e9 if enq else 0.0,
            "gbs": reals * (w.precision // 8) * w.Vh * enq / (best * 1e-3) / 1e9 if enq else 0.0}


def cg_mixed_leg(torch, w64, w32, mu=0.05, tol=1e-10, inner_tol=1e-4, maxiter=2000):
    """lqcd_cg_solve_tm_mixed: the same fp64 system as cg_leg(w64), iterated in fp32 with fp64 defect correction."""
    b = w64.inp[1]
    x = torch.empty_like(b)
    ws = torch.empty(w64.ctx.cg_mixed_workspace_bytes(w32.ctx), dtype=torch.uint8, device=w64.dev)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    best = None
    for _ in range(2):
        torch.cuda.synchronize()
        e0.record()
        it, outer, res = w64.ctx.cg_solve_tm_mixed(w32.ctx, x, w64.gauge, w32.gauge, b, w64.kappa, mu, tol, inner_tol, maxiter, ws)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        best = ms if best is None else min(best, ms)
    return {"inner_iterations": it, "outer_corrections": outer, "true_relres": res, "tol": tol, "inner_tol": inner_tol,
            "ms": best}


def cpu_baseline_leg(cfg_id, precision):
    """The oracle as it stands on the host cores: full-lattice dslash_eo of the same workload,
    one warm-up then best of 3 (about 2-5 s of CPU work on 8+ cores)."""
    import numpy as np
    import lattice_inputs as li
    import oracle
    c = li.CONFIGS[cfg_id]
    cd = np.complex64 if precision == 32 else np.complex128
    U = li.links_for_config(cfg_id, dtype=cd)
    psi = li.gaussian_spinor(c["dims"], dtype=cd)
    Vh = int(np.prod(c["dims"])) // 2
    oracle.dslash_eo(U, psi, c["dims"], c["bc"], 0)
    best = None
    for _ in range(3):
        t0 = time.perf_counter()
        oracle.dslash_eo(U, psi, c["dims"], c["bc"], 0)
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    nthreads = oracle.num_threads()
    oracle.set_num_threads(1)
    t0 = time.perf_counter()
    oracle.dslash_eo(U, psi, c["dims"], c["bc"], 0)
    one = time.perf_counter() - t0
    oracle.set_num_threads(nthreads)
    return {"value": Vh * FLOP_PER_SITE / best / 1e9, "unit": "GFLOP/s", "cores": nthreads,
            "value_1_thread": Vh * FLOP_PER_SITE / one / 1e9, "kind": "oracle",
            "sample": f"config {cfg_id}: one full oracle.dslash_eo (V/2 = {Vh} output sites, fp64 arithmetic on "
                      f"fp{precision} inputs), best of 3 after one warm-up, {best * 1e3:.0f} ms"}


def run_b200(args):
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the CUDA path is the only implementation; no CPU fallback)")
    import __graft_entry__ as ge
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    # LQCD_BENCH_DEVICE / LQCD_BENCH_BACKEND=gloo: functional test of the N > 1 path on a box with one GPU
    # (all ranks share the device, host-side barrier and max over ranks through gloo); numbers are then meaningless
    local = int(os.environ.get("LQCD_BENCH_DEVICE", local))
    backend = os.environ.get("LQCD_BENCH_BACKEND", "nccl")
    reduce_device = "cuda" if backend == "nccl" else "cpu"
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist_
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        if backend == "nccl":
            dist_.init_process_group("nccl", device_id=dev)
        else:
            dist_.init_process_group(backend)
        dist = dist_
    if rank == 0:
        ge.build()
    if dist is not None:
        dist.barrier()
    import paper_1112_5280_b200 as L
    L._lib()
    peak, peak_src = measured_peaks()

    w = Workload(args.config, args.precision, args.recon, dev, args.block)
    sampler = ClockSampler(local) if rank == 0 else None
    t0 = time.time()
    main = kernel_leg(torch, dist, w, args.steps, args.warmup, world, reduce_device)
    # the same region four more times, so the line also shows the spread (value = first region)
    repeats = [main["ms_per_step"]] + [kernel_leg(torch, dist, w, args.steps, 0, world, reduce_device)["ms_per_step"] for _ in range(4)]
    # keep the same launches running until nvidia-smi has seen >= 1.5 s of them (clocks under load)
    while time.time() - t0 < 1.5:
        for _ in range(20):
            w.step()
        torch.cuda.synchronize()
    t1 = time.time()
    clocks = sampler.stop(t0, t1) if sampler else None
    if clocks is not None:
        clocks["window"] = "warm-up + the five timed regions + untimed continuation of the same launches to >= 1.5 s"

    line = {
        "metric": METRIC, "value": main["gflops"], "unit": "GFLOP/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": main["ms_per_step"], "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32 (f16 storage)" if args.precision == 16 else f"f{args.precision}", "data": "synthetic",
        "config": {
            "workload": f"config {args.config}: {'x'.join(map(str, w.dims))} even-odd dslash, recon-{args.recon}, "
                        f"fp{args.precision}, random SU(3) links seed 1, Gaussian spinors seed 2.., bc (+,+,+,-)",
            "step": f"{w.nbuf} lqcd_dslash_eo launches (out_parity 0,1,0,1) over {w.nbuf} distinct in/out half spinors",
            "sites_per_step": w.sites_per_step(),
            "l2": "inputs larger than L2: links %.0f MB streamed per launch (one parity's half of the packed field) + "
                  "%.0f MB of rotating spinor buffers; no flush"
                  % (w.ctx.gauge_bytes() / 2e6, 2 * w.nbuf * w.ctx.spinor_bytes(True) / 1e6),
            "parallelism": "replicas only (no sharding, no collective)" if world > 1 else "single GPU",
        },
        "gpu_launches": main["launches"],
        "achieved_gbs": main["gbs"],
        # community "no-reuse" convention (8 neighbour spinors + output + 8 links per site: counts L2 hits; the
        # paper's 105 GB/s on an AMD 5870, is by inference quoted this way with 18-real links)
        "effective_gbs_no_reuse": main["gbs"] * (8 * 24 + 24 + 8 * args.recon) / REALS_PER_SITE[args.recon],
        "us_per_launch": main["us_per_launch"],
        "ms_per_step_5_regions": {"all": repeats, "median": sorted(repeats)[2], "min": min(repeats)},
        "clocks": clocks,
        "roofline": {
            "bound": "hbm", "achieved": main["gbs"], "peak": peak, "unit": "GB/s", "frac": main["gbs"] / peak,
            "traffic": ncu_traffic(args.precision, args.recon), "peak_source": peak_src,
            "kernel": f"dslash_kernel<fp{args.precision}, recon {args.recon}>",
            "model": f"compulsory bytes, each operand once: {w.bytes_per_launch() // w.Vh} B per site x V/2 = {w.bytes_per_launch()} B per launch",
            "frac_of_nominal_8TBs": main["gbs"] / NOMINAL_HBM_GBS,
        },
    }

    legs = set() if args.no_extras else set(args.legs.split(","))
    want = lambda name: "all" in legs or name in legs
    if rank == 0:
        if want("matrix"):
            line["matrix"] = matrix_leg(torch, w)
        if want("cg"):
            line["cg"] = cg_leg(torch, w)
        if want("e2e"):
            line["e2e"] = e2e_leg(torch, w, max(1, min(args.steps, 10)), 1)
    if want("other"):
        other = 32 if args.precision == 64 else 64
        w2 = Workload(args.config, other, args.recon, dev, args.block, keep_host=False)
        r2 = kernel_leg(torch, dist, w2, max(1, args.steps // 2), args.warmup, world, reduce_device)
        line[f"fp{other}"] = {"gflops": r2["gflops"], "achieved_gbs": r2["gbs"], "frac": r2["gbs"] / peak,
                              "frac_of_nominal_8TBs": r2["gbs"] / NOMINAL_HBM_GBS, "us_per_launch": r2["us_per_launch"],
                              "traffic": ncu_traffic(other, args.recon)}
        if want("fp16") and args.recon == 12:
            w16 = Workload(args.config, 16, 12, dev, args.block, keep_host=False)
            r16 = kernel_leg(torch, dist, w16, max(1, args.steps // 2), args.warmup, world, reduce_device)
            line["fp16_storage"] = {"gflops": r16["gflops"], "achieved_gbs": r16["gbs"], "frac": r16["gbs"] / peak,
                                    "us_per_launch": r16["us_per_launch"],
                                    "model": "296 B per site: 2 x (24 halfs + fp32 norm) + 8 x 12 halfs; fp32 arithmetic"}
            del w16
            w32h = Workload(args.config, 32, 12, dev, args.block, keep_host=False, link_precision=16)
            r = kernel_leg(torch, dist, w32h, max(1, args.steps // 2), args.warmup, world, reduce_device)
            nbytes = (48 * 4 + 8 * 24) * w32h.Vh
            line["fp32_half_links"] = {"gflops": r["gflops"], "us_per_launch": r["us_per_launch"],
                                       "achieved_gbs": nbytes / (r["us_per_launch"] * 1e-6) / 1e9,
                                       "model": "384 B per site: fp32 spinors in and out + 8 x 12 halfs"}
            del w32h
        if rank == 0 and want("cgmixed"):
            w64, w32 = (w2, w) if other == 64 else (w, w2)
            line["cg_fp64"] = cg_leg(torch, w64, tol=1e-10)
            line["cg_mixed"] = cg_mixed_leg(torch, w64, w32, tol=1e-10)
            if args.recon == 12:
                w32h = Workload(args.config, 32, 12, dev, args.block, keep_host=False, nbuf=1, link_precision=16)
                line["cg_mixed_half_links"] = cg_mixed_leg(torch, w64, w32h, tol=1e-10)
                del w32h
        del w2
    del w
    torch.cuda.empty_cache()
    if want("cpu") or args.chain:
        if rank == 0:
            if args.chain:  # config 5; opt-in: generating its 3 GB A11 link field takes minutes of host time
                import numpy as np
                import lattice_inputs as li
                U5 = li.links_for_config(5, dtype=np.complex64)
                line["chain"] = [chain_leg(torch, 5, 32, rc, dev, U=U5) for rc in (12, 18)]
                del U5
            if want("cpu"):
                line["cpu_baseline"] = cpu_baseline_leg(args.config, args.precision)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line))


# ------------------------------------------------------------------------------------------------
# reference arm: the CPU oracle on the host cores (this tier has no reference implementation)
# ------------------------------------------------------------------------------------------------
def run_reference(args):
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import numpy as np
    import lattice_inputs as li
    import oracle
    oracle.build()
    c = li.CONFIGS[args.config]
    dims, bc = c["dims"], c["bc"]
    cd = np.complex64 if args.precision == 32 else np.complex128
    U = li.links_for_config(args.config, dtype=cd)
    psi = li.gaussian_spinor(dims, dtype=cd)
    X, Y, Z, T = dims
    V = X * Y * Z * T
    # a step = oracle.dslash_sites on a bounded sample of the workload's output sites (every `stride`-th
    # lexicographic site), sized from one calibration call so K + W steps end within ~2 minutes
    def sites_for(n):
        lex = np.linspace(0, V - 1, n).astype(np.int64)
        return np.stack([lex % X, (lex // X) % Y, (lex // (X * Y)) % Z, lex // (X * Y * Z)], axis=1).astype(np.int32)
    probe = sites_for(65536)
    oracle.dslash_sites(U, psi, dims, bc, probe)
    t0 = time.perf_counter()
    oracle.dslash_sites(U, psi, dims, bc, probe)
    per_site = (time.perf_counter() - t0) / len(probe)
    budget = 120.0 / max(1, args.steps + args.warmup)
    n = int(max(1024, min(V // 2, budget / per_site)))
    sites = sites_for(n)
    for _ in range(args.warmup):
        oracle.dslash_sites(U, psi, dims, bc, sites)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.dslash_sites(U, psi, dims, bc, sites)
    dt = (time.perf_counter() - t0) / args.steps
    val = n * FLOP_PER_SITE / dt / 1e9
    sample = f"{n} output sites of config {args.config} per step via oracle.dslash_sites (fp64 arithmetic on fp{args.precision} inputs)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": "GFLOP/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"config {args.config}: {'x'.join(map(str, dims))} even-odd dslash (CPU oracle, host cores)",
                   "sample": sample},
        "gpu_launches": 0,
        "cpu_baseline": {"value": val, "unit": "GFLOP/s", "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "GFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_b200(args)


if __name__ == "__main__":
    main()
