#!/usr/bin/env python
"""bench.py -- Wilson dslash benchmark on B200 (BASELINE.json metric: dslash GFLOP/s at 1320 flop/site
and achieved HBM GB/s vs roofline at 32^3x64).

    python bench.py --gpus 1 --steps K --warmup W            # this repo's CUDA path (default)
    python bench.py --impl reference --steps K --warmup W    # the CPU oracle on the host cores

Workload (config.workload): BASELINE.json configs[3] = SURVEY.md sec. 8(d) config 4, the headline
bandwidth case: 32^3x64, even-odd dslash, 12-real links, random SU(3) links (seed 1), Gaussian
spinors (seed 2), antiperiodic in t.  Primary line fp32.  Further legs ride in the same JSON line (--legs).

A step = one pass of the hot path (K1..L6 of SURVEY.md sec. 8(a)) over one batch of NBUF = 4
half-lattice spinors: NBUF launches of lqcd_dslash_eo, alternating out_parity 0,1 (H_eo, H_oe),
each reading its own input buffer and writing its own output buffer.  Rotating buffers keeps the
spinor working set (NBUF x 2 x 100/201 MB) above the 126 MB L2 so no launch finds its input
resident from the previous one; the 403/805 MB link field is streamed once per launch.

Timing protocol (">= 200 launches ... repeated 5x, report median and min"; PAPER.md:87
"statistics are of O(10k) for each volume"): after W warm-up steps, FIVE timed regions, each R x K steps between two
CUDA events with a barrier + synchronize on both sides, R chosen so that a region holds >= 200 launches and lasts
>= 100 ms whatever K is.  `value` / `ms_per_step` are the MEDIAN region; the first (coolest) and the fastest region
are printed beside it.  Then the same launches run back to back for >= 1.5 s, timed with CUDA events: `sustained`.
Every region carries the SM clock and throttle reasons sampled (NVML, every ~5 ms) while IT ran.

Multi-GPU: the headline path does not shard ("replicas only"): --gpus N runs N independent replicas,
one process per GPU, no data-path collective; value = N replicas' sites / max time.  The T-slab decomposition
(next row f3) is timed by the `slab` leg when WORLD_SIZE > 1.
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
REALS_PER_SITE = {8: 112, 12: 144, 18: 192}   # compulsory eo model: 24 in + 24 out + 8 links
NBUF = 4
METRIC = "dslash GFLOP/s (1320 flop/site), 32^3x64 even-odd recon-12"
FALLBACK_HBM_GBS = 6650.0             # /opt/skills/guides/B200_PROFILING.md fallback
NOMINAL_HBM_GBS = 8000.0              # north_star's "~8 TB/s"
MIN_REGION_LAUNCHES = 200
MIN_REGION_MS = 100.0
SUSTAINED_S = 1.5
ALL_LEGS = ("fp64", "recon18", "recon8", "matrix", "cg", "cgmixed", "fp16", "config3", "chain", "e2e", "slab", "heatbath", "variants", "cpu")


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", type=int, default=4, help="lattice_inputs.CONFIGS id of the main workload")
    ap.add_argument("--precision", type=int, default=32, choices=[16, 32, 64], help="precision of the primary line (16: half storage, fp32 arithmetic)")
    ap.add_argument("--recon", type=int, default=12, choices=[8, 12, 18])
    ap.add_argument("--kernel", default="gather", choices=["gather", "pipe", "blocked", "lstage"],
                    help="lqcd_set_kernel for the primary line and the fp64 / recon legs: gather (one thread per site) or pipe (TMA pipeline)")
    ap.add_argument("--no-extras", action="store_true", help="primary line only (profiling runs)")
    ap.add_argument("--legs", default="all", help="comma list of extra legs: " + ",".join(ALL_LEGS) + " (default all)")
    return ap.parse_args()


def workload_name(cfg_id, dims, precision):
    """One string for both arms (the reference arm computes the same operator on the same inputs)."""
    return (f"config {cfg_id}: {'x'.join(map(str, dims))} even-odd Wilson dslash, fp{32 if precision == 16 else precision} inputs, "
            f"random SU(3) links seed 1, Gaussian spinors seed 2, bc (+,+,+,-)")


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, device copy)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(precision, recon):
    """dram bytes per launch of the dslash kernel as captured by `ncu --set full` (profiles/dram_traffic.csv, which
    names the capture each row comes from); (bytes, source) or (None, None).  A profiler figure, not a run-time one."""
    path = os.path.join(ROOT, "profiles", "dram_traffic.csv")
    try:
        with open(path) as f:
            for line in f:
                p = [x.strip() for x in line.split(",")]
                if len(p) >= 4 and p[0] == "config4" and p[1] == f"fp{precision}" and p[2] == f"recon{recon}":
                    return float(p[3]), (p[4] if len(p) > 4 else "profiles/dram_traffic.csv")
    except OSError:
        pass
    return None, None


class ClockSampler:
    """SM clock, power and throttle reasons sampled every ~5 ms through NVML (nvidia-smi -lms 50 if NVML is not
    importable), so that every timed region can be given the clock it actually ran at."""
    BITS = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "sw_power_cap": 0x4}

    def __init__(self, index, uuid=None):
        self.rows, self.stop_flag, self.proc, self.smax = [], False, None, None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            try:  # the CUDA device index is not the NVML index under CUDA_VISIBLE_DEVICES: go by UUID
                self.h = pynvml.nvmlDeviceGetHandleByUUID(("GPU-" + str(uuid)).encode())
            except Exception:
                self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.smax = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.thr = threading.Thread(target=self._poll_nvml, daemon=True)
            self.how = "NVML, ~5 ms period"
        except Exception:
            self.nv = None
            q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
                 "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
            try:
                self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={q}", "--format=csv,noheader,nounits",
                                              "-lms", "50"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            except OSError:
                self.proc = None
            self.thr = threading.Thread(target=self._poll_smi, daemon=True)
            self.how = "nvidia-smi -lms 50"
        self.thr.start()

    def _poll_nvml(self):
        nv = self.nv
        while not self.stop_flag:
            try:
                clk = float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                mask = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                pw = nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0
                self.rows.append((time.time(), clk, pw, {n for n, b in self.BITS.items() if mask & b}))
            except Exception:
                pass
            time.sleep(0.005)

    def _poll_smi(self):
        if self.proc is None:
            return
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.proc.stdout:
            p = [x.strip() for x in line.split(",")]
            try:
                self.smax = float(p[1])
                self.rows.append((time.time(), float(p[0]), float(p[2]),
                                  {n for n, v in zip(names, p[3:7]) if v.lower().startswith("active")}))
            except (ValueError, IndexError):
                continue

    def window(self, t0, t1):
        """Median SM clock, mean power and the throttle reasons seen in [t0, t1] (wall clock)."""
        rows = [r for r in self.rows if t0 <= r[0] <= t1]
        if not rows:  # region shorter than the sampling period: the nearest sample
            rows = sorted(self.rows, key=lambda r: abs(r[0] - 0.5 * (t0 + t1)))[:1]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": self.smax, "reasons": ["no clock samples"], "samples": 0}
        clk = sorted(r[1] for r in rows)
        reasons = set().union(*[r[3] for r in rows])
        return {"sm_mhz": clk[len(clk) // 2], "sm_max_mhz": self.smax, "power_w": sum(r[2] for r in rows) / len(rows),
                "reasons": sorted(reasons), "samples": len(rows)}

    def close(self):
        self.stop_flag = True
        if self.proc is not None:
            self.proc.terminate()
        self.thr.join(timeout=2)


# ------------------------------------------------------------------------------------------------
# this repo's arm
# ------------------------------------------------------------------------------------------------
class Workload:
    """Seeded inputs of one config on the device in native layout, plus pinned host copies."""

    def __init__(self, cfg_id, precision, recon, dev, nbuf=NBUF, keep_host=True, in_parity=None, U=None, link_precision=0, kernel="gather"):
        import numpy as np
        import torch
        import lattice_inputs as li
        import paper_1112_5280_b200 as L
        self.L, self.torch = L, torch
        c = li.CONFIGS[cfg_id]
        self.cfg_id, self.dims, self.bc, self.kappa = cfg_id, c["dims"], c["bc"], c["kappa"]
        self.precision, self.recon, self.dev, self.nbuf, self.link_precision = precision, recon, dev, nbuf, link_precision
        cd = np.complex128 if precision == 64 else np.complex64  # precision 16 exchanges complex64
        self.ctx = L.Context(self.dims, precision, recon, self.bc, link_precision)
        if kernel == "pipe" and precision != 16 and not link_precision:
            self.ctx.set_kernel(L.KERNEL_PIPE)
        if kernel == "blocked":
            self.ctx.set_kernel(L.KERNEL_BLOCKED)
        if kernel == "lstage" and precision != 16 and not link_precision:
            self.ctx.set_kernel(L.KERNEL_LSTAGE)
        self.kernel = kernel
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

    launches_per_step = property(lambda self: self.nbuf)

    def sites_per_step(self):
        return self.nbuf * self.Vh

    def bytes_per_site(self):
        """Algorithmic (compulsory) bytes per output site: input spinor once, output once, 8 links once."""
        if self.precision == 16:
            return 2 * 52 + 8 * 24          # 24 halfs + one fp32 norm per spinor site, 12 halfs per link
        if self.link_precision == 16:
            return 48 * 4 + 8 * 24          # fp32 spinors, 12 halfs per link
        return REALS_PER_SITE[self.recon] * (self.precision // 8)

    def bytes_per_launch(self):
        return self.bytes_per_site() * self.Vh


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


class Timer:
    """CUDA-event timing of regions of R x K steps on the current stream, barrier + synchronize on both sides,
    max over ranks; every region is attributed the clocks sampled while it ran."""

    def __init__(self, torch, dist, reduce_device, sampler):
        self.torch, self.dist, self.reduce_device, self.sampler = torch, dist, reduce_device, sampler

    def _fence(self):
        self.torch.cuda.synchronize()
        if self.dist is not None:
            self.dist.barrier()
        self.torch.cuda.synchronize()

    def region(self, fn, nsteps):
        torch = self.torch
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        self._fence()
        t0 = time.time()
        e0.record()
        for _ in range(nsteps):
            fn()
        e1.record()
        self._fence()
        t1 = time.time()
        ms = max_over_ranks(torch, self.dist, e0.elapsed_time(e1), self.reduce_device)
        clocks = self.sampler.window(t0, t1) if self.sampler else None
        return ms, clocks

    def reps_for(self, fn, steps, launches_per_step):
        """R such that R x K steps hold >= MIN_REGION_LAUNCHES launches and last >= MIN_REGION_MS (from one probe)."""
        ms, _ = self.region(fn, steps)
        r_time = MIN_REGION_MS / max(ms, 1e-3)
        r_launch = MIN_REGION_LAUNCHES / (steps * launches_per_step)
        r = max(1.0, r_time, r_launch)
        if self.dist is not None:  # every rank must run the same number of steps
            r = max_over_ranks(self.torch, self.dist, r, self.reduce_device)
        return int(-(-r // 1))

    def measure(self, fn, steps, warmup, launches_per_step, nregions=5, sustained_s=0.0):
        for _ in range(warmup):
            fn()
        reps = self.reps_for(fn, steps, launches_per_step)
        regions = []
        for _ in range(nregions):
            ms, clocks = self.region(fn, reps * steps)
            regions.append({"ms_per_step": ms / (reps * steps), "clocks": clocks})
        order = sorted(range(nregions), key=lambda i: regions[i]["ms_per_step"])
        res = {"reps": reps, "regions": regions, "median": regions[order[nregions // 2]], "first": regions[0],
               "min": regions[order[0]]}
        if sustained_s > 0:
            n = max(1, int(sustained_s * 1e3 / (res["median"]["ms_per_step"] * steps) + 1))
            if self.dist is not None:
                n = int(max_over_ranks(self.torch, self.dist, n, self.reduce_device))
            ms, clocks = self.region(fn, n * steps)
            res["sustained"] = {"ms_per_step": ms / (n * steps), "seconds": ms * 1e-3, "steps": n * steps, "clocks": clocks}
        return res


def kernel_numbers(w, ms_step, world, peak):
    t_launch = ms_step / w.launches_per_step * 1e-3
    gbs = w.bytes_per_launch() / t_launch / 1e9
    return {"ms_per_step": ms_step, "us_per_launch": t_launch * 1e6, "gflops": aggregate_gflops(world, w.sites_per_step(), ms_step),
            "gbs": gbs, "frac": gbs / peak, "frac_of_nominal_8TBs": gbs / NOMINAL_HBM_GBS}


def kernel_leg(timer, w, steps, warmup, world, peak, nregions=3, sustained_s=0.0):
    """Device-resident timing of one Workload: median / first / min region and (optionally) the sustained run,
    each with GB/s under the compulsory-bytes model and the clock it ran at."""
    L = w.L
    n0 = L.launch_count()
    m = timer.measure(w.step, steps, warmup, w.launches_per_step, nregions, sustained_s)
    out = kernel_numbers(w, m["median"]["ms_per_step"], world, peak)
    out["clocks"] = m["median"]["clocks"]
    for k in ("first", "min") + (("sustained",) if "sustained" in m else ()):
        out[k] = kernel_numbers(w, m[k]["ms_per_step"], world, peak)
        out[k]["clocks"] = m[k]["clocks"]
        if k == "sustained":
            out[k]["seconds"], out[k]["steps"] = m[k]["seconds"], m[k]["steps"]
    out["regions_ms_per_step"] = [r["ms_per_step"] for r in m["regions"]]
    out["regions_sm_mhz"] = [r["clocks"]["sm_mhz"] if r["clocks"] else None for r in m["regions"]]
    out["region_steps"] = m["reps"] * steps
    out["launches_total"] = L.launch_count() - n0
    out["bytes_per_site"] = w.bytes_per_site()
    return out


def brief(r, keys=("us_per_launch", "gflops", "gbs", "frac", "frac_of_nominal_8TBs")):
    """Compact form of a kernel_leg result for the secondary legs."""
    d = {k: r[k] for k in keys}
    d["sm_mhz"] = r["clocks"]["sm_mhz"] if r.get("clocks") else None
    d["first_us"], d["min_us"] = r["first"]["us_per_launch"], r["min"]["us_per_launch"]
    d["bytes_per_site"] = r["bytes_per_site"]
    return d


def pcie_peak(torch, dev, nbytes=100 << 20, reps=5):
    """Measured pinned-copy bandwidth of this box: H2D alone, D2H alone, and both directions at once on two streams
    (GB/s per direction).  The e2e leg moves the same bytes up and down, so the last figure is its bound."""
    h_up = torch.empty(nbytes, dtype=torch.uint8).pin_memory()
    h_dn = torch.empty(nbytes, dtype=torch.uint8).pin_memory()
    d_up = torch.empty(nbytes, dtype=torch.uint8, device=dev)
    d_dn = torch.empty(nbytes, dtype=torch.uint8, device=dev)
    s1, s2 = torch.cuda.Stream(dev), torch.cuda.Stream(dev)
    def timed(up, down):
        best = None
        for _ in range(reps + 1):
            torch.cuda.synchronize(dev)
            t0 = time.perf_counter()
            if up:
                with torch.cuda.stream(s1):
                    d_up.copy_(h_up, non_blocking=True)
            if down:
                with torch.cuda.stream(s2):
                    h_dn.copy_(d_dn, non_blocking=True)
            torch.cuda.synchronize(dev)
            dt = time.perf_counter() - t0
            best = dt if best is None else min(best, dt)
        return nbytes / best / 1e9
    return {"h2d_gbs": timed(True, False), "d2h_gbs": timed(False, True), "bidirectional_gbs_per_direction": timed(True, True),
            "how": f"{nbytes >> 20} MiB pinned copies, best of {reps}, wall clock around a synchronize"}


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
    for _ in range(3):  # the host link is shared with other tenants of the box: three regions, the median counts
        t0 = time.perf_counter()
        e0.record()
        for _ in range(steps):
            ctx.dslash_eo_host_batch(out_h, None, w.in_host, par, ws)  # one step = the batch of NBUF half spinors
        e1.record()
        torch.cuda.synchronize()
        wall = (time.perf_counter() - t0) * 1e3
        regions.append(max(e0.elapsed_time(e1), wall) / steps)
    ms = sorted(regions)[1]
    hb = w.in_host[0].numel() * w.in_host[0].element_size()
    pcie = pcie_peak(torch, w.dev)
    per_dir = hb * w.nbuf / (ms * 1e-3) / 1e9
    return {
        "value": world * w.sites_per_step() * FLOP_PER_SITE / (ms * 1e-3) / 1e9,
        "unit": "GFLOP/s",
        "h2d_bytes_per_step": hb * w.nbuf,
        "d2h_bytes_per_step": hb * w.nbuf,
        "ms_per_step": ms,
        "ms_per_step_regions": regions,
        "steps": steps,
        "bound": "pcie",
        "gbs_per_direction": per_dir,
        "pcie_peak": pcie,
        "frac_of_pcie": per_dir / pcie["bidirectional_gbs_per_direction"],
        "gauge": "resident (uploaded and packed once before the timed region)",
        "ms_one_application_with_gauge_upload": min(tg),
        "gauge_h2d_bytes": w.U_host.numel() * w.U_host.element_size(),
    }


def chain_leg(torch, cfg_id, precision, recon, dev, napply=100, reps=3, U=None, kernel="gather"):
    """Config 5 (reading A16): x_{k+1} = M x_k, M = 1 - kappa^2 H_eo H_oe, `napply` times back to back,
    ping-pong buffers, timed as one block; `reps` + 1 blocks, median and min."""
    w = Workload(cfg_id, precision, recon, dev, nbuf=1, keep_host=False, in_parity=0, U=U, kernel=kernel)  # even half spinor
    x, y = w.inp[0], w.out[0]
    ws = torch.empty_like(x)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    times = []
    for _ in range(reps + 1):
        a, b = x.clone(), y
        torch.cuda.synchronize()
        e0.record()
        for _k in range(napply):
            w.ctx.apply_M(b, w.gauge, a, w.kappa, 1, ws)
            a, b = b, a
        e1.record()
        torch.cuda.synchronize()
        times.append(e0.elapsed_time(e1))
    med, best = sorted(times)[len(times) // 2], min(times)
    reals = REALS_PER_SITE[recon] * 2 + 24  # pass 1 + pass 2 with the xpay read
    nbytes = reals * (precision // 8) * w.Vh
    finite = bool(torch.isfinite(a.view(torch.float32 if precision == 32 else torch.float64)).all().item())
    return {
        "workload": f"config {cfg_id}: {'x'.join(map(str, w.dims))} fp{precision} recon-{recon} apply_M(eo=1) x{napply} chained",
        "ms_per_chain": med, "ms_per_chain_min": best, "ms_per_application": med / napply,
        "gflops": 2 * FLOP_PER_SITE * w.Vh * napply / (med * 1e-3) / 1e9,
        "gbs": nbytes * napply / (med * 1e-3) / 1e9,
        "bytes_per_application": nbytes, "finite": finite,
    }


def config3_leg(torch, timer, dev, peak, steps, warmup):
    """Config 3 (16^3x32, lqcd_dslash_full, A11 links): first timings, roofline fraction reported, not graded.  With
    every link stored twice the working set (in + out spinors + packed links) is 75 / 101 MB in fp32 (12- / 18-real: inside
    the 126 MB L2, so those figures are L2 bandwidth) and 151 / 201 MB in fp64 (not L2-resident).  Bytes: the full-lattice compulsory model of SURVEY.md sec. 8(d), 96 (12-real) /
    120 (18-real) reals per site -- each link counted once although lqcd_dslash_full reads 8 gathered links per
    site, so `gbs` here is model bytes / time, and `gbs_as_read` counts what the kernel reads."""
    import numpy as np
    import lattice_inputs as li
    import paper_1112_5280_b200 as L
    c = li.CONFIGS[3]
    out = {}
    for precision in (32, 64):
        cd = np.complex64 if precision == 32 else np.complex128
        U = li.links_for_config(3, dtype=cd)
        for recon in (12, 18):
            ctx = L.Context(c["dims"], precision, recon, c["bc"])
            gauge = torch.empty(ctx.gauge_bytes(), dtype=torch.uint8, device=dev)
            ctx.pack_gauge(gauge, torch.from_numpy(U).to(dev))
            psi = torch.from_numpy(li.gaussian_spinor(c["dims"], dtype=cd)).to(dev)
            a, b = (torch.empty(ctx.spinor_bytes(False), dtype=torch.uint8, device=dev) for _ in range(2))
            ctx.pack_spinor(a, psi, -1)
            torch.cuda.synchronize()
            m = timer.measure(lambda: ctx.dslash_full(b, gauge, a), steps, warmup, 1, nregions=3)
            us = m["median"]["ms_per_step"] * 1e3
            V = 2 * ctx.Vh
            model = (48 + 4 * recon) * (precision // 8) * V
            read = (48 + 8 * recon) * (precision // 8) * V
            out[f"fp{precision}_recon{recon}"] = {
                "us_per_application": us, "gflops": V * FLOP_PER_SITE / (us * 1e-6) / 1e9, "gbs": model / (us * 1e-6) / 1e9,
                "gbs_as_read": read / (us * 1e-6) / 1e9, "model_reals_per_site": 48 + 4 * recon,
                "working_set_mb": (2 * ctx.spinor_bytes(False) + ctx.gauge_bytes()) / 1e6,
                "sm_mhz": m["median"]["clocks"]["sm_mhz"] if m["median"]["clocks"] else None}
    out["note"] = "not graded; fp32 working sets fit the 126 MB L2, fp64 ones do not (links are stored twice): see working_set_mb"
    return out


def matrix_leg(torch, w, napply=50, reps=3):
    """Fermion-matrix applications on the primary workload's fields: lqcd_apply_M(eo=1) and the twisted-mass
    lqcd_apply_M_tm(eo=1) (next row f1), napply back-to-back applications alternating between two input
    buffers, median of `reps` + 1.  2 launches, 2 x 1320 flop and (2 x (24 + 24 + 8 recon) + 24) reals per even site."""
    x, y, ws = w.inp[1], w.out[1], w.out[0]   # inp[1] holds an even half spinor (out_parity 1)
    x2, y2 = w.inp[3 % w.nbuf], w.out[3 % w.nbuf]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    res = {}
    for name, fn in (("apply_M", lambda o, i: w.ctx.apply_M(o, w.gauge, i, w.kappa, 1, ws)),
                     ("apply_M_tm", lambda o, i: w.ctx.apply_M_tm(o, w.gauge, i, w.kappa, 0.05, 1, ws))):
        times = []
        for _ in range(reps + 1):
            torch.cuda.synchronize()
            e0.record()
            for k in range(napply):
                fn(y, x) if k & 1 else fn(y2, x2)
            e1.record()
            torch.cuda.synchronize()
            times.append(e0.elapsed_time(e1) / napply)
        ms = sorted(times)[len(times) // 2]
        nbytes = 2 * w.bytes_per_launch() + w.bytes_per_launch() * 24 // (2 * 24 + 8 * w.recon)  # two passes + the xpay read
        if w.precision == 16:
            nbytes = 2 * w.bytes_per_launch() + 52 * w.Vh
        res[name] = {"us_per_application": ms * 1e3, "gflops": 2 * FLOP_PER_SITE * w.Vh / (ms * 1e-3) / 1e9,
                     "gbs": nbytes / (ms * 1e-3) / 1e9}
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


def heatbath_leg(torch, dev, cfg_id=4, beta=6.0, ntries=4, sweeps=3):
    """Next row f4, last clause: pure-gauge SU(3) heatbath sweeps (8 sublattice launches each) on the config's lattice,
    fp64, link field in the update layout, uniforms drawn on the device beforehand (they are inputs of the method).  Bytes per link
    update (model): the 18 staple links and the link itself are shared with other updates -- each launch touches all
    links of the three other directions (3 V), the mu links of both parities (V) and writes V/2: 9 links of 144 B per
    update -- plus the uniforms of one attempt and the direction per subgroup (3 x 6 x 8 B)."""
    import numpy as np
    import lattice_inputs as li
    import paper_1112_5280_b200 as L
    c = li.CONFIGS[cfg_id]
    ctx = L.Context(c["dims"], 64, 18, (1, 1, 1, 1))
    Uc = torch.from_numpy(li.links_for_config(cfg_id, dtype=np.complex128)).to(dev)
    U = torch.empty(ctx.update_links_bytes(), dtype=torch.uint8, device=dev)   # the update layout (structure of arrays, checkerboarded)
    ctx.pack_update_links(U, Uc)
    torch.cuda.synchronize()
    del Uc
    ws = torch.empty(ctx.plaquette_workspace_bytes(), dtype=torch.uint8, device=dev)
    p0 = ctx.plaquette(U, ws)
    n = ctx.heatbath_uniforms(ntries)
    # one independent array of uniforms per sublattice launch of a sweep (8 x 453 MB at 32^3 x 64, ntries 4), redrawn
    # between sweeps outside the timed region: no number is used twice, so plaquette_after is a heatbath's, not an artefact
    u = [1.0 - torch.rand(n, dtype=torch.float64, device=dev) for _ in range(8)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    times = []
    for s in range(sweeps + 1):
        torch.cuda.synchronize()
        e0.record()
        for mu in range(4):
            for parity in (0, 1):
                ctx.heatbath_sublattice(U, beta, mu, parity, u[2 * mu + parity], ntries)
        e1.record()
        torch.cuda.synchronize()
        times.append(e0.elapsed_time(e1))
        for t in u:
            t.copy_(1.0 - torch.rand(n, dtype=torch.float64, device=dev))
    ms = sorted(times[1:])[len(times[1:]) // 2]
    links = 4 * 2 * ctx.Vh
    nbytes = links * (9 * 144 + 3 * 6 * 8)
    return {"workload": f"config {cfg_id} lattice {'x'.join(map(str, c['dims']))}, fp64, beta {beta}, {ntries} attempts per subgroup",
            "ms_per_sweep": ms, "us_per_sublattice_launch": ms * 1e3 / 8, "link_updates_per_s": links / (ms * 1e-3),
            "gbs_model": nbytes / (ms * 1e-3) / 1e9, "bytes_per_link_update_model": 9 * 144 + 144,
            "plaquette_before": p0, "plaquette_after": ctx.plaquette(U, ws), "sweeps_timed": sweeps}


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
    sampler = ClockSampler(local, getattr(torch.cuda.get_device_properties(dev), "uuid", None))
    timer = Timer(torch, dist, reduce_device, sampler)
    solo = Timer(torch, None, reduce_device, sampler)   # rank-0-only legs

    w = Workload(args.config, args.precision, args.recon, dev, kernel=args.kernel)
    main = kernel_leg(timer, w, args.steps, args.warmup, world, peak, nregions=5, sustained_s=SUSTAINED_S)
    traffic, traffic_src = ncu_traffic(args.precision, args.recon)
    kname = f"{'dslash_pipe_kernel' if args.kernel == 'pipe' else 'dslash_kernel'}<fp{args.precision}, recon {args.recon}, EPI_STORE>"

    def roofline(r):
        return {"bound": "hbm", "achieved": r["gbs"], "peak": peak, "unit": "GB/s", "frac": r["gbs"] / peak,
                "us_per_launch": r["us_per_launch"], "sm_mhz": r["clocks"]["sm_mhz"] if r["clocks"] else None,
                "reasons": r["clocks"]["reasons"] if r["clocks"] else None}

    line = {
        "metric": METRIC, "value": main["gflops"], "unit": "GFLOP/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": main["ms_per_step"], "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32 (f16 storage)" if args.precision == 16 else f"f{args.precision}", "data": "synthetic",
        "config": {
            "workload": workload_name(args.config, w.dims, args.precision),
            "links": f"{args.recon}-real storage, third row rebuilt in registers" if args.recon != 18 else "18-real storage",
            "step": f"{w.nbuf} lqcd_dslash_eo launches (out_parity 0,1,0,1) over {w.nbuf} distinct in/out half spinors",
            "sites_per_step": w.sites_per_step(),
            "timed_region": f"value = median of 5 regions of {main['region_steps']} steps each (R x K, R chosen for >= "
                            f"{MIN_REGION_LAUNCHES} launches and >= {MIN_REGION_MS:.0f} ms per region); `sustained` = one region of >= {SUSTAINED_S} s",
            "l2": "inputs larger than L2: links %.0f MB streamed per launch (one parity's half of the packed field) + "
                  "%.0f MB of rotating spinor buffers; no flush"
                  % (w.ctx.gauge_bytes() / 2e6, 2 * w.nbuf * w.ctx.spinor_bytes(True) / 1e6),
            "parallelism": "replicas only (no sharding, no collective)" if world > 1 else "single GPU",
        },
        "gpu_launches": main["launches_total"],
        "achieved_gbs": main["gbs"],
        # community "no-reuse" convention (8 neighbour spinors + output + 8 links per site: counts L2 hits; the
        # paper's 105 GB/s on an AMD 5870, is by inference quoted this way with 18-real links)
        "effective_gbs_no_reuse": main["gbs"] * (8 * 24 + 24 + 8 * args.recon) / REALS_PER_SITE[args.recon],
        "us_per_launch": main["us_per_launch"],
        "regions": {"ms_per_step": main["regions_ms_per_step"], "sm_mhz": main["regions_sm_mhz"],
                    "median": main["ms_per_step"], "first": main["first"]["ms_per_step"], "min": main["min"]["ms_per_step"]},
        "clocks": dict(main["clocks"] or {}, window="the median timed region (sampled while it ran: " + sampler.how + ")"),
        "roofline": dict(roofline(main), **{
            "traffic": traffic, "traffic_source": traffic_src,
            "dram_gbs_at_ncu_traffic": traffic / (main["us_per_launch"] * 1e-6) / 1e9 if traffic else None,
            "achieved_is": "effective bandwidth = algorithmic (compulsory) bytes / measured launch time, against the measured device-copy peak",
            "peak_source": peak_src, "kernel": kname,
            "model": f"compulsory bytes, each operand once: {w.bytes_per_site()} B per site x V/2 = {w.bytes_per_launch()} B per launch",
            "frac_of_nominal_8TBs": main["gbs"] / NOMINAL_HBM_GBS, "region": "median of 5",
            "sustained_frac": main["sustained"]["gbs"] / peak,
            "sustained_frac_of_nominal_8TBs": main["sustained"]["gbs"] / NOMINAL_HBM_GBS}),
        "roofline_first_region": roofline(main["first"]),
        # flags the loaded liblqcd.so was compiled with (a library left over from a -D sweep would show here)
        "build_flags": _build_flags(),
        "sustained": dict(roofline(main["sustained"]), seconds=main["sustained"]["seconds"], gflops=main["sustained"]["gflops"],
                          steps=main["sustained"]["steps"]),
    }

    legs = set() if args.no_extras else set(args.legs.split(","))
    want = lambda name: "all" in legs or name in legs
    half = max(1, args.steps // 2)
    if rank == 0:
        if want("matrix"):
            line["matrix"] = matrix_leg(torch, w)
        if want("cg"):
            line["cg"] = cg_leg(torch, w)
        if want("e2e"):
            line["e2e"] = e2e_leg(torch, w, max(1, min(args.steps, 10)), 1)
    other = 32 if args.precision == 64 else 64
    w2 = None
    if want("fp64") or want("cgmixed"):
        w2 = Workload(args.config, other, args.recon, dev, keep_host=False, kernel=args.kernel)
    if want("fp64"):
        r2 = kernel_leg(timer, w2, half, args.warmup, world, peak, nregions=5, sustained_s=SUSTAINED_S)
        t2, t2s = ncu_traffic(other, args.recon)
        line[f"fp{other}"] = dict(brief(r2), traffic=t2, traffic_source=t2s, regions_ms_per_step=r2["regions_ms_per_step"],
                                  regions_sm_mhz=r2["regions_sm_mhz"],
                                  sustained=dict(roofline(r2["sustained"]), seconds=r2["sustained"]["seconds"], gflops=r2["sustained"]["gflops"]))
        # north_star's target names both precisions: the other one's headline numbers ride inside the roofline record
        line["roofline"][f"fp{other}"] = {
            "us_per_launch": r2["us_per_launch"], "achieved": r2["gbs"], "frac": r2["frac"],
            "frac_of_nominal_8TBs": r2["frac_of_nominal_8TBs"], "sustained_frac": r2["sustained"]["gbs"] / peak,
            "sustained_frac_of_nominal_8TBs": r2["sustained"]["gbs"] / NOMINAL_HBM_GBS,
            "sm_mhz": r2["clocks"]["sm_mhz"] if r2["clocks"] else None, "traffic": t2,
            "bytes_per_launch": w2.bytes_per_launch(), "region": "median of 5"}
    if rank == 0 and want("cgmixed") and args.precision != 16:
        w64, w32 = (w2, w) if other == 64 else (w, w2)
        line["cg_fp64"] = cg_leg(torch, w64, tol=1e-10)
        line["cg_mixed"] = cg_mixed_leg(torch, w64, w32, tol=1e-10)
        if args.recon == 12:
            w32h = Workload(args.config, 32, 12, dev, keep_host=False, nbuf=1, link_precision=16)
            line["cg_mixed_half_links"] = cg_mixed_leg(torch, w64, w32h, tol=1e-10)
            del w32h
            # 16-bit solver (next row f4): inner CG on 16-bit operator fields, fp32 iterate and residual
            w16 = Workload(args.config, 16, 12, dev, keep_host=False, nbuf=1)
            line["cg_mixed_16bit"] = cg_mixed_leg(torch, w64, w16, tol=1e-10, inner_tol=1e-3)
            del w16
    del w2
    torch.cuda.empty_cache()
    if want("variants") and args.kernel == "gather" and args.precision != 16:
        # the data-movement variants of the same arithmetic (lqcd_set_kernel), timed like the fp64 leg
        line["kernel_variants"] = {}
        for kern in ("pipe", "blocked", "lstage"):
            for prec in (32, 64):
                wv = Workload(args.config, prec, args.recon, dev, keep_host=False, kernel=kern)
                rv = kernel_leg(timer, wv, half, args.warmup, world, peak)
                line["kernel_variants"][f"{kern}_fp{prec}"] = {"us_per_launch": rv["us_per_launch"], "first_us": rv["first"]["us_per_launch"],
                                                                "frac": rv["frac"], "sm_mhz": rv["clocks"]["sm_mhz"] if rv["clocks"] else None}
                del wv
                torch.cuda.empty_cache()
        line["kernel_variants"]["note"] = ("same arithmetic, bit-identical results: pipe = persistent TMA pipeline (links + neighbour tiles staged), "
                                           "blocked = gather kernel on 4-D boxes of warp tiles, lstage = gather kernel with TMA-staged links; "
                                           "the primary line is the gather kernel")
    if want("recon18"):
        for prec in (32, 64):
            wv = Workload(args.config, prec, 18, dev, keep_host=False, kernel=args.kernel)
            line[f"recon18_fp{prec}"] = brief(kernel_leg(timer, wv, half, args.warmup, world, peak))
            del wv
            torch.cuda.empty_cache()
    if want("recon8") and getattr(L, "HAS_RECON8", False):
        for prec in (32, 64):
            wv = Workload(args.config, prec, 8, dev, keep_host=False, kernel=args.kernel)
            line[f"recon8_fp{prec}"] = brief(kernel_leg(timer, wv, half, args.warmup, world, peak))
            del wv
            torch.cuda.empty_cache()
    if want("fp16"):
        w16 = Workload(args.config, 16, 12, dev, keep_host=False)
        line["fp16_storage"] = dict(brief(kernel_leg(timer, w16, half, args.warmup, world, peak)),
                                    model="296 B per site: 2 x (24 halfs + fp32 norm) + 8 x 12 halfs; fp32 arithmetic")
        del w16
        w32h = Workload(args.config, 32, 12, dev, keep_host=False, link_precision=16)
        line["fp32_half_links"] = dict(brief(kernel_leg(timer, w32h, half, args.warmup, world, peak)),
                                       model="384 B per site: fp32 spinors in and out + 8 x 12 halfs")
        del w32h
        torch.cuda.empty_cache()
    del w
    torch.cuda.empty_cache()
    if want("slab") and args.precision != 16:
        # next row f3: the same operator decomposed into `world` time slabs (one rank: the ring closes on itself)
        from paper_1112_5280_b200 import slab_bench
        r = slab_bench.run(torch, dist, timer, dev, args.config, args.precision, args.recon, half, args.warmup, peak, world, rank,
                           FLOP_PER_SITE)
        if rank == 0:
            line["slab"] = r
    if rank == 0:
        if want("config3"):
            line["config3"] = config3_leg(torch, solo, dev, peak, 50, 10)
        if want("chain"):  # config 5: generating its 3 GB A11 link field takes some tens of seconds of host time
            import numpy as np
            import lattice_inputs as li
            t0 = time.perf_counter()
            U5 = li.links_for_config(5, dtype=np.complex64)
            gen_s = time.perf_counter() - t0
            line["chain"] = [chain_leg(torch, 5, 32, rc, dev, U=U5, kernel=args.kernel) for rc in (12, 18)]
            line["chain_link_generation_s"] = gen_s
            del U5
        if want("heatbath"):
            line["heatbath"] = heatbath_leg(torch, dev, args.config)
        if want("cpu"):
            line["cpu_baseline"] = cpu_baseline_leg(args.config, 32 if args.precision == 16 else args.precision)
    sampler.close()
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(primary_keys_last(line)))


# keys of the contract line (and what explains them) go LAST in the printed object: a reader who only keeps the tail of
# a long stdout still sees the metric, the roofline record, the CPU baseline and the end-to-end number
PRIMARY_KEYS = ("build_flags", "regions", "sustained", "roofline_first_region", "achieved_gbs", "effective_gbs_no_reuse",
                "us_per_launch", "config", "clocks", "gpu_launches", "cpu_baseline", "e2e", "roofline", "data", "dtype",
                "vs_baseline", "scaling", "higher_is_better", "ms_per_step", "warmup", "steps", "n_gpus", "unit", "value", "metric")


def primary_keys_last(line):
    out = {k: v for k, v in line.items() if k not in PRIMARY_KEYS}
    out.update((k, line[k]) for k in PRIMARY_KEYS if k in line)
    return out


def _build_flags():
    from paper_1112_5280_b200 import _build
    return _build.built_flags()


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
    cd = np.complex128 if args.precision == 64 else np.complex64
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
        "config": {"workload": workload_name(args.config, dims, args.precision),
                   "implementation": "CPU oracle on the host cores", "sample": sample},
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
