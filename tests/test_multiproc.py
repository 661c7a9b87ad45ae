"""N > 1 host logic of bench.py on CPU: world_size-2 gloo processes (the path is "replicas only",
DESIGN.md section 8: no data-path collective; the only exchange is the max-over-ranks of the step time)."""
import os
import socket
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms = bench.max_over_ranks(torch, dist, 10.0 * (rank + 1), "cpu")  # rank r "measured" 10 (r + 1) ms
        dist.barrier()
        out[rank] = (ms, bench.aggregate_gflops(world, 1000, ms))
    finally:
        dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_world2():
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0][0] == res[1][0] == 20.0  # the slowest rank's time, on every rank
    # two replicas of 1000 sites per step in 20 ms: 2 * 1000 * 1320 flop / 0.02 s
    assert abs(res[0][1] - 2 * 1000 * 1320 / 0.02 / 1e9) < 1e-12


def test_single_process_needs_no_process_group():
    import bench
    assert bench.max_over_ranks(torch, None, 3.5, "cpu") == 3.5


def test_reference_arm_runs_on_rank0_only():
    """Under torchrun the other ranks exit 0 without work and print nothing."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


def _slab_worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    from paper_1112_5280_b200.slab import TimeSlab
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        s = TimeSlab((8, 8, 8, 16), 32, 12, (1, 1, 1, -1), rank, world)   # host-only: no CUDA call is made
        sb = s.slice_bytes
        f = torch.empty((s.Tl + 2) * sb, dtype=torch.uint8)
        for tl in range(s.Tl + 2):                       # byte pattern = 16 * rank + local slice; ghosts 255
            s.slice_view(f, tl).fill_(255 if tl in (0, s.Tl + 1) else 16 * rank + tl)
        s.exchange(f, dist)
        out[rank] = (int(s.slice_view(f, 0)[0]), int(s.slice_view(f, 0)[-1]), int(s.slice_view(f, s.Tl + 1)[0]),
                     int(s.slice_view(f, s.Tl + 1)[-1]), int(s.slice_view(f, 1)[0]), s.time_indices(), s.local_parity(0))
    finally:
        dist.destroy_process_group()


def test_time_slab_ghost_exchange_world2():
    """Ring exchange of the time-slab decomposition (paper_1112_5280_b200/slab.py) over gloo on CPU tensors:
    ghost 0 receives the left neighbour's last interior slice, ghost Tl + 1 the right neighbour's first."""
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_slab_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    Tl = 8
    for r in range(2):
        other = 1 - r
        g0a, g0b, g1a, g1b, own, tidx, lp = res[r]
        assert g0a == g0b == 16 * other + Tl      # left neighbour (= the other rank on a ring of 2): its slice Tl
        assert g1a == g1b == 16 * other + 1       # right neighbour: its slice 1
        assert own == 16 * r + 1                  # interior untouched
        assert tidx == [(r * Tl - 1 + k) % 16 for k in range(Tl + 2)] and lp == 1


def test_reference_arm_prints_the_contract_line():
    """bench.py --impl reference: one JSON line with the base contract's keys plus impl / cpu_baseline / e2e."""
    import json
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0",
                        "--config", "2"], capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-500:]
    lines = [l for l in r.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "impl", "cpu_baseline", "e2e", "gpu_launches"):
        assert k in d, k
    assert d["impl"] == "reference" and d["gpu_launches"] == 0 and d["value"] > 0 and d["vs_baseline"] is None
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
