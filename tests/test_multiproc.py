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
