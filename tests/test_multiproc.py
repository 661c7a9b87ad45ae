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
    from paper_1112_5280_b200.slab import TimeSlab, SendRecvTransport
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        s = TimeSlab((8, 8, 8, 16), 32, 12, (1, 1, 1, -1), rank, world)   # host-only: no CUDA call is made
        tr = SendRecvTransport(s, dist, "cpu")
        assert tr.send_up.numel() == s.halo_bytes == 8 * 8 * 8 // 2 * 12 * 4   # projected half spinors: 12 reals per face site
        tr.send_up.fill_(10 * rank + 1)       # byte patterns: which rank, which face
        tr.send_down.fill_(10 * rank + 2)
        tr.from_up.fill_(255)
        tr.from_down.fill_(255)
        tr.exchange(s)
        out[rank] = (int(tr.from_up[0]), int(tr.from_up[-1]), int(tr.from_down[0]), int(tr.from_down[-1]), s.above(), s.below(),
                     s.time_indices(), s.t_below())
    finally:
        dist.destroy_process_group()


def _check_ring(world):
    port = _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_slab_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    Tl = 16 // world
    for r in range(world):
        fu0, fu1, fd0, fd1, above, below, tidx, tb = res[r]
        assert (above, below) == ((r + 1) % world, (r - 1) % world)
        assert fu0 == fu1 == 10 * above + 2      # from_up: the DOWNWARD face (first slice) of the rank above
        assert fd0 == fd1 == 10 * below + 1      # from_down: the UPWARD face (last slice) of the rank below
        assert tidx == list(range(r * Tl, (r + 1) * Tl)) and tb == (r * Tl - 1) % 16


def test_time_slab_face_exchange_world2():
    """Ring exchange of the projected faces (paper_1112_5280_b200/slab.py, SendRecvTransport) over gloo on CPU tensors.  On
    a ring of two both neighbours are the same rank, so the pairing of the two faces is what this pins."""
    _check_ring(2)


def test_time_slab_face_exchange_world4():
    _check_ring(4)


def _transport_worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    from paper_1112_5280_b200.slab import TimeSlab, SendRecvTransport, make_transport
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        s = TimeSlab((8, 8, 8, 16), 32, 12, (1, 1, 1, -1), rank, world)

        class FakePeer:                       # stands in for PeerMemoryTransport: comes up on rank 0 only / everywhere
            def __init__(self, slab, dist_, device, fail_on=()):
                if slab.rank in fail_on:
                    raise RuntimeError("no peer mapping on this rank")

        res = {}
        t, name = make_transport(s, dist, "cpu", "auto")
        res["auto"] = type(t).__name__
        t, name = make_transport(s, dist, "cpu", "peer_or_sendrecv", peer_factory=lambda *a: FakePeer(*a, fail_on=(1,)))
        res["fallback"] = (type(t).__name__, "unavailable" in name)
        t, name = make_transport(s, dist, "cpu", "peer_or_sendrecv", peer_factory=lambda *a: FakePeer(*a))
        res["all_ok"] = type(t).__name__
        try:
            make_transport(s, dist, "cpu", "peer", peer_factory=lambda *a: FakePeer(*a, fail_on=(1,)))
            res["peer"] = "returned"
        except RuntimeError as e:
            res["peer"] = "raised: " + str(e)
        # the transport agreed on works: one ring exchange after the fallback
        tr = make_transport(s, dist, "cpu", "peer_or_sendrecv", peer_factory=lambda *a: FakePeer(*a, fail_on=(0,)))[0]
        tr.send_up.fill_(10 * rank + 1)
        tr.send_down.fill_(10 * rank + 2)
        tr.exchange(s)
        res["exchange"] = (int(tr.from_up[0]), int(tr.from_down[0]))
        out[rank] = res
    finally:
        dist.destroy_process_group()


def test_transport_choice_is_agreed_on_by_every_rank_world2():
    """make_transport: if the peer-memory set-up fails on ONE rank, both ranks use send/recv ("peer_or_sendrecv") or both
    raise ("peer") -- never one rank spinning on peer flags while the other posts ncclSend.  "auto" is send/recv."""
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_transport_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    for r in range(world):
        assert res[r]["auto"] == "SendRecvTransport"
        assert res[r]["fallback"] == ("SendRecvTransport", True), res[r]
        assert res[r]["all_ok"] == "FakePeer"
        assert res[r]["peer"].startswith("raised: peer-memory transport unavailable"), res[r]
        other = 1 - r
        assert res[r]["exchange"] == (10 * other + 2, 10 * other + 1)
    assert "no peer mapping" in res[1]["peer"] and "another rank" in res[0]["peer"]


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
