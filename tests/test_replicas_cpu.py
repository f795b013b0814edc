"""Multi-GPU is "replicas only": N independent problems, no data-path collective.
These tests cover the rank logic of bench.py with world_size 2 on the CPU (gloo, 127.0.0.1)."""
import json
import os
import socket
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import argparse

    import torch.distributed as dist

    sys.path.insert(0, ROOT)
    import bench

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    args = argparse.Namespace(config=0, scale=10, theta=None, order=None)
    w = bench.workload(args, rank)
    # every rank draws its own replica of the same recipe
    ms, inter = bench.reduce_over_ranks(dist, 10.0 * (rank + 1), 1000 * (rank + 1), "cpu")
    q.put((rank, float(w.pos.astype(np.float64).sum()), w.n, w.eps, w.theta, w.order, ms, inter))
    dist.destroy_process_group()


def test_two_replicas_draw_different_sets_and_reduce_max_time_sum_work():
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, s0, n0, e0, t0, o0, ms0, i0), (r1, s1, n1, e1, t1, o1, ms1, i1) = res
    assert n0 == n1 == 1024 and (e0, t0, o0) == (e1, t1, o1)   # same recipe, same parameters
    assert s0 != s1                                            # different seeds: independent replicas
    assert ms0 == ms1 == 20.0 and i0 == i1 == 3000.0           # slowest rank's time, everybody's work


def test_reference_arm_under_torchrun_prints_one_line_from_rank_0():
    port = _free_port()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--config", "0",
           "--scale", "10", "--steps", "1", "--warmup", "0"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["unit"] == "Ginteractions/s" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
