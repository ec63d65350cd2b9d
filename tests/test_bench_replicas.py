"""bench.py's multi-rank plumbing on CPU (gloo, world_size 2): replicas only, so
the only cross-rank step is the max-over-ranks of the step time, and only rank 0 of the reference
arm does any work."""
import json
import os
import socket
import subprocess
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms = [12.5, 40.25][rank]                       # rank 1 is the slow replica
    got = bench.rank_max(ms, world, "cpu")
    q.put((rank, got, bench.job_value(24 * 20, world, got)))
    dist.barrier()
    dist.destroy_process_group()


def test_rank_max_and_job_value_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, got, val in res:
        assert got == 40.25                            # every rank sees the slowest rank's time
        assert val == pytest.approx(2 * 480 / 40.25e-3)


def test_single_rank_is_identity():
    import bench
    assert bench.rank_max(3.5, 1, "cpu") == 3.5
    assert bench.job_value(480, 1, 10.0) == pytest.approx(48000.0)


def test_reference_arm_only_rank0_prints():
    """--impl reference under a 2-rank launch: rank 0 times the oracle and prints one JSON line,
    rank 1 exits 0 without work."""
    outs = []
    for rank in (0, 1):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", LOCAL_RANK=str(rank))
        r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                            "--steps", "1", "--warmup", "3"], capture_output=True, text=True, env=env, timeout=600)
        assert r.returncode == 0, r.stderr
        outs.append(r.stdout.strip())
    line = json.loads(outs[0].splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["value"] > 0
    assert outs[1] == ""
