"""-m "not gpu": host logic of bench.py.

The path does not shard ("replicas only"), so the only N > 1 logic is the
whole-job reduction: value = (pair tests all ranks processed) / (max over ranks of the timed region).
It is covered here with world_size = 2 over gloo on the CPU.
"""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r processed 1000 * (r + 1) units per step in 10 * (r + 1) ms over 4 steps
    value, ms = bench.aggregate(1000.0 * (rank + 1), 4, 10.0 * (rank + 1), world, dist)
    q.put((rank, value, ms))
    dist.barrier()
    dist.destroy_process_group()


def test_aggregate_world2_gloo():
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
    # units = (1000 + 2000) * 4 ; time = max(10, 20) ms
    for _, value, ms in res:
        assert value == pytest.approx(12000.0 / 20e-3)
        assert ms == pytest.approx(20.0 / 4)


def test_aggregate_single_rank():
    sys.path.insert(0, ROOT)
    import bench
    value, ms = bench.aggregate(500.0, 10, 25.0, 1)
    assert value == pytest.approx(5000.0 / 25e-3) and ms == pytest.approx(2.5)


def test_reference_arm_prints_one_json_line_and_other_ranks_stay_silent():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0",
                          "--steps", "1", "--warmup", "0", "--gpus", "2"], env=env, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0 and out.stdout.strip() == ""
    env = dict(os.environ, RANK="0", WORLD_SIZE="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0",
                          "--steps", "1", "--warmup", "0", "--ref-sample", "200"], env=env, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == "element_face_pair_tests_per_s"
    assert line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0
