"""CPU tests of bench.py's N > 1 host logic (the path is "replicas only": DESIGN.md section 8): the max-over-ranks
reduction under a world_size-2 gloo group, the aggregate value, and the reference arm's rank-0-only rule."""
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


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist

    sys.path.insert(0, ROOT)
    import bench

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, dist, torch.device("cpu"))  # rank 1 is the slow one: 15 ms
    dist.barrier()
    dist.destroy_process_group()
    out[rank] = ms


def test_max_over_ranks_gloo_world2():
    import torch.multiprocessing as mp

    port = _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
        assert out[0] == 15.0 and out[1] == 15.0


def test_replicas_value_is_the_whole_job_aggregate():
    sys.path.insert(0, ROOT)
    import bench

    one = bench.replicas_value(2.0e12, 1000.0, 1)
    assert one == pytest.approx(2.0)
    assert bench.replicas_value(2.0e12, 1000.0, 8) == pytest.approx(8 * one)
    assert bench.max_over_ranks(3.5, None, None) == 3.5


def test_reference_arm_prints_on_rank0_only():
    """bench.py --impl reference: under torchrun (N > 1) rank 0 alone runs and prints; the others exit 0 silently."""
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "tiny", "--gpus", "2",
           "--steps", "1", "--warmup", "0"]
    outs = []
    for rank in (0, 1):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2")
        r = subprocess.run(cmd, env=env, capture_output=True, text=True, timeout=300)
        assert r.returncode == 0, r.stderr
        outs.append(r.stdout.strip())
    assert outs[1] == ""
    line = json.loads(outs[0])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
