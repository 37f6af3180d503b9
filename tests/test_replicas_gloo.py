"""N > 1 is "replicas only": one independent context per rank, no data-path collective; the only
exchange is the reduction of the timings in bench.py.  That rank logic is covered here with world_size 2 on CPU
(gloo), and the reference arm's rule that only rank 0 works."""
from __future__ import annotations

import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, q) -> None:
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # rank 1 is the slow one; rank 0 has a non-finite state in the second call
        ms, e2e, ok = bench.reduce_over_ranks(10.0 + 5.0 * rank, 40.0 - 3.0 * rank, True, dist, "cpu")
        ms2, _, ok2 = bench.reduce_over_ranks(1.0, 1.0, rank != 0, dist, "cpu")
        q.put((rank, ms, e2e, ok, ms2, ok2))
    finally:
        dist.destroy_process_group()


def test_timing_reduction_is_max_over_ranks_world_size_2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, e2e, ok, ms2, ok2 in got:
        assert ms == 15.0 and e2e == 40.0 and ok is True          # slowest rank decides, on every rank
        assert ms2 == 1.0 and ok2 is False                        # one bad replica invalidates the job


def test_whole_job_value_counts_every_replica():
    sys.path.insert(0, ROOT)
    import bench
    one = bench.whole_job_grind(9.0, 256 ** 3, 1, 7)
    assert bench.whole_job_grind(9.0, 256 ** 3, 8, 7) == pytest.approx(one / 8)      # weak scaling: 8 x the cells
    assert one == pytest.approx(9.0e6 / (256 ** 3 * 7 * 3))


def test_reference_arm_runs_on_rank_0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0"], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
    env0 = dict(os.environ, RANK="0", WORLD_SIZE="2", LOCAL_RANK="0")
    r0 = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                         "--warmup", "0", "--ref-n", "24"], capture_output=True, text=True, env=env0, timeout=600)
    assert r0.returncode == 0, r0.stderr
    line = json.loads(r0.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["gpu_launches"] == 0
