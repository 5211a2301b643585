"""The N>1 timing plumbing of bench.py on CPU: world_size-2 gloo process groups.

bench.py --gpus N slab-decomposes ONE grid over the N ranks (strong scaling; the exchange itself is covered by
tests/test_dist_plumbing.py); what bench.py adds is the barrier and the max-over-ranks of the timed region and the
whole-job rate.  These tests run that host logic with two real processes.
"""
import json
import os
import socket
import subprocess
import sys

import pytest
import torch
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
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), WORLD_SIZE=str(world),
                      RANK=str(rank), LOCAL_RANK=str(rank))
    sys.path.insert(0, ROOT)
    import bench
    w, r, lr = bench.dist_env()
    dist = bench.dist_init(w, "gloo")
    dist.barrier()
    # rank r "measured" (10 + 5 r) ms per step: the job is as slow as its slowest replica
    ms = bench.max_over_ranks(10.0 + 5.0 * r, dist)
    value = bench.job_gflops((64, 64, 64), ms * 1e-3)
    dist.barrier()
    dist.destroy_process_group()
    q.put((r, w, lr, ms, value))


def test_max_over_ranks_and_job_value_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    import bench
    one = bench.flops_pair((64, 64, 64)) / 15e-3 / 1e9
    for r, (rank, world, local_rank, ms, value) in enumerate(out):
        assert (rank, world, local_rank) == (r, 2, r)
        assert ms == 15.0                                  # max over ranks, seen by every rank
        assert value == pytest.approx(one)                 # strong scaling: ONE grid over the ranks in the slowest rank's time


def test_single_process_needs_no_group():
    import bench
    assert bench.dist_init(1, "gloo") is None
    assert bench.max_over_ranks(3.5, None) == 3.5
    n = 1024 ** 3
    assert bench.flops_pair((1024, 1024, 1024)) == 5.0 * n * 30          # 5 N^3 log2 N^3, BASELINE.json metric
    assert bench.job_gflops((1024,) * 3, 1.0) == pytest.approx(5.0 * n * 30 / 1e9)


def test_reference_arm_under_torchrun_prints_one_line():
    """bench.py --impl reference with 2 ranks: rank 0 alone times the oracle and prints ONE JSON line."""
    env = dict(os.environ)
    env.pop("RANK", None)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()),
           os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
           "--size", "32"]
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [ln for ln in res.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["unit"] == "GFLOP/s"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"] > 0
    assert d["e2e"] == {"value": d["value"], "unit": "GFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["higher_is_better"] is True and d["vs_baseline"] is None


def test_gpus_must_match_the_launchers_world_size():
    """`bench.py --gpus 4` started as a single process must not print an n_gpus = 1 line: it exits non-zero and says how
    to launch it (the driver starts N > 1 under torchrun, which sets WORLD_SIZE)."""
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "4", "--steps", "1"],
                         capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert res.returncode != 0
    assert "torch.distributed.run" in res.stderr and "--nproc-per-node 4" in res.stderr
    assert not [ln for ln in res.stdout.splitlines() if ln.startswith("{")]
