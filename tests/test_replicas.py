"""N > 1 host logic (replicas only) on CPU: two processes, gloo backend."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    from paper_1408_5853_b200 import replicas as R
    r, lr, w = R.rank_env()
    assert (r, lr, w) == (rank, rank, world)
    dist = R.init("gloo", lr, w)
    R.barrier(dist)
    ms_local = 10.0 + 5.0 * rank            # rank 1 is the slow one
    ms_max = R.max_over_ranks(ms_local, dist)
    R.barrier(dist)
    out[rank] = (ms_max, R.job_gcups(1 << 20, 7, ms_max * 1e-3, w))
    dist.destroy_process_group()


def test_two_replicas_report_the_slowest_rank_and_the_whole_job():
    import torch.multiprocessing as mp
    world, port = 2, 29500 + os.getpid() % 2000
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0] == res[1]
    ms_max, value = res[0]
    assert ms_max == 15.0
    assert value == pytest.approx(2 * (1 << 20) * 7 / 15e-3 / 1e9)


def test_single_process_needs_no_group():
    sys.path.insert(0, ROOT)
    from paper_1408_5853_b200 import replicas as R
    assert R.init("gloo", 0, 1) is None
    assert R.max_over_ranks(3.5, None) == 3.5
    R.barrier(None)
    assert R.job_gcups(1000, 10, 1e-3, 1) == pytest.approx(1e-2)


def test_reference_arm_runs_on_rank_0_only():
    """bench.py --impl reference under torchrun: ranks > 0 exit 0 without work or output."""
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_reference_arm_prints_one_json_line():
    env = dict(os.environ, RANK="0", LOCAL_RANK="0", WORLD_SIZE="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "GCUPS" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
