"""Host logic of bench.py that needs no GPU: the max-over-ranks timing of the N > 1 replicas path on a
world_size-2 gloo group, and the reference arm (the oracle timed on the host cores; rank 0 alone prints)."""
import json
import os
import subprocess
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _rank_main(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms_local = 10.0 + 5.0 * rank                       # rank 1 is the slow one
    ms = bench.max_over_ranks(ms_local, world, torch.device("cpu"))
    out[rank] = (ms, bench.whole_job_value(world, 1000, ms))
    dist.barrier()
    dist.destroy_process_group()


def test_replicas_timing_is_max_over_ranks_and_value_is_whole_job_gloo_world2():
    world, port = 2, 29000 + os.getpid() % 2000
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_rank_main, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0][0] == res[1][0] == 15.0              # every rank reports the slowest rank's time
    assert res[0][1] == pytest.approx(2 * 1000 / 15e-3)  # two replicas' timesteps over that time


def test_single_rank_needs_no_process_group():
    import bench
    assert bench.max_over_ranks(3.5, 1, torch.device("cpu")) == 3.5
    assert bench.whole_job_value(1, 500, 50.0) == pytest.approx(1e4)


def _run_reference(rank):
    env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", LOCAL_RANK=str(rank))
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "C1",
                           "--gpus", "2", "--steps", "2", "--warmup", "1"], env=env, cwd=ROOT,
                          capture_output=True, text=True, timeout=300)


def test_reference_arm_rank0_prints_one_line_other_ranks_exit_silently():
    r0, r1 = _run_reference(0), _run_reference(1)
    assert r0.returncode == 0 and r1.returncode == 0
    assert r1.stdout.strip() == ""
    lines = [l for l in r0.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "timesteps/s" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert d["n_gpus"] == 2 and d["steps"] == 2 and d["warmup"] == 1
