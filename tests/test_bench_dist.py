"""Host-side logic of bench.py's N > 1 path ("replicas only": no data-path collective, only the
max-over-ranks timing), covered with world_size-2 gloo on CPU; and the --impl reference arm."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = [10.0, 14.0][rank]
    ms_max = bench.max_over_ranks(ms, world, "cpu")
    out[rank] = (ms_max, bench.whole_job_gflops(world, 5, 1000, ms_max))
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value_gloo_world2():
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(2, 29517, out), nprocs=2, join=True)
    want = 2 * 5 * 4 * 1000 * 1320 / (14.0e-3) / 1e9
    for rank in (0, 1):
        ms_max, value = out[rank]
        assert ms_max == 14.0                      # the slower rank sets the time on every rank
        assert abs(value - want) < 1e-12 * want    # value = units all ranks processed / that time


def test_reference_arm_prints_one_json_line_rank0_only():
    env = dict(os.environ, OMP_NUM_THREADS="4")
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "1",
           "--steps", "101", "--warmup", "3"]          # > 100 steps -> the small bounded sample
    r = subprocess.run(cmd, capture_output=True, text=True, env=env, timeout=600)
    assert r.returncode == 0, r.stderr
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    j = json.loads(lines[0])
    assert j["impl"] == "reference" and j["unit"] == "GFLOPS" and j["value"] > 0
    assert j["cpu_baseline"]["kind"] == "oracle" and j["cpu_baseline"]["cores"] >= 1
    assert j["e2e"]["h2d_bytes_per_step"] == 0 and j["e2e"]["value"] == j["value"]
    # a non-zero rank does no work and prints nothing
    r = subprocess.run(cmd, capture_output=True, text=True, env=dict(env, RANK="1", WORLD_SIZE="2"), timeout=60)
    assert r.returncode == 0 and r.stdout.strip() == ""


import pytest


@pytest.mark.gpu
def test_strong_scaling_arm_runs_the_slab_cg_on_one_gpu():
    """bench.py --scaling strong at N = 1: the slab decomposition's stages with the rank as its own neighbour; the
    line carries the contract's keys, "scaling": "strong", and the last solve made progress."""
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--scaling", "strong", "--gpus", "1", "--steps", "12", "--warmup", "4"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    j = json.loads(lines[0])
    assert j["scaling"] == "strong" and j["n_gpus"] == 1 and j["unit"] == "GFLOPS" and j["value"] > 0
    assert j["config"]["ranks"] == 1 and j["config"]["local_lattice"] == [32, 32, 32, 64]
    assert j["gpu_launches"] > 0 and j["last_solve"]["iterations"] == 12
    assert 0 < j["last_solve"]["rel_resid_true"] < 1.0
