"""Host-side logic of bench.py's N > 1 path ("replicas only"), on CPU with gloo, world size 2."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = [10.0, 14.0][rank]            # rank 1 is the slow one
    kernel = [9.0, 8.0][rank]
    ms_max, k_max = bench.reduce_max_over_ranks([ms, kernel], torch.device("cpu"), world)
    dist.barrier()
    out[rank] = (ms_max, k_max, bench.whole_job_value(world, 1000, 5, ms_max * 1e-3))
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, 29541, out), nprocs=world, join=True)
        res = dict(out)
    for r in range(world):
        ms_max, k_max, value = res[r]
        assert ms_max == 14.0 and k_max == 9.0
        assert abs(value - 2 * 1000 * 5 / 0.014) < 1e-6


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_algorithmic_bytes_match_design():
    import bench
    from paper_2110_08650_b200 import workloads as W
    wl = W.CONFIGS["thermal_128"]
    assert abs(bench.algorithmic_bytes_per_particle_step(wl, W.n_particles(wl)) - 66.79) < 0.01
