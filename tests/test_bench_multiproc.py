"""CPU-only: the N > 1 logic of bench.py (replicas only) with two gloo processes:
the step time is the MAX over ranks, the value the whole job's; under --impl reference only rank 0 works."""
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
    dist.barrier()
    ms = bench.reduce_max_ms(10.0 * (rank + 1), dist, "cpu")          # rank 1 is the slow replica
    out[rank] = (ms, bench.whole_job_value(1000, world, ms))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_take_the_max_and_sum_the_work():
    world, port = 2, 29500 + os.getpid() % 2000
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0] == res[1]
    ms, value = res[0]
    assert ms == 20.0 and abs(value - 2 * 1000 / 20e-3 / 1e6) < 1e-12


def test_single_process_needs_no_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_max_ms(3.5, None, "cpu") == 3.5
    assert bench.whole_job_value(2_000_000, 1, 1.0) == 2000.0


def test_reference_arm_other_ranks_exit_quietly():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--config", "tiny",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
