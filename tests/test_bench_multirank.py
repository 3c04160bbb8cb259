"""The N > 1 path of bench.py (replicas only) on CPU: two gloo ranks agree on the
max-over-ranks time and the whole-job value; the reference arm runs on rank 0 only."""
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % port, rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, world)          # rank 1 is the slower one
    val = bench.whole_job_value(1.0e6, ms, world)
    dist.barrier()
    out[rank] = (ms, val)
    dist.destroy_process_group()


def test_two_ranks_take_the_slowest_time_and_sum_the_work():
    world = 2
    with mp.Manager() as man:
        out = man.dict()
        mp.spawn(_worker, args=(world, 29531 + os.getpid() % 200, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0] == res[1]
    ms, val = res[0]
    assert ms == 15.0
    assert val == 2 * 1.0e6 / 15.0e-3


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, 1) == 3.5
    assert bench.whole_job_value(2.0e6, 4.0, 1) == 2.0e6 / 4.0e-3
    assert bench.cell_updates([4, 8], [1, 2]) == 512.0 * (4 + 16)


def test_reference_arm_is_silent_on_other_ranks():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       capture_output=True, text=True, env=env, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
