"""The N > 1 path of bench.py on CPU: two processes over gloo (127.0.0.1).

The build is defined on one device (replicas only, no data-path collective), so what
the ranks share is host logic: every rank draws its own particle set, the step time is the maximum over the
ranks, the reported value is the whole job's throughput, and `--impl reference` runs on rank 0 alone.
"""
import os
import subprocess
import sys

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from paper_2307_06345_b200 import workloads as W

    cfg = bench.rank_workload(W.CONFIGS[3], rank)
    x, y, z = cfg.generate(4096)
    my_ms = 4.0 + 3.0 * rank                                  # rank 1 is the slow one
    ms = bench.max_over_ranks(my_ms, world, "cpu")
    value = bench.whole_job_value(4096, world, ms)
    sums = [None] * world
    dist.all_gather_object(sums, W.checksum(x, y, z))
    out[rank] = (ms, value, sums, cfg.seed)
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_share_the_slowest_time_and_draw_different_particles():
    world, port = 2, 29500 + os.getpid() % 500
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert set(res) == {0, 1}
    for r in (0, 1):
        ms, value, sums, seed = res[r]
        assert ms == 7.0                                      # max over ranks, on every rank
        assert value == pytest.approx(2 * 4096 / 7.0e-3 / 1e6)   # whole job: both ranks' particles per step
        assert sums[0] != sums[1]                             # replicas build different trees
    assert res[0][3] != res[1][3]


def test_single_rank_needs_no_process_group():
    import bench
    assert bench.max_over_ranks(3.5, 1, "cpu") == 3.5
    assert bench.whole_job_value(1 << 26, 1, 4.0) == pytest.approx((1 << 26) / 4.0e-3 / 1e6)


def test_reference_arm_runs_on_rank_zero_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0"], capture_output=True, text=True, env=env, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
