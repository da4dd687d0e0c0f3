"""The N > 1 path on CPU: two processes over gloo (127.0.0.1).

What the ranks share is host logic: every rank draws its own particle set, the step time is the maximum over the
ranks, the reported value is the whole job's throughput, `--impl reference` runs on rank 0 alone -- and, for the
distributed build of PAPER.md:198-204 (paper_2307_06345_b200/distributed.py), the exchange steps themselves: the
min / max all-reduce of the boxes, the broadcast of the start array and the all-reduce(sum) of the leaf counts between
f and g in every round.  No CUDA kernel can run here, so f and g are the oracle's (this is a test of the plumbing
around them; the kernels are compared with the oracle in tests/test_gpu_global.py).
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


def _global_tree_worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    from paper_2307_06345_b200 import distributed as D
    from paper_2307_06345_b200 import workloads as W

    bucket = 16
    x, y, z = W.plummer(3000 + 2000 * rank, W.BASE_SEED + 100 + rank)       # ranks hold different numbers of particles
    box = D.allreduce_box(torch.from_numpy(oracle.box(x, y, z)))
    P = oracle.sort(oracle.keys(x, y, z, box.numpy()))[0]
    start = None
    if rank == 0:
        start = torch.from_numpy(oracle.leaves_topdown(P, bucket)[0].view(np.int64))
    start = D.broadcast_leaves(start, "cpu")

    def count(K):
        Ku = K.numpy().view(np.uint64)
        return torch.from_numpy(oracle.round_(P, Ku, bucket)["N"].view(np.int32).copy())      # f on this rank's keys

    def rebalance(K, N):
        Ku = K.numpy().view(np.uint64)
        # g on the summed counts: a one-shard "global round" whose particle keys realise exactly those counts
        keys = np.repeat(Ku[:-1], N.numpy().view(np.uint32))
        r = oracle.round_(keys, Ku, bucket, cap=1 << 20)
        return torch.from_numpy(r["K"].view(np.int64).copy()), bool(np.any(r["O"] != 1))

    K, N, rounds = D.global_leaves(count, rebalance, start)
    gathered = [None] * world
    dist.all_gather_object(gathered, P)
    out[rank] = (box.numpy().copy(), K.numpy().view(np.uint64).copy(), N.numpy().view(np.uint32).copy(), rounds, gathered)
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_build_one_global_tree_with_the_real_all_reduce():
    import oracle
    world, port = 2, 30100 + os.getpid() % 500
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_global_tree_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    box0, K0, N0, rounds0, shards = res[0]
    box1, K1, N1, rounds1, _ = res[1]
    assert np.array_equal(box0, box1) and np.array_equal(K0, K1) and np.array_equal(N0, N1) and rounds0 == rounds1
    Pall = np.sort(np.concatenate(shards), kind="stable")
    Ktop, Ntop = oracle.leaves_topdown(Pall, 16)               # the fixpoint is the balanced tree of ALL particles
    assert np.array_equal(K0, Ktop) and np.array_equal(N0, Ntop)
    assert int(N0.sum()) == 3000 + 5000
    assert 2 <= rounds0 <= 6                                   # rank 0's own tree is a start a few levels short
