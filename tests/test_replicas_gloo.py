"""The N > 1 path of bench.py (replicas only) on CPU: world_size 2, gloo."""
import os
import socket

import torch
import torch.multiprocessing as mp

from paper_2605_31057_b200 import replicas


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    r, w, local, dist = replicas.setup("gloo")
    assert (r, w, local) == (rank, world, rank) and dist is not None
    dist.barrier()
    # rank-dependent timings: the job is as slow as its slowest replica
    ms_step, kern_ms, e2e_ms = replicas.max_over_ranks(dist, [10.0 + rank, 9.0 - rank, 30.0 + 2 * rank])
    value = replicas.job_throughput(w, 4.0e13, ms_step)
    # head-sharded mode (bench.py --shard heads): 5 heads over 2 ranks = 3 + 2; the job did the work of
    # all heads in the time of the slowest shard
    h_lo, h_hi = replicas.head_shard(5, w, rank)
    (job_units,) = replicas.sum_over_ranks(dist, [1.0e13 * (h_hi - h_lo)])
    sharded = replicas.job_throughput_sharded(job_units, ms_step)
    q.put((rank, ms_step, kern_ms, e2e_ms, value, (h_lo, h_hi), job_units, sharded))
    dist.barrier()
    dist.destroy_process_group()


def test_two_replicas_take_the_max_time_and_sum_the_work():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms_step, kern_ms, e2e_ms, value, heads, job_units, sharded in got:
        assert (ms_step, kern_ms, e2e_ms) == (11.0, 9.0, 32.0)           # max over ranks, element-wise
        assert abs(value - 2 * 4.0e13 / 11.0e-3) <= 1e-3 * value         # whole-job aggregate
        assert heads == ((0, 3), (3, 5))[rank]                            # H not divisible by N
        assert job_units == 5.0e13                                        # every head counted once
        assert abs(sharded - 5.0e13 / 11.0e-3) <= 1e-3 * sharded          # strong scaling: total work / slowest shard


def test_head_shards_partition_the_heads():
    """bench.py --shard heads: the shards are contiguous, disjoint, cover [0, H) and differ by at most one head
    (H = 12 / 40 / 16 are the BASELINE.json head counts; 8 GPUs is the paper's device count)."""
    import pytest
    for H in (1, 5, 12, 16, 40):
        for world in range(1, min(H, 8) + 1):
            cuts = [replicas.head_shard(H, world, r) for r in range(world)]
            assert cuts[0][0] == 0 and cuts[-1][1] == H
            assert all(cuts[r][1] == cuts[r + 1][0] for r in range(world - 1))
            sizes = [b - a for a, b in cuts]
            assert min(sizes) >= 1 and max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    assert [replicas.head_shard(12, 8, r) for r in range(8)] == [(0, 2), (2, 4), (4, 6), (6, 8), (8, 9), (9, 10), (10, 11), (11, 12)]
    with pytest.raises(ValueError):
        replicas.head_shard(4, 5, 0)
    with pytest.raises(ValueError):
        replicas.head_shard(4, 2, 2)
    assert replicas.sum_over_ranks(None, [1.5, 2.5]) == [1.5, 2.5]
    assert replicas.job_throughput_sharded(10.0, 1000.0) == 10.0


def test_single_process_is_the_identity():
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK"):
        os.environ.pop(k, None)
    r, w, local, dist = replicas.setup("gloo")
    assert (r, w, local, dist) == (0, 1, 0, None)
    assert replicas.max_over_ranks(None, [1.5, 2.5]) == [1.5, 2.5]
    assert replicas.job_throughput(1, 10.0, 1000.0) == 10.0


def test_reference_arm_runs_on_rank0_only(tmp_path):
    """bench.py --impl reference: ranks other than 0 exit 0 without work (task contract)."""
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""
