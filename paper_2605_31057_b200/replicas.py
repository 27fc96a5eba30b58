"""Multi-GPU plumbing of bench.py: replicas, or head shards of one call.

The hot path has no exchange step: heads and batches are independent and the block index is
head-independent, so N GPUs run N independent replicas of the call (what a Ulysses-style head
sharding of a full model would give each GPU).  `torch.distributed` is used for the
barrier around the timed region and for the max-over-ranks time only; there is no data-path
collective.  Backend "nccl" on GPUs, "gloo" in the CPU tests.

`bench.py --shard heads` is the strong-scaling view of the same fact: every rank builds the same
index and runs heads [h_lo, h_hi) of the SAME seeded call (what one device of the paper's 8-device
Ulysses run holds between its two all-to-alls); the call takes as long as the slowest
shard and the job did the work of all of them.
"""
from __future__ import annotations

import os

import torch


def env_ranks():
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def setup(backend: str = "nccl"):
    """(rank, world, local_rank, dist or None); initialises the process group when WORLD_SIZE > 1
    (MASTER_ADDR / MASTER_PORT from the environment, as torchrun sets them)."""
    rank, world, local = env_ranks()
    if world <= 1:
        return rank, world, local, None
    import torch.distributed as dist
    if backend == "nccl":
        torch.cuda.set_device(local)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    else:
        dist.init_process_group(backend)
    return rank, world, local, dist


def max_over_ranks(dist, values, device="cpu"):
    """Element-wise maximum of a list of per-rank floats over all ranks (identity when dist is None)."""
    if dist is None:
        return [float(v) for v in values]
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def job_throughput(world: int, units_per_rank_step: float, ms_step_max: float) -> float:
    """Whole-job aggregate: every rank processed units_per_rank_step per step (weak scaling), and a
    step takes as long as the slowest rank."""
    return world * units_per_rank_step / (ms_step_max * 1e-3)


def head_shard(H: int, world: int, rank: int):
    """Heads [h_lo, h_hi) of rank `rank` when H heads are dealt to `world` ranks as evenly as possible
    (the first H % world ranks hold one head more).  Needs world <= H: a rank without heads has no call."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    if world > H:
        raise ValueError(f"cannot shard {H} heads over {world} ranks")
    base, extra = divmod(H, world)
    h_lo = rank * base + min(rank, extra)
    return h_lo, h_lo + base + (1 if rank < extra else 0)


def sum_over_ranks(dist, values, device="cpu"):
    """Element-wise sum of a list of per-rank floats over all ranks (identity when dist is None)."""
    if dist is None:
        return [float(v) for v in values]
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return [float(x) for x in t]


def job_throughput_sharded(total_units_step: float, ms_step_max: float) -> float:
    """Strong scaling: the ranks together processed total_units_step (the sum of their shards) per step,
    and the step takes as long as the slowest shard."""
    return total_units_step / (ms_step_max * 1e-3)
