"""Multi-GPU = scenario sharding (44K scenarios split over 8 GPUs).

Scenarios are independent (no agent, roadgraph point or metric of scenario b reads anything
of scenario b'), so ranks take disjoint slices of the scenario ids and run the same path with
NO data-path collective.  torch.distributed is used only for the benchmark's barrier and the
max-over-ranks timing (NCCL on the GPU box, gloo in the CPU tests).
"""
import os

import torch
import torch.distributed as dist


def rank_world():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def shard_ids(per_rank_B, rank, world):
    """Weak scaling: rank r owns scenario ids [r*B, (r+1)*B); ids are global, so every scenario
    of the job is distinct and reproducible whatever the number of ranks."""
    assert 0 <= rank < world
    return list(range(rank * per_rank_B, (rank + 1) * per_rank_B))


def split_ids(total_B, rank, world):
    """Strong scaling helper: contiguous, balanced split of [0, total_B)."""
    base, rem = divmod(total_B, world)
    start = rank * base + min(rank, rem)
    return list(range(start, start + base + (1 if rank < rem else 0)))


def init_process_group(backend=None):
    rank, world = rank_world()
    if world > 1 and not dist.is_initialized():
        if backend is None:
            backend = "nccl" if torch.cuda.is_available() else "gloo"
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29512")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, world


def barrier():
    if dist.is_initialized():
        dist.barrier()


def max_over_ranks(value, device="cpu"):
    """Max of a python float over ranks (timing is the slowest rank's)."""
    if not dist.is_initialized():
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value, device="cpu"):
    if not dist.is_initialized():
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())
