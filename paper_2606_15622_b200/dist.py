"""Multi-GPU plumbing of the benchmark: independent replicas, one per rank.

The hot path has no exchange step on one node: every rank advances its own ensemble (its own seed), so the only
collectives are the barrier around the timed region and the MAX reduction of the per-rank time.  This module holds
that host logic so that it can be exercised on CPU with the gloo backend (tests/test_dist_cpu.py).
"""
import os

import torch
import torch.distributed as dist


def world():
    return int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0"))


def replica_seed(base_seed, rank):
    """Seed of rank's replica: distinct ensembles, same shape (weak scaling)."""
    return int(base_seed) + int(rank)


def init(backend, device=None):
    ws, _, _ = world()
    if ws > 1 and not dist.is_initialized():
        if backend == "nccl":
            dist.init_process_group("nccl", device_id=device)
        else:
            dist.init_process_group(backend)
    return ws


def barrier():
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def max_over_ranks(value, device="cpu"):
    """MAX of a python float over all ranks (identity for a single process)."""
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized():
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(units_per_rank, steps, ms_max, world_size):
    """Whole-job units/s: every rank processed units_per_rank * steps in at most ms_max milliseconds."""
    return world_size * units_per_rank * steps / (ms_max * 1e-3)


def shutdown():
    if dist.is_available() and dist.is_initialized():
        dist.destroy_process_group()
