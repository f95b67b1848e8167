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


# ---------------------------------------------------------------------------------------------------------------
# one domain cut into slabs of whole rows, one particle exchange per step (include/fpcl.h
# "fp_set_slab").  Host logic only -- the partition, the cell sort and the collision step are the library's kernels.
# The exchange keeps the SOURCE order (receive buffer = concatenation over source slabs in ascending order, the
# slab's own stayers in their place): that is what makes the cut run bit-identical to the uncut one.
# Unmeasured on hardware: this pool offers one GPU per call, so the NCCL path is exercised on CPU with gloo
# (tests/test_dist_cpu.py) and the device kernels with several slabs on one GPU (tests/test_gpu_slab.py).
# ---------------------------------------------------------------------------------------------------------------
FIELDS = ("x", "y", "vx", "vy", "vz", "pid")


def slab_row_bounds(ny, nslabs):
    """First rows of nslabs slabs of (nearly) equal height covering rows 0 .. ny."""
    if not 1 <= nslabs <= min(ny, 64):
        raise ValueError("need 1 <= nslabs <= min(ny, 64)")
    return [(ny * s) // nslabs for s in range(nslabs + 1)]


def exchange_slab_particles(parts, starts, group=None):
    """All-to-all of partitioned particles between the ranks of ``group`` (one slab per rank).

    parts: dict of 1-D tensors (FIELDS) holding this rank's particles grouped by destination slab;
    starts: list of nslabs+1 offsets (host ints) of those groups.  Returns a dict of tensors with the particles this
    rank now owns, in ascending source-rank order.  Two collectives per step: the counts, then one
    all_to_all_single per field (NCCL on GPUs, gloo on CPU)."""
    ws = dist.get_world_size(group)
    assert len(starts) == ws + 1
    send_counts = [int(starts[s + 1] - starts[s]) for s in range(ws)]
    dev = parts["x"].device
    sc = torch.tensor(send_counts, dtype=torch.int64, device=dev)
    rc = torch.empty_like(sc)
    dist.all_to_all_single(rc, sc, group=group)
    recv_counts = [int(v) for v in rc.tolist()]
    out = {}
    for k in FIELDS:
        src = parts[k][: starts[-1]].contiguous()
        wire = src.view(torch.int32)                       # 4-byte fields; the collectives have no uint32
        dst = torch.empty(sum(recv_counts), dtype=torch.int32, device=dev)
        dist.all_to_all_single(dst, wire, output_split_sizes=recv_counts, input_split_sizes=send_counts, group=group)
        out[k] = dst.view(src.dtype)
    return out, recv_counts


def exchange_in_process(parts_by_slab, starts_by_slab):
    """The same exchange between slabs held by one process (several contexts on one device): plain slicing and
    concatenation in ascending source order.  parts_by_slab[s] / starts_by_slab[s]: slab s's partitioned particles."""
    n = len(parts_by_slab)
    out = []
    for dst in range(n):
        out.append({k: torch.cat([parts_by_slab[src][k][starts_by_slab[src][dst]:starts_by_slab[src][dst + 1]] for src in range(n)])
                    for k in FIELDS})
    return out
