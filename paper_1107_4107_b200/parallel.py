"""Multi-GPU plumbing: trajectories are independent, so the path shards
by image rows with no communication during integration.  The only exchange step is the sum of the
per-rank density histograms (exact integer counts, order-independent): one all-reduce of 4 MiB.

One process per GPU (torchrun); `torch.distributed` with NCCL on GPUs, gloo in the CPU tests.
"""
import torch
import torch.distributed as dist


def strip_bounds(lo, hi, world, rank):
    """Rank r's horizontal strip [lo_y, hi_y) of the action square: equal heights, exact end points."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    h = (hi - lo) / world
    lo_y = lo + rank * h
    hi_y = hi if rank == world - 1 else lo + (rank + 1) * h
    return lo_y, hi_y


def shard_rows(gy, world, rank):
    """Contiguous row range [j0, j1) of a gy-row image owned by `rank` (strong-scaling split)."""
    base, rem = divmod(gy, world)
    j0 = rank * base + min(rank, rem)
    return j0, j0 + base + (1 if rank < rem else 0)


def allreduce_hist(hist):
    """In-place sum of the uint32 histogram over all ranks.  The tensor holds the uint32 bits as int32;
    two's-complement addition is the same bit pattern as unsigned addition mod 2^32."""
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(hist, op=dist.ReduceOp.SUM)
    return hist


def gather_image(local_rows, world, rank, dst=0):
    """Concatenate per-rank image strips in rank order on `dst` (returns None elsewhere)."""
    if not (dist.is_available() and dist.is_initialized()) or world == 1:
        return local_rows
    parts = [None] * world if rank == dst else None
    dist.gather_object(local_rows.cpu(), parts, dst=dst)
    if rank != dst:
        return None
    return torch.cat(parts, dim=0)
