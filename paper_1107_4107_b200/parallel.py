"""Multi-GPU plumbing: trajectories are independent, so the path shards by
contiguous ranges of the global trajectory index with no communication during integration.  A rank holds the slice
[k0, k0 + n) of the ensemble the grid describes (include/aw.h, aw_grid.k0): grid position and every random draw are
functions of the GLOBAL index, so a rank's rows are bit-identical to the same rows of the single-GPU result.

The only exchange steps are the sum of the per-rank density histograms (exact integer counts, order-independent:
one all-reduce of 4 MiB) and the rank-ordered concatenation of the image strips (one gather).  Both run on the
tensors where they live (NCCL on device tensors; gloo on CPU tensors in the tests).

One process per GPU (torchrun); `torch.distributed` with NCCL on GPUs, gloo in the CPU tests.
"""
import torch
import torch.distributed as dist


def shard_rows(gy, world, rank):
    """Contiguous row range [j0, j1) of a gy-row image owned by `rank` (strong scaling: the whole job is fixed)."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    base, rem = divmod(gy, world)
    j0 = rank * base + min(rank, rem)
    return j0, j0 + base + (1 if rank < rem else 0)


def slice_of(gx, gy, world, rank, scaling="weak"):
    """(gx, gy_total, k0, n) of rank's slice.  weak: every rank owns a full gx x gy block of a gx x (gy*world)
    ensemble over the same action rectangle (per-GPU work fixed); strong: the gx x gy ensemble is split by rows."""
    if scaling == "weak":
        if not (0 <= rank < world):
            raise ValueError("rank out of range")
        return gx, gy * world, rank * gx * gy, gx * gy
    if scaling != "strong":
        raise ValueError("scaling must be 'weak' or 'strong'")
    j0, j1 = shard_rows(gy, world, rank)
    return gx, gy, j0 * gx, (j1 - j0) * gx


def _active():
    return dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1


def allreduce_hist(hist):
    """In-place sum of the uint32 histogram over all ranks.  The tensor holds the uint32 bits as int32;
    two's-complement addition is the same bit pattern as unsigned addition mod 2^32."""
    if _active():
        dist.all_reduce(hist, op=dist.ReduceOp.SUM)
    return hist


def gather_image(local, counts, dst=0):
    """Concatenate the per-rank image slices (1-D tensors of counts[r] elements, any dtype) in rank order on `dst`
    (returns None elsewhere).  One collective on the tensors where they live: NCCL gather on device tensors (gloo on
    CPU tensors); ragged slices are padded to the longest one for the collective and trimmed afterwards."""
    if not _active():
        return local
    world, rank = dist.get_world_size(), dist.get_rank()
    if len(counts) != world or local.numel() != counts[rank]:
        raise ValueError("counts must list every rank's slice length")
    longest = max(counts)
    send = local.contiguous()
    if send.numel() < longest:
        send = torch.cat([send, send.new_zeros(longest - send.numel())])
    parts = [torch.empty(longest, dtype=local.dtype, device=local.device) for _ in range(world)] \
        if rank == dst else None
    dist.gather(send, parts, dst=dst)
    if rank != dst:
        return None
    return torch.cat([p[:c] for p, c in zip(parts, counts)])
