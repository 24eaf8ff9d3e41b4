"""Batch sharding of the LETKF local analysis across GPUs.

Every grid point is an independent local problem (Procedure 3 line 5,
PAPER.md:256), so the path shards with NO data-path collective: rank g owns the contiguous batch
slice [g*B/G, (g+1)*B/G) -- the paper's n_x in [m*Nx/M, (m+1)*Nx/M).  This module holds only the
host logic (slice bounds, gather of per-rank results for checking); the per-rank compute is one
call of the C-ABI library on the rank's slice.  torch.distributed is used for plumbing only.
"""
import torch
import torch.distributed as dist


def shard_bounds(batch, world_size, rank):
    """[lo, hi) of rank's contiguous slice; sizes differ by at most one, low ranks get the extra."""
    if world_size < 1 or not 0 <= rank < world_size or batch < 0:
        raise ValueError("bad (batch, world_size, rank)")
    q, r = divmod(batch, world_size)
    lo = rank * q + min(rank, r)
    return lo, lo + q + (1 if rank < r else 0)


def all_bounds(batch, world_size):
    return [shard_bounds(batch, world_size, g) for g in range(world_size)]


def local_slice(t, world_size, rank):
    """The rank's view (no copy) of a batch-outermost tensor."""
    lo, hi = shard_bounds(t.shape[0], world_size, rank)
    return t[lo:hi]


def gather_batch(local, batch, group=None):
    """all_gather of ragged per-rank slices back into [batch, ...] order (checking / output
    assembly; not on the timed path).  Works with gloo (CPU tensors) and nccl (CUDA tensors)."""
    world = dist.get_world_size(group)
    bounds = all_bounds(batch, world)
    cap = max(hi - lo for lo, hi in bounds)
    pad = torch.zeros((cap,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    pad[: local.shape[0]] = local
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad, group=group)
    return torch.cat([parts[g][: hi - lo] for g, (lo, hi) in enumerate(bounds)], dim=0)


def max_over_ranks(value, device=None, group=None):
    """Max of a python float over the ranks (device-side timing: the slowest rank counts)."""
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())
