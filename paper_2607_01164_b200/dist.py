"""Multi-GPU plumbing of the hot path (one process per GPU, torch.distributed).

The path shards by SAMPLES: every rank holds the whole model and processes its own batch of query
points (a brick range of the grid, or a slice of the point list); the forward needs no exchange and
the backward needs exactly one: the sum over ranks of the per-Gaussian gradients (DESIGN.md
"Multi-GPU").  Nothing here computes anything of the method; it splits work and calls all_reduce.
"""
from __future__ import annotations

GRAD_KEYS = ("dmean", "dscale", "dquat", "dopacity", "dscalar", "err")


def shard_bricks(brick_cnt, rank: int, world: int):
    """Split a grid's bricks into `world` contiguous z-slabs (brick-aligned batches).
    Returns (brick_lo, brick_cnt) of this rank's batch; the count along z may be 0 for trailing ranks."""
    nz = int(brick_cnt[2])
    per = (nz + world - 1) // world
    z0 = min(rank * per, nz)
    z1 = min(z0 + per, nz)
    return (0, 0, z0), (int(brick_cnt[0]), int(brick_cnt[1]), z1 - z0)


def shard_points(num_points: int, rank: int, world: int):
    """Contiguous slice [lo, hi) of the point list owned by this rank (sizes differ by at most one)."""
    base, rem = divmod(int(num_points), world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def allreduce_grads(grads: dict, flat=None):
    """Sum the gradient tensors over all ranks, in place, with ONE collective on a flat staging buffer.
    `flat` (optional) is a preallocated 1-D float32 tensor of at least sum(numel) elements."""
    import torch
    import torch.distributed as dist

    keys = [k for k in GRAD_KEYS if grads.get(k) is not None]
    total = sum(grads[k].numel() for k in keys)
    if flat is None or flat.numel() < total:
        flat = torch.empty(total, dtype=torch.float32, device=grads[keys[0]].device)
    off = 0
    for k in keys:
        n = grads[k].numel()
        flat[off:off + n].copy_(grads[k].reshape(-1))
        off += n
    dist.all_reduce(flat[:total], op=dist.ReduceOp.SUM)
    off = 0
    for k in keys:
        n = grads[k].numel()
        grads[k].reshape(-1).copy_(flat[off:off + n])
        off += n
    return grads
