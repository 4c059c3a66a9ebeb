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


GRAD_COLS = dict(dmean=3, dscale=3, dquat=4, dopacity=1, dscalar=1, err=1)


def flat_layout(n: int):
    """Offsets (in floats) of the six gradient tensors of n Gaussians inside one flat buffer; every section starts on a
    multiple of 4 floats (16 bytes: gs_grads.dquat needs it).  Returns ({name: (offset, columns)}, total floats)."""
    off, o = {}, 0
    for k in GRAD_KEYS:
        off[k] = (o, GRAD_COLS[k])
        o += (n * GRAD_COLS[k] + 3) // 4 * 4
    return off, o


def allreduce_grads(grads: dict, loss=None):
    """Sum the gradient tensors (and, if given, the loss scalar) over all ranks, in place.  With grads["flat"] (see
    api.Context.alloc_grads(flat=True)) the six tensors are views of one buffer and the exchange is ONE collective with no
    packing; otherwise they are packed into a staging buffer first."""
    import torch
    import torch.distributed as dist

    if grads.get("flat") is not None:
        dist.all_reduce(grads["flat"], op=dist.ReduceOp.SUM)
    else:
        keys = [k for k in GRAD_KEYS if grads.get(k) is not None]
        flat = torch.cat([grads[k].reshape(-1) for k in keys])
        dist.all_reduce(flat, op=dist.ReduceOp.SUM)
        o = 0
        for k in keys:
            n = grads[k].numel()
            grads[k].reshape(-1).copy_(flat[o:o + n])
            o += n
    if loss is not None:
        dist.all_reduce(loss, op=dist.ReduceOp.SUM)
    return grads
