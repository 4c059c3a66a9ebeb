"""World-size-2 gloo tests (CPU) of the multi-GPU plumbing: sample sharding and the one gradient all-reduce.
The oracle shows that gradients are additive over disjoint sample shards, which is what makes the
data-parallel split of the path exact."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2607_01164_b200 import dist as gsdist
from paper_2607_01164_b200 import inputs


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    n = 37
    rng = np.random.default_rng(rank)
    grads = {k: torch.from_numpy(rng.standard_normal((n, c) if c > 1 else n).astype(np.float32))
             for k, c in (("dmean", 3), ("dscale", 3), ("dquat", 4), ("dopacity", 1), ("dscalar", 1), ("err", 1))}
    mine = {k: v.clone() for k, v in grads.items()}
    gsdist.allreduce_grads(grads)
    # reference: gather everyone's local tensors and add
    for k in grads:
        parts = [torch.empty_like(mine[k]) for _ in range(world)]
        dist.all_gather(parts, mine[k])
        assert torch.allclose(grads[k], sum(parts), atol=1e-6), k
    lo, hi = gsdist.shard_points(1001, rank, world)
    t = torch.tensor([hi - lo], dtype=torch.int64)
    dist.all_reduce(t)
    assert int(t.item()) == 1001
    out.put((rank, lo, hi))
    dist.destroy_process_group()


def test_allreduce_and_sharding_world2():
    ctxm = mp.get_context("spawn")
    q = ctxm.Queue()
    port = _free_port()
    procs = [ctxm.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    got = sorted(q.get(timeout=5) for _ in range(2))
    assert got[0][1] == 0 and got[0][2] == got[1][1] and got[1][2] == 1001


def test_brick_shards_cover_grid():
    for world in (1, 2, 3, 8):
        cnt = (4, 5, 7)
        seen = []
        for r in range(world):
            lo, c = gsdist.shard_bricks(cnt, r, world)
            assert lo[:2] == (0, 0) and c[:2] == cnt[:2]
            seen += list(range(lo[2], lo[2] + c[2]))
        assert seen == list(range(cnt[2]))


def test_gradients_add_over_sample_shards(oracle):
    # the exchange step is a plain sum: oracle gradients over two disjoint shards add up to the full-batch ones
    g = inputs.c1_gaussians(seed=0, n=256)
    xyz = oracle.grid_points(inputs.c1_grid(16))
    rng = np.random.default_rng(0)
    target = rng.uniform(0, 1, len(xyz)).astype(np.float32)
    fwd = oracle.forward(g, xyz, 0.01, mode=1)
    _, a, _ = oracle.mse(fwd["phi"], fwd["I"], target, 0.01)
    full = oracle.backward(g, xyz, fwd["phi"], fwd["I"], a, None, target, 0.01, mode=1)
    parts = []
    for r in range(2):
        lo, hi = gsdist.shard_points(len(xyz), r, 2)
        parts.append(oracle.backward(g, xyz[lo:hi], fwd["phi"][lo:hi], fwd["I"][lo:hi], a[lo:hi], None, target[lo:hi], 0.01, mode=1))
    for k in full:
        np.testing.assert_allclose(parts[0][k] + parts[1][k], full[k], rtol=1e-9, atol=1e-15)


def _bench_worker(rank, world, port, out):
    """bench.py's N > 1 arm on CPU: its own sharding function, the oracle in place of the CUDA library, the flat gradient
    buffer and allreduce_grads over gloo.  Every rank holds the same model; the loss mean runs over the GLOBAL sample count."""
    import bench
    from oracle import wveg_oracle as oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    res = {}
    for kind in ("grid", "points"):
        g = inputs.c1_gaussians(seed=0, n=300)
        if kind == "grid":
            grid = inputs.Grid((24, 20, 28), (0.0, 0.0, 0.0), (1 / 24, 1 / 24, 1 / 28))
            target = np.random.default_rng(1).uniform(0, 1, grid.num_points).astype(np.float32)
            wl = dict(name="t", kind="grid", g=g, grid=grid, target=target)
        else:
            xyz = np.random.default_rng(2).uniform(0, 1, (3001, 3)).astype(np.float32)
            target = np.random.default_rng(3).uniform(0, 1, 3001).astype(np.float32)
            wl = dict(name="t", kind="points", g=g, batches=[(xyz, target)])
        shards, P_total = bench.shard_workload(wl, rank, world)
        off, total = gsdist.flat_layout(g.n)
        flat = torch.zeros(total, dtype=torch.float32)
        grads = {k: flat[o:o + g.n * c].view((g.n, c) if c > 1 else (g.n,)) for k, (o, c) in off.items()}
        grads["flat"] = flat
        loss = torch.zeros(1, dtype=torch.float64)
        npts = 0
        for s in shards:
            pts = oracle.grid_points(s["grid"]) if kind == "grid" else s["xyz"]
            npts += len(pts)
            fwd = oracle.forward(g, pts, 0.01, mode=1)
            res_ = fwd["phi"] - s["target"]
            covered = fwd["I"].astype(np.float32) > np.float32(0.01)
            a = np.where(covered, 2.0 * res_ / P_total, 0.0)     # what gs_set_sample_count(P_total) makes the fused MSE do
            loss += float((res_ ** 2).sum() / P_total)
            gr = oracle.backward(g, pts, fwd["phi"], fwd["I"], a, None, s["target"], 0.01, mode=1)
            for k, v in gr.items():
                grads[k] += torch.from_numpy(v.astype(np.float32)).view(grads[k].shape)
        gsdist.allreduce_grads(grads, loss)
        cnt = torch.tensor([npts], dtype=torch.int64)
        dist.all_reduce(cnt)
        assert int(cnt.item()) == P_total
        res[kind] = ({k: grads[k].numpy().copy() for k in gsdist.GRAD_KEYS}, float(loss.item()))
    out.put((rank, res))
    dist.destroy_process_group()


def test_bench_sharding_dry_run_world2(oracle):
    ctxm = mp.get_context("spawn")
    q = ctxm.Queue()
    port = _free_port()
    procs = [ctxm.Process(target=_bench_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = dict(q.get(timeout=240) for _ in range(2))
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    # one-batch reference
    g = inputs.c1_gaussians(seed=0, n=300)
    grid = inputs.Grid((24, 20, 28), (0.0, 0.0, 0.0), (1 / 24, 1 / 24, 1 / 28))
    cases = {"grid": (oracle.grid_points(grid), np.random.default_rng(1).uniform(0, 1, grid.num_points).astype(np.float32)),
             "points": (np.random.default_rng(2).uniform(0, 1, (3001, 3)).astype(np.float32),
                        np.random.default_rng(3).uniform(0, 1, 3001).astype(np.float32))}
    for kind, (pts, target) in cases.items():
        fwd = oracle.forward(g, pts, 0.01, mode=1)
        loss, a, _ = oracle.mse(fwd["phi"], fwd["I"], target, 0.01)
        full = oracle.backward(g, pts, fwd["phi"], fwd["I"], a, None, target, 0.01, mode=1)
        for r in range(2):   # both ranks hold the all-reduced result
            grads, l = got[r][kind]
            assert l == pytest.approx(loss, rel=1e-9)
            for k, v in full.items():
                np.testing.assert_allclose(grads[k].reshape(v.shape), v, rtol=2e-4, atol=1e-6 * np.abs(v).max())
