"""-m gpu parity at BASELINE.json's full size, in the launch configuration bench.py times:
configs[1] (C2): 256^3 Marschner-Lobb grid, 262,144 Gaussians, one whole-grid forward+backward.
The oracle finishes this size in seconds (cell-grid cull, OpenMP), so every output is compared element
by element: all 16.8 M intersection sets and the 2.56 M sorted pair keys bit-exact, Phi within 1e-5,
every gradient tensor within 1e-4 relative L2.
configs[2] (C3) is checked the same way on one 2^20-point batch (the oracle needs about a minute for it)."""
import numpy as np
import pytest

from paper_2607_01164_b200 import inputs
from gpu_util import TAU, GpuRun, check_forward, check_grads, check_sets

pytestmark = pytest.mark.gpu


def test_c2_full_size(oracle):
    grid = inputs.c2_grid(256)
    g = inputs.c2_gaussians(seed=2, n_grid=256, n=262144)
    target = inputs.c2_target(grid)
    xyz = oracle.grid_points(grid)
    fwd = oracle.forward(g, xyz, TAU, mode=1)
    loss, a, serr = oracle.mse(fwd["phi"], fwd["I"], target, TAU)
    gr = oracle.backward(g, xyz, fwd["phi"], fwd["I"], a, None, target, TAU, mode=1)
    run = GpuRun(g, "grid", grid, target)
    api = run.api
    # integer stages
    M, aabb, valid = oracle.preprocess_f32(g, TAU)
    assert np.array_equal(run.ctx.debug_get(api.DBG_AABB, np.float32, 6).view(np.uint32), aabb.view(np.uint32))
    blo, bhi, cnt = oracle.brick_ranges(aabb, valid, grid)
    keys, start = oracle.brick_keys(blo, bhi, cnt, grid)
    pb = run.ctx.debug_get(api.DBG_PAIR_BRICK, np.uint32)
    pg = run.ctx.debug_get(api.DBG_PAIR_GAUSS, np.uint32)
    assert len(keys) > 2_000_000
    assert np.array_equal((pb.astype(np.uint64) << np.uint64(32)) | pg.astype(np.uint64), keys)
    assert np.array_equal(run.ctx.debug_get(api.DBG_BRICK_START, np.uint32).astype(np.int64), start)
    tested, hits = check_sets(run, fwd)
    assert hits > 90_000_000
    # values
    near, e_phi, e_I = check_forward(run, fwd)
    assert near <= 16  # samples whose I sits within rounding of tau (excluded from the Phi comparison)
    assert float(run.loss.item()) == pytest.approx(loss, rel=1e-6)
    errs = check_grads(run, gr)
    # properties that hold at any size (sum rules of Eq. 2)
    got = run.grads_np()
    covered = fwd["I"].astype(np.float32) > np.float32(TAU)
    assert got["dscalar"].sum() == pytest.approx(a[covered].sum(), rel=1e-4, abs=1e-7)
    assert got["err"].sum() == pytest.approx(serr[covered].sum(), rel=1e-4)
    print("C2 full size: T", len(keys), "hits", hits, "tested", tested, "phi err", e_phi, "grad errs", errs)


def test_c3_full_size(oracle):
    # BASELINE.json configs[2] at full size: 2,000,000 points, 1,048,576 Gaussians, one 2^20-point batch without
    # replacement, LBVH + query sort + cull lists rebuilt by gs_build_accel (what `bench.py --workload c3` times)
    xyz_all, t_all = inputs.c3_points()
    g = inputs.c3_gaussians(xyz_all, t_all)
    idx = inputs.batch_indices(3, 0, len(xyz_all), 1 << 20)
    xyz, target = np.ascontiguousarray(xyz_all[idx]), np.ascontiguousarray(t_all[idx])
    dom = inputs.points_domain(xyz_all)
    fwd = oracle.forward(g, xyz, TAU, mode=1)
    loss, a, serr = oracle.mse(fwd["phi"], fwd["I"], target, TAU)
    gr = oracle.backward(g, xyz, fwd["phi"], fwd["I"], a, None, target, TAU, mode=1)
    run = GpuRun(g, "points", xyz, target, domain=dom, fused=True)
    api = run.api
    M, aabb, valid = oracle.preprocess_f32(g, TAU)
    codes = oracle.morton_codes(g.mean, dom[0], dom[1], valid)
    order, keys = oracle.morton_order(codes)
    assert np.array_equal(run.ctx.debug_get(api.DBG_LEAF_MORTON, np.uint32), codes[order])
    assert np.array_equal(run.ctx.debug_get(api.DBG_LEAF_ORDER, np.uint32), order)
    pcodes = oracle.morton_codes(xyz, dom[0], dom[1])
    porder, _ = oracle.morton_order(pcodes)
    assert np.array_equal(run.ctx.debug_get(api.DBG_POINT_ORDER, np.uint32), porder)
    tested, hits = check_sets(run, fwd)   # all 2^20 intersection sets, bit-exact
    assert hits > 400_000_000
    near, e_phi, e_I = check_forward(run, fwd)
    assert near <= 16
    assert float(run.loss.item()) == pytest.approx(loss, rel=1e-6)
    errs = check_grads(run, gr)
    got = run.grads_np()
    covered = fwd["I"].astype(np.float32) > np.float32(TAU)
    assert got["dscalar"].sum() == pytest.approx(a[covered].sum(), rel=1e-4, abs=1e-7)
    assert got["err"].sum() == pytest.approx(serr[covered].sum(), rel=1e-4)
    print("C3 full size: hits", hits, "tested", tested, "phi err", e_phi, "grad errs", errs)


def test_c4_like_batches(oracle):
    # configs[3] shape at reduced size: a 64^3 grid decoded in two brick-aligned batches with one preprocess;
    # anisotropic model with 5 % needles; the second batch re-uses the records (gs_build_accel repeated)
    import torch
    from paper_2607_01164_b200 import api
    n_grid = 64
    field = inputs.c4_field(seed=4)
    g = inputs.c4_gaussians(seed=4, n_grid=n_grid, n=16384, field=field)
    full = inputs.c4_grid(n_grid)
    ctx = api.Context()
    dev = [torch.from_numpy(x).cuda() for x in (g.mean, g.scale, g.quat, g.opacity, g.scalar)]
    ctx.gs_preprocess(*dev)
    for lo, cnt in (((0, 0, 0), (8, 8, 4)), ((0, 0, 4), (8, 8, 4))):
        batch = full.batch(lo, cnt)
        q = api.grid_query(batch)
        ctx.gs_build_accel(q)
        P = batch.num_points
        phi = torch.empty(P, device="cuda")
        I = torch.empty(P, device="cuda")
        ctx.gs_sample_fwd(q, phi, I)  # forward-only decode
        xyz = oracle.grid_points(batch)
        ref = oracle.forward(g, xyz, TAU, mode=1)
        cnt_, hs, hx, tested, hits = ctx.debug_point_sets(q)
        assert np.array_equal(cnt_, ref["count"]) and np.array_equal(hs, ref["hsum"]) and np.array_equal(hx, ref["hxor"])
        near = np.abs(ref["I"] - TAU) <= 2e-6 * TAU
        assert np.abs(phi.cpu().numpy() - ref["phi"])[~near].max() <= 1e-5
    ctx.close()
