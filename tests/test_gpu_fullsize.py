"""-m gpu parity at BASELINE.json's full size, in the launch configuration bench.py times:
configs[1] (C2): 256^3 Marschner-Lobb grid, 262,144 Gaussians, one whole-grid forward+backward.
The oracle finishes this size in seconds (cell-grid cull, OpenMP), so every output is compared element
by element: all 16.8 M intersection sets and the 2.56 M sorted pair keys bit-exact, Phi within 1e-5,
every gradient tensor within 1e-4 relative L2.
configs[2] (C3) is checked the same way on one 2^20-point batch (the oracle needs about a minute for it).
configs[3] (C4): the full 4,194,304-Gaussian model, two 128^3 brick-aligned batches of the 1024^3 grid with one
gs_preprocess; configs[4] (C5): the full 8,388,608-Gaussian model, one 2^24-point batch -- forward AND backward, every
output element against oracle mode 1 (whose cost is proportional to the hit pairs: ~5e6 and ~3e8)."""
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


class _Shim:
    """What gpu_util.check_* need of a run, for flows that are not one GpuRun (several batches per preprocess)."""

    def __init__(self, ctx, q, P, phi, I, grads):
        self.ctx, self.q, self.P, self.phi, self.I, self.grads = ctx, q, P, phi, I, grads

    def np(self, t):
        return t.detach().cpu().numpy()[: self.P]

    def grads_np(self):
        return {k: v.detach().cpu().numpy().astype(np.float64) for k, v in self.grads.items()}

    def sets(self):
        return self.ctx.debug_point_sets(self.q)


def test_c4_full_batch(oracle):
    # BASELINE.json configs[3] at its stated size: 4,194,304 Gaussians (5 % needles of axis ratio 20:1) on a 1024^3 grid,
    # decoded in 128^3 brick-aligned batches (16^3 bricks) with ONE gs_preprocess: an interior batch and the upper corner
    import torch
    from paper_2607_01164_b200 import api
    field = inputs.c4_field(seed=4)
    g = inputs.c4_gaussians(seed=4, n_grid=1024, n=4_194_304, field=field)
    full = inputs.c4_grid(1024)
    ctx = api.Context()
    dev = [torch.from_numpy(x).cuda() for x in (g.mean, g.scale, g.quat, g.opacity, g.scalar)]
    ctx.gs_preprocess(*dev)
    M, aabb, valid = oracle.preprocess_f32(g, TAU)
    assert np.array_equal(ctx.debug_get(api.DBG_AABB, np.float32, 6).view(np.uint32), aabb.view(np.uint32))
    grads = ctx.alloc_grads(g.n)
    for lo in ((48, 48, 48), (112, 112, 112)):
        batch = full.batch(lo, (16, 16, 16))
        P = batch.num_points
        assert P == 128 ** 3
        target = inputs.c4_target(batch, field)
        xyz = oracle.grid_points(batch)
        fwd = oracle.forward(g, xyz, TAU, mode=1)
        loss, a, serr = oracle.mse(fwd["phi"], fwd["I"], target, TAU)
        gr = oracle.backward(g, xyz, fwd["phi"], fwd["I"], a, None, target, TAU, mode=1)
        q = api.grid_query(batch)
        ctx.gs_build_accel(q)
        # integer stage: the sorted (brick, gaussian) keys of this batch
        blo, bhi, cnt = oracle.brick_ranges(aabb, valid, batch)
        keys, start = oracle.brick_keys(blo, bhi, cnt, batch)
        pb = ctx.debug_get(api.DBG_PAIR_BRICK, np.uint32)
        pg = ctx.debug_get(api.DBG_PAIR_GAUSS, np.uint32)
        assert len(keys) > 50_000
        assert np.array_equal((pb.astype(np.uint64) << np.uint64(32)) | pg.astype(np.uint64), keys)
        assert np.array_equal(ctx.debug_get(api.DBG_BRICK_START, np.uint32).astype(np.int64), start)
        phi = torch.full((P,), -7.0, device="cuda")
        I = torch.full((P,), -7.0, device="cuda")
        dphi = torch.full((P,), -7.0, device="cuda")
        lossd = torch.zeros(1, dtype=torch.float64, device="cuda")
        t = torch.from_numpy(target).cuda()
        ctx.gs_sample_fwd(q, phi, I, target=t, loss=lossd, dL_dphi=dphi)
        for v in grads.values():
            v.fill_(-7.0)
        ctx.gs_sample_bwd(q, None, None, None, grads)   # backward of the fused MSE (what bench.py times)
        torch.cuda.synchronize()
        run = _Shim(ctx, q, P, phi, I, grads)
        tested, hits = check_sets(run, fwd)
        assert hits > 3_000_000
        near, e_phi, e_I = check_forward(run, fwd)
        assert near <= 16
        assert float(lossd.item()) == pytest.approx(loss, rel=1e-6)
        errs = check_grads(run, gr)
        # the general backward (explicit dL/dPhi array) on the same batch
        for v in grads.values():
            v.fill_(-7.0)
        ctx.gs_sample_bwd(q, phi, I, dphi, grads, target=t)
        torch.cuda.synchronize()
        errs2 = check_grads(run, gr)
        print("C4 batch", lo, "T", len(keys), "hits", hits, "tested", tested, "phi err", e_phi, "grad errs", errs, errs2)
    ctx.close()


_C5 = {}


def _c5_pool():
    """configs[4] as BASELINE.json states it: the 200,000,000-point set (2.4 GB of positions, drawn once per test session by
    a pool of threads) and the 8,388,608 Gaussians centred on points of THAT set."""
    if not _C5:
        xyz_all, t_all = inputs.c5_points(seed=5)
        assert len(xyz_all) == 200_000_000
        _C5.update(xyz=xyz_all, t=t_all, g=inputs.c5_gaussians(xyz_all, t_all), dom=inputs.points_domain(xyz_all))
    return _C5["xyz"], _C5["t"], _C5["g"], _C5["dom"]


def test_c5_full_batch(oracle):
    # BASELINE.json configs[4] at its stated size: 8,388,608 Gaussians (sigma 0.0005-0.002) centred on points of the
    # shell-and-fragments distribution; one batch of 2^24 random points of the 200 M-point set, forward + backward; LBVH,
    # query sort and cull lists rebuilt by gs_build_accel
    xyz_all, t_all, g, dom = _c5_pool()
    assert g.n == 8_388_608
    idx = inputs.batch_indices(5, 0, len(xyz_all), 1 << 24)
    xyz, target = np.ascontiguousarray(xyz_all[idx]), np.ascontiguousarray(t_all[idx])
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
    tested, hits = check_sets(run, fwd)   # all 2^24 intersection sets, bit-exact
    assert hits > 200_000_000
    near, e_phi, e_I = check_forward(run, fwd)
    assert near <= 64
    assert float(run.loss.item()) == pytest.approx(loss, rel=1e-6)
    errs = check_grads(run, gr)
    got = run.grads_np()
    covered = fwd["I"].astype(np.float32) > np.float32(TAU)
    assert got["dscalar"].sum() == pytest.approx(a[covered].sum(), rel=1e-4, abs=1e-7)
    assert got["err"].sum() == pytest.approx(serr[covered].sum(), rel=1e-4)
    print("C5 full batch: hits", hits, "tested", tested, "phi err", e_phi, "grad errs", errs)


def test_c5_decode_first_and_last_chunk(oracle):
    # configs[4]'s "full forward decode of all points": the 200 M points go through the sampler in 12 chunks of <= 2^24 in
    # set order, after ONE gs_preprocess -- the first gs_build_accel builds the LBVH over the Gaussians, the later ones reuse it
    # and only sort and cull their own points.  The first and the last chunk (ragged: 15,450,624 points) are compared with the
    # oracle, every intersection set and every value; bench.py times all twelve.
    import torch
    from paper_2607_01164_b200 import api
    xyz_all, t_all, g, dom = _c5_pool()
    chunk = 1 << 24
    starts = list(range(0, len(xyz_all), chunk))
    assert len(starts) == 12 and len(xyz_all) - starts[-1] == 15_450_624
    ctx = api.Context()
    dev = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (g.mean, g.scale, g.quat, g.opacity, g.scalar)]
    ctx.gs_preprocess(*dev, domain=dom, tau=TAU)
    for a in (starts[0], starts[-1]):
        xyz = np.ascontiguousarray(xyz_all[a:a + chunk])
        P = len(xyz)
        fwd = oracle.forward(g, xyz, TAU, mode=1)
        x = torch.from_numpy(xyz).cuda()
        q = api.points_query(x)
        ctx.gs_build_accel(q)
        phi, I = torch.full((P,), -7.0, device="cuda"), torch.full((P,), -7.0, device="cuda")
        ctx.gs_sample_fwd(q, phi, I)
        torch.cuda.synchronize()
        run = _Shim(ctx, q, P, phi, I, None)
        tested, hits = check_sets(run, fwd)
        assert hits > 10 * P
        near, e_phi, e_I = check_forward(run, fwd)
        assert near <= 64
        print("C5 decode chunk at", a, "P", P, "hits", hits, "tested", tested, "phi err", e_phi, "I err", e_I)
        del x, phi, I
    ctx.close()
