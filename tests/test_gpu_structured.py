"""-m gpu parity: structured path (S1, S2, S4, S6, S7, S8) through the C ABI vs the oracle.

Bar (BASELINE.json north_star): integer stages bit-exact (AABB / records feed them, so those are
compared bit-exactly too), per-point intersection ID sets bit-exact, forward max abs error <= 1e-5
of the scalar range, gradient relative L2 error <= 1e-4 per parameter tensor.
"""
import numpy as np
import pytest

from paper_2607_01164_b200 import inputs
from gpu_util import TAU, GpuRun, check_forward, check_grads, check_sets

pytestmark = pytest.mark.gpu


def _oracle_all(oracle, g, grid, target, dL_dI=None):
    xyz = oracle.grid_points(grid)
    fwd = oracle.forward(g, xyz, TAU, mode=1)
    loss, a, serr = oracle.mse(fwd["phi"], fwd["I"], target, TAU)
    gr = oracle.backward(g, xyz, fwd["phi"], fwd["I"], a, dL_dI, target, TAU, mode=1)
    return xyz, fwd, loss, a, serr, gr


def _check_integer_stages(oracle, run, g, grid):
    api = run.api
    M, aabb, valid = oracle.preprocess_f32(g, TAU)
    rec = run.ctx.debug_get(api.DBG_RECORDS, np.float32, 16).reshape(4, g.n, 4)  # float4 planes [4][N]
    gaabb = run.ctx.debug_get(api.DBG_AABB, np.float32, 6)
    v = valid.astype(bool)
    assert np.array_equal(gaabb.view(np.uint32), aabb.view(np.uint32)), "AABBs are not bit-exact"
    gM = np.concatenate([rec[1][:, :3], rec[2][:, :3], rec[3][:, :3]], axis=1)
    assert np.array_equal(gM[v].view(np.uint32), M[v].view(np.uint32)), "whitening matrices are not bit-exact"
    assert np.array_equal(rec[0][v, :3], g.mean[v]) and np.array_equal(rec[0][v, 3], g.opacity[v]) and np.array_equal(rec[1][v, 3], g.scalar[v])
    assert np.all(np.isnan(rec[0][~v, 0]))
    blo, bhi, cnt = oracle.brick_ranges(aabb, valid, grid)
    keys, start = oracle.brick_keys(blo, bhi, cnt, grid)
    assert np.array_equal(run.ctx.debug_get(api.DBG_BRICK_COUNT, np.uint32), cnt)
    pb = run.ctx.debug_get(api.DBG_PAIR_BRICK, np.uint32)
    pg = run.ctx.debug_get(api.DBG_PAIR_GAUSS, np.uint32)
    gkeys = (pb.astype(np.uint64) << np.uint64(32)) | pg.astype(np.uint64)
    assert np.array_equal(gkeys, keys), "sorted (brick, gaussian) keys differ"
    assert np.array_equal(run.ctx.debug_get(api.DBG_BRICK_START, np.uint32).astype(np.int64), start)
    return len(keys)


def test_c1_tiny_structured_full(oracle):
    # BASELINE.json configs[0]: 1,024 Gaussians, 32^3 voxel-centre grid, target from a second seeded set
    g = inputs.c1_gaussians(seed=0, n=1024)
    grid = inputs.c1_grid(32)
    g2 = inputs.c1_gaussians(seed=1, n=1024)
    xyz = oracle.grid_points(grid)
    target = oracle.forward(g2, xyz, TAU, mode=1, want_sets=False)["phi"].astype(np.float32)
    xyz, fwd, loss, a, serr, gr = _oracle_all(oracle, g, grid, target)
    run = GpuRun(g, "grid", grid, target)
    T = _check_integer_stages(oracle, run, g, grid)
    assert T > 1024
    tested, hits = check_sets(run, fwd)
    assert hits > 40000 and (fwd["count"] == 0).sum() > 1000  # exercises the empty path
    near, e_phi, e_I = check_forward(run, fwd)
    assert near == 0
    assert float(run.loss.item()) == pytest.approx(loss, rel=1e-6)
    np.testing.assert_allclose(run.np(run.dphi), a, rtol=2e-5, atol=2e-5 / len(a))  # dL/dPhi = 2 res / P, |d res| <= 1e-5
    np.testing.assert_allclose(run.np(run.serr), serr, atol=1e-5)
    check_grads(run, gr)


def test_ragged_batch_anisotropic(oracle):
    # grid whose dims are not multiples of 8, sampled in a sub-box batch; 20:1 elongated Gaussians; dL/dI present
    gridfull = inputs.Grid((44, 29, 21), (-0.1, 0.2, 0.0), (1 / 40, 1 / 32, 1 / 20))
    g = inputs.c4_gaussians(seed=7, n_grid=40, n=3000)
    g.quat[:] = (g.quat * np.random.default_rng(1).uniform(0.3, 3.0, (g.n, 1))).astype(np.float32)  # non-unit quaternions
    rng = np.random.default_rng(3)
    for grid in (gridfull, gridfull.batch((1, 1, 0), (3, 3, 3)), gridfull.batch((5, 3, 2), (1, 1, 1))):
        P = grid.num_points
        target = rng.uniform(0, 1, P).astype(np.float32)
        dI = rng.standard_normal(P) * 1e-3
        xyz, fwd, loss, a, serr, gr = _oracle_all(oracle, g, grid, target, dI)
        run = GpuRun(g, "grid", grid, target, dL_dI=dI.astype(np.float32))
        _check_integer_stages(oracle, run, g, grid)
        check_sets(run, fwd)
        check_forward(run, fwd)
        assert float(run.loss.item()) == pytest.approx(loss, rel=1e-6)
        check_grads(run, gr)


def test_invalid_empty_and_degenerate(oracle):
    import torch
    from paper_2607_01164_b200 import api
    grid = inputs.c1_grid(16)
    g = inputs.c1_gaussians(seed=4, n=200)
    g.scale[0, 1] = 0.0
    g.quat[1] = 0.0
    g.mean[2, 0] = np.nan
    g.opacity[3] = np.inf
    g.scale[4] = -1.0
    target = np.full(grid.num_points, 0.5, np.float32)
    xyz, fwd, loss, a, serr, gr = _oracle_all(oracle, g, grid, target)
    run = GpuRun(g, "grid", grid, target)
    _check_integer_stages(oracle, run, g, grid)
    check_sets(run, fwd)
    check_forward(run, fwd)
    check_grads(run, gr)
    got = run.grads_np()
    for k in got:
        assert np.all(got[k][:5] == 0.0), k  # invalid Gaussians receive zero gradient
    # a model that covers nothing: every sample takes the empty value, loss = mean(t^2), no gradient
    far = inputs.c1_gaussians(seed=5, n=8)
    far.mean[:] += 10.0
    run = GpuRun(far, "grid", grid, target)
    assert np.all(run.np(run.phi) == 0.0) and np.all(run.np(run.I) == 0.0) and np.all(run.np(run.dphi) == 0.0)
    assert float(run.loss.item()) == pytest.approx(0.25, rel=1e-6)
    assert all(np.all(v == 0.0) for v in run.grads_np().values())
    # N = 0
    empty = far.subset(np.arange(0))
    run = GpuRun(empty, "grid", grid, target)
    assert np.all(run.np(run.phi) == 0.0) and float(run.loss.item()) == pytest.approx(0.25, rel=1e-6)
    # single Gaussian at a voxel centre: contribution at its mean is exactly w (Eq. 3, G(mu) = 1)
    one = inputs.Gaussians(np.array([[0.53125, 0.46875, 0.59375]], np.float32), np.array([[0.05, 0.02, 0.09]], np.float32),
                           np.array([[0.2, -0.4, 0.1, 0.7]], np.float32), np.array([0.75], np.float32), np.array([0.3], np.float32))
    run = GpuRun(one, "grid", grid, target)
    c = (9 * 16 + 7) * 16 + 8
    assert run.np(run.I)[c] == np.float32(0.75) and abs(run.np(run.phi)[c] - np.float32(0.3)) < 1e-7
    # error handling: calls out of order / bad arguments
    ctx = api.Context()
    q = api.grid_query(grid)
    with pytest.raises(api.GsError) as ei:
        ctx.gs_build_accel(q)
    assert ei.value.status == api.GS_ERR_STATE
    dev = [torch.from_numpy(x).cuda() for x in (g.mean, g.scale, g.quat, g.opacity, g.scalar)]
    with pytest.raises(api.GsError) as ei:
        ctx.gs_preprocess(*dev, tau=1.5)
    assert ei.value.status == api.GS_ERR_INVALID_ARG
    ctx.gs_preprocess(*dev)
    phi = torch.zeros(grid.num_points, device="cuda")
    with pytest.raises(api.GsError) as ei:
        ctx.gs_sample_fwd(q, phi, phi.clone())
    assert ei.value.status == api.GS_ERR_STATE
    bad = api.grid_query(inputs.Grid((16, 16, 16), (0, 0, 0), (1 / 16,) * 3, (1, 0, 0), (2, 2, 2)))
    with pytest.raises(api.GsError) as ei:
        ctx.gs_build_accel(bad)
    assert ei.value.status == api.GS_ERR_INVALID_ARG
    ctx.close()


def test_step_host_matches_device_path(oracle):
    # the HOST-buffer entry point (bench.py's e2e leg) gives the same results as the device-pointer calls
    from paper_2607_01164_b200 import api
    g = inputs.c1_gaussians(seed=0, n=512)
    grid = inputs.c1_grid(24)
    rng = np.random.default_rng(0)
    target = rng.uniform(0, 1, grid.num_points).astype(np.float32)
    xyz, fwd, loss, a, serr, gr = _oracle_all(oracle, g, grid, target)
    ctx = api.Context()
    P, n = grid.num_points, g.n
    phi, I = np.zeros(P, np.float32), np.zeros(P, np.float32)
    grads = dict(dmean=np.zeros((n, 3), np.float32), dscale=np.zeros((n, 3), np.float32), dquat=np.zeros((n, 4), np.float32),
                 dopacity=np.zeros(n, np.float32), dscalar=np.zeros(n, np.float32), err=np.zeros(n, np.float32))
    gh = dict(mean=g.mean, scale=g.scale, quat=g.quat, opacity=g.opacity, scalar=g.scalar)
    got_loss = ctx.gs_step_host(gh, api.grid_query(grid), target, phi, I, grads)
    assert got_loss == pytest.approx(loss, rel=1e-6)
    assert np.abs(phi - fwd["phi"]).max() <= 1e-5
    from gpu_util import rel_l2
    for k, v in gr.items():
        assert rel_l2(grads[k], v) <= 1e-4, k
    ctx.close()


def test_fused_mse_backward(oracle):
    # gs_sample_bwd(dL_dphi = NULL): the backward of the forward's fused MSE loss (coefficients kept by the forward)
    # gives the same gradients as the explicit dL_dphi form; misuse is a state error
    import torch
    from paper_2607_01164_b200 import api
    g = inputs.c4_gaussians(seed=11, n_grid=40, n=2500)
    grid = inputs.Grid((40, 37, 26), (0.0, 0.0, 0.0), (1 / 40, 1 / 40, 1 / 40))
    rng = np.random.default_rng(5)
    target = rng.uniform(0, 1, grid.num_points).astype(np.float32)
    xyz, fwd, loss, a, serr, gr = _oracle_all(oracle, g, grid, target)
    run = GpuRun(g, "grid", grid, target, fused=True)
    check_forward(run, fwd)
    assert float(run.loss.item()) == pytest.approx(loss, rel=1e-6)
    check_grads(run, gr)
    # a forward without target leaves no coefficients: the fused backward must refuse
    ctx = run.ctx
    ctx.gs_sample_fwd(run.q, run.phi, run.I)
    with pytest.raises(api.GsError) as ei:
        ctx.gs_sample_bwd(run.q, None, None, None, run.grads)
    assert ei.value.status == api.GS_ERR_STATE
    # dL_dI cannot be combined with the fused form
    ctx.gs_sample_fwd(run.q, run.phi, run.I, target=run.target)
    with pytest.raises(api.GsError) as ei:
        ctx.gs_sample_bwd(run.q, None, None, None, run.grads, dL_dI=torch.zeros_like(run.phi))
    assert ei.value.status == api.GS_ERR_STATE


def test_long_brick_runs_sorted(oracle):
    # brick runs of every length class of the per-brick sort (<= 32 shuffles, <= 128 rank sort, <= 1024 bitonic in
    # shared memory, longer in global memory): 5,000 Gaussians several bricks wide over a 3 x 2 x 2 brick grid,
    # plus many that are smaller than a brick; the sorted (brick, gaussian) list must be bit-exact either way
    rng = np.random.default_rng(11)
    grid = inputs.Grid((24, 16, 12), (0.0, 0.0, 0.0), (1 / 24, 1 / 24, 1 / 24))
    n_big, n_small = 5000, 600
    g = inputs.c1_gaussians(seed=12, n=n_big + n_small)
    g.mean[:] = rng.uniform((0, 0, 0), (1.0, 16 / 24, 0.5), (g.n, 3)).astype(np.float32)
    g.scale[:n_big] = rng.uniform(0.08, 0.2, (n_big, 3)).astype(np.float32)
    g.scale[n_big:] = rng.uniform(0.004, 0.01, (n_small, 3)).astype(np.float32)
    perm = rng.permutation(g.n)
    for a in (g.mean, g.scale, g.quat, g.opacity, g.scalar):
        a[:] = a[perm]
    for sub in (grid, grid.batch((2, 1, 1), (1, 1, 1))):
        run = GpuRun(g, "grid", sub, None)
        T = _check_integer_stages(oracle, run, g, sub)
        start = run.ctx.debug_get(run.api.DBG_BRICK_START, np.uint32).astype(np.int64)
        lens = np.diff(start)
        assert T == start[-1] and lens.max() > 1024
    # a second grid whose runs fall in the middle classes
    g2 = inputs.c1_gaussians(seed=13, n=1500)
    g2.scale[:] = rng.uniform(0.02, 0.06, (g2.n, 3)).astype(np.float32)
    run = GpuRun(g2, "grid", inputs.c1_grid(32), None)
    _check_integer_stages(oracle, run, g2, inputs.c1_grid(32))
    lens = np.diff(run.ctx.debug_get(run.api.DBG_BRICK_START, np.uint32).astype(np.int64))
    assert ((lens > 32) & (lens <= 128)).any() and ((lens > 128) & (lens <= 1024)).any()


def test_structured_path_is_deterministic(oracle):
    # the brick lists are filled through atomics but every run is sorted, and the backward uses no atomics: two passes
    # over the same inputs give bit-identical samples and gradients (the loss scalar is summed with atomics: not compared)
    grid = inputs.Grid((44, 29, 21), (-0.1, 0.2, 0.0), (1 / 40, 1 / 32, 1 / 20))
    g = inputs.c4_gaussians(seed=9, n_grid=40, n=4000)
    target = np.random.default_rng(4).uniform(0, 1, grid.num_points).astype(np.float32)
    runs = [GpuRun(g, "grid", grid, target, fused=True) for _ in range(2)]
    a, b = runs
    assert np.array_equal(a.np(a.phi).view(np.uint32), b.np(b.phi).view(np.uint32))
    assert np.array_equal(a.np(a.I).view(np.uint32), b.np(b.I).view(np.uint32))
    ga, gb = a.grads_np(), b.grads_np()
    for k in ga:
        assert np.array_equal(ga[k], gb[k]), k
    pa = a.ctx.debug_get(a.api.DBG_PAIR_GAUSS, np.uint32)
    assert np.array_equal(pa, b.ctx.debug_get(b.api.DBG_PAIR_GAUSS, np.uint32))


@pytest.mark.parametrize("fused", [False, True])
def test_jittered_grid(oracle, fused):
    """In-cell jitter (D26): one random sample position per voxel instead of its centre, drawn by the same
    counter-based generator on both sides.  ID sets bit-exact, forward / gradients to the usual tolerances, on C1 and on
    a ragged sub-box batch with elongated Gaussians."""
    rng = np.random.default_rng(21)
    cases = [(inputs.c1_gaussians(seed=0, n=1024), inputs.c1_grid(32), 5)]
    gridfull = inputs.Grid((44, 29, 21), (-0.1, 0.2, 0.0), (1 / 40, 1 / 32, 1 / 20))
    cases.append((inputs.c4_gaussians(seed=7, n_grid=40, n=3000), gridfull.batch((1, 1, 0), (3, 3, 3)), 2 ** 40 + 17))
    for g, grid, seed in cases:
        xyz = oracle.grid_points(grid, jitter_seed=seed)
        assert not np.array_equal(xyz, oracle.grid_points(grid))
        P = grid.num_points
        target = rng.uniform(0, 1, P).astype(np.float32)
        dI = None if fused else (rng.standard_normal(P) * 1e-3)
        fwd = oracle.forward(g, xyz, TAU, mode=1)
        loss, a, serr = oracle.mse(fwd["phi"], fwd["I"], target, TAU)
        gr = oracle.backward(g, xyz, fwd["phi"], fwd["I"], a, dI, target, TAU, mode=1)
        run = GpuRun(g, "grid", grid, target, dL_dI=None if dI is None else dI.astype(np.float32), fused=fused, jitter_seed=seed)
        _check_integer_stages(oracle, run, g, grid)   # the brick lists do not depend on the jitter
        check_sets(run, fwd)
        check_forward(run, fwd)
        assert float(run.loss.item()) == pytest.approx(loss, rel=1e-6)
        check_grads(run, gr)
        # another seed gives other samples
        run2 = GpuRun(g, "grid", grid, target, fused=True, jitter_seed=seed + 1)
        assert not np.array_equal(run2.np(run2.phi), run.np(run.phi))


def test_small_batches_use_the_coarse_index(oracle):
    # From the second small batch after a gs_preprocess on, the build looks only at the Gaussians of the coarse cells
    # (16^3 bricks) the batch overlaps.  Batches that straddle 8 / 2 / 1 coarse cells must give the same sorted keys, counts,
    # ID sets and gradients as the oracle (a Gaussian listed in several cells is handled exactly once).
    import torch
    from paper_2607_01164_b200 import api
    n_grid = 512
    g = inputs.c4_gaussians(seed=11, n_grid=n_grid, n=70000)
    g.scale[:] = (g.scale * 6.0).astype(np.float32)      # many Gaussians overlap several coarse cells
    g.scale[5, 2] = np.nan                                # an invalid one
    full = inputs.c4_grid(n_grid)
    ctx = api.Context()
    dev = [torch.from_numpy(x).cuda() for x in (g.mean, g.scale, g.quat, g.opacity, g.scalar)]
    ctx.gs_preprocess(*dev)
    M, aabb, valid = oracle.preprocess_f32(g, TAU)
    rng = np.random.default_rng(0)
    for lo, cnt in (((3, 3, 3), (2, 2, 2)),          # first batch: full pass
                    ((10, 26, 12), (12, 8, 10)),     # straddles 2 x 2 x 2 coarse cells
                    ((16, 32, 5), (4, 3, 6)),        # one coarse cell, aligned at its corner
                    ((30, 40, 50), (5, 2, 2)),       # 2 x 1 x 1
                    ((60, 60, 60), (4, 4, 4))):      # upper corner of the grid
        batch = full.batch(lo, cnt)
        P = batch.num_points
        q = api.grid_query(batch)
        ctx.gs_build_accel(q)
        blo, bhi, bc = oracle.brick_ranges(aabb, valid, batch)
        keys, start = oracle.brick_keys(blo, bhi, bc, batch)
        assert np.array_equal(ctx.debug_get(api.DBG_BRICK_COUNT, np.uint32), bc)
        pb = ctx.debug_get(api.DBG_PAIR_BRICK, np.uint32)
        pg = ctx.debug_get(api.DBG_PAIR_GAUSS, np.uint32)
        assert np.array_equal((pb.astype(np.uint64) << np.uint64(32)) | pg.astype(np.uint64), keys)
        assert np.array_equal(ctx.debug_get(api.DBG_BRICK_START, np.uint32).astype(np.int64), start)
        target = rng.uniform(0, 1, P).astype(np.float32)
        xyz = oracle.grid_points(batch)
        fwd = oracle.forward(g, xyz, TAU, mode=1)
        _, a, _ = oracle.mse(fwd["phi"], fwd["I"], target, TAU)
        gr = oracle.backward(g, xyz, fwd["phi"], fwd["I"], a, None, target, TAU, mode=1)
        phi, I = torch.empty(P, device="cuda"), torch.empty(P, device="cuda")
        loss = torch.zeros(1, dtype=torch.float64, device="cuda")
        ctx.gs_sample_fwd(q, phi, I, target=torch.from_numpy(target).cuda(), loss=loss)
        grads = ctx.alloc_grads(g.n)
        for v in grads.values():
            v.fill_(-7.0)
        ctx.gs_sample_bwd(q, None, None, None, grads)
        cnt_, hs, hx, tested, hits = ctx.debug_point_sets(q)
        assert np.array_equal(cnt_, fwd["count"]) and np.array_equal(hs, fwd["hsum"]) and np.array_equal(hx, fwd["hxor"])
        assert hits > 0
        for k, v in gr.items():
            got = grads[k].cpu().numpy().astype(np.float64)
            assert np.linalg.norm(got - v) <= 1e-4 * max(np.linalg.norm(v), 1e-30), k
    assert ctx.gs_status_query()["num_gaussians"] == 70000
    ctx.close()


def test_coarse_index_follows_a_change_of_grid(oracle):
    # two different grids queried in small batches against ONE preprocess: the coarse index is rebuilt for the new geometry
    import torch
    from paper_2607_01164_b200 import api
    g = inputs.c4_gaussians(seed=12, n_grid=256, n=66000)
    g.scale[:] = (g.scale * 3.0).astype(np.float32)
    ctx = api.Context()
    ctx.gs_preprocess(*[torch.from_numpy(x).cuda() for x in (g.mean, g.scale, g.quat, g.opacity, g.scalar)])
    M, aabb, valid = oracle.preprocess_f32(g, TAU)
    for n_grid, batches in ((256, (((2, 2, 2), (3, 3, 3)), ((14, 15, 16), (4, 4, 4)))), (384, (((1, 1, 1), (2, 2, 2)), ((30, 31, 15), (5, 3, 4)), ((0, 0, 0), (3, 2, 2))))):
        full = inputs.c4_grid(n_grid)
        for lo, cnt in batches:
            batch = full.batch(lo, cnt)
            q = api.grid_query(batch)
            ctx.gs_build_accel(q)
            blo, bhi, bc = oracle.brick_ranges(aabb, valid, batch)
            keys, start = oracle.brick_keys(blo, bhi, bc, batch)
            assert np.array_equal(ctx.debug_get(api.DBG_BRICK_COUNT, np.uint32), bc)
            pb = ctx.debug_get(api.DBG_PAIR_BRICK, np.uint32)
            pg = ctx.debug_get(api.DBG_PAIR_GAUSS, np.uint32)
            assert np.array_equal((pb.astype(np.uint64) << np.uint64(32)) | pg.astype(np.uint64), keys)
            ref = oracle.forward(g, oracle.grid_points(batch), TAU, mode=1)
            cnt_, hs, hx, tested, hits = ctx.debug_point_sets(q)
            assert np.array_equal(cnt_, ref["count"]) and np.array_equal(hs, ref["hsum"]) and np.array_equal(hx, ref["hxor"])
    ctx.close()
