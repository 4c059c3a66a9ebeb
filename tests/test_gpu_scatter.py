"""-m gpu parity of the SCATTER mode of a point query: the paper's own unstructured formulation (section 5.1,
PAPER.md:184-196: a wide tree over the sample positions, one warp per Gaussian, atomics into the samples, register sums
in the backward), selected with gs_set_option(GS_OPT_POINTS_ACCEL, GS_POINTS_SCATTER).  Same bar as the gather mode:
ID sets bit-exact, Phi <= 1e-5, gradients <= 1e-4 per tensor; the two modes are also compared with each other."""
import numpy as np
import pytest

from paper_2607_01164_b200 import inputs
from gpu_util import TAU, GpuRun, check_forward, check_grads, check_sets

pytestmark = pytest.mark.gpu
SCATTER = 1


def _oracle_all(oracle, g, xyz, target, dL_dI=None):
    fwd = oracle.forward(g, xyz, TAU, mode=1)
    loss, a, serr = oracle.mse(fwd["phi"], fwd["I"], target, TAU)
    gr = oracle.backward(g, xyz, fwd["phi"], fwd["I"], a, dL_dI, target, TAU, mode=1)
    return fwd, loss, a, serr, gr


@pytest.mark.parametrize("presorted", [False, True])
def test_scatter_c3_reduced(oracle, presorted):
    xyz_all, t_all = inputs.c3_points(seed=3, p=60000)
    g = inputs.c3_gaussians(xyz_all, t_all, seed=3, n=20000, sigma_lo=0.004, sigma_hi=0.04)
    idx = inputs.batch_indices(3, 0, len(xyz_all), 40003)   # many leaves, several tree levels, a ragged tail
    xyz, target = np.ascontiguousarray(xyz_all[idx]), np.ascontiguousarray(t_all[idx])
    dom = inputs.points_domain(xyz_all)
    fwd, loss, a, serr, gr = _oracle_all(oracle, g, xyz, target)
    run = GpuRun(g, "points", xyz, target, domain=dom, presorted=presorted, points_accel=SCATTER)
    api = run.api
    # the processing order of the Gaussians is their Morton order, as in gather mode; the tree over them is not built
    M, aabb, valid = oracle.preprocess_f32(g, TAU)
    order, _ = oracle.morton_order(oracle.morton_codes(g.mean, dom[0], dom[1], valid))
    assert np.array_equal(run.ctx.debug_get(api.DBG_LEAF_ORDER, np.uint32), order)
    with pytest.raises(api.GsError):
        run.ctx.debug_get(api.DBG_NODE_LEFT, np.int32)
    if not presorted:
        porder, _ = oracle.morton_order(oracle.morton_codes(xyz, dom[0], dom[1]))
        assert np.array_equal(run.ctx.debug_get(api.DBG_POINT_ORDER, np.uint32), porder)
    tested, hits = check_sets(run, fwd)
    assert hits > 20 * len(xyz) and tested >= hits
    check_forward(run, fwd)
    assert float(run.loss.item()) == pytest.approx(loss, rel=1e-6)
    np.testing.assert_allclose(run.np(run.serr), serr, atol=1e-5)
    check_grads(run, gr)
    if not presorted:   # fused-MSE backward, and agreement with the gather mode
        check_grads(GpuRun(g, "points", xyz, target, domain=dom, fused=True, points_accel=SCATTER), gr)
        other = GpuRun(g, "points", xyz, target, domain=dom, points_accel=0)
        assert np.abs(run.np(run.phi) - other.np(other.phi)).max() <= 2e-6
        for k, v in other.grads_np().items():
            assert np.linalg.norm(run.grads_np()[k] - v) <= 2e-5 * np.linalg.norm(v), k


def test_scatter_sparse_with_dI_and_nonfinite_points(oracle):
    xyz_all, t_all = inputs.c5_points(seed=5, p=50000, clusters=64, chunk=1 << 15)
    g = inputs.c3_gaussians(xyz_all, t_all, seed=5, n=6000, sigma_lo=0.002, sigma_hi=0.01)
    g.scale[17, 1] = 0.0          # invalid Gaussians have empty support
    g.quat[18] = 0.0
    rng = np.random.default_rng(9)
    extra = rng.uniform(0, 1, (3000, 3)).astype(np.float32)  # queries far from any Gaussian
    xyz = np.concatenate([xyz_all[:30001], extra])
    target = np.concatenate([t_all[:30001], np.zeros(3000, np.float32)])
    bad = rng.choice(len(xyz), 30, replace=False)
    xyz[bad[:10], 0] = np.nan
    xyz[bad[10:20], 1] = np.inf
    xyz[bad[20:], 2] = -np.inf
    dI = rng.standard_normal(len(xyz)) * 1e-3
    dom = (np.zeros(3, np.float32), np.ones(3, np.float32))
    # a non-finite sample lies in no support: the oracle sees the finite ones only (its loss mean still runs over all P)
    good = np.setdiff1d(np.arange(len(xyz)), bad)
    xg, tg = np.ascontiguousarray(xyz[good]), np.ascontiguousarray(target[good])
    fwd = oracle.forward(g, xg, TAU, mode=1)
    assert (fwd["count"] == 0).sum() > 1000
    res = fwd["phi"] - tg
    covered = fwd["I"].astype(np.float32) > np.float32(TAU)
    a = np.where(covered, 2.0 * res / len(xyz), 0.0)
    gr = oracle.backward(g, xg, fwd["phi"], fwd["I"], a, dI[good], tg, TAU, mode=1)
    run = GpuRun(g, "points", xyz, target, domain=dom, dL_dI=dI.astype(np.float32), points_accel=SCATTER)
    phi, I = run.np(run.phi), run.np(run.I)
    assert np.all(phi[bad] == 0.0) and np.all(I[bad] == 0.0)
    cnt, hs, hx, tested, hits = run.sets()
    assert np.all(cnt[bad] == 0)
    assert np.array_equal(cnt[good], fwd["count"]) and np.array_equal(hs[good], fwd["hsum"]) and np.array_equal(hx[good], fwd["hxor"])
    near = np.abs(fwd["I"] - TAU) <= 2e-6 * TAU
    assert np.abs(phi[good] - fwd["phi"])[~near].max() <= 1e-5
    check_grads(run, gr)
    got = run.grads_np()
    assert all(np.all(np.isfinite(v)) for v in got.values())
    assert np.all(got["dmean"][17:19] == 0.0) and np.all(got["dscalar"][17:19] == 0.0)


def test_scatter_degenerate(oracle):
    rng = np.random.default_rng(2)
    dom = (np.zeros(3, np.float32), np.ones(3, np.float32))
    xyz = rng.uniform(0, 1, (1000, 3)).astype(np.float32)
    target = rng.uniform(0, 1, 1000).astype(np.float32)
    base = inputs.c1_gaussians(seed=6, n=64)
    base.scale[:] = (base.scale * 4).astype(np.float32)
    for n in (0, 1, 3):
        g = base.subset(np.arange(n))
        run = GpuRun(g, "points", xyz, target, domain=dom, points_accel=SCATTER)
        if n:
            fwd, loss, a, serr, gr = _oracle_all(oracle, g, xyz, target)
            check_sets(run, fwd)
            check_forward(run, fwd)
            floor = {k: float(np.linalg.norm(gr["dscalar"])) for k in ("dmean", "dscale", "dquat", "dopacity")}
            check_grads(run, gr, zero_floor=floor)
        else:
            assert np.all(run.np(run.phi) == 0.0) and np.all(run.np(run.I) == 0.0)
    g = base.subset(np.arange(40))
    for P in (0, 1, 33, 65):
        run = GpuRun(g, "points", xyz[:P], target[:P], domain=dom, points_accel=SCATTER)
        if P:
            fwd, loss, a, serr, gr = _oracle_all(oracle, g, xyz[:P], target[:P])
            check_sets(run, fwd)
            check_forward(run, fwd)
            check_grads(run, gr, zero_floor={k: float(np.linalg.norm(gr["dscalar"])) for k in ("dmean", "dscale", "dquat", "dopacity")})


def test_scatter_c3_full_size(oracle):
    # BASELINE.json configs[2] at full size through the scatter mode (what `bench.py --workload c3` times in its A/B leg)
    xyz_all, t_all = inputs.c3_points()
    g = inputs.c3_gaussians(xyz_all, t_all)
    idx = inputs.batch_indices(3, 0, len(xyz_all), 1 << 20)
    xyz, target = np.ascontiguousarray(xyz_all[idx]), np.ascontiguousarray(t_all[idx])
    dom = inputs.points_domain(xyz_all)
    fwd, loss, a, serr, gr = _oracle_all(oracle, g, xyz, target)
    run = GpuRun(g, "points", xyz, target, domain=dom, fused=True, points_accel=SCATTER)
    tested, hits = check_sets(run, fwd)
    assert hits > 400_000_000
    near, e_phi, e_I = check_forward(run, fwd)
    assert near <= 16
    assert float(run.loss.item()) == pytest.approx(loss, rel=1e-6)
    errs = check_grads(run, gr)
    print("C3 full size, scatter mode: hits", hits, "tested", tested, "phi err", e_phi, "grad errs", errs)


def test_gaussian_side_is_reused_between_queries_of_one_preprocess(oracle):
    # gs.h (gs_build_accel): the Gaussian side of a point accel (Morton order, LBVH, records in leaf order) is built by the first
    # point query after a gs_preprocess and reused by the following ones.  Three different queries after ONE preprocess, with
    # the mode switched in between (the scatter mode builds the Morton order only, the gather mode then adds the tree), must
    # give what fresh contexts give; a new preprocess (a moved model) must not see the old tree.
    import torch
    from paper_2607_01164_b200 import api
    xyz_all, t_all = inputs.c3_points(seed=3, p=30000)
    g = inputs.c3_gaussians(xyz_all, t_all, seed=3, n=8000, sigma_lo=0.004, sigma_hi=0.04)
    dom = inputs.points_domain(xyz_all)
    chunks = [np.ascontiguousarray(xyz_all[a:b]) for a, b in ((0, 9001), (9001, 20000), (20000, 30000))]
    refs = [oracle.forward(g, c, TAU, mode=1) for c in chunks]
    dev = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (g.mean, g.scale, g.quat, g.opacity, g.scalar)]
    ctx = api.Context()
    ctx.gs_preprocess(*dev, domain=dom)
    modes = [api.POINTS_SCATTER, api.POINTS_GATHER, api.POINTS_GATHER]
    for c, ref, mode in zip(chunks, refs, modes):
        ctx.gs_set_option(api.OPT_POINTS_ACCEL, mode)
        xd = torch.from_numpy(c).cuda()
        q = api.points_query(xd)
        ctx.gs_build_accel(q)
        phi, I = torch.empty(len(c), device="cuda"), torch.empty(len(c), device="cuda")
        ctx.gs_sample_fwd(q, phi, I)
        cnt, hs, hx, _, _ = ctx.debug_point_sets(q)
        assert np.array_equal(cnt, ref["count"]) and np.array_equal(hs, ref["hsum"]) and np.array_equal(hx, ref["hxor"])
        near = np.abs(ref["I"] - TAU) <= 2e-6 * TAU
        assert np.abs(phi.cpu().numpy() - ref["phi"])[~near].max() <= 1e-5
    # the model moves: the next query must rebuild
    g2 = g.subset(np.arange(g.n))
    g2.mean[:] = (g.mean + np.float32(0.01)).astype(np.float32)
    dev2 = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (g2.mean, g2.scale, g2.quat, g2.opacity, g2.scalar)]
    ctx.gs_preprocess(*dev2, domain=dom)
    xd = torch.from_numpy(chunks[0]).cuda()
    q = api.points_query(xd)
    ctx.gs_build_accel(q)
    ref2 = oracle.forward(g2, chunks[0], TAU, mode=1)
    cnt, hs, hx, _, _ = ctx.debug_point_sets(q)
    assert np.array_equal(cnt, ref2["count"]) and np.array_equal(hs, ref2["hsum"]) and np.array_equal(hx, ref2["hxor"])
    ctx.close()
