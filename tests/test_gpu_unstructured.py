"""-m gpu parity: unstructured path (S1, S3, S5, S6, S7, S8) through the C ABI vs the oracle.

Integer stages (Morton keys, leaf order, radix-tree topology, node boxes, query order, per-point ID
sets) are bit-exact; fp32 values within the north_star tolerances.
"""
import numpy as np
import pytest

from paper_2607_01164_b200 import inputs
from gpu_util import TAU, GpuRun, check_forward, check_grads, check_sets

pytestmark = pytest.mark.gpu


def _oracle_all(oracle, g, xyz, target, dL_dI=None):
    fwd = oracle.forward(g, xyz, TAU, mode=1)
    loss, a, serr = oracle.mse(fwd["phi"], fwd["I"], target, TAU)
    gr = oracle.backward(g, xyz, fwd["phi"], fwd["I"], a, dL_dI, target, TAU, mode=1)
    return fwd, loss, a, serr, gr


def _check_lbvh(oracle, run, g, xyz, dom, presorted=False):
    api = run.api
    M, aabb, valid = oracle.preprocess_f32(g, TAU)
    codes = oracle.morton_codes(g.mean, dom[0], dom[1], valid)
    order, keys = oracle.morton_order(codes)
    assert np.array_equal(run.ctx.debug_get(api.DBG_LEAF_MORTON, np.uint32), codes[order]), "sorted Morton codes differ"
    assert np.array_equal(run.ctx.debug_get(api.DBG_LEAF_ORDER, np.uint32), order), "BVH leaf order differs"
    if g.n >= 2:
        tree = oracle.lbvh_build(keys, aabb[order])
        assert np.array_equal(run.ctx.debug_get(api.DBG_NODE_LEFT, np.int32), tree["left"])
        assert np.array_equal(run.ctx.debug_get(api.DBG_NODE_RIGHT, np.int32), tree["right"])
        assert np.array_equal(run.ctx.debug_get(api.DBG_NODE_PARENT, np.int32), tree["parent"])
        assert np.array_equal(run.ctx.debug_get(api.DBG_LEAF_PARENT, np.int32), tree["leaf_parent"])
        nb = run.ctx.debug_get(api.DBG_NODE_AABB, np.float32, 6)
        assert np.array_equal(nb.view(np.uint32), tree["node_aabb"].view(np.uint32)), "node boxes are not the exact min/max"
    if not presorted and len(xyz):
        pcodes = oracle.morton_codes(xyz, dom[0], dom[1])
        porder, _ = oracle.morton_order(pcodes)
        assert np.array_equal(run.ctx.debug_get(api.DBG_POINT_ORDER, np.uint32), porder), "query coherence order differs"
        assert np.array_equal(run.ctx.debug_get(api.DBG_POINT_MORTON, np.uint32), pcodes[porder])


@pytest.mark.parametrize("presorted", [False, True])
def test_c3_reduced(oracle, presorted):
    # reduced copy of BASELINE.json configs[2]: same distributions, sizes the oracle finishes in seconds;
    # 40,003 points = many packets and a ragged tail
    xyz_all, t_all = inputs.c3_points(seed=3, p=60000)
    g = inputs.c3_gaussians(xyz_all, t_all, seed=3, n=20000, sigma_lo=0.004, sigma_hi=0.04)
    idx = inputs.batch_indices(3, 0, len(xyz_all), 40003)
    xyz, target = np.ascontiguousarray(xyz_all[idx]), np.ascontiguousarray(t_all[idx])
    dom = inputs.points_domain(xyz_all)
    fwd, loss, a, serr, gr = _oracle_all(oracle, g, xyz, target)
    run = GpuRun(g, "points", xyz, target, domain=dom, presorted=presorted)
    _check_lbvh(oracle, run, g, xyz, dom, presorted)
    tested, hits = check_sets(run, fwd)
    assert hits > 20 * len(xyz)
    check_forward(run, fwd)
    assert float(run.loss.item()) == pytest.approx(loss, rel=1e-6)
    np.testing.assert_allclose(run.np(run.serr), serr, atol=1e-5)
    check_grads(run, gr)
    if not presorted:  # fused-MSE backward (dL_dphi = NULL) gives the same gradients
        check_grads(GpuRun(g, "points", xyz, target, domain=dom, fused=True), gr)


def test_c5_like_sparse_with_dI(oracle):
    # shell-and-fragments distribution (configs[4] shape): most of the box is empty, many uncovered samples
    xyz_all, t_all = inputs.c5_points(seed=5, p=50000, clusters=64, chunk=1 << 15)
    g = inputs.c3_gaussians(xyz_all, t_all, seed=5, n=6000, sigma_lo=0.002, sigma_hi=0.01)
    rng = np.random.default_rng(9)
    extra = rng.uniform(0, 1, (3000, 3)).astype(np.float32)  # queries far from any Gaussian
    xyz = np.concatenate([xyz_all[:30001], extra])
    target = np.concatenate([t_all[:30001], np.zeros(3000, np.float32)])
    dI = rng.standard_normal(len(xyz)) * 1e-3
    dom = (np.zeros(3, np.float32), np.ones(3, np.float32))
    fwd, loss, a, serr, gr = _oracle_all(oracle, g, xyz, target, dI)
    assert (fwd["count"] == 0).sum() > 1000
    run = GpuRun(g, "points", xyz, target, domain=dom, dL_dI=dI.astype(np.float32))
    _check_lbvh(oracle, run, g, xyz, dom)
    check_sets(run, fwd)
    check_forward(run, fwd)
    check_grads(run, gr)


def test_cull_pool_growth_and_context_reuse(oracle):
    # every Gaussian reaches every packet: the per-packet lists (gs_build_accel) outgrow the initial pool, so the
    # count-and-repeat path runs; then the same context serves a light query (lists shrink, pool is re-used)
    rng = np.random.default_rng(11)
    n = 1500
    g = inputs.c1_gaussians(seed=12, n=n)
    g.scale[:] = rng.uniform(0.3, 0.6, (n, 3)).astype(np.float32)
    xyz = rng.uniform(0, 1, (20011, 3)).astype(np.float32)
    target = rng.uniform(0, 1, len(xyz)).astype(np.float32)
    dom = (np.zeros(3, np.float32), np.ones(3, np.float32))
    fwd, loss, a, serr, gr = _oracle_all(oracle, g, xyz, target)
    assert fwd["count"].astype(np.int64).sum() > 256 * len(xyz)   # more than the initial 256 list entries per point
    run = GpuRun(g, "points", xyz, target, domain=dom)
    check_sets(run, fwd)
    check_forward(run, fwd)
    check_grads(run, gr)
    # light query on the same context
    import torch
    xyz2 = np.ascontiguousarray(xyz[:777])
    q2 = run.api.points_query(torch.from_numpy(xyz2).cuda())
    run.ctx.gs_build_accel(q2)
    phi, I = torch.empty(777, device="cuda"), torch.empty(777, device="cuda")
    run.ctx.gs_sample_fwd(q2, phi, I)
    ref = oracle.forward(g, xyz2, TAU, mode=1)
    assert np.abs(phi.cpu().numpy() - ref["phi"]).max() <= 1e-5
    assert np.abs(I.cpu().numpy() - ref["I"]).max() <= 2e-5 * max(1.0, float(ref["I"].max()))


def test_nonfinite_query_points(oracle):
    # NaN / infinite coordinates: such a sample hits nothing (Phi = 0, I = 0) and must not disturb the finite
    # samples that share its packet (their packet box then culls nothing)
    rng = np.random.default_rng(4)
    xyz_all, t_all = inputs.c3_points(seed=3, p=8000)
    g = inputs.c3_gaussians(xyz_all, t_all, seed=3, n=3000, sigma_lo=0.01, sigma_hi=0.05)
    xyz = np.ascontiguousarray(xyz_all[:2000]).copy()
    bad = rng.choice(len(xyz), 40, replace=False)
    xyz[bad[:15], 0] = np.nan
    xyz[bad[15:30], 1] = np.inf
    xyz[bad[30:], 2] = -np.inf
    good = np.setdiff1d(np.arange(len(xyz)), bad)
    dom = inputs.points_domain(xyz_all)
    ref = oracle.forward(g, np.ascontiguousarray(xyz[good]), TAU, mode=0)
    run = GpuRun(g, "points", xyz, None, domain=dom)
    phi, I = run.np(run.phi), run.np(run.I)
    assert np.all(phi[bad] == 0.0) and np.all(I[bad] == 0.0)
    cnt, hs, hx, tested, hits = run.sets()
    assert np.all(cnt[bad] == 0)
    assert np.array_equal(cnt[good], ref["count"]) and np.array_equal(hs[good], ref["hsum"]) and np.array_equal(hx[good], ref["hxor"])
    near = np.abs(ref["I"] - TAU) <= 2e-6 * TAU
    assert np.abs(phi[good] - ref["phi"])[~near].max() <= 1e-5


def test_degenerate_unstructured(oracle):
    rng = np.random.default_rng(2)
    dom = (np.zeros(3, np.float32), np.ones(3, np.float32))
    xyz = rng.uniform(0, 1, (1000, 3)).astype(np.float32)
    target = rng.uniform(0, 1, 1000).astype(np.float32)
    base = inputs.c1_gaussians(seed=6, n=64)
    base.scale[:] = (base.scale * 4).astype(np.float32)
    for n in (0, 1, 2, 3):
        g = base.subset(np.arange(n))
        run = GpuRun(g, "points", xyz, target, domain=dom)
        if n:
            fwd, loss, a, serr, gr = _oracle_all(oracle, g, xyz, target)
            _check_lbvh(oracle, run, g, xyz, dom)
            check_sets(run, fwd)
            check_forward(run, fwd)
            # one Gaussian (or a few that do not overlap): Phi = v wherever covered, so every gradient except
            # dL/dv vanishes exactly; compare those against the size of the terms that cancel (~ |dL/dv|)
            floor = {k: float(np.linalg.norm(gr["dscalar"])) for k in ("dmean", "dscale", "dquat", "dopacity")}
            check_grads(run, gr, zero_floor=floor)
        else:
            assert np.all(run.np(run.phi) == 0.0) and np.all(run.np(run.I) == 0.0)
    # identical means (equal Morton codes: the id in the low word keeps keys unique), invalid Gaussians, P = 0 / 1 / 33
    g = base.subset(np.arange(40))
    g.mean[5:25] = g.mean[5]
    g.scale[30, 0] = np.nan
    g.quat[31] = 0
    for P in (0, 1, 33):
        run = GpuRun(g, "points", xyz[:P], target[:P], domain=dom)
        if P:
            fwd, loss, a, serr, gr = _oracle_all(oracle, g, xyz[:P], target[:P])
            _check_lbvh(oracle, run, g, xyz[:P], dom)
            check_sets(run, fwd)
            check_forward(run, fwd)
            check_grads(run, gr, zero_floor={k: float(np.linalg.norm(gr["dscalar"])) for k in ("dmean", "dscale", "dquat", "dopacity")})
    # a point query without a domain is a state error
    from paper_2607_01164_b200 import api
    import torch
    ctx = api.Context()
    dev = [torch.from_numpy(x).cuda() for x in (g.mean, g.scale, g.quat, g.opacity, g.scalar)]
    ctx.gs_preprocess(*dev)
    with pytest.raises(api.GsError) as ei:
        ctx.gs_build_accel(api.points_query(torch.from_numpy(xyz).cuda()))
    assert ei.value.status == api.GS_ERR_STATE
    ctx.close()


def test_backward_with_and_without_hit_masks(oracle):
    # GS_OPT_BWD_HIT_MASKS (gs.h): the forward leaves one hit bit per cull-list entry and the backward evaluates only the entries
    # that hit, compacted across chunks.  Same per-entry arithmetic: both forms agree with each other far inside the 1e-4 they
    # each meet against the oracle, in the fused and the general form; a backward WITHOUT a forward on the accel falls back.
    import torch
    from paper_2607_01164_b200 import api
    from gpu_util import rel_l2
    xyz_all, t_all = inputs.c5_points(seed=7, p=90000)
    g = inputs.c5_gaussians(xyz_all, t_all, seed=7, n=30000)
    idx = inputs.batch_indices(7, 0, len(xyz_all), 50021)      # ragged tail: 50021 = 1563 packets + 5 points
    xyz, target = np.ascontiguousarray(xyz_all[idx]), np.ascontiguousarray(t_all[idx])
    dom = inputs.points_domain(xyz_all)
    fwd, loss, a, serr, gr = _oracle_all(oracle, g, xyz, target)
    runs = {}
    for fused in (True, False):
        run = GpuRun(g, "points", xyz, target, domain=dom, fused=fused)            # masks on (default)
        check_grads(run, gr)
        runs[fused] = run
    ctx = api.Context()
    ctx.gs_set_option(api.OPT_BWD_HIT_MASKS, 0)
    dev = [torch.from_numpy(np.ascontiguousarray(x)).cuda() for x in (g.mean, g.scale, g.quat, g.opacity, g.scalar)]
    ctx.gs_preprocess(*dev, domain=dom, tau=TAU)
    q = api.points_query(runs[False].xyz)
    ctx.gs_build_accel(q)
    grads = ctx.alloc_grads(g.n)
    # general form straight after the build, no forward on this context: phi / I / dL_dphi come from the other run
    r = runs[False]
    ctx.gs_sample_bwd(q, r.phi, r.I, r.dphi, grads, target=r.target)
    torch.cuda.synchronize()
    for k, v in r.grads.items():
        assert rel_l2(grads[k].cpu().numpy(), v.cpu().numpy()) <= 1e-5, k   # the order of the atomic additions only
    # and with masks on but no forward since the build: the fallback, same numbers
    ctx.gs_set_option(api.OPT_BWD_HIT_MASKS, 1)
    ctx.gs_build_accel(q)
    for v in grads.values():
        v.fill_(-7.0)
    ctx.gs_sample_bwd(q, r.phi, r.I, r.dphi, grads, target=r.target)
    torch.cuda.synchronize()
    for k, v in r.grads.items():
        assert rel_l2(grads[k].cpu().numpy(), v.cpu().numpy()) <= 1e-5, k   # the order of the atomic additions only
    for k, v in runs[True].grads.items():
        assert rel_l2(v.cpu().numpy(), r.grads[k].cpu().numpy()) <= 2e-4, k    # fused vs general form: each is within 1e-4 of the oracle
    ctx.close()
