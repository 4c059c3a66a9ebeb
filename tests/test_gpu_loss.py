"""-m gpu parity: gs_sample_fwd_loss (L1 / MSE over the defined samples, Eq. 4 false-negative and Eq. 5 false-positive
terms fused into the forward epilogue) and the backward of that loss, vs the oracle."""
import numpy as np
import pytest

from paper_2607_01164_b200 import inputs
from gpu_util import TAU, check_grads, to_dev

pytestmark = pytest.mark.gpu

LAM_FN, EPS_FN, LAM_FP = 0.8, 0.5, 0.3


def _run(oracle, g, kind_name, query_kind, query_obj, xyz, target, defined, domain=None):
    import torch
    from paper_2607_01164_b200 import api
    P = len(xyz)
    # ---- oracle: forward, loss, backward
    fwd = oracle.forward(g, xyz, TAU, mode=1)
    # keep the L1 kink and the class thresholds away from fp32 noise (a flipped sign / class is a different, equally
    # valid result): move the few targets that sit on a residual of ~0
    res = fwd["phi"] - target
    close = np.abs(res) < 1e-4
    target = np.where(close, target + np.float32(0.01), target).astype(np.float32)
    If = fwd["I"].astype(np.float32)
    thr = np.float32(1.0 + EPS_FN) * np.float32(TAU)
    near = (np.abs(fwd["I"] - TAU) <= 4e-6 * TAU) | (np.abs(fwd["I"] - float(thr)) <= 4e-6 * float(thr))
    assert near.sum() == 0, "pick another seed: a sample sits on a class threshold"
    nd = int(defined.sum()) if defined is not None else P
    ref = oracle.loss(fwd["phi"], fwd["I"], target, defined, TAU, kind_name, LAM_FN, EPS_FN, LAM_FP)
    assert ref["counts"][0] == nd
    gr = oracle.backward(g, xyz, fwd["phi"], fwd["I"], ref["dL_dphi"], ref["dL_dI"], target, TAU, mode=1)
    # ---- GPU
    ctx = api.Context()
    dev = to_dev(torch, g.mean, g.scale, g.quat, g.opacity, g.scalar)
    ctx.gs_preprocess(*dev, domain=domain, tau=TAU)
    if query_kind == "grid":
        q = api.grid_query(query_obj)
    else:
        xyz_d = to_dev(torch, query_obj)[0]
        q = api.points_query(xyz_d)
    ctx.gs_build_accel(q)
    f32 = dict(dtype=torch.float32, device="cuda")
    phi, I, dphi, dI, serr = (torch.full((P,), -7.0, **f32) for _ in range(5))
    terms = torch.full((3,), -7.0, dtype=torch.float64, device="cuda")
    t_d = to_dev(torch, target)[0]
    def_d = to_dev(torch, defined)[0] if defined is not None else None
    kind = api.LOSS_L1 if kind_name == "l1" else api.LOSS_MSE
    ctx.gs_sample_fwd_loss(q, phi, I, t_d, kind=kind, lambda_fn=LAM_FN, eps_fn=EPS_FN, lambda_fp=LAM_FP, defined=def_d,
                           num_defined=nd, loss_terms=terms, dL_dphi=dphi, dL_dI=dI, sample_err=serr)
    grads = ctx.alloc_grads(g.n)
    ctx.gs_sample_bwd(q, phi, I, dphi, grads, dL_dI=dI, target=t_d)
    torch.cuda.synchronize()
    got_terms = terms.cpu().numpy()
    # ---- compare
    assert ref["counts"][1] > 0 and (defined is None or ref["counts"][2] > 0), "the case must exercise the terms"
    np.testing.assert_allclose(got_terms, ref["loss"], rtol=2e-5, atol=1e-12)
    np.testing.assert_allclose(phi.cpu().numpy(), fwd["phi"], atol=1e-5)
    b = dI.cpu().numpy().astype(np.float64)
    # class membership is an integer decision: the sets D- and U+ must be the oracle's
    assert np.array_equal(b < 0, ref["dL_dI"] < 0) and np.array_equal(b > 0, ref["dL_dI"] > 0)
    np.testing.assert_allclose(b, ref["dL_dI"], rtol=1e-6)
    a = dphi.cpu().numpy().astype(np.float64)
    np.testing.assert_allclose(a, ref["dL_dphi"], rtol=3e-5, atol=3e-5 / nd)
    np.testing.assert_allclose(serr.cpu().numpy(), ref["sample_err"], atol=1e-5)

    class R:  # the shape check_grads expects
        pass
    r = R()
    r.grads_np = lambda: {k: v.detach().cpu().numpy().astype(np.float64) for k, v in grads.items()}
    # err (D10) is defined through |Phi - t| of covered samples with a target: undefined samples would need the mask,
    # which gs_sample_bwd does not take; compare the parameter gradients only
    gr = {k: v for k, v in gr.items() if k != "err"}
    errs = check_grads(r, gr)
    if query_kind == "grid":
        # on a grid the forward kept the backward coefficients: gs_sample_bwd(dL_dphi = NULL) must give the same gradients
        grads2 = ctx.alloc_grads(g.n)
        ctx.gs_sample_fwd_loss(q, phi, I, t_d, kind=kind, lambda_fn=LAM_FN, eps_fn=EPS_FN, lambda_fp=LAM_FP, defined=def_d,
                               num_defined=nd, loss_terms=terms)
        ctx.gs_sample_bwd(q, None, None, None, grads2)
        torch.cuda.synchronize()
        r2 = R()
        r2.grads_np = lambda: {k: v.detach().cpu().numpy().astype(np.float64) for k, v in grads2.items()}
        check_grads(r2, gr)
    else:
        with pytest.raises(api.GsError):   # a point query keeps no coefficients
            ctx.gs_sample_bwd(q, None, None, None, grads)
    ctx.close()
    return errs, ref


@pytest.mark.parametrize("kind", ["l1", "mse"])
def test_grid_losses(oracle, kind):
    # ragged grid (dims not multiples of 8), anisotropic Gaussians, 70 % of the samples defined
    grid = inputs.Grid((44, 29, 21), (-0.1, 0.2, 0.0), (1 / 40, 1 / 32, 1 / 20))
    g = inputs.c4_gaussians(seed=7, n_grid=40, n=2500)
    rng = np.random.default_rng(5)
    xyz = oracle.grid_points(grid)
    P = grid.num_points
    target = rng.uniform(0, 1, P).astype(np.float32)
    defined = (rng.uniform(0, 1, P) < 0.7).astype(np.uint8)
    _run(oracle, g, kind, "grid", grid, xyz, target, defined)


def test_grid_l1_all_defined(oracle):
    # defined = NULL: every sample is in D (the structured case of the paper, L1 + Eq. 4)
    grid = inputs.c1_grid(32)
    g = inputs.c1_gaussians(seed=0, n=1024)
    rng = np.random.default_rng(6)
    target = rng.uniform(0, 1, grid.num_points).astype(np.float32)
    _run(oracle, g, "l1", "grid", grid, oracle.grid_points(grid), target, None)


@pytest.mark.parametrize("kind", ["l1", "mse"])
def test_points_losses(oracle, kind):
    # unstructured: points of the C3 mixture (defined) plus uniform points of the bounding box, most of which fall
    # outside the data's support (undefined: Eq. 5 penalises influence there)
    xyz_all, t_all = inputs.c3_points(seed=31, p=6000)
    g = inputs.c3_gaussians(xyz_all, t_all, seed=31, n=1500)
    g.scale[:] = (g.scale * 4.0).astype(np.float32)  # keep a C3-like overlap at this reduced count
    rng = np.random.default_rng(8)
    extra = rng.uniform(0, 1, (3000, 3)).astype(np.float32)
    xyz = np.ascontiguousarray(np.concatenate([xyz_all[:5000], extra]))
    target = np.concatenate([t_all[:5000], np.zeros(3000, np.float32)]).astype(np.float32)
    defined = np.concatenate([np.ones(5000, np.uint8), np.zeros(3000, np.uint8)])
    perm = rng.permutation(len(xyz))
    xyz, target, defined = np.ascontiguousarray(xyz[perm]), np.ascontiguousarray(target[perm]), np.ascontiguousarray(defined[perm])
    _run(oracle, g, kind, "points", xyz, xyz, target, defined, domain=inputs.points_domain(xyz))


def test_loss_argument_errors(oracle):
    import torch
    from paper_2607_01164_b200 import api
    grid = inputs.c1_grid(16)
    g = inputs.c1_gaussians(seed=0, n=64)
    ctx = api.Context()
    ctx.gs_preprocess(*to_dev(torch, g.mean, g.scale, g.quat, g.opacity, g.scalar), tau=TAU)
    q = api.grid_query(grid)
    ctx.gs_build_accel(q)
    P = grid.num_points
    phi, I, t = (torch.zeros(P, device="cuda") for _ in range(3))
    for kw in (dict(kind=7), dict(lambda_fn=-1.0), dict(eps_fn=float("nan")), dict(num_defined=0), dict(num_defined=P - 1)):
        with pytest.raises(api.GsError):
            ctx.gs_sample_fwd_loss(q, phi, I, t, **kw)
    with pytest.raises(api.GsError):
        ctx.gs_sample_fwd_loss(q, phi, I, None)
    # a valid call with every optional output absent
    ctx.gs_sample_fwd_loss(q, phi, I, t, kind=api.LOSS_L1, lambda_fn=1.0, eps_fn=0.1)
    torch.cuda.synchronize()
    ctx.close()
