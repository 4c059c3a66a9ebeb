"""Pins of the oracle's analytic gradients (PAPER.md:130, :140 name them; the paper prints no formulas).

* central finite differences of the oracle's own forward, in double, with the hit and coverage
  sets frozen (Phi is discontinuous where a support boundary or the I = tau threshold crosses a
  sample; the analytic gradient ignores that, like the paper's);
* sum rules that follow from Eq. 2 alone (partition of unity, degree-0 homogeneity in w);
* the constant-scalar model has no gradient except through dL/dI.
"""
import numpy as np
import pytest

from paper_2607_01164_b200 import inputs

TAU = 0.01


def _setup(seed=0, n=24, res=7):
    g = inputs.c1_gaussians(seed=seed, n=n)
    # larger Gaussians so that every one of them has many hits on a coarse grid
    g.scale[:] = (g.scale * 4.0).astype(np.float32)
    # non-unit quaternions: the normalisation Jacobian must be exercised
    rng = np.random.default_rng(seed + 100)
    g.quat[:] = (g.quat * rng.uniform(0.5, 2.0, (n, 1))).astype(np.float32)
    return g, rng


def _loss(oracle, g, xyz, ca, cb, mask, covered):
    out = oracle.forward(g, xyz, TAU, mode=0, hit_mask_in=mask, covered_in=covered, want_sets=False)
    return float(np.dot(ca, out["phi"]) + np.dot(cb, out["I"]))


@pytest.mark.parametrize("with_b", [False, True])
def test_finite_differences(oracle, with_b):
    g, rng = _setup()
    xyz = oracle.grid_points(inputs.c1_grid(7))
    P = xyz.shape[0]
    base = oracle.forward(g, xyz, TAU, mode=0, want_mask=True)
    mask = base["hit_mask"]
    covered = (base["I"].astype(np.float32) > np.float32(TAU)).astype(np.uint8)
    assert covered.sum() > P // 2 and mask.sum() > 20 * g.n
    ca = rng.standard_normal(P)
    cb = rng.standard_normal(P) if with_b else np.zeros(P)
    grads = oracle.backward(g, xyz, base["phi"], base["I"], ca, cb if with_b else None, None, TAU, mode=0,
                            hit_mask_in=mask, covered_in=covered)
    fields = dict(mean="dmean", scale="dscale", quat="dquat", opacity="dopacity", scalar="dscalar")
    for name, gname in fields.items():
        arr = getattr(g, name)
        ana = grads[gname].reshape(arr.shape)
        num = np.zeros(arr.shape, np.float64)
        it = np.nditer(arr, flags=["multi_index"])
        for _ in it:
            idx = it.multi_index
            if idx[0] >= 6:  # six Gaussians, every component
                continue
            x0 = arr[idx]
            # step is an exactly representable fp32 increment
            h = np.float32(abs(x0) * 2e-5 + 2e-6)
            xp, xm = np.float32(x0 + h), np.float32(x0 - h)
            arr[idx] = xp
            lp = _loss(oracle, g, xyz, ca, cb, mask, covered)
            arr[idx] = xm
            lm = _loss(oracle, g, xyz, ca, cb, mask, covered)
            arr[idx] = x0
            num[idx] = (lp - lm) / (float(xp) - float(xm))
        sel = (slice(0, 6),) + (slice(None),) * (arr.ndim - 1)
        scale = np.abs(ana[sel]).max() + 1e-30
        err = np.abs(num[sel] - ana[sel]).max() / scale
        assert err < 2e-5, (name, err, num[sel], ana[sel])
        assert np.abs(ana[sel]).max() > 0


def test_sum_rules(oracle):
    g = inputs.c1_gaussians(seed=0, n=1024)
    grid = inputs.c1_grid(20)
    xyz = oracle.grid_points(grid)
    P = xyz.shape[0]
    rng = np.random.default_rng(5)
    target = rng.uniform(0, 1, P).astype(np.float32)
    fwd = oracle.forward(g, xyz, TAU, mode=1)
    loss, a, serr = oracle.mse(fwd["phi"], fwd["I"], target, TAU)
    covered = fwd["I"].astype(np.float32) > np.float32(TAU)
    gr = oracle.backward(g, xyz, fwd["phi"], fwd["I"], a, None, target, TAU, mode=1)
    # partition of unity: sum_i w_i G_ic / I_c = 1  =>  sum_i dL/dv_i = sum_{c covered} a_c
    assert gr["dscalar"].sum() == pytest.approx(a[covered].sum(), rel=1e-10)
    # Phi is homogeneous of degree 0 in the weights: sum_i w_i dL/dw_i = 0 when dL/dI = 0
    wdw = g.opacity.astype(np.float64) * gr["dopacity"]
    assert abs(wdw.sum()) < 1e-12 * np.abs(wdw).sum()
    # error statistic (DESIGN D10) distributes each covered sample's |res| over its contributors
    assert gr["err"].sum() == pytest.approx(serr[covered].sum(), rel=1e-10)
    assert np.all(gr["err"] >= 0)
    # quaternion gradient is orthogonal to q (Phi does not depend on |q|)
    qdot = (g.quat.astype(np.float64) * gr["dquat"]).sum(1)
    assert np.abs(qdot).max() < 1e-12 * (np.abs(gr["dquat"]).max() + 1e-30)
    # all-pairs and culled backward agree
    gr0 = oracle.backward(g, xyz, fwd["phi"], fwd["I"], a, None, target, TAU, mode=0)
    for k in gr:
        np.testing.assert_allclose(gr[k], gr0[k], rtol=1e-9, atol=1e-18, err_msg=k)


def test_constant_scalar_has_no_shape_gradient(oracle):
    g = inputs.c1_gaussians(seed=9, n=256)
    g.scalar[:] = 0.375
    xyz = oracle.grid_points(inputs.c1_grid(12))
    rng = np.random.default_rng(2)
    a = rng.standard_normal(xyz.shape[0])
    fwd = oracle.forward(g, xyz, TAU, mode=1)
    gr = oracle.backward(g, xyz, fwd["phi"], fwd["I"], a, None, None, TAU, mode=1)
    ref = np.abs(a).sum()
    for k in ("dmean", "dscale", "dquat", "dopacity"):
        assert np.abs(gr[k]).max() < 1e-9 * ref, k
    assert np.abs(gr["dscalar"]).max() > 0
    # with dL/dI present the shape gradients come alive
    b = rng.standard_normal(xyz.shape[0])
    gr = oracle.backward(g, xyz, fwd["phi"], fwd["I"], a, b, None, TAU, mode=1)
    assert np.abs(gr["dmean"]).max() > 1e-3


def test_dI_gradient_of_total_influence(oracle):
    # L = sum_c I_c for one isotropic Gaussian has a closed form per sample: dI/dw = G
    g = inputs.Gaussians(np.array([[0.5, 0.5, 0.5]], np.float32), np.array([[0.2, 0.2, 0.2]], np.float32),
                         np.array([[1, 0, 0, 0]], np.float32), np.array([0.5], np.float32), np.array([0.25], np.float32))
    xyz = oracle.grid_points(inputs.c1_grid(6))
    fwd = oracle.forward(g, xyz, TAU, mode=0)
    P = xyz.shape[0]
    gr = oracle.backward(g, xyz, fwd["phi"], fwd["I"], np.zeros(P), np.ones(P), None, TAU, mode=0)
    d = xyz.astype(np.float64) - 0.5
    s = float(np.float32(0.2))
    d2 = (d ** 2).sum(1)
    hit = fwd["count"] == 1
    G = np.exp(-0.5 * d2 / s ** 2) * hit
    assert gr["dopacity"][0] == pytest.approx(G.sum(), rel=1e-12)
    # dI/dmu = w G d / sigma^2 ; dI/dsigma_j = w G d_j^2 / sigma^3
    np.testing.assert_allclose(gr["dmean"][0], (0.5 * G[:, None] * d / s ** 2).sum(0), rtol=1e-10, atol=1e-12)
    np.testing.assert_allclose(gr["dscale"][0], (0.5 * G[:, None] * d ** 2 / s ** 3).sum(0), rtol=1e-10)
    assert gr["dscalar"][0] == 0.0
