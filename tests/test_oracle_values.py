"""Pins of the oracle's VALUE arithmetic (forward) against what the paper and mathematics fix.

None of these retypes the oracle's formula: they use closed forms, scipy's multivariate normal pdf
and rotation routines, hand-computed special cases, and structural properties of Eq. 2.
Citations are PAPER.md:<line>.
"""
import math
import os

import numpy as np
import pytest

from paper_2607_01164_b200 import inputs

TAU = 0.01


def _golden():
    out = {}
    path = os.path.join(os.path.dirname(__file__), "golden", "paper_constants.txt")
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        name, value = line.split()[:2]
        out[name] = value
    return out


def _one(mean=(0.5, 0.5, 0.5), scale=(0.1, 0.1, 0.1), quat=(1, 0, 0, 0), w=0.7, v=0.3):
    return inputs.Gaussians(np.array([mean], np.float32), np.array([scale], np.float32), np.array([quat], np.float32),
                            np.array([w], np.float32), np.array([v], np.float32))


def test_cutoff_constant(oracle):
    # tau_1 = 0.01; support G >= tau <=> |u|^2 <= -2 ln tau
    assert float(_golden()["tau1"]) == TAU
    assert abs(oracle.r2(TAU) - (-2.0 * math.log(0.01))) < 1e-6
    assert abs(oracle.r2(TAU) - 9.2103404) < 1e-6


def test_weight_at_mean(oracle):
    # Eq. 3: G_i(mu_i) = e^0 = 1, so I = w exactly and Phi = v
    g = _one(w=0.7, v=0.3, scale=(0.03, 0.2, 0.07), quat=(0.3, -0.5, 0.1, 0.8))
    out = oracle.forward(g, g.mean, TAU, mode=0)
    assert out["I"][0] == float(np.float32(0.7))
    assert out["phi"][0] == pytest.approx(float(np.float32(0.3)), rel=1e-15)
    assert out["count"][0] == 1


def test_single_isotropic_closed_form(oracle):
    # I(p) = w exp(-|p-mu|^2 / (2 sigma^2)); Phi = v where I > tau, else the empty value 0
    sigma, w, v = 0.1, 0.7, 0.3
    g = _one(scale=(sigma,) * 3, w=w, v=v)
    rng = np.random.default_rng(1)
    xyz = (0.5 + rng.uniform(-0.45, 0.45, (400, 3))).astype(np.float32)
    out = oracle.forward(g, xyz, TAU, mode=0)
    d2 = ((xyz.astype(np.float64) - g.mean.astype(np.float64)) ** 2).sum(1)
    s64 = float(np.float32(sigma))
    G = np.exp(-0.5 * d2 / s64 ** 2)
    inside = G >= TAU * (1 + 1e-5)
    outside = G <= TAU * (1 - 1e-5)
    assert inside.sum() > 50 and outside.sum() > 50
    w64, v64 = float(np.float32(w)), float(np.float32(v))
    np.testing.assert_allclose(out["I"][inside], w64 * G[inside], rtol=1e-12)
    assert np.all(out["I"][outside] == 0.0) and np.all(out["count"][outside] == 0)
    covered = inside & (w64 * G > TAU * (1 + 1e-5))
    np.testing.assert_allclose(out["phi"][covered], v64, rtol=1e-12)
    # hit but w*G <= tau: influence is reported, value is the empty value (DESIGN D5)
    weak = inside & (w64 * G < TAU * (1 - 1e-5))
    assert weak.sum() > 0
    assert np.all(out["phi"][weak] == 0.0) and np.all(out["I"][weak] > 0.0)


def test_support_radius(oracle):
    # G = tau exactly at Mahalanobis radius sqrt(-2 ln tau) = 3.0348543
    sigma = 0.05
    g = _one(scale=(sigma,) * 3, w=1.0, v=1.0)
    r = math.sqrt(-2.0 * math.log(TAU))
    assert abs(r - 3.0348543) < 1e-6
    s64 = float(np.float32(sigma))
    dirs = np.array([[1, 0, 0], [0, 1, 0], [0, 0, 1], [1, 1, 1], [-1, 2, 0.5]], np.float64)
    dirs /= np.linalg.norm(dirs, axis=1, keepdims=True)
    pin = (0.5 + dirs * r * s64 * (1 - 1e-4)).astype(np.float32)
    pout = (0.5 + dirs * r * s64 * (1 + 1e-4)).astype(np.float32)
    oin = oracle.forward(g, pin, TAU, mode=0)
    oout = oracle.forward(g, pout, TAU, mode=0)
    assert np.all(oin["count"] == 1) and np.all(oout["count"] == 0)
    np.testing.assert_allclose(oin["I"], TAU, rtol=2e-3)


def test_rotation_convention_by_hand(oracle):
    # DESIGN D1 (Eq. 3 read literally, u = S^-1 R d): q = rotation by 90 deg about z maps world x onto
    # principal axis 1, so the fall-off along world x uses sigma_1 (= b), along world y sigma_0 (= a).
    a, b, c = 0.02, 0.08, 0.05
    q = (math.cos(math.pi / 4), 0.0, 0.0, math.sin(math.pi / 4))
    g = _one(scale=(a, b, c), quat=q, w=1.0, v=1.0)
    t = 0.03
    xyz = np.array([[0.5 + t, 0.5, 0.5], [0.5, 0.5 + t, 0.5], [0.5, 0.5, 0.5 + t]], np.float32)
    out = oracle.forward(g, xyz, TAU, mode=0)
    d = xyz.astype(np.float64) - 0.5
    a64, b64, c64 = (float(np.float32(s)) for s in (a, b, c))
    expect = [math.exp(-0.5 * (d[0, 0] / b64) ** 2), math.exp(-0.5 * (d[1, 1] / a64) ** 2), math.exp(-0.5 * (d[2, 2] / c64) ** 2)]
    np.testing.assert_allclose(out["I"], expect, rtol=1e-6)  # rtol: fp32 quaternion (cos, sin) rounding


def test_against_scipy_normal_pdf(oracle):
    # Eq. 3: R^T S^-2 R is the inverse covariance, so G = pdf * (2 pi)^{3/2} |Sigma|^{1/2}
    scipy_stats = pytest.importorskip("scipy.stats")
    from scipy.spatial.transform import Rotation
    rng = np.random.default_rng(7)
    for trial in range(5):
        q = rng.standard_normal(4)
        q /= np.linalg.norm(q)
        s = np.exp(rng.uniform(np.log(0.05), np.log(0.3), 3))
        g = _one(scale=tuple(s), quat=tuple(q), w=1.0, v=1.0)
        q32 = g.quat[0].astype(np.float64)
        q32 /= np.linalg.norm(q32)
        R = Rotation.from_quat([q32[1], q32[2], q32[3], q32[0]]).as_matrix()  # scipy is scalar-last
        S2 = np.diag(g.scale[0].astype(np.float64) ** 2)
        cov = R.T @ S2 @ R  # inverse of R^T S^-2 R
        xyz = (0.5 + rng.uniform(-0.1, 0.1, (200, 3))).astype(np.float32)
        out = oracle.forward(g, xyz, TAU, mode=0)
        pdf = scipy_stats.multivariate_normal(mean=g.mean[0].astype(np.float64), cov=cov).pdf(xyz.astype(np.float64))
        G = pdf * (2 * np.pi) ** 1.5 * np.sqrt(np.linalg.det(cov))
        hit = out["count"] == 1
        assert hit.sum() > 20
        np.testing.assert_allclose(out["I"][hit], G[hit], rtol=1e-10)
        # membership: G >= tau, except within rounding of the boundary
        assert np.all(hit[G > TAU * (1 + 1e-4)]) and not np.any(hit[G < TAU * (1 - 1e-4)])


def test_constant_scalar_collection(oracle):
    # Eq. 2 is a weighted average: a collection with one common scalar reproduces it
    # wherever it is covered; uncovered points return the empty value 0 (DESIGN D5).
    g = inputs.c1_gaussians(seed=0, n=512)
    g.scalar[:] = 0.625
    xyz = oracle.grid_points(inputs.c1_grid(16))
    out = oracle.forward(g, xyz, TAU, mode=1)
    covered = out["I"].astype(np.float32) > np.float32(TAU)
    assert covered.sum() > 100 and (~covered).sum() > 100
    np.testing.assert_allclose(out["phi"][covered], 0.625, rtol=1e-13)
    assert np.all(out["phi"][~covered] == 0.0)


def test_convexity_and_set_definition(oracle):
    # Phi_c lies between the min and max scalar of the Gaussians whose support contains c (Eq. 2)
    g = inputs.c1_gaussians(seed=3, n=300)
    xyz = oracle.grid_points(inputs.c1_grid(12))
    out = oracle.forward(g, xyz, TAU, mode=0, want_mask=True)
    mask = out["hit_mask"].astype(bool)
    assert np.array_equal(mask.sum(1), out["count"])
    v = g.scalar.astype(np.float64)
    covered = out["I"].astype(np.float32) > np.float32(TAU)
    vmin = np.where(mask, v[None, :], np.inf).min(1)
    vmax = np.where(mask, v[None, :], -np.inf).max(1)
    assert np.all(out["phi"][covered] >= vmin[covered] - 1e-12)
    assert np.all(out["phi"][covered] <= vmax[covered] + 1e-12)
    # membership agrees with the double-precision Mahalanobis test away from the boundary (scipy rotation)
    from scipy.spatial.transform import Rotation
    q = g.quat.astype(np.float64)
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    R = Rotation.from_quat(np.concatenate([q[:, 1:], q[:, :1]], axis=1)).as_matrix()
    d = xyz.astype(np.float64)[:, None, :] - g.mean.astype(np.float64)[None, :, :]
    u = np.einsum("njk,pnk->pnj", R, d) / g.scale.astype(np.float64)[None, :, :]
    qd = (u ** 2).sum(-1)
    r2 = -2.0 * math.log(TAU)
    assert np.all(mask[qd < r2 * (1 - 1e-5)]) and not np.any(mask[qd > r2 * (1 + 1e-5)])
    # and the values follow Eq. 2 with that kernel
    wG = np.where(mask, g.opacity.astype(np.float64)[None, :] * np.exp(-0.5 * qd), 0.0)
    np.testing.assert_allclose(out["I"], wG.sum(1), rtol=1e-9, atol=1e-300)
    np.testing.assert_allclose(out["phi"][covered], ((wG * v[None, :]).sum(1) / wG.sum(1))[covered], rtol=1e-9)


def test_weight_split_invariance(oracle):
    # relocating k copies onto one Gaussian with weight w/k keeps Eq. 2 "exactly equal"
    g = inputs.c1_gaussians(seed=5, n=64)
    g.opacity[:] = (g.opacity * 0.5 + 0.25).astype(np.float32)
    xyz = oracle.grid_points(inputs.c1_grid(10))
    base = oracle.forward(g, xyz, TAU, mode=0)
    k = 4
    idx = np.concatenate([np.arange(64), np.repeat(np.arange(8), k - 1)])
    g2 = g.subset(idx)
    split = np.isin(idx, np.arange(8))
    g2.opacity[split] = (g2.opacity[split].astype(np.float64) / k).astype(np.float32)  # /4 is exact in fp32
    out = oracle.forward(g2, xyz, TAU, mode=0)
    np.testing.assert_allclose(out["I"], base["I"], rtol=1e-13)
    np.testing.assert_allclose(out["phi"], base["phi"], rtol=1e-12, atol=0)


def test_culled_equals_all_pairs(oracle):
    # the cell-grid cull only removes pairs the plain all-pairs definition rejects too
    for seed, n, res in ((0, 1024, 20), (11, 200, 9)):
        g = inputs.c1_gaussians(seed=seed, n=n)
        xyz = oracle.grid_points(inputs.c1_grid(res))
        a = oracle.forward(g, xyz, TAU, mode=0)
        b = oracle.forward(g, xyz, TAU, mode=1)
        for k in ("count", "hsum", "hxor"):
            assert np.array_equal(a[k], b[k]), k
        assert np.array_equal(a["I"], b["I"]) and np.array_equal(a["phi"], b["phi"])  # same order (ascending id)
    # unstructured points, anisotropic model
    xyz, t = inputs.c3_points(seed=3, p=4000)
    g = inputs.c3_gaussians(xyz, t, seed=3, n=500, sigma_lo=0.01, sigma_hi=0.08)
    a = oracle.forward(g, xyz, TAU, mode=0)
    b = oracle.forward(g, xyz, TAU, mode=1)
    assert a["count"].sum() > 10000
    for k in ("count", "hsum", "hxor", "I", "phi"):
        assert np.array_equal(a[k], b[k]), k


def test_invalid_gaussians_are_empty(oracle):
    g = inputs.c1_gaussians(seed=2, n=32)
    ref = oracle.forward(g.subset(np.arange(4, 32)), oracle.grid_points(inputs.c1_grid(8)), TAU, mode=0)
    g.scale[0, 1] = 0.0
    g.quat[1] = 0.0
    g.mean[2, 0] = np.nan
    g.opacity[3] = np.inf
    out = oracle.forward(g, oracle.grid_points(inputs.c1_grid(8)), TAU, mode=0)
    np.testing.assert_array_equal(out["I"], ref["I"])
    np.testing.assert_array_equal(out["count"], ref["count"])


def test_mse_epilogue(oracle):
    rng = np.random.default_rng(0)
    phi = rng.uniform(0, 1, 1000)
    I = rng.uniform(0, 0.02, 1000)
    t = rng.uniform(0, 1, 1000).astype(np.float32)
    loss, d, e = oracle.mse(phi, I, t, TAU)
    assert loss == pytest.approx(float(np.mean((phi - t) ** 2)), rel=1e-13)
    cov = I.astype(np.float32) > np.float32(TAU)
    # derivative of the mean-squared error, zero where the sample is uncovered (DESIGN D5)
    h = 1e-6
    num = np.array([(np.mean((phi + h * (np.arange(1000) == c) - t) ** 2) - np.mean((phi - h * (np.arange(1000) == c) - t) ** 2)) / (2 * h)
                    for c in range(0, 1000, 97)])
    np.testing.assert_allclose(d[::97], np.where(cov[::97], num, 0.0), rtol=1e-6, atol=1e-12)
    np.testing.assert_allclose(e, np.abs(phi - t), rtol=1e-15)


def test_jittered_grid_positions(oracle):
    """In-cell jitter: every sample stays inside its voxel's cell, the generator is the splitmix64
    finaliser written out here with Python integers, positions are uniform in the cell and independent per axis."""
    from paper_2607_01164_b200 import inputs
    M = (1 << 64) - 1

    def mix(z):
        z = (z + 0x9E3779B97F4A7C15) & M
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & M
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & M
        return z ^ (z >> 31)

    for seed, L, a in ((0, 0, 0), (7, 123456789, 2), (2 ** 63 + 5, 2 ** 40 + 3, 1)):
        want = ((mix((seed + L) & M) >> (21 * a)) & (2 ** 21 - 1)) / 2.0 ** 21 - 0.5
        assert oracle.jitter(seed, L, a) == want and -0.5 <= want < 0.5
    grid = inputs.Grid((20, 13, 9), (-0.3, 0.1, 0.0), (0.05, 0.04, 0.1))
    sub = grid.batch((1, 0, 0), (1, 2, 1))
    centres = oracle.grid_points(sub).astype(np.float64)
    a = oracle.grid_points(sub, jitter_seed=11).astype(np.float64)
    b = oracle.grid_points(sub, jitter_seed=12).astype(np.float64)
    assert np.array_equal(a, oracle.grid_points(sub, jitter_seed=11).astype(np.float64)) and not np.array_equal(a, b)
    frac = (a - centres) / np.asarray(grid.spacing)
    assert np.all(np.abs(frac) <= 0.5 + 1e-5)
    # the batch's samples are those of the whole grid (the counter is the GLOBAL voxel index)
    full = oracle.grid_points(grid, jitter_seed=11).reshape(9, 13, 20, 3)
    assert np.array_equal(a.reshape(8, 13, 8, 3), full[0:8, 0:13, 8:16].astype(np.float64))
    big = inputs.Grid((64, 64, 32), (0, 0, 0), (1, 1, 1))
    f = oracle.grid_points(big, jitter_seed=3).astype(np.float64) - oracle.grid_points(big).astype(np.float64)
    assert abs(f.mean()) < 2e-3 and abs(f.var() - 1 / 12) < 2e-3             # uniform on [-0.5, 0.5)
    assert np.all(np.abs(np.corrcoef(f.T) - np.eye(3)) < 0.01)               # axes independent
