"""Pins of the rendering oracle (oracle/wveg_render.py): closed forms of the
emission-absorption quadrature for piecewise-constant media, front-to-back order, the transfer table, the float32 fma."""
import numpy as np
import pytest

from paper_2607_01164_b200 import inputs
from oracle import wveg_render

TAU = 0.01


def _one(mean, sigma, w, v):
    n = len(w)
    quat = np.tile(np.array([1, 0, 0, 0], np.float32), (n, 1))
    return inputs.Gaussians(np.asarray(mean, np.float32), np.repeat(np.asarray(sigma, np.float32)[:, None], 3, axis=1), quat,
                            np.asarray(w, np.float32), np.asarray(v, np.float32))


def test_fmaf32_is_correctly_rounded():
    rng = np.random.default_rng(0)
    a, b, c = (rng.standard_normal(20000).astype(np.float32) for _ in range(3))
    c[::7] = (-a[::7].astype(np.float64) * b[::7].astype(np.float64)).astype(np.float32)   # heavy cancellation
    got = wveg_render._fmaf32(a, b, c)
    from fractions import Fraction
    for i in range(0, 20000, 97):
        exact = Fraction(float(a[i])) * Fraction(float(b[i])) + Fraction(float(c[i]))
        lo, hi = np.nextafter(got[i], np.float32(-np.inf)), np.nextafter(got[i], np.float32(np.inf))
        err = abs(Fraction(float(got[i])) - exact)
        assert err <= abs(Fraction(float(lo)) - exact) and err <= abs(Fraction(float(hi)) - exact)


def test_transfer_table_interpolates_linearly():
    tab = np.array([[0, 0, 0, 0], [1, 2, 3, 4], [3, 2, 1, 0]], np.float32)
    got = wveg_render.transfer(tab, np.array([-1.0, 0.0, 0.25, 0.5, 0.75, 1.0, 7.0]))
    want = np.array([[0, 0, 0, 0], [0, 0, 0, 0], [.5, 1, 1.5, 2], [1, 2, 3, 4], [2, 2, 2, 2], [3, 2, 1, 0], [3, 2, 1, 0]])
    np.testing.assert_allclose(got, want, atol=1e-15)


def test_constant_medium_closed_form():
    # one isotropic Gaussian: Phi = v wherever covered (Eq. 2), covered iff w exp(-r^2 / 2 s^2) > tau, i.e. inside the
    # sphere of radius s sqrt(2 ln(w / tau)).  A ray through the centre sees a constant medium over the covered chord:
    # A = 1 - exp(-sigma(v) * n_cov * dt), C = rgb(v) * A  (prod (1 - alpha) telescopes exactly)
    s, w, v = 0.1, 0.8, 0.65
    g = _one([[0.5, 0.5, 0.5]], [s], [w], [v])
    R = s * np.sqrt(2.0 * np.log(np.float32(w) / np.float32(TAU)))
    o = np.array([[0.5, 0.5, -1.0], [0.5, 0.5 + 0.5 * R, -1.0], [0.5, 0.5 + 1.5 * R, -1.0]], np.float32)
    d = np.tile(np.array([0, 0, 1], np.float32), (3, 1))
    tr = np.tile(np.array([1.0, 2.0], np.float32), (3, 1))
    spp = 400
    tab = inputs.diverging_transfer(64, extinction=9.0)
    out = wveg_render.render(g, o, d, tr, spp, tab, TAU, mode=0)
    dt = 1.0 / spp
    z = 1.0 + (np.arange(spp) + 0.5) * dt - 1.0
    col = wveg_render.transfer(tab, np.float64(np.float32(v)))
    for ray, off in enumerate((0.0, 0.5 * R, 1.5 * R)):
        rr = np.sqrt((z - 0.5) ** 2 + off ** 2)
        ncov = int((rr < R - 1e-6).sum())
        assert int(out["covered"][ray].sum()) in (ncov, ncov + 1, ncov + 2)   # samples within 1e-6 of the sphere may go either way
        ncov = int(out["covered"][ray].sum())
        A = 1.0 - np.exp(-col[3] * ncov * float(np.float32(dt)))
        np.testing.assert_allclose(out["rgba"][ray, 3], A, rtol=1e-6, atol=1e-12)
        np.testing.assert_allclose(out["rgba"][ray, :3], col[:3] * A, rtol=1e-6, atol=1e-12)
    assert out["rgba"][2].max() == 0.0 and out["covered"][2].sum() == 0    # the third ray misses the support


def test_front_to_back_order():
    # two disjoint constant media along the ray: C = c1 A1 + (1 - A1) c2 A2; marching back to front gives another colour
    g = _one([[0.5, 0.5, 0.3], [0.5, 0.5, 0.7]], [0.04, 0.04], [0.9, 0.9], [0.1, 0.9])
    o = np.array([[0.5, 0.5, 0.0]], np.float32)
    d = np.array([[0, 0, 1]], np.float32)
    tr = np.array([[0.0, 1.0]], np.float32)
    spp = 500
    tab = inputs.diverging_transfer(32, extinction=30.0)
    out = wveg_render.render(g, o, d, tr, spp, tab, TAU, mode=0)
    cov, phi = out["covered"][0], out["phi"][0]
    first, second = cov & (np.arange(spp) < spp // 2), cov & (np.arange(spp) >= spp // 2)
    assert first.sum() > 20 and second.sum() > 20
    np.testing.assert_allclose(phi[first], np.float32(0.1), rtol=1e-12)
    np.testing.assert_allclose(phi[second], np.float32(0.9), rtol=1e-12)
    dt = float(np.float32(1.0) / np.float32(spp))
    c1, c2 = wveg_render.transfer(tab, float(np.float32(0.1))), wveg_render.transfer(tab, float(np.float32(0.9)))
    A1, A2 = 1 - np.exp(-c1[3] * first.sum() * dt), 1 - np.exp(-c2[3] * second.sum() * dt)
    np.testing.assert_allclose(out["rgba"][0, :3], c1[:3] * A1 + (1 - A1) * c2[:3] * A2, rtol=1e-9)
    np.testing.assert_allclose(out["rgba"][0, 3], 1 - (1 - A1) * (1 - A2), rtol=1e-9)
    wrong = c2[:3] * A2 + (1 - A2) * c1[:3] * A1
    assert np.abs(out["rgba"][0, :3] - wrong).max() > 1e-3


def test_rays_that_miss_the_box_are_empty():
    g = inputs.c1_gaussians(seed=0, n=64)
    o, d, tr = inputs.camera_rays(6, 5, eye=(3.0, 3.0, 3.0), look_at=(9.0, 9.0, 9.0))   # looking away from the unit box
    assert np.all(tr[:, 1] <= tr[:, 0])
    out = wveg_render.render(g, o, d, tr, 16, inputs.diverging_transfer(), TAU, mode=0)
    assert np.all(out["rgba"] == 0.0)


def test_camera_rays_by_hand():
    o, d, tr = inputs.camera_rays(3, 3, eye=(0.5, -2.0, 0.5), look_at=(0.5, 0.5, 0.5), up=(0, 0, 1), fov_y_deg=90.0)
    np.testing.assert_allclose(d[4], [0, 1, 0], atol=1e-7)                       # centre pixel looks along +y
    np.testing.assert_allclose(tr[4], [2.0, 3.0], atol=1e-6)                     # enters the unit box at y = 0, leaves at y = 1
    c = np.array([-2 / 3, 1, 2 / 3]); c /= np.linalg.norm(c)                      # top-left pixel: x = -2/3 tan45, z = +2/3
    np.testing.assert_allclose(d[0], c, atol=1e-6)
