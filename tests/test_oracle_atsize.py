"""Pins of the oracle at the sizes the GPU parity tests use it at ("oracle loose ends").

* At configs[1] / configs[2] scale the oracle only ever runs with its cell-grid cull (mode = 1,
  oracle/wveg_oracle.c cellgrid_*), the one part of it that is not checkable by eye.  Here the plain
  all-pairs definition (mode = 0: every point against every Gaussian, Eq. 2/3 PAPER.md:84-89 with
  the per-pair cutoff of PAPER.md:116) is run against the FULL 1,048,576-Gaussian configs[2] model
  and the FULL 262,144-Gaussian configs[1] model on point subsets small enough for all-pairs, and
  must give identical ID sets, I and Phi, and the same gradients.
* The per-Gaussian error statistic E_i (DESIGN D10; north_star's, the paper defines none) gets two
  closed forms beside its sum rule: Gaussians with disjoint supports (E_i = sum over its covered
  samples of |v_i - t_c|, since Phi = v_i and w_i G / I = 1 there) and coincident Gaussians (Phi is the
  weighted mean of the values and the error is shared in proportion to the weights).
"""
import numpy as np
import pytest

from paper_2607_01164_b200 import inputs

TAU = 0.01


def _same_forward(a, b):
    assert np.array_equal(a["count"], b["count"])
    assert np.array_equal(a["hsum"], b["hsum"])
    assert np.array_equal(a["hxor"], b["hxor"])
    # the same pairs are summed in the same (ascending id) order: bit-identical doubles
    assert np.array_equal(a["I"], b["I"])
    assert np.array_equal(a["phi"], b["phi"])


def test_cull_equals_all_pairs_full_c3_model(oracle):
    xyz_all, t_all = inputs.c3_points()
    g = inputs.c3_gaussians(xyz_all, t_all)
    assert g.n == 1_048_576
    idx = inputs.batch_indices(33, 0, len(xyz_all), 4096)
    xyz, target = np.ascontiguousarray(xyz_all[idx]), np.ascontiguousarray(t_all[idx])
    plain = oracle.forward(g, xyz, TAU, mode=0)
    culled = oracle.forward(g, xyz, TAU, mode=1)
    assert int(plain["count"].astype(np.int64).sum()) > 1_000_000   # ~445 hits per point
    _same_forward(plain, culled)
    _, a, _ = oracle.mse(plain["phi"], plain["I"], target, TAU)
    b = np.random.default_rng(5).standard_normal(len(xyz)) * 1e-3
    g0 = oracle.backward(g, xyz, plain["phi"], plain["I"], a, b, target, TAU, mode=0)
    g1 = oracle.backward(g, xyz, plain["phi"], plain["I"], a, b, target, TAU, mode=1)
    for k in g0:
        # the cell grid visits a Gaussian's points in another order: equal up to double rounding
        scale = max(np.abs(g0[k]).max(), 1e-300)
        assert np.abs(g0[k] - g1[k]).max() <= 1e-12 * scale, k


def test_cull_equals_all_pairs_full_c2_model(oracle):
    g = inputs.c2_gaussians(seed=2, n_grid=256, n=262144)
    grid = inputs.c2_grid(256)
    # a 32^3 batch away from the grid's corner, so that Gaussians reach it from every side
    sub = grid.batch((9, 17, 5), (4, 4, 4))
    xyz = oracle.grid_points(sub)
    target = inputs.c2_target(sub)
    plain = oracle.forward(g, xyz, TAU, mode=0)
    culled = oracle.forward(g, xyz, TAU, mode=1)
    assert int(plain["count"].astype(np.int64).sum()) > 150_000     # ~6 hits per sample
    _same_forward(plain, culled)
    _, a, _ = oracle.mse(plain["phi"], plain["I"], target, TAU)
    g0 = oracle.backward(g, xyz, plain["phi"], plain["I"], a, None, target, TAU, mode=0)
    g1 = oracle.backward(g, xyz, plain["phi"], plain["I"], a, None, target, TAU, mode=1)
    touched = 0
    for k in g0:
        scale = max(np.abs(g0[k]).max(), 1e-300)
        assert np.abs(g0[k] - g1[k]).max() <= 1e-12 * scale, k
        touched = max(touched, int(np.count_nonzero(g0[k].reshape(g.n, -1).any(axis=1))))
    assert 500 < touched < g.n // 50   # a small batch of a large model: most Gaussians miss it (the skip path)


def _two(mean, scale, w, v):
    n = len(w)
    quat = np.tile(np.array([1, 0, 0, 0], np.float32), (n, 1))
    return inputs.Gaussians(np.asarray(mean, np.float32), np.asarray(scale, np.float32), quat, np.asarray(w, np.float32),
                            np.asarray(v, np.float32))


def test_error_statistic_disjoint_gaussians(oracle):
    # two Gaussians 0.5 apart with sigma 0.04: supports (radius 3.03 sigma = 0.12) do not meet
    g = _two([[0.25, 0.5, 0.5], [0.75, 0.5, 0.5]], [[0.04] * 3, [0.04] * 3], [0.6, 0.3], [0.2, 0.9])
    xyz = oracle.grid_points(inputs.c1_grid(24))
    rng = np.random.default_rng(0)
    target = rng.uniform(0, 1, len(xyz)).astype(np.float32)
    fwd = oracle.forward(g, xyz, TAU, mode=0, want_mask=True)
    assert not np.any(fwd["hit_mask"][:, 0] & fwd["hit_mask"][:, 1])
    covered = fwd["I"].astype(np.float32) > np.float32(TAU)
    _, a, _ = oracle.mse(fwd["phi"], fwd["I"], target, TAU)
    gr = oracle.backward(g, xyz, fwd["phi"], fwd["I"], a, None, target, TAU, mode=0)
    for i in range(2):
        mine = covered & (fwd["hit_mask"][:, i] != 0)
        assert mine.sum() > 20
        # where only Gaussian i reaches, Phi = v_i and its share w_i G / I is 1: E_i = sum |v_i - t|
        want = np.abs(np.float64(g.scalar[i]) - target[mine].astype(np.float64)).sum()
        assert gr["err"][i] == pytest.approx(want, rel=1e-12)


def test_error_statistic_coincident_gaussians(oracle):
    # three Gaussians with the same mean, scale and rotation: Phi = sum w v / sum w wherever covered and every sample's
    # error is shared in proportion to the weights
    w = np.array([0.5, 0.25, 0.125])
    v = np.array([0.1, 0.7, 0.4])
    g = _two([[0.5, 0.5, 0.5]] * 3, [[0.05, 0.08, 0.11]] * 3, w, v)
    w, v = g.opacity.astype(np.float64), g.scalar.astype(np.float64)   # the fp32 values the oracle sees
    xyz = oracle.grid_points(inputs.c1_grid(20))
    rng = np.random.default_rng(1)
    target = rng.uniform(0, 1, len(xyz)).astype(np.float32)
    fwd = oracle.forward(g, xyz, TAU, mode=0)
    covered = fwd["I"].astype(np.float32) > np.float32(TAU)
    assert covered.sum() > 50
    mean_v = float((w * v).sum() / w.sum())
    assert np.abs(fwd["phi"][covered] - mean_v).max() < 1e-12
    total = np.abs(mean_v - target[covered].astype(np.float64)).sum()
    _, a, _ = oracle.mse(fwd["phi"], fwd["I"], target, TAU)
    gr = oracle.backward(g, xyz, fwd["phi"], fwd["I"], a, None, target, TAU, mode=0)
    for i in range(3):
        assert gr["err"][i] == pytest.approx(w[i] / w.sum() * total, rel=1e-10)
