"""Pins of the oracle's pruning and sample-error densification (oracle.prune, oracle.densify_select, oracle.densify;
PAPER.md:144, :154, :166) against plain loops on tiny inputs and the properties the paper states."""
import numpy as np


def test_prune_by_plain_loop(oracle):
    rng = np.random.default_rng(0)
    n = 40
    p = dict(mean=rng.uniform(0, 1, (n, 3)), raw_scale=rng.uniform(-5, -3, (n, 3)), quat=rng.standard_normal((n, 4)),
             raw_opacity=rng.standard_normal(n), raw_scalar=rng.standard_normal(n))
    m, v = rng.standard_normal(12 * n), rng.uniform(0, 1, 12 * n)
    w = rng.uniform(0, 0.01, n).astype(np.float32)
    w[3] = np.float32(0.005)  # exactly the threshold stays ("below" is removed)
    p2, m2, v2, keep = oracle.prune(p, m, v, w, 0.005)
    want = [i for i in range(n) if float(w[i]) >= float(np.float32(0.005))]
    assert keep.tolist() == want and 3 in want and 0 < len(want) < n
    n2 = len(want)
    for j, i in enumerate(want):  # every kept Gaussian carries its parameters and both moments of every element
        assert np.array_equal(p2["quat"][j], p["quat"][i]) and p2["raw_scalar"][j] == p["raw_scalar"][i]
        assert np.array_equal(m2[3 * j:3 * j + 3], m[3 * i:3 * i + 3])                          # mean block
        assert np.array_equal(m2[6 * n2 + 4 * j:6 * n2 + 4 * j + 4], m[6 * n + 4 * i:6 * n + 4 * i + 4])  # quat block
        assert v2[11 * n2 + j] == v[11 * n + i] and v2[10 * n2 + j] == v[10 * n + i]
    assert len(m2) == 12 * n2 == len(v2)


def test_select_order(oracle):
    # errors (0.5, 0.9, 0.1, 0.9, 0.3, 0.7); sample 4 is a false negative (I <= tau), sample 5 is not defined
    err = np.array([0.5, 0.9, 0.1, 0.9, 0.3, 0.7], np.float32)
    I = np.array([0.2, 0.2, 0.2, 0.2, 0.01, 0.2], np.float32)
    d = np.array([1, 1, 1, 1, 1, 0], np.uint8)
    # false negative first, then highest error, ties by index; undefined never
    assert oracle.densify_select(err, I, d, 4).tolist() == [4, 1, 3, 0]
    assert oracle.densify_select(err, I, d, 99).tolist() == [4, 1, 3, 0, 2]
    assert oracle.densify_select(err, I, None, 3).tolist() == [4, 1, 3]
    assert oracle.densify_select(err, I, None, 6).tolist() == [4, 1, 3, 5, 0, 2]
    # I = tau exactly is uncovered (strict coverage rule)
    rng = np.random.default_rng(1)
    e = rng.uniform(0, 1, 500).astype(np.float32)
    Ii = rng.uniform(0, 0.02, 500).astype(np.float32)
    sel = oracle.densify_select(e, Ii, None, 50)
    nfn = int((Ii <= np.float32(0.01)).sum())
    assert np.all(Ii[sel[:min(50, nfn)]] <= np.float32(0.01))
    assert np.all(np.diff(e[sel[:min(50, nfn)]]) <= 0)  # by error inside the false negatives


def test_densify_appends_initialised_gaussians(oracle):
    rng = np.random.default_rng(2)
    n = 5
    p = dict(mean=rng.uniform(0, 1, (n, 3)), raw_scale=rng.uniform(-5, -3, (n, 3)), quat=rng.standard_normal((n, 4)),
             raw_opacity=rng.standard_normal(n), raw_scalar=rng.standard_normal(n))
    m, v = rng.standard_normal(12 * n), rng.uniform(0, 1, 12 * n)
    pos = rng.uniform(0, 1, (10, 3)).astype(np.float32)
    t = np.array([0.25, 0.5, 0.0, 1.0, 0.75, 0.1, 0.2, 0.3, 0.4, 0.6], np.float32)
    sel = np.array([4, 2, 3])
    p2, m2, v2 = oracle.densify(p, m, v, pos, t, sel, np.log(0.02), np.log(0.01 / 0.99))
    assert len(p2["raw_opacity"]) == 8 and np.array_equal(p2["mean"][:5], p["mean"])
    assert np.array_equal(p2["mean"][5:], pos[sel].astype(np.float64))
    # sigmoid(raw_scalar) is the ground-truth value, clipped away from 0 and 1 where the logit diverges
    np.testing.assert_allclose(1 / (1 + np.exp(-p2["raw_scalar"][5:])), [0.75, 1e-4, 1 - 1e-4], rtol=1e-7)
    np.testing.assert_allclose(1 / (1 + np.exp(-p2["raw_opacity"][5:])), 0.01, rtol=1e-6)  # initial weight 0.01
    np.testing.assert_allclose(np.exp(p2["raw_scale"][5:]), 0.02, rtol=1e-6)
    assert np.array_equal(p2["quat"][5:], np.tile([1.0, 0, 0, 0], (3, 1)))
    # moments: old ones in place inside the re-laid-out blocks, new ones zero
    assert np.array_equal(m2[:15], m[:15]) and not m2[15:24].any()
    assert np.array_equal(v2[6 * 8:6 * 8 + 20], v[6 * 5:6 * 5 + 20]) and not v2[6 * 8 + 20:6 * 8 + 32].any()
    assert len(m2) == 96
