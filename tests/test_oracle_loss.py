"""Pins of the oracle's training losses (oracle.loss: L1 / MSE reconstruction over the defined samples, Eq. 4
false-negative term, Eq. 5 false-positive term) against values worked out by hand from
the equations, against central differences, and against the sum rules the normalisations imply."""
import numpy as np
import pytest

TAU = 0.01


def test_eq4_false_negative_by_hand(oracle):
    # Eq. 4 with tau = 0.01, eps = 0.5: threshold (1 + eps) tau = 0.015.
    # I = (0.005, 0.012, 0.02, 0.0149, 0.3): D- = {0, 1, 3}; sum of (0.015 - I) = 0.010 + 0.003 + 0.0001 = 0.0131
    # L_FN = lambda * 0.0131 / 3 with lambda = 6  ->  0.0262
    I = np.array([0.005, 0.012, 0.02, 0.0149, 0.3])
    phi = np.array([0.0, 0.4, 0.5, 0.6, 0.7])
    t = phi.astype(np.float32)  # zero reconstruction residual where covered
    r = oracle.loss(phi, I, t, None, TAU, "l1", lambda_fn=6.0, eps_fn=0.5)
    assert r["counts"] == (5, 3, 0)
    assert r["loss"][1] == pytest.approx(0.0262, rel=1e-6)  # thresholds are fp32: 0.015f differs from 0.015 by 4e-10
    assert r["loss"][2] == 0.0
    np.testing.assert_allclose(r["dL_dI"], [-2.0, -2.0, 0.0, -2.0, 0.0])  # -lambda / |D-|
    # nothing is below the threshold: the term vanishes instead of dividing by zero
    r = oracle.loss(phi, np.full(5, 0.5), t, None, TAU, "l1", lambda_fn=6.0, eps_fn=0.5)
    assert r["loss"][1] == 0.0 and not r["dL_dI"].any()


def test_eq5_false_positive_by_hand(oracle):
    # Eq. 5: U = samples not defined in the volume, U+ = { I_u >= tau }.
    # defined = (1, 0, 0, 0, 1), I = (0.5, 0.01, 0.009, 0.03, 0.2): U+ = {1, 3} (I = tau counts: ">=");
    # L_FP = lambda (0.01 + 0.03) / 2 = 0.02 lambda, lambda = 5 -> 0.1
    I = np.array([0.5, np.float32(0.01), 0.009, 0.03, 0.2], dtype=np.float64)
    d = np.array([1, 0, 0, 0, 1], np.uint8)
    phi = np.array([0.3, 0.0, 0.0, 0.8, 0.1])
    t = np.array([0.1, 9.0, 9.0, 9.0, 0.4], np.float32)  # targets of undefined samples must not matter
    r = oracle.loss(phi, I, t, d, TAU, "l1", lambda_fp=5.0)
    assert r["counts"] == (2, 0, 2)
    assert r["loss"][2] == pytest.approx(0.1, rel=1e-6)
    np.testing.assert_allclose(r["dL_dI"], [0.0, 2.5, 0.0, 2.5, 0.0])
    # L1 over the two defined samples: (|0.3 - 0.1| + |0.1 - 0.4|) / 2 = 0.25; gradient sign / 2 where covered
    assert r["loss"][0] == pytest.approx(0.25, rel=1e-6)
    np.testing.assert_allclose(r["dL_dphi"], [0.5, 0.0, 0.0, 0.0, -0.5])
    np.testing.assert_allclose(r["sample_err"], [0.2, 0.0, 0.0, 0.0, 0.3], rtol=1e-6)


def test_l1_uncovered_defined_sample(oracle):
    # a defined sample with I <= tau is a false negative: it reads Phi = 0, enters the loss as |0 - t| and passes no
    # gradient through Phi (DESIGN D5); strict coverage rule I > tau
    I = np.array([np.float32(0.01), 0.02])
    phi = np.array([0.0, 0.75])
    t = np.array([0.5, 0.25], np.float32)
    r = oracle.loss(phi, I, t, None, TAU, "l1")
    assert r["loss"][0] == pytest.approx((0.5 + 0.5) / 2)
    np.testing.assert_allclose(r["dL_dphi"], [0.0, 0.5])


def test_reduces_to_mse(oracle):
    rng = np.random.default_rng(0)
    P = 1000
    phi, I = rng.uniform(0, 1, P), rng.uniform(0, 0.05, P)
    t = rng.uniform(0, 1, P).astype(np.float32)
    l0, a0, e0 = oracle.mse(phi, I, t, TAU)
    r = oracle.loss(phi, I, t, None, TAU, "mse")
    assert r["loss"] == (pytest.approx(l0, rel=1e-14), 0.0, 0.0)
    np.testing.assert_allclose(r["dL_dphi"], a0, rtol=1e-14)
    np.testing.assert_allclose(r["sample_err"], e0, rtol=0)
    assert not r["dL_dI"].any()


@pytest.mark.parametrize("kind", ["l1", "mse"])
def test_gradients_by_central_differences(oracle, kind):
    rng = np.random.default_rng(1)
    P = 60
    phi = rng.uniform(0.1, 0.9, P)
    t = rng.uniform(0.1, 0.9, P).astype(np.float32)
    I = rng.choice([0.004, 0.012, 0.018, 0.03, 0.4], P) * rng.uniform(0.95, 1.05, P)   # around tau and (1 + eps) tau
    d = (rng.uniform(0, 1, P) < 0.6).astype(np.uint8)
    kw = dict(tau=TAU, kind=kind, lambda_fn=3.0, eps_fn=1.0, lambda_fp=0.7)
    # keep every sample away from the kinks so that a +-h step changes no membership: |res| and the three thresholds
    h = 1e-6
    ok = (np.abs(phi - t) > 1e-3) & (np.abs(I - 0.01) > 1e-4) & (np.abs(I - 0.02) > 1e-4)
    assert ok.sum() > 40
    r = oracle.loss(phi, I, t, d, **kw)
    covered = I.astype(np.float32) > np.float32(TAU)
    phi = np.where(covered, phi, 0.0)  # an uncovered sample outputs the empty value; its Phi is not a variable
    r = oracle.loss(phi, I, t, d, **kw)
    total = lambda p, i: sum(oracle.loss(p, i, t, d, **kw)["loss"])
    for c in np.flatnonzero(ok)[:40]:
        if covered[c]:
            pp, pm = phi.copy(), phi.copy()
            pp[c] += h
            pm[c] -= h
            assert (total(pp, I) - total(pm, I)) / (2 * h) == pytest.approx(r["dL_dphi"][c], rel=1e-6, abs=1e-9)
        else:
            assert r["dL_dphi"][c] == 0.0
        ip, im = I.copy(), I.copy()
        ip[c] += h
        im[c] -= h
        assert (total(phi, ip) - total(phi, im)) / (2 * h) == pytest.approx(r["dL_dI"][c], rel=1e-6, abs=1e-9)


def test_sum_rules(oracle):
    # the normalisations of Eq. 4 / Eq. 5 make the I-gradients of each term sum to -lambda_FN and +lambda_FP
    rng = np.random.default_rng(2)
    P = 5000
    phi, t = rng.uniform(0, 1, P), rng.uniform(0, 1, P).astype(np.float32)
    I = rng.uniform(0, 0.04, P)
    d = (rng.uniform(0, 1, P) < 0.5).astype(np.uint8)
    r = oracle.loss(phi, I, t, d, TAU, "l1", lambda_fn=2.0, eps_fn=0.25, lambda_fp=0.5)
    b = r["dL_dI"]
    assert b[b < 0].sum() == pytest.approx(-2.0) and b[b > 0].sum() == pytest.approx(0.5)
    nD, nFN, nFP = r["counts"]
    If = I.astype(np.float32)
    assert nD == int(d.sum())
    assert nFN == int(((If < np.float32(1.25) * np.float32(TAU)) & (d == 1)).sum())
    assert nFP == int(((If >= np.float32(TAU)) & (d == 0)).sum())
    # L1: every covered defined sample with a non-zero residual carries |dL/dPhi| = 1 / nD
    a = r["dL_dphi"]
    assert np.abs(a).sum() == pytest.approx(((If > np.float32(TAU)) & (d == 1)).sum() / nD)
