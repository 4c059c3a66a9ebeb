"""Pins of the oracle's training-step completion (oracle.activate, oracle.adam_step; PAPER.md:140 activations,
PAPER.md:231 Adam with the paper's learning rates): closed forms, a library Adam (torch.optim.Adam on CPU in float64),
and central differences for the chain rule through the activations."""
import numpy as np
import pytest


def _params(rng, n):
    return dict(mean=rng.uniform(0, 1, (n, 3)), raw_scale=rng.uniform(-5, -3, (n, 3)), quat=rng.standard_normal((n, 4)),
                raw_opacity=rng.standard_normal(n), raw_scalar=rng.standard_normal(n))


def _grads(rng, n, scale=1.0):
    return dict(dmean=scale * rng.standard_normal((n, 3)), dscale=scale * rng.standard_normal((n, 3)),
                dquat=scale * rng.standard_normal((n, 4)), dopacity=scale * rng.standard_normal(n),
                dscalar=scale * rng.standard_normal(n))


def test_activations_closed_forms(oracle):
    # exp(0) = 1, sigmoid(0) = 1/2, sigmoid(-x) = 1 - sigmoid(x), sigmoid(ln 3) = 3/4; exp(ln 0.02) = 0.02
    rs = np.array([[0.0, np.log(0.02), -1.0]], np.float32)
    s, w, v = oracle.activate(rs, np.array([0.0], np.float32), np.array([np.log(3.0)], np.float32))
    assert s[0, 0] == 1.0 and s[0, 1] == pytest.approx(0.02, rel=1e-7) and s[0, 2] == pytest.approx(np.exp(-1.0), rel=1e-15)
    assert w[0] == 0.5 and v[0] == pytest.approx(0.75, rel=1e-7)
    x = np.linspace(-6, 6, 25).astype(np.float32)
    _, a, _ = oracle.activate(np.zeros((25, 3), np.float32), x, x)
    _, b, _ = oracle.activate(np.zeros((25, 3), np.float32), -x, x)
    np.testing.assert_allclose(a + b, 1.0, rtol=1e-15)
    assert np.all((a > 0) & (a < 1))  # "constrain them within [0,1)"


def test_first_step_moves_by_lr_against_the_gradient_sign(oracle):
    # t = 1: m_hat = g, v_hat = g^2, so the step is lr * g / (|g| + eps) = lr * sign(g) up to eps / |g|
    rng = np.random.default_rng(0)
    n = 50
    p = _params(rng, n)
    p0 = {k: v.copy() for k, v in p.items()}
    g = _grads(rng, n)
    m, v = np.zeros(12 * n), np.zeros(12 * n)
    oracle.adam_step(p, g, m, v, 1)
    lr = dict(mean=0.00016, raw_scale=0.001, quat=0.0001, raw_opacity=0.025, raw_scalar=0.0025)
    for k, gk in (("mean", "dmean"), ("quat", "dquat")):
        np.testing.assert_allclose(p[k] - p0[k], -lr[k] * g[gk] / (np.abs(g[gk]) + 1e-8), rtol=1e-9)
        big = np.abs(g[gk]) > 0.1
        np.testing.assert_allclose((p[k] - p0[k])[big], (-lr[k] * np.sign(g[gk]))[big], rtol=2e-7)
    # activated tensors: the sign of the raw gradient is the sign of the activated one (exp' > 0, sigmoid' > 0)
    for k, gk in (("raw_scale", "dscale"), ("raw_opacity", "dopacity"), ("raw_scalar", "dscalar")):
        assert np.array_equal(np.sign(p[k] - p0[k]), -np.sign(g[gk]))
        assert np.all(np.abs(p[k] - p0[k]) <= lr[k] * (1 + 1e-12))
    # moments after one step: m = (1 - b1) g, v = (1 - b2) g^2 (raw-space gradient for the activated tensors)
    np.testing.assert_allclose(m[:3 * n], 0.1 * g["dmean"].ravel(), rtol=1e-12)
    w = 1 / (1 + np.exp(-p0["raw_opacity"]))
    np.testing.assert_allclose(m[10 * n:11 * n], 0.1 * g["dopacity"] * w * (1 - w), rtol=1e-12)
    np.testing.assert_allclose(v[3 * n:6 * n], 0.001 * (g["dscale"] * np.exp(p0["raw_scale"])).ravel() ** 2, rtol=1e-12)


def test_matches_library_adam(oracle):
    # five steps with changing gradients against torch.optim.Adam (float64, CPU); the raw-space gradients are formed
    # here with torch's own exp / sigmoid derivatives (autograd through the activations)
    torch = pytest.importorskip("torch")
    rng = np.random.default_rng(1)
    n = 20
    p = _params(rng, n)
    tp = {k: torch.tensor(v.copy(), dtype=torch.float64, requires_grad=True) for k, v in p.items()}
    lrs = dict(mean=0.00016, raw_scale=0.001, quat=0.0001, raw_opacity=0.025, raw_scalar=0.0025)
    opt = torch.optim.Adam([{"params": [tp[k]], "lr": lrs[k]} for k in lrs], betas=(0.9, 0.999), eps=1e-8)
    m, v = np.zeros(12 * n), np.zeros(12 * n)
    for t in range(1, 6):
        g = _grads(rng, n, scale=10.0 ** rng.uniform(-4, 0))
        # a loss that is linear in the ACTIVATED values with coefficients g: its gradient w.r.t. them is g
        opt.zero_grad()
        loss = ((tp["mean"] * torch.tensor(g["dmean"])).sum() + (torch.exp(tp["raw_scale"]) * torch.tensor(g["dscale"])).sum()
                + (tp["quat"] * torch.tensor(g["dquat"])).sum() + (torch.sigmoid(tp["raw_opacity"]) * torch.tensor(g["dopacity"])).sum()
                + (torch.sigmoid(tp["raw_scalar"]) * torch.tensor(g["dscalar"])).sum())
        loss.backward()
        opt.step()
        oracle.adam_step(p, g, m, v, t)
        for k in lrs:
            np.testing.assert_allclose(p[k], tp[k].detach().numpy(), rtol=1e-10, atol=1e-13)


def test_chain_rule_by_central_differences(oracle):
    # d/d raw of c . act(raw) by central differences of the oracle's own activation = what the Adam step feeds its moments
    rng = np.random.default_rng(2)
    n = 8
    p = _params(rng, n)
    g = _grads(rng, n)
    m, v = np.zeros(12 * n), np.zeros(12 * n)
    q = {k: a.copy() for k, a in p.items()}
    oracle.adam_step(q, g, m, v, 1)
    h = 1e-3  # raw parameters enter the oracle's activation as float32: steps must survive that rounding
    f32 = lambda a: a.astype(np.float32)
    def lin(rs, rw, rv):
        s, w, vv = oracle.activate(f32(rs), f32(rw), f32(rv))
        return (s * g["dscale"]).sum() + (w * g["dopacity"]).sum() + (vv * g["dscalar"]).sum()
    base = {k: f32(p[k]).astype(np.float64) for k in ("raw_scale", "raw_opacity", "raw_scalar")}
    for i in range(n):
        for k in range(3):
            d = np.zeros((n, 3)); d[i, k] = h
            fd = (lin(base["raw_scale"] + d, base["raw_opacity"], base["raw_scalar"]) -
                  lin(base["raw_scale"] - d, base["raw_opacity"], base["raw_scalar"])) / (2 * float(np.float32(h)))
            assert m[3 * n + 3 * i + k] / 0.1 == pytest.approx(fd, rel=2e-3, abs=1e-6)
        d = np.zeros(n); d[i] = h
        fd = (lin(base["raw_scale"], base["raw_opacity"] + d, base["raw_scalar"]) -
              lin(base["raw_scale"], base["raw_opacity"] - d, base["raw_scalar"])) / (2 * float(np.float32(h)))
        assert m[10 * n + i] / 0.1 == pytest.approx(fd, rel=2e-3, abs=1e-6)


def test_constant_gradient_walks_linearly(oracle):
    # with a constant gradient m_hat = g and v_hat = g^2 at every t, so each step moves by lr * sign(g)
    n = 4
    p = dict(mean=np.zeros((n, 3)), raw_scale=np.zeros((n, 3)), quat=np.ones((n, 4)), raw_opacity=np.zeros(n), raw_scalar=np.zeros(n))
    g = dict(dmean=np.full((n, 3), 0.3), dscale=np.zeros((n, 3)), dquat=np.full((n, 4), -2.0), dopacity=np.zeros(n), dscalar=np.zeros(n))
    m, v = np.zeros(12 * n), np.zeros(12 * n)
    for t in range(1, 11):
        oracle.adam_step(p, g, m, v, t)
    np.testing.assert_allclose(p["mean"], -10 * 0.00016, rtol=1e-6)
    np.testing.assert_allclose(p["quat"], 1 + 10 * 0.0001, rtol=1e-6)
    assert not p["raw_scale"].any() and not p["raw_opacity"].any()  # zero gradient: no move (0 / (0 + eps))
