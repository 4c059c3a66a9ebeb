"""-m gpu parity: gs_prune and gs_densify (PAPER.md:144 pruning by the weight threshold; PAPER.md:154, :166 sample-error
densification, false negatives first) vs the oracle.  Integer work (kept set, selected samples, copied values) is
compared bit for bit; the logit of the new scalars to 1e-6."""
import numpy as np
import pytest

from paper_2607_01164_b200 import inputs
from gpu_util import TAU, to_dev

pytestmark = pytest.mark.gpu

KEYS = ("mean", "raw_scale", "quat", "raw_opacity", "raw_scalar")
W = dict(mean=3, raw_scale=3, quat=4, raw_opacity=1, raw_scalar=1)


def _random_model(rng, n, cap):
    raw = dict(mean=rng.uniform(0, 1, (cap, 3)), raw_scale=rng.uniform(-5, -3, (cap, 3)), quat=rng.standard_normal((cap, 4)),
               raw_opacity=rng.standard_normal(cap) - 4.0, raw_scalar=rng.standard_normal(cap))
    raw = {k: a.astype(np.float32) for k, a in raw.items()}
    m = rng.standard_normal(12 * cap).astype(np.float32)
    v = rng.uniform(0, 1, 12 * cap).astype(np.float32)
    return raw, m, v


def _check_model(torch, rd, m_d, v_d, n, want_p, want_m, want_v, exact_upto=None):
    """Device arrays (first n Gaussians; moment blocks laid out for n) against the oracle's float64 copies."""
    for k in KEYS:
        got = rd[k].cpu().numpy().reshape(len(rd[k]), -1)[:n]
        ref = np.asarray(want_p[k]).reshape(n, -1)
        e = n if exact_upto is None else exact_upto
        assert np.array_equal(got[:e].astype(np.float64), ref[:e]), k
        if e < n:
            if k == "raw_scalar":
                np.testing.assert_allclose(got[e:], ref[e:], rtol=2e-6, atol=2e-6)
            else:
                assert np.array_equal(got[e:].astype(np.float64), ref[e:]), k
    assert np.array_equal(m_d.cpu().numpy()[:12 * n].astype(np.float64), want_m)
    assert np.array_equal(v_d.cpu().numpy()[:12 * n].astype(np.float64), want_v)


def test_prune(oracle):
    import torch
    from paper_2607_01164_b200 import api
    rng = np.random.default_rng(0)
    n = 20000
    raw, m, v = _random_model(rng, n, n)
    w = (1 / (1 + np.exp(-raw["raw_opacity"].astype(np.float64)))).astype(np.float32)
    w[7] = np.float32(0.005)  # exactly the threshold is kept
    ctx = api.Context()
    rd = {k: to_dev(torch, raw[k])[0] for k in KEYS}
    m_d, v_d, w_d = to_dev(torch, m, v, w)
    n2 = ctx.gs_prune(rd, n, m_d, v_d, w_d, 0.005)
    p2, m2, v2, keep = oracle.prune({k: raw[k].astype(np.float64) for k in KEYS}, m.astype(np.float64), v.astype(np.float64), w, 0.005)
    assert n2 == len(keep) and 0 < n2 < n and 7 in keep
    _check_model(torch, rd, m_d, v_d, n2, p2, m2, v2)
    # nothing below the threshold: unchanged; everything below: empty model
    assert ctx.gs_prune(rd, n2, m_d, v_d, torch.ones(n2, device="cuda"), 0.005) == n2
    _check_model(torch, rd, m_d, v_d, n2, p2, m2, v2)
    assert ctx.gs_prune(rd, n2, m_d, v_d, torch.zeros(n2, device="cuda"), 0.005) == 0
    ctx.close()


@pytest.mark.parametrize("kind", ["grid", "grid_jitter", "points"])
def test_densify(oracle, kind):
    import torch
    from paper_2607_01164_b200 import api
    rng = np.random.default_rng(1)
    n, cap, k = 700, 1500, 600
    g = inputs.c1_gaussians(seed=3, n=n)
    raw, m, v = _random_model(rng, n, cap)
    raw["mean"][:n] = g.mean
    raw["raw_scale"][:n] = np.log(g.scale)
    raw["quat"][:n] = g.quat
    ctx = api.Context()
    if kind.startswith("grid"):
        grid = inputs.Grid((29, 18, 21), (0.0, 0.1, 0.0), (1 / 29, 1 / 24, 1 / 21)).batch((1, 0, 0), (2, 2, 3))
        seed = 77 if kind == "grid_jitter" else None   # new Gaussians sit at the jittered samples (D26)
        xyz = oracle.grid_points(grid, jitter_seed=seed)
        q, dom = api.grid_query(grid, jitter_seed=seed), None
    else:
        xyz = rng.uniform(0, 1, (5000, 3)).astype(np.float32)
        xyz_d = to_dev(torch, xyz)[0]
        q, dom = api.points_query(xyz_d), inputs.points_domain(xyz)
    P = len(xyz)
    ctx.gs_preprocess(*to_dev(torch, g.mean, g.scale, g.quat, g.opacity, g.scalar), domain=dom, tau=TAU)
    ctx.gs_build_accel(q)
    # seeded per-sample inputs (not taken from the CUDA forward): errors with many exact ties, I around tau
    err = (rng.integers(0, 40, P) / 40.0).astype(np.float32)
    I = rng.choice([0.0, 0.004, np.float32(0.01), 0.02, 0.5], P, p=[0.03, 0.03, 0.04, 0.45, 0.45]).astype(np.float32)
    target = rng.choice([0.0, 1.0, 0.3, 0.77, 0.5], P).astype(np.float32)
    defined = (rng.uniform(0, 1, P) < 0.8).astype(np.uint8)
    rs_init, rw_init = float(np.float32(np.log(0.02))), float(np.float32(np.log(0.01 / 0.99)))
    rd = {k: to_dev(torch, raw[k])[0] for k in KEYS}
    m_full, v_full = np.zeros(12 * cap, np.float32), np.zeros(12 * cap, np.float32)
    m_full[:12 * n], v_full[:12 * n] = m[:12 * n], v[:12 * n]   # blocks laid out for n
    m_d, v_d = to_dev(torch, m_full, v_full)
    e_d, I_d, t_d, d_d = to_dev(torch, err, I, target, defined)
    n2 = ctx.gs_densify(rd, n, m_d, v_d, cap, q, e_d, I_d, t_d, k, rs_init, rw_init, defined=d_d, num_defined=int(defined.sum()))
    sel = oracle.densify_select(err, I, defined, k, TAU)
    assert n2 == n + len(sel) == n + k
    assert (I[sel] <= np.float32(TAU)).sum() > 50 and (I[sel] > np.float32(TAU)).sum() > 50  # both classes are selected
    p_old = {kk: raw[kk][:n].astype(np.float64) for kk in KEYS}
    p2, m2, v2 = oracle.densify(p_old, m[:12 * n].astype(np.float64), v[:12 * n].astype(np.float64), xyz, target, sel, rs_init, rw_init)
    _check_model(torch, rd, m_d, v_d, n2, p2, m2, v2, exact_upto=n)
    # capacity and candidate limits
    n3 = ctx.gs_densify(rd, n2, m_d, v_d, n2 + 5, q, e_d, I_d, t_d, 100, rs_init, rw_init, defined=d_d, num_defined=int(defined.sum()))
    assert n3 == n2 + 5
    with pytest.raises(api.GsError):
        ctx.gs_densify(rd, n2, m_d, v_d, n2 - 1, q, e_d, I_d, t_d, 1, rs_init, rw_init)
    ctx.close()
