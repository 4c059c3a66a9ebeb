"""-m gpu: randomised parity of the CUDA path with the oracle.  Every case draws a model and a query from one seed --
model size, anisotropy, scale relative to the sampling distance, grid shape (ragged, anisotropic spacing, shifted origin),
batch position, point count, list / build options -- and checks what every parity test checks: ID sets bit for bit,
Phi to 1e-5, I to 2e-5, the loss to 1e-6, gradients to 1e-4 relative L2 per tensor.  The cases are seeded and fixed; they
exist to reach the corners the hand-written cases do not (a stale buffer after a change of shape, an empty batch, a list
that grows between two builds on one context)."""
import numpy as np
import pytest

from paper_2607_01164_b200 import inputs
from gpu_util import TAU, GpuRun, check_forward, check_grads, check_sets

pytestmark = pytest.mark.gpu


def _model(rng, n, lo, hi, sig_lo, sig_hi, needle_frac):
    mean = rng.uniform(lo, hi, (n, 3)).astype(np.float32)
    scale = np.exp(rng.uniform(np.log(sig_lo), np.log(sig_hi), (n, 3))).astype(np.float32)
    needles = rng.uniform(0, 1, n) < needle_frac
    scale[needles, 2] = (scale[needles, 0] * 20.0).astype(np.float32)
    quat = rng.standard_normal((n, 4)).astype(np.float32)
    quat *= rng.uniform(0.5, 2.0, (n, 1)).astype(np.float32)       # not unit: the library normalises
    opacity = (1.0 / (1.0 + np.exp(-rng.standard_normal(n)))).astype(np.float32)
    scalar = rng.uniform(0, 1, n).astype(np.float32)
    return inputs.Gaussians(mean, scale, quat, opacity, scalar)


def _oracle_all(oracle, g, xyz, target, dI):
    fwd = oracle.forward(g, xyz, TAU, mode=1)
    loss, a, serr = oracle.mse(fwd["phi"], fwd["I"], target, TAU)
    gr = oracle.backward(g, xyz, fwd["phi"], fwd["I"], a, dI, target, TAU, mode=1)
    return fwd, loss, gr


def _tol_I(g):
    # I has no north_star tolerance; its fp32 error is |dq| / 2 with |dq| <~ 2 |u| |M||d| 2^-24, which grows
    # with the ratio of the longest to the shortest axis: 2e-5 at the 20:1 of the configs, in proportion beyond
    aniso = float((g.scale.max(axis=1) / g.scale.min(axis=1)).max())
    return 2e-5 * max(1.0, aniso / 20.0)


def _check_loss(run, loss):
    # L = mean (Phi - t)^2 with Phi to 1e-5: |dL| <= 2 mean|res| 1e-5 <= 2 sqrt(L) 1e-5; the 1e-6 relative figure of the other
    # tests holds once the rounding errors of thousands of samples average out, not for P = 1
    got = float(run.loss.item())
    assert abs(got - loss) <= 1e-6 * loss + (2e-5 * np.sqrt(loss) if run.P < 1000 else 0.0) + 1e-12, (got, loss, run.P)


FLOORED = []   # (test, seed, tensor) of every comparison that used a cancellation floor instead of the plain 1e-4: printed below


def _floors(gr, g, tag):
    # A gradient tensor whose EXACT value vanishes by cancellation (an isolated Gaussian, where Phi = v wherever it is covered, so
    # every term of dL/dmu, dL/ds, dL/dq, dL/dw cancels against its neighbour) cannot be held to a relative error: fp32 leaves the
    # rounding of the terms that cancel.  Only then -- the oracle's tensor is below 1e-6 of the size of those terms, i.e. zero to
    # fp32 -- is the result compared against that size instead of against the tensor's own norm; everything else is held to the
    # plain 1e-4.  Size of the cancelling terms, per Gaussian that is hit at all: |dL/dv_i| times what the chain rule multiplies it
    # by (1 / sigma_min,i for the mean and the scales, the Gaussian's own anisotropy for the rotation, 1 / w_i for the weight).
    dv = np.abs(np.asarray(gr["dscalar"], np.float64).ravel())
    hit = dv > 0
    if not hit.any():
        return {}
    smin, smax = g.scale.min(axis=1).astype(np.float64), g.scale.max(axis=1).astype(np.float64)
    mult = {"dmean": 1.0 / smin, "dscale": 1.0 / smin, "dquat": smax / smin, "dopacity": 1.0 / g.opacity.astype(np.float64)}
    out = {}
    for k, m in mult.items():
        size = float(np.linalg.norm((dv * m)[hit]))
        if float(np.linalg.norm(gr[k])) < 1e-6 * size:
            out[k] = size
            FLOORED.append((*tag, k))
    return out


# seeds beyond the first twelve: the ones that failed under the fixed 1e-5 / 2e-5 / 1e-6 / 1e-4 bounds when a wider range was
# run by hand in round 2 (P = 1 losses, I at > 20:1 anisotropy, isolated Gaussians), kept as fixed cases
SEEDS = list(range(12)) + [45, 53, 79, 111, 116, 132, 251]


@pytest.mark.parametrize("seed", SEEDS)
def test_random_grid_case(oracle, seed):
    import torch
    rng = np.random.default_rng(1000 + seed)
    dims = tuple(int(x) for x in rng.integers(9, 70, 3))
    spacing = tuple(float(x) for x in rng.uniform(0.7, 1.4, 3) / max(dims))
    origin = tuple(float(x) for x in rng.uniform(-0.3, 0.3, 3))
    full = inputs.Grid(dims, origin, spacing)
    nb = full.brick_cnt
    lo = tuple(int(rng.integers(0, b)) for b in nb)
    cnt = tuple(int(rng.integers(1, b - l + 1)) for b, l in zip(nb, lo))
    batch = full.batch(lo, cnt) if seed % 3 else full
    ext = np.asarray(dims) * np.asarray(spacing)
    n = int(rng.choice([1, 7, 300, 4000, 20000]))
    vox = float(np.mean(spacing))
    g = _model(rng, n, np.asarray(origin) - 0.05 * ext, np.asarray(origin) + 1.05 * ext, 0.4 * vox, float(rng.choice([2.0, 5.0])) * vox,
               needle_frac=0.05 if seed % 2 else 0.0)
    xyz = oracle.grid_points(batch)
    target = rng.uniform(0, 1, len(xyz)).astype(np.float32)
    dI = (rng.standard_normal(len(xyz)) * 1e-3).astype(np.float32) if seed % 4 == 1 else None
    fwd, loss, gr = _oracle_all(oracle, g, xyz, target, dI)
    run = GpuRun(g, "grid", batch, target, dL_dI=dI, fused=(dI is None and seed % 2 == 0))
    if seed % 5 == 0:   # the same context after another batch shape (buffers sized for something else), asynchronous builds on
        api = run.api
        run.ctx.gs_set_option(api.OPT_ASYNC_BUILD, 1)
        other = full.batch((0, 0, 0), (1, 1, 1))
        run.ctx.gs_build_accel(api.grid_query(other))
        run.ctx.gs_build_accel(run.q)
        run.ctx.gs_sample_fwd(run.q, run.phi, run.I, target=run.target, loss=run.loss.zero_(), dL_dphi=run.dphi, sample_err=run.serr)
        torch.cuda.synchronize()
    check_sets(run, fwd)
    check_forward(run, fwd, tol_I=_tol_I(g))
    _check_loss(run, loss)
    check_grads(run, gr, zero_floor=_floors(gr, g, ("grid", seed)))


@pytest.mark.parametrize("seed", SEEDS)
def test_random_points_case(oracle, seed):
    rng = np.random.default_rng(2000 + seed)
    P = int(rng.choice([1, 31, 32, 33, 1000, 20011, 70000]))
    n = int(rng.choice([1, 2, 50, 3000, 30000]))
    clustered = seed % 2 == 0
    if clustered:
        centres = rng.uniform(0.1, 0.9, (8, 3))
        xyz = (centres[rng.integers(0, 8, P)] + rng.standard_normal((P, 3)) * 0.03).astype(np.float32)
    else:
        xyz = rng.uniform(0, 1, (P, 3)).astype(np.float32)
    sig = float(rng.choice([0.003, 0.01, 0.04]))
    g = _model(rng, n, 0.0, 1.0, 0.5 * sig, 3.0 * sig, needle_frac=0.05 if seed % 3 == 0 else 0.0)
    if n > 10:
        g.mean[: n // 2] = xyz[rng.integers(0, P, n // 2)]          # half of the Gaussians sit on samples
    target = rng.uniform(0, 1, P).astype(np.float32)
    dI = (rng.standard_normal(P) * 1e-3).astype(np.float32) if seed % 4 == 2 else None
    dom = (np.full(3, -0.25, np.float32), np.full(3, 1.25, np.float32))
    fwd, loss, gr = _oracle_all(oracle, g, xyz, target, dI)
    from paper_2607_01164_b200 import api
    run = GpuRun(g, "points", xyz, target, domain=dom, dL_dI=dI, fused=(dI is None and seed % 2 == 1), presorted=False,
                 points_accel=api.POINTS_SCATTER if seed % 6 == 5 else None)
    check_sets(run, fwd)
    check_forward(run, fwd, tol_I=_tol_I(g))
    _check_loss(run, loss)
    check_grads(run, gr, zero_floor=_floors(gr, g, ("points", seed)))


def test_zz_report_floored_comparisons():
    # not a check of the kernels: says how many of the comparisons above used a cancellation floor (run with -s to see them)
    print(f"\ncancellation floors used in {len(FLOORED)} tensor comparisons: {FLOORED}")
    assert len(FLOORED) <= 2 * len(SEEDS), "floors are for the rare exact cancellation, not the rule"
