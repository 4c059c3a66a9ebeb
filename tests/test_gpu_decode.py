"""-m gpu: gs_decode_grid, the forward-only decode of a grid region in brick-aligned batches on several streams (gs.h;
BASELINE.json configs[3]).  Its output must be, bit for bit, what gs_build_accel + gs_sample_fwd give batch by batch, in
batch-major order; one batch is also compared with the oracle."""
import numpy as np
import pytest

from paper_2607_01164_b200 import inputs
from gpu_util import TAU

pytestmark = pytest.mark.gpu


def _dev(torch, *arrays):
    return [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrays]


def _batches(region, bb):
    """The batches of gs_decode_grid's enumeration (x fastest), as inputs.Grid objects."""
    out = []
    nb = [(c + b - 1) // b for c, b in zip(region.brick_cnt, bb)]
    for z in range(nb[2]):
        for y in range(nb[1]):
            for x in range(nb[0]):
                lo = tuple(l + i * b for l, i, b in zip(region.brick_lo, (x, y, z), bb))
                cnt = tuple(min(b, l0 + c - l) for b, l0, c, l in zip(bb, region.brick_lo, region.brick_cnt, lo))
                out.append(inputs.Grid(region.dims, region.origin, region.spacing, lo, cnt))
    return out


def _reference(api, torch, dev, batches):
    ctx = api.Context()
    ctx.gs_preprocess(*dev)
    P = sum(b.num_points for b in batches)
    phi, I = torch.empty(P, device="cuda"), torch.empty(P, device="cuda")
    off = 0
    for b in batches:
        q = api.grid_query(b)
        ctx.gs_build_accel(q)
        ctx.gs_sample_fwd(q, phi[off:off + b.num_points], I[off:off + b.num_points])
        off += b.num_points
    torch.cuda.synchronize()
    ctx.close()
    return phi, I


@pytest.mark.parametrize("streams", [1, 3])
def test_decode_equals_batch_by_batch(oracle, streams):
    import torch
    from paper_2607_01164_b200 import api
    # a ragged grid (60 x 64 x 52 voxels: the last bricks along x and z are clipped), a region that is not the whole grid, batches
    # of 3 x 2 x 2 bricks that do not divide it
    g = inputs.c4_gaussians(seed=11, n_grid=64, n=30000)
    full = inputs.Grid((60, 64, 52), (0.0, 0.0, 0.0), (1 / 64, 1 / 64, 1 / 64))
    region = full.batch((1, 0, 1), (7, 8, 6))
    bb = (3, 2, 2)
    batches = _batches(region, bb)
    assert len(batches) == 3 * 4 * 3 and len({b.num_points for b in batches}) > 1
    dev = _dev(torch, g.mean, g.scale, g.quat, g.opacity, g.scalar)
    phi_ref, I_ref = _reference(api, torch, dev, batches)
    ctx = api.Context()
    P = region.num_points
    assert P == sum(b.num_points for b in batches)
    phi, I = torch.full((P,), -7.0, device="cuda"), torch.full((P,), -7.0, device="cuda")
    for rep in range(2):    # the second call re-uses the worker contexts
        ctx.gs_decode_grid(*dev, api.grid_query(region), bb, phi, I, streams=streams)
        assert torch.equal(phi, phi_ref) and torch.equal(I, I_ref)
        phi.fill_(-7.0)
    # one batch against the oracle (the per-batch forward itself is covered by tests/test_gpu_structured.py)
    k = 17
    off = sum(b.num_points for b in batches[:k])
    ref = oracle.forward(g, oracle.grid_points(batches[k]), TAU, mode=1)
    near = np.abs(ref["I"] - TAU) <= 2e-6 * TAU
    assert np.abs(phi_ref[off:off + batches[k].num_points].cpu().numpy() - ref["phi"])[~near].max() <= 1e-5
    ctx.close()


def test_decode_repeats_a_batch_that_outgrew_the_speculative_buffer(oracle):
    import torch
    from paper_2607_01164_b200 import api
    # all Gaussians sit in the upper half of the grid: every worker sizes its pair list on a (nearly) empty batch, so the first
    # dense batch overflows the speculative capacity, does nothing and must be repeated by gs_decode_grid
    g = inputs.c4_gaussians(seed=12, n_grid=64, n=40000, elongated_frac=0.0)   # radius <= 3.03 * 4 voxels: none reaches z < 0.3
    g.mean[:, 2] = (0.5 + 0.5 * g.mean[:, 2]).astype(np.float32)
    full = inputs.Grid((64, 64, 64), (0.0, 0.0, 0.0), (1 / 64, 1 / 64, 1 / 64))
    bb = (4, 4, 1)
    batches = _batches(full, bb)
    dev = _dev(torch, g.mean, g.scale, g.quat, g.opacity, g.scalar)
    phi_ref, I_ref = _reference(api, torch, dev, batches)
    assert float(I_ref[: 64 * 64 * 8].max().item()) == 0.0 and float(I_ref.max().item()) > 0.0
    ctx = api.Context()
    phi, I = torch.full_like(phi_ref, -7.0), torch.full_like(I_ref, -7.0)
    ctx.gs_decode_grid(*dev, api.grid_query(full), bb, phi, I, streams=2)
    assert torch.equal(phi, phi_ref) and torch.equal(I, I_ref)
    assert ctx.gs_status_query()["decode_repeats"] >= 1   # the overflow path did run
    with pytest.raises(api.GsError) as e:
        ctx.gs_decode_grid(*dev, api.grid_query(full), (0, 4, 4), phi, I)
    assert e.value.status == api.GS_ERR_INVALID_ARG
    # a region that reaches beyond the grid is refused before any batch runs (it used to fail inside a worker thread, after
    # other batches had written their part of phi / I)
    phi.fill_(-7.0)
    over = inputs.Grid(full.dims, full.origin, full.spacing, (0, 0, 4), (8, 8, 5))
    with pytest.raises(api.GsError) as e:
        ctx.gs_decode_grid(*dev, api.grid_query(over), bb, phi, I, streams=2)
    assert e.value.status == api.GS_ERR_INVALID_ARG and "beyond the grid" in str(e.value)
    torch.cuda.synchronize()
    assert float(phi.max().item()) == -7.0
    ctx.close()
