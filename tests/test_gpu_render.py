"""-m gpu parity of the ray marcher (gs_render) against oracle/wveg_render.py on
the same rays, transfer table and model: RGBA within 2e-5 for every pixel whose ray has no sample sitting on the coverage
threshold (those may legitimately flip, as in the forward tests); the image also goes to a PPM file, the headless stand-in
for a window."""
import os

import numpy as np
import pytest

from paper_2607_01164_b200 import inputs

pytestmark = pytest.mark.gpu
TAU = 0.01


@pytest.mark.parametrize("mode", [0, 1])
def test_render_matches_oracle(oracle, mode):
    import torch
    from oracle import wveg_render
    from paper_2607_01164_b200 import api
    g = inputs.c1_gaussians(seed=0, n=600)
    g.scale[:] = (g.scale * 2.0).astype(np.float32)
    W, H, spp = 48, 36, 96
    o, d, tr = inputs.camera_rays(W, H, eye=(1.9, -1.4, 1.3), look_at=(0.5, 0.5, 0.45), fov_y_deg=38.0)
    assert (tr[:, 1] > tr[:, 0]).sum() > W * H // 3 and (tr[:, 1] <= tr[:, 0]).sum() > 10   # rays that hit the box, rays that miss it
    table = inputs.diverging_transfer(64, extinction=25.0)
    ref = wveg_render.render(g, o, d, tr, spp, table, TAU, mode=1)
    ctx = api.Context()
    ctx.gs_set_option(api.OPT_POINTS_ACCEL, mode)
    dev = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (g.mean, g.scale, g.quat, g.opacity, g.scalar)]
    ctx.gs_preprocess(*dev, domain=((0, 0, 0), (1, 1, 1)), tau=TAU)
    od, dd, td, tab = (torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (o, d, tr, table))
    rgba = torch.full((W * H, 4), -7.0, device="cuda")
    ctx.gs_render(od, dd, td, spp, tab, rgba)
    torch.cuda.synchronize()
    got = rgba.cpu().numpy().astype(np.float64)
    near = (np.abs(ref["I"] - TAU) <= 2e-6 * TAU).any(axis=1)
    assert near.sum() <= 4
    assert ref["rgba"][:, 3].max() > 0.5 and (ref["rgba"][:, 3] == 0).sum() > 10
    err = np.abs(got - ref["rgba"])[~near].max()
    assert err <= 2e-5, err
    assert np.all(got[tr[:, 1] <= tr[:, 0]] == 0.0)
    # a caller's accel does not survive gs_render: the next forward must be preceded by gs_build_accel
    q = api.grid_query(inputs.c1_grid(8))
    with pytest.raises(api.GsError):
        ctx.gs_sample_fwd(q, torch.empty(512, device="cuda"), torch.empty(512, device="cuda"))
    # headless image: PPM over a white background
    out = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out")
    os.makedirs(out, exist_ok=True)
    img = np.clip(got[:, :3] + (1.0 - got[:, 3:4]), 0, 1).reshape(H, W, 3)
    with open(os.path.join(out, f"render_mode{mode}.ppm"), "wb") as f:
        f.write(b"P6\n%d %d\n255\n" % (W, H))
        f.write((img * 255 + 0.5).astype(np.uint8).tobytes())
    ctx.close()


def test_render_chunks_and_errors():
    import torch
    from paper_2607_01164_b200 import api
    g = inputs.c1_gaussians(seed=1, n=200)
    dev = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (g.mean, g.scale, g.quat, g.opacity, g.scalar)]
    table = torch.from_numpy(inputs.diverging_transfer(16)).cuda()
    o, d, tr = inputs.camera_rays(40, 30, eye=(1.8, 1.7, 1.5), look_at=(0.5, 0.5, 0.5))
    od, dd, td = (torch.from_numpy(a).cuda() for a in (o, d, tr))
    ctx = api.Context()
    rgba = torch.empty((1200, 4), device="cuda")
    with pytest.raises(api.GsError) as e:
        ctx.gs_render(od, dd, td, 8, table, rgba)
    assert e.value.status == api.GS_ERR_STATE
    ctx.gs_preprocess(*dev, tau=TAU)                      # no domain
    with pytest.raises(api.GsError) as e:
        ctx.gs_render(od, dd, td, 8, table, rgba)
    assert e.value.status == api.GS_ERR_STATE
    ctx.gs_preprocess(*dev, domain=((0, 0, 0), (1, 1, 1)), tau=TAU)
    with pytest.raises(api.GsError) as e:
        ctx.gs_render(od, dd, td, 0, table, rgba)
    assert e.value.status == api.GS_ERR_INVALID_ARG
    # many samples per ray: 1200 rays x 20000 samples = 2.4e7 > 2^24, i.e. two chunks; equals the one-chunk halves
    ctx.gs_render(od, dd, td, 20000, table, rgba)
    half = torch.empty((600, 4), device="cuda")
    ctx.gs_render(od[600:], dd[600:], td[600:], 20000, table, half)
    torch.cuda.synchronize()
    assert torch.allclose(rgba[600:], half, atol=1e-6)
    ctx.close()
