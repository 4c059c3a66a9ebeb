"""-m gpu tests of the C-ABI boundary's contract (include/gs.h "Conventions"): unaligned per-sample views, the
invalid-Gaussian count of gs_status_query, per-context launch counters, a Gaussian spanning a 2048-voxel batch axis,
and the multi-GPU decomposition run on ONE GPU: two sample shards through the library add up to the one-batch result."""
import numpy as np
import pytest

from paper_2607_01164_b200 import inputs
from gpu_util import TAU, GpuRun, check_grads, rel_l2

pytestmark = pytest.mark.gpu


def _dev(torch, *arrays):
    return [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrays]


def test_unaligned_sample_views(oracle):
    # gs.h: per-sample arrays may be 4-byte-aligned views (tensor[1:]); even x extent => the kernel would otherwise take
    # its float2 path.  Results must equal the aligned call bit for bit (same arithmetic, scalar moves).
    import torch
    from paper_2607_01164_b200 import api
    g = inputs.c1_gaussians(seed=0, n=1024)
    grid = inputs.c1_grid(32)
    P = grid.num_points
    target = np.random.default_rng(2).uniform(0, 1, P).astype(np.float32)
    ref = GpuRun(g, "grid", grid, target)
    ctx = api.Context()
    ctx.gs_preprocess(*_dev(torch, g.mean, g.scale, g.quat, g.opacity, g.scalar))
    q = api.grid_query(grid)
    ctx.gs_build_accel(q)
    big = [torch.full((P + 1,), -7.0, device="cuda") for _ in range(5)]
    phi, I, dphi, serr, t = (b[1:] for b in big)
    assert phi.data_ptr() % 8 == 4
    t.copy_(torch.from_numpy(target))
    loss = torch.zeros(1, dtype=torch.float64, device="cuda")
    ctx.gs_sample_fwd(q, phi, I, target=t, loss=loss, dL_dphi=dphi, sample_err=serr)
    grads = ctx.alloc_grads(g.n)
    ctx.gs_sample_bwd(q, phi, I, dphi, grads, target=t)
    torch.cuda.synchronize()
    for got, want in ((phi, ref.phi), (I, ref.I), (dphi, ref.dphi), (serr, ref.serr)):
        assert torch.equal(got, want[:P])
    assert float(loss.item()) == pytest.approx(float(ref.loss.item()), rel=1e-7)   # float partial sums in another order
    for b in big:
        assert float(b[0].item()) == -7.0   # nothing written in front of the view
    for k, v in grads.items():
        assert torch.equal(v, ref.grads[k]), k
    # only one of the arrays unaligned
    phi2 = torch.full((P,), -7.0, device="cuda")
    ctx.gs_sample_fwd(q, phi2, I, target=t)
    torch.cuda.synchronize()
    assert torch.equal(phi2, ref.phi[:P])
    ctx.close()


def test_status_query_counts_invalid_gaussians():
    import torch
    from paper_2607_01164_b200 import api
    g = inputs.c1_gaussians(seed=3, n=500)
    g.scale[7, 1] = 0.0
    g.scale[8, 0] = -1.0
    g.quat[100] = 0.0
    g.mean[200, 2] = np.nan
    g.opacity[300] = np.inf
    ctx = api.Context()
    assert ctx.gs_status_query()["num_gaussians"] == 0
    ctx.gs_preprocess(*_dev(torch, g.mean, g.scale, g.quat, g.opacity, g.scalar))
    st = ctx.gs_status_query()
    assert st["num_gaussians"] == 500 and st["invalid_gaussians"] == 5
    q = api.grid_query(inputs.c1_grid(16))
    ctx.gs_build_accel(q)
    st = ctx.gs_status_query()
    assert st["grid_pairs"] > 0 and 0 < st["grid_touched"] <= 495
    g2 = inputs.c1_gaussians(seed=4, n=300)
    ctx.gs_preprocess(*_dev(torch, g2.mean, g2.scale, g2.quat, g2.opacity, g2.scalar))
    st = ctx.gs_status_query()
    assert st["num_gaussians"] == 300 and st["invalid_gaussians"] == 0   # reset by every gs_preprocess
    ctx.close()


def test_launch_counters_are_per_context():
    import torch
    from paper_2607_01164_b200 import api
    g = inputs.c1_gaussians(seed=0, n=256)
    dev = _dev(torch, g.mean, g.scale, g.quat, g.opacity, g.scalar)
    a, b = api.Context(), api.Context()
    a.profile_read(); b.profile_read()
    a.gs_preprocess(*dev)
    a.gs_preprocess(*dev)
    b.gs_preprocess(*dev)
    assert a.profile_read()[2] == 2
    assert b.profile_read()[2] == 1
    assert a.profile_read()[2] == 0
    a.close(); b.close()


def test_gaussian_spanning_a_2048_voxel_axis(oracle):
    # the backward's cell-count packing must hold 1024 cells along z (a batch may span 2048 voxels per axis)
    grid = inputs.Grid((8, 8, 2048), (0.0, 0.0, 0.0), (1 / 8, 1 / 8, 1 / 2048))
    mean = np.array([[0.5, 0.5, 0.5], [0.3, 0.6, 0.2]], np.float32)
    scale = np.array([[0.08, 0.08, 0.4], [0.05, 0.05, 0.01]], np.float32)   # the first one reaches beyond both z ends
    quat = np.array([[1, 0, 0, 0], [1, 0, 0, 0]], np.float32)
    g = inputs.Gaussians(mean, scale, quat, np.array([0.5, 0.7], np.float32), np.array([0.2, 0.9], np.float32))
    P = grid.num_points
    target = np.random.default_rng(0).uniform(0, 1, P).astype(np.float32)
    xyz = oracle.grid_points(grid)
    fwd = oracle.forward(g, xyz, TAU, mode=1)
    _, a, _ = oracle.mse(fwd["phi"], fwd["I"], target, TAU)
    gr = oracle.backward(g, xyz, fwd["phi"], fwd["I"], a, None, target, TAU, mode=1)
    assert np.abs(gr["dscale"][0]).max() > 0
    for fused in (False, True):
        run = GpuRun(g, "grid", grid, target, fused=fused)
        check_grads(run, gr)


def test_two_sample_shards_add_up_on_one_gpu(oracle):
    # DESIGN.md section 10 on one GPU: the grid's bricks are split into two z-slabs (dist.shard_bricks), each slab runs
    # through the C ABI as its own batch with the GLOBAL sample count as the loss normaliser (gs_set_sample_count); the
    # per-shard losses and gradients must ADD UP to the one-batch ones and Phi / I must concatenate bit-exactly.
    import torch
    from paper_2607_01164_b200 import api, dist as gsdist
    g = inputs.c4_gaussians(seed=9, n_grid=48, n=6000)
    grid = inputs.Grid((48, 40, 44), (0.0, 0.0, 0.0), (1 / 48, 1 / 48, 1 / 48))
    P = grid.num_points
    target = np.random.default_rng(5).uniform(0, 1, P).astype(np.float32)
    one = GpuRun(g, "grid", grid, target, fused=True)
    dev = _dev(torch, g.mean, g.scale, g.quat, g.opacity, g.scalar)
    total = {k: torch.zeros_like(v) for k, v in one.grads.items()}
    loss_sum = 0.0
    phis, Is = [], []
    bd = grid.batch_dims
    t3 = target.reshape(bd[2], bd[1], bd[0])
    for r in range(2):
        lo, cnt = gsdist.shard_bricks(grid.brick_cnt, r, 2)
        sub = grid.batch(lo, cnt)
        ctx = api.Context()
        ctx.gs_set_sample_count(P)
        ctx.gs_preprocess(*dev)
        q = api.grid_query(sub)
        ctx.gs_build_accel(q)
        Pr = sub.num_points
        z0 = 8 * lo[2]
        t = torch.from_numpy(np.ascontiguousarray(t3[z0:z0 + sub.batch_dims[2]].ravel())).cuda()
        phi, I = torch.empty(Pr, device="cuda"), torch.empty(Pr, device="cuda")
        loss = torch.zeros(1, dtype=torch.float64, device="cuda")
        ctx.gs_sample_fwd(q, phi, I, target=t, loss=loss)
        grads = ctx.alloc_grads(g.n, flat=True)
        ctx.gs_sample_bwd(q, None, None, None, grads)
        torch.cuda.synchronize()
        for k in total:
            total[k] += grads[k]
        loss_sum += float(loss.item())
        phis.append(phi); Is.append(I)
        ctx.close()
    assert torch.equal(torch.cat(phis), one.phi[:P]) and torch.equal(torch.cat(Is), one.I[:P])
    assert loss_sum == pytest.approx(float(one.loss.item()), rel=1e-9)
    for k in total:
        assert rel_l2(total[k].cpu().numpy(), one.grads[k].cpu().numpy()) <= 1e-5, k
    # ... and against the oracle's one-batch gradients
    xyz = oracle.grid_points(grid)
    fwd = oracle.forward(g, xyz, TAU, mode=1)
    _, a, _ = oracle.mse(fwd["phi"], fwd["I"], target, TAU)
    gr = oracle.backward(g, xyz, fwd["phi"], fwd["I"], a, None, target, TAU, mode=1)
    for k, v in gr.items():
        assert rel_l2(total[k].cpu().numpy(), v) <= 1e-4, k


def test_async_build_matches_synchronous_and_reports_overflow(oracle):
    # GS_OPT_ASYNC_BUILD (gs.h): steady-state grid builds without a host round trip give bit-identical results; a batch whose
    # pair list outgrows the speculative capacity does nothing and the NEXT call reports GS_ERR_OVERFLOW
    import torch
    from paper_2607_01164_b200 import api
    g = inputs.c4_gaussians(seed=3, n_grid=64, n=20000)
    full = inputs.Grid((64, 64, 64), (0.0, 0.0, 0.0), (1 / 64, 1 / 64, 1 / 64))
    P = full.num_points
    target = np.random.default_rng(1).uniform(0, 1, P).astype(np.float32)
    ref = GpuRun(g, "grid", full, target, fused=True)
    ctx = api.Context()
    ctx.gs_set_option(api.OPT_ASYNC_BUILD, 1)
    dev = _dev(torch, g.mean, g.scale, g.quat, g.opacity, g.scalar)
    t = torch.from_numpy(target).cuda()
    q = api.grid_query(full)
    phi, I = torch.empty(P, device="cuda"), torch.empty(P, device="cuda")
    grads = ctx.alloc_grads(g.n)
    loss = torch.zeros(1, dtype=torch.float64, device="cuda")
    for step in range(4):   # step 0 is the synchronous sizing build, 1..3 run without a host round trip
        loss.zero_()
        for v in grads.values():
            v.fill_(-7.0)
        ctx.gs_preprocess(*dev)
        ctx.gs_build_accel(q)
        ctx.gs_sample_fwd(q, phi, I, target=t, loss=loss)
        ctx.gs_sample_bwd(q, None, None, None, grads)
        torch.cuda.synchronize()
        assert torch.equal(phi, ref.phi[:P]) and torch.equal(I, ref.I[:P])
        assert float(loss.item()) == float(ref.loss.item())
        for k, v in grads.items():
            assert torch.equal(v, ref.grads[k]), (step, k)
    st = ctx.gs_status_query()
    assert st["grid_pairs"] == ref.ctx.gs_status_query()["grid_pairs"] and st["grid_touched"] == ref.ctx.gs_status_query()["grid_touched"]
    # overflow: size the buffer with a one-brick batch, then ask for the whole grid asynchronously
    small = full.batch((3, 3, 3), (1, 1, 1))
    ctx2 = api.Context()
    ctx2.gs_set_option(api.OPT_ASYNC_BUILD, 1)
    ctx2.gs_preprocess(*dev)
    qs = api.grid_query(small)
    ctx2.gs_build_accel(qs)                      # synchronous: capacity = 1.5 x a few hundred pairs
    ctx2.gs_build_accel(q)                       # asynchronous: T is far beyond the capacity
    phi.fill_(-7.0)
    ctx2.gs_sample_fwd(q, phi, I)                # does nothing
    torch.cuda.synchronize()
    assert float(phi.min().item()) == -7.0 and float(phi.max().item()) == -7.0
    # with a loss and a backward, the batch that did not happen says so in band: NaN loss, zero gradients (never the
    # -7 "previous step" values), long before the status reaches the host
    loss.zero_()
    for v in grads.values():
        v.fill_(-7.0)
    ctx2.gs_sample_fwd(q, phi, I, target=t, loss=loss)
    ctx2.gs_sample_bwd(q, None, None, None, grads)
    torch.cuda.synchronize()
    assert np.isnan(float(loss.item()))
    for k, v in grads.items():
        assert float(v.abs().max().item()) == 0.0, k
    with pytest.raises(api.GsError) as e:
        ctx2.gs_build_accel(q)
    assert e.value.status == api.GS_ERR_OVERFLOW
    ctx2.gs_build_accel(q)                       # synchronous again: grows the buffer
    ctx2.gs_sample_fwd(q, phi, I)
    torch.cuda.synchronize()
    assert torch.equal(phi, ref.phi[:P])
    ctx.close(); ctx2.close()


def test_async_sizing_build_keeps_a_list_that_fitted(oracle):
    # A sizing build under GS_OPT_ASYNC_BUILD whose pair list FITS the buffer it finds (T <= capacity < 1.5 T + headroom): the
    # list is written by the first fill, which consumes the histogram, so the fill must not be repeated -- the buffer is grown
    # around its contents instead.  (The situation arises when the option is switched on for a context that has built before,
    # or when the model grows a little between two sizing builds; it used to write out of bounds.)
    import torch
    from paper_2607_01164_b200 import api
    g = inputs.c4_gaussians(seed=5, n_grid=64, n=30000)
    full = inputs.Grid((64, 64, 64), (0.0, 0.0, 0.0), (1 / 64, 1 / 64, 1 / 64))
    P = full.num_points
    ref = GpuRun(g, "grid", full, None)
    ctx = api.Context()
    dev = _dev(torch, g.mean, g.scale, g.quat, g.opacity, g.scalar)
    q = api.grid_query(full)
    phi, I = torch.empty(P, device="cuda"), torch.empty(P, device="cuda")
    ctx.gs_preprocess(*dev)
    ctx.gs_build_accel(q)                         # synchronous, option off: the buffer holds exactly T pairs (+ 12 % slack)
    ctx.gs_set_option(api.OPT_ASYNC_BUILD, 1)
    for step in range(3):                         # step 0: sizing build that finds T <= capacity < 1.5 T; 1, 2: asynchronous
        phi.fill_(-7.0)
        ctx.gs_build_accel(q)
        ctx.gs_sample_fwd(q, phi, I)
        torch.cuda.synchronize()
        assert torch.equal(phi, ref.phi[:P]) and torch.equal(I, ref.I[:P]), step
    assert ctx.gs_status_query()["grid_pairs"] == ref.ctx.gs_status_query()["grid_pairs"]
    ctx.close()


def test_contexts_on_their_own_streams_run_side_by_side(oracle):
    # Contexts are independent (gs.h: a context is bound to the stream given to gs_create; all scratch is context-owned): batches
    # of one grid dealt round-robin to three contexts on three CUDA streams give exactly the output of one context doing them
    # in turn.  This is how `bench.py` overlaps the builds and forwards of a configs[3] decode.
    import torch
    from paper_2607_01164_b200 import api
    g = inputs.c4_gaussians(seed=7, n_grid=64, n=40000)
    full = inputs.Grid((64, 64, 64), (0.0, 0.0, 0.0), (1 / 64, 1 / 64, 1 / 64))
    dev = _dev(torch, g.mean, g.scale, g.quat, g.opacity, g.scalar)
    batches = [full.batch((2 * x, 2 * y, 2 * z), (2, 2, 2)) for z in range(4) for y in range(4) for x in range(4)]
    qs = [api.grid_query(b) for b in batches]
    Pb = api.query_num_points(qs[0])
    one = api.Context()
    one.gs_preprocess(*dev)
    phi1, I1 = torch.empty(len(qs) * Pb, device="cuda"), torch.empty(len(qs) * Pb, device="cuda")
    for k, q in enumerate(qs):
        one.gs_build_accel(q)
        one.gs_sample_fwd(q, phi1[k * Pb:(k + 1) * Pb], I1[k * Pb:(k + 1) * Pb])
    torch.cuda.synchronize()
    ref = oracle.forward(g, oracle.grid_points(batches[5]), TAU, mode=1)    # one batch against the oracle, the rest against `one`
    assert np.abs(phi1[5 * Pb:6 * Pb].cpu().numpy() - ref["phi"]).max() <= 1e-5
    streams = [torch.cuda.Stream() for _ in range(3)]
    ctxs = [api.Context(stream=s_) for s_ in streams]
    for c, s_ in zip(ctxs, streams):
        s_.wait_stream(torch.cuda.current_stream())
        c.gs_set_option(api.OPT_ASYNC_BUILD, 1)
        c.gs_preprocess(*dev)
    phi3, I3 = torch.full_like(phi1, -7.0), torch.full_like(I1, -7.0)
    for s_ in streams:
        s_.wait_stream(torch.cuda.current_stream())
    for rep in range(2):
        for k, q in enumerate(qs):
            c = ctxs[k % 3]
            c.gs_build_accel(q)
            c.gs_sample_fwd(q, phi3[k * Pb:(k + 1) * Pb], I3[k * Pb:(k + 1) * Pb])
    torch.cuda.synchronize()
    assert torch.equal(phi3, phi1) and torch.equal(I3, I1)
    for c in ctxs + [one]:
        c.close()
