"""Pins of the oracle's integer stages: AABBs, brick keys, Morton codes and the
LBVH (north_star (2)).  Each is checked against an independent brute-force statement in numpy /
pure Python on tiny inputs, or against invariants that hold at any size.
"""
import math

import numpy as np

from paper_2607_01164_b200 import inputs

TAU = 0.01


def test_aabb_is_conservative_and_tight(oracle):
    # the cutoff ellipsoid's exact half-extent along world axis k is r sqrt(Sigma_kk), Sigma = R^T S^2 R
    from scipy.spatial.transform import Rotation
    g = inputs.c4_gaussians(seed=4, n_grid=64, n=2000)
    M, aabb, valid = oracle.preprocess_f32(g, TAU)
    assert valid.all()
    q = g.quat.astype(np.float64)
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    R = Rotation.from_quat(np.concatenate([q[:, 1:], q[:, :1]], axis=1)).as_matrix()
    S2 = g.scale.astype(np.float64) ** 2
    cov_diag = np.einsum("njk,nj->nk", R ** 2, S2)
    e = math.sqrt(-2 * math.log(TAU)) * np.sqrt(cov_diag)
    half = 0.5 * (aabb[:, 3:].astype(np.float64) - aabb[:, :3])
    assert np.all(half >= e) and np.all(half <= e * (1 + 2 ** -8 + 1e-5) + 1e-7)
    np.testing.assert_allclose(0.5 * (aabb[:, 3:].astype(np.float64) + aabb[:, :3]), g.mean, atol=1e-6)
    # whitening matrix reproduces the inverse covariance of Eq. 3: M^T M = R^T S^-2 R
    Mm = M.reshape(-1, 3, 3).astype(np.float64)
    conic = np.einsum("nji,njk->nik", Mm, Mm)
    ref = np.einsum("nji,nj,njk->nik", R, 1.0 / S2, R)
    np.testing.assert_allclose(conic, ref, rtol=2e-5, atol=2e-5 * np.abs(ref).max())


def test_every_hit_lies_inside_the_aabb(oracle):
    g = inputs.c4_gaussians(seed=1, n_grid=32, n=400)  # includes 20:1 elongated ones
    xyz = oracle.grid_points(inputs.c1_grid(32))
    M, aabb, valid = oracle.preprocess_f32(g, TAU)
    out = oracle.forward(g, xyz, TAU, mode=0, want_mask=True)
    mask = out["hit_mask"].astype(bool)
    inside = np.all((xyz[:, None, :] >= aabb[None, :, :3]) & (xyz[:, None, :] <= aabb[None, :, 3:]), axis=2)
    assert mask.sum() > 10000
    assert not np.any(mask & ~inside)


def test_brick_keys_brute_force(oracle):
    g = inputs.c1_gaussians(seed=0, n=300)
    g.mean[:5] = np.array([[-0.2, 0.5, 0.5], [1.3, 0.5, 0.5], [0.001, 0.001, 0.999], [0.5, -1, 0.5], [0.5, 0.5, 5]], np.float32)
    grid = inputs.Grid((40, 27, 19), (0.0, 0.0, 0.0), (1 / 40, 1 / 27, 1 / 19))  # ragged: 5 x 4 x 3 bricks
    for batch in (grid, grid.batch((1, 0, 1), (3, 2, 2))):
        M, aabb, valid = oracle.preprocess_f32(g, TAU)
        blo, bhi, cnt = oracle.brick_ranges(aabb, valid, batch)
        keys, start = oracle.brick_keys(blo, bhi, cnt, batch)
        # brute force: Gaussian i is listed for brick b iff its AABB interval meets the brick's slab on every axis
        expect = []
        lo3, cnt3 = batch.brick_lo, batch.brick_cnt
        for bz in range(cnt3[2]):
            for by in range(cnt3[1]):
                for bx in range(cnt3[0]):
                    bid = (bz * cnt3[1] + by) * cnt3[0] + bx
                    b = (bx + lo3[0], by + lo3[1], bz + lo3[2])
                    ok = np.ones(g.n, bool)
                    for k in range(3):
                        e0 = batch.origin[k] + 8 * b[k] * batch.spacing[k]
                        e1 = batch.origin[k] + 8 * (b[k] + 1) * batch.spacing[k]
                        ok &= (aabb[:, k].astype(np.float64) < e1) & (aabb[:, 3 + k].astype(np.float64) >= e0)
                    expect += [(bid << 32) | int(i) for i in np.nonzero(ok)[0]]
        assert len(expect) > 150
        assert np.array_equal(keys, np.array(sorted(expect), np.uint64))
        assert np.array_equal(np.sort(keys), keys) and len(np.unique(keys)) == len(keys)
        nb = cnt3[0] * cnt3[1] * cnt3[2]
        assert start[0] == 0 and start[nb] == len(keys)
        bricks = (keys >> np.uint64(32)).astype(np.int64)
        for b in range(nb):
            assert np.all(bricks[start[b]:start[b + 1]] == b)
        assert cnt.sum() == len(keys)


def test_brick_lists_cover_every_hit(oracle):
    # a hit pair must appear in the list of the brick holding the voxel (the cull is conservative)
    g = inputs.c4_gaussians(seed=2, n_grid=24, n=150)
    grid = inputs.c1_grid(24)
    xyz = oracle.grid_points(grid)
    M, aabb, valid = oracle.preprocess_f32(g, TAU)
    blo, bhi, cnt = oracle.brick_ranges(aabb, valid, grid)
    keys, start = oracle.brick_keys(blo, bhi, cnt, grid)
    keyset = set(int(k) for k in keys)
    out = oracle.forward(g, xyz, TAU, mode=0, want_mask=True)
    pts, gs = np.nonzero(out["hit_mask"])
    x, y, z = pts % 24, (pts // 24) % 24, pts // 576
    bid = ((z // 8) * 3 + (y // 8)) * 3 + (x // 8)
    assert len(pts) > 5000
    assert all(((int(b) << 32) | int(i)) in keyset for b, i in zip(bid, gs))


def _morton_py(q):
    code = 0
    for b in range(10):
        for k in range(3):
            code |= ((int(q[k]) >> b) & 1) << (3 * b + k)
    return code


def test_morton_codes(oracle):
    lo, hi = np.zeros(3, np.float32), np.ones(3, np.float32)
    pts = np.array([[0, 0, 0], [0.99999994, 0.99999994, 0.99999994], [1.0, 1.0, 1.0], [-3, 0.5, 2], [1 / 1024, 0, 0],
                    [0, 1 / 1024, 0], [0, 0, 1 / 1024], [0.5, 0.25, 0.125]], np.float32)
    codes = oracle.morton_codes(pts, lo, hi)
    assert list(codes[:3]) == [0, 2 ** 30 - 1, 2 ** 30 - 1]
    assert codes[3] == _morton_py((0, 512, 1023))
    assert list(codes[4:7]) == [1, 2, 4]  # x is the lowest bit of each triple (DESIGN D8)
    assert codes[7] == _morton_py((512, 256, 128))
    rng = np.random.default_rng(0)
    lo = np.array([-1.0, 0.25, 3.0], np.float32)
    hi = np.array([2.0, 0.75, 3.5], np.float32)
    pts = (lo + (hi - lo) * rng.uniform(-0.1, 1.1, (2000, 3))).astype(np.float32)
    codes = oracle.morton_codes(pts, lo, hi)
    # cell index = trunc of the position in 1024ths of the box, clamped (away from cell edges: exact in double too)
    t = (pts.astype(np.float64) - lo) / (hi.astype(np.float64) - lo) * 1024
    safe = np.all(np.abs(t - np.round(t)) > 1e-3, axis=1)
    q = np.clip(np.floor(t), 0, 1023).astype(np.int64)
    expect = np.array([_morton_py(r) for r in q], np.uint32)
    assert safe.sum() > 1900 and np.array_equal(codes[safe], expect[safe])
    valid = np.ones(2000, np.uint8)
    valid[7] = 0
    assert oracle.morton_codes(pts, lo, hi, valid)[7] == 1 << 30
    order, keys = oracle.morton_order(codes)
    assert np.array_equal(order, np.lexsort((np.arange(2000), codes)))
    assert np.array_equal(keys, (codes[order].astype(np.uint64) << np.uint64(32)) | order.astype(np.uint64))


def _check_tree(keys, tree, leaf_aabb):
    n = len(keys)
    left, right, parent = tree["left"], tree["right"], tree["parent"]
    assert parent[0] == -1

    def walk(node):  # returns (lo, hi) leaf range; checks the radix-tree property on the way
        ranges = []
        for child in (left[node], right[node]):
            if child < 0:
                leaf = ~child
                assert tree["leaf_parent"][leaf] == node
                ranges.append((leaf, leaf))
            else:
                assert parent[child] == node
                ranges.append(walk(child))
        (l0, l1), (r0, r1) = ranges
        assert l1 + 1 == r0  # contiguous, ordered
        lo, hi = l0, r1
        assert (tree["range_lo"][node], tree["range_hi"][node]) == (lo, hi)
        # Karras numbering: left child is internal node l1 (its last key), right child r0 (its first)
        if left[node] >= 0:
            assert left[node] == l1
        if right[node] >= 0:
            assert right[node] == r0
        # all keys of the node share a prefix that the two children split at its first differing bit
        full = int(keys[lo]) ^ int(keys[hi])
        split_bit = full.bit_length() - 1
        assert all(((int(keys[k]) >> split_bit) & 1) == 0 for k in range(l0, l1 + 1))
        assert all(((int(keys[k]) >> split_bit) & 1) == 1 for k in range(r0, r1 + 1))
        bb = tree["node_aabb"][node]
        assert np.array_equal(bb[:3], leaf_aabb[lo:hi + 1, :3].min(0)) and np.array_equal(bb[3:], leaf_aabb[lo:hi + 1, 3:].max(0))
        return lo, hi

    assert walk(0) == (0, n - 1)


def test_lbvh_topology(oracle):
    import sys
    sys.setrecursionlimit(10000)
    rng = np.random.default_rng(3)
    for n in (2, 3, 7, 64, 500):
        pts = rng.uniform(0, 1, (n, 3)).astype(np.float32)
        if n == 500:
            pts[100:300] = pts[100]  # many equal codes: the id in the low word keeps keys unique
        codes = oracle.morton_codes(pts, np.zeros(3, np.float32), np.ones(3, np.float32))
        order, keys = oracle.morton_order(codes)
        half = rng.uniform(0.01, 0.05, (n, 3)).astype(np.float32)
        leaf_aabb = np.concatenate([pts - half, pts + half], axis=1)[order]
        tree = oracle.lbvh_build(keys, leaf_aabb)
        assert len(tree["left"]) == n - 1
        _check_tree(keys, tree, leaf_aabb)
    assert len(oracle.lbvh_build(np.array([5], np.uint64), np.zeros((1, 6), np.float32))["left"]) == 0
    assert len(oracle.lbvh_build(np.zeros(0, np.uint64), np.zeros((0, 6), np.float32))["left"]) == 0


def test_grid_points(oracle):
    grid = inputs.Grid((20, 9, 17), (0.25, -1.0, 3.0), (0.1, 0.2, 0.05), (1, 0, 1), (2, 2, 1))
    xyz = oracle.grid_points(grid)
    assert grid.batch_dims == (12, 9, 8) and xyz.shape[0] == 12 * 9 * 8
    np.testing.assert_allclose(xyz, inputs.voxel_centres(grid), rtol=3e-7, atol=1e-7)
    # x fastest
    assert xyz[1, 0] > xyz[0, 0] and xyz[1, 1] == xyz[0, 1] and xyz[12, 1] > xyz[0, 1]
