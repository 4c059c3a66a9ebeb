"""ctypes binding of the CPU oracle (oracle/wveg_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It shares nothing with the CUDA path (paper_2607_01164_b200/csrc).
The wrappers only marshal numpy arrays; all arithmetic lives in the C file.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "wveg_oracle.c")
_LIB = os.path.join(_HERE, "libwveg_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C, OpenMP, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Gaussians(C.Structure):
    _fields_ = [("n", C.c_int64), ("mean", C.c_void_p), ("scale", C.c_void_p), ("quat", C.c_void_p),
                ("opacity", C.c_void_p), ("scalar", C.c_void_p)]


class _Grid(C.Structure):
    _fields_ = [("dims", C.c_int32 * 3), ("origin", C.c_float * 3), ("spacing", C.c_float * 3),
                ("brick_lo", C.c_int32 * 3), ("brick_cnt", C.c_int32 * 3)]


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.wo_r2_f32.restype = C.c_float
        _lib.wo_r2_f32.argtypes = [C.c_float]
        _lib.wo_r_f32.restype = C.c_float
        _lib.wo_r_f32.argtypes = [C.c_float]
        _lib.wo_num_threads.restype = C.c_int
        _lib.wo_jitter.restype = C.c_float
        _lib.wo_grid_num_points.restype = C.c_int64
        _lib.wo_brick_keys.restype = C.c_int64
        _lib.wo_forward.restype = C.c_int
        _lib.wo_backward.restype = C.c_int
        _lib.wo_lbvh_build.restype = C.c_int
    return _lib


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _p(a):
    return None if a is None else C.c_void_p(a.ctypes.data)


def _gs(g):
    """g: object with mean/scale/quat/opacity/scalar arrays.  Returns (struct, keepalive)."""
    arrs = [_f32(g.mean), _f32(g.scale), _f32(g.quat), _f32(g.opacity), _f32(g.scalar)]
    s = _Gaussians(arrs[0].shape[0], *[a.ctypes.data for a in arrs])
    return s, arrs


def _grid(grid):
    s = _Grid()
    for k in range(3):
        s.dims[k] = int(grid.dims[k])
        s.origin[k] = float(grid.origin[k])
        s.spacing[k] = float(grid.spacing[k])
        s.brick_lo[k] = int(grid.brick_lo[k])
        s.brick_cnt[k] = int(grid.brick_cnt[k])
    return s


def num_threads() -> int:
    return int(lib().wo_num_threads())


def r2(tau: float) -> float:
    return float(lib().wo_r2_f32(C.c_float(tau)))


def preprocess_f32(g, tau: float = 0.01):
    """fp32 whitening matrices M [N,9], cutoff AABBs [N,6] (lo, hi), valid [N] (decision precision)."""
    s, keep = _gs(g)
    n = s.n
    M = np.zeros((n, 9), np.float32)
    aabb = np.zeros((n, 6), np.float32)
    valid = np.zeros(n, np.uint8)
    lib().wo_preprocess_f32(C.byref(s), C.c_float(tau), _p(M), _p(aabb), _p(valid))
    return M, aabb, valid


def hit_f32(M9, mu, p, tau: float = 0.01) -> bool:
    M9, mu, p = _f32(M9), _f32(mu), _f32(p)
    lib().wo_hit_f32.restype = C.c_int
    return bool(lib().wo_hit_f32(_p(M9), _p(mu), _p(p), C.c_float(tau)))


def grid_points(grid, jitter_seed=None) -> np.ndarray:
    """[P,3] f32 sample positions of a grid batch (x fastest): voxel centres, or with jitter_seed one random position
    inside every voxel's cell (counter-based generator, DESIGN D26)."""
    s = _grid(grid)
    P = int(lib().wo_grid_num_points(C.byref(s)))
    xyz = np.zeros((P, 3), np.float32)
    if jitter_seed is None:
        lib().wo_grid_points(C.byref(s), _p(xyz))
    else:
        lib().wo_grid_points_jitter(C.byref(s), C.c_uint64(int(jitter_seed)), _p(xyz))
    return xyz


def jitter(seed: int, voxel_linear: int, axis: int) -> float:
    return float(lib().wo_jitter(C.c_uint64(int(seed)), C.c_uint64(int(voxel_linear)), C.c_int(axis)))


def forward(g, xyz, tau: float = 0.01, mode: int = 1, hit_mask_in=None, covered_in=None, want_mask: bool = False,
            want_sets: bool = True):
    """Returns dict(phi f64 [P], I f64 [P], count u32, hsum u64, hxor u64[, hit_mask u8 [P,N]])."""
    s, keep = _gs(g)
    xyz = _f32(xyz)
    P = xyz.shape[0]
    out = dict(phi=np.zeros(P, np.float64), I=np.zeros(P, np.float64))
    if want_sets:
        out.update(count=np.zeros(P, np.uint32), hsum=np.zeros(P, np.uint64), hxor=np.zeros(P, np.uint64))
    if want_mask:
        out["hit_mask"] = np.zeros((P, s.n), np.uint8)
    if hit_mask_in is not None:
        hit_mask_in = np.ascontiguousarray(hit_mask_in, np.uint8)
        assert hit_mask_in.shape == (P, s.n)
    if covered_in is not None:
        covered_in = np.ascontiguousarray(covered_in, np.uint8)
    rc = lib().wo_forward(C.byref(s), _p(xyz), C.c_int64(P), C.c_float(tau), C.c_int(mode), _p(hit_mask_in),
                          _p(covered_in), _p(out["phi"]), _p(out["I"]), _p(out.get("count")), _p(out.get("hsum")),
                          _p(out.get("hxor")), _p(out.get("hit_mask")))
    if rc != 0:
        raise RuntimeError("wo_forward failed")
    return out


def mse(phi, I, target, tau: float = 0.01):
    """Returns (loss, dL_dphi f64 [P], sample_err f64 [P])."""
    phi = np.ascontiguousarray(phi, np.float64)
    I = np.ascontiguousarray(I, np.float64)
    target = _f32(target)
    P = phi.shape[0]
    loss = C.c_double(0.0)
    d = np.zeros(P, np.float64)
    e = np.zeros(P, np.float64)
    lib().wo_mse(_p(phi), _p(I), _p(target), C.c_int64(P), C.c_float(tau), C.byref(loss), _p(d), _p(e))
    return float(loss.value), d, e


def loss(phi, I, target, defined=None, tau: float = 0.01, kind: str = "l1", lambda_fn: float = 0.0, eps_fn: float = 0.0,
         lambda_fp: float = 0.0):
    """The paper's training losses (L1 or MSE reconstruction over the defined samples, Eq. 4 false-negative and Eq. 5
    false-positive terms).  Returns dict(loss (rec, fn, fp), dL_dphi, dL_dI, sample_err f64 [P], counts (nD, nFN, nFP))."""
    phi = np.ascontiguousarray(phi, np.float64)
    I = np.ascontiguousarray(I, np.float64)
    target = _f32(target)
    P = phi.shape[0]
    dmask = None if defined is None else np.ascontiguousarray(defined, np.uint8)
    l3 = np.zeros(3, np.float64)
    c3 = np.zeros(3, np.int64)
    a = np.zeros(P, np.float64)
    b = np.zeros(P, np.float64)
    e = np.zeros(P, np.float64)
    lib().wo_loss(_p(phi), _p(I), _p(target), _p(dmask), C.c_int64(P), C.c_float(tau), C.c_int({"mse": 0, "l1": 1}[kind]),
                  C.c_float(lambda_fn), C.c_float(eps_fn), C.c_float(lambda_fp), _p(l3), _p(a), _p(b), _p(e), _p(c3))
    return dict(loss=tuple(float(x) for x in l3), dL_dphi=a, dL_dI=b, sample_err=e, counts=tuple(int(x) for x in c3))


PAPER_LR = (0.00016, 0.001, 0.0001, 0.025, 0.0025)  # mean, scale, quat, opacity (weights), scalar (values): PAPER.md:231


def activate(raw_scale, raw_opacity, raw_scalar):
    """exp / sigmoid / sigmoid activations.  Returns (scale [n,3], opacity [n], scalar [n]) in f64."""
    rs, rw, rv = _f32(raw_scale), _f32(raw_opacity), _f32(raw_scalar)
    n = rw.shape[0]
    s, w, v = np.zeros((n, 3)), np.zeros(n), np.zeros(n)
    lib().wo_activate(C.c_int64(n), _p(rs), _p(rw), _p(rv), _p(s), _p(w), _p(v))
    return s, w, v


def adam_step(params: dict, grads: dict, m, v, t: int, lr=PAPER_LR, beta1=0.9, beta2=0.999, eps=1e-8):
    """One Adam step on the raw parameters (dict mean, raw_scale, quat, raw_opacity, raw_scalar: f64 arrays, updated in
    place) from the gradients w.r.t. the ACTIVATED values (dict dmean, dscale, dquat, dopacity, dscalar).  m, v: f64
    [12 n] moment blocks (mean | scale | quat | opacity | scalar), updated in place."""
    n = params["raw_opacity"].shape[0]
    for k in ("mean", "raw_scale", "quat", "raw_opacity", "raw_scalar"):
        assert params[k].dtype == np.float64 and params[k].flags["C_CONTIGUOUS"]
    g = {k: np.ascontiguousarray(grads[k], np.float64) for k in ("dmean", "dscale", "dquat", "dopacity", "dscalar")}
    lr = np.ascontiguousarray(lr, np.float64)
    lib().wo_adam_step(C.c_int64(n), _p(params["mean"]), _p(params["raw_scale"]), _p(params["quat"]), _p(params["raw_opacity"]),
                       _p(params["raw_scalar"]), _p(g["dmean"]), _p(g["dscale"]), _p(g["dquat"]), _p(g["dopacity"]),
                       _p(g["dscalar"]), _p(m), _p(v), _p(lr), C.c_double(beta1), C.c_double(beta2), C.c_double(eps), C.c_int(t))


PARAM_KEYS = ("mean", "raw_scale", "quat", "raw_opacity", "raw_scalar")
_WIDTH = dict(mean=3, raw_scale=3, quat=4, raw_opacity=1, raw_scalar=1)


def _moment_blocks(m, n):
    """Views of a [12 n] moment block: mean 3n | scale 3n | quat 4n | opacity n | scalar n."""
    out, o = {}, 0
    for k in PARAM_KEYS:
        out[k] = m[o:o + _WIDTH[k] * n]
        o += _WIDTH[k] * n
    return out


def prune(params: dict, m, v, opacity, tau2: float = 0.005):
    """Pruning: "periodically removes Gaussians below a chosen ... threshold", here the weight threshold
    0.005.  Keeps, in their order, the Gaussians with opacity >= tau2 (decided on the float32 activated opacity);
    their parameters and Adam moments move with them.  Returns (params, m, v, kept indices)."""
    keep = np.flatnonzero(np.asarray(opacity, np.float32) >= np.float32(tau2))
    n, n2 = len(opacity), len(keep)
    mb, vb = _moment_blocks(np.asarray(m), n), _moment_blocks(np.asarray(v), n)
    p2 = {k: np.ascontiguousarray(np.asarray(params[k]).reshape(n, -1)[keep]).reshape((n2,) + np.asarray(params[k]).shape[1:]) for k in PARAM_KEYS}
    m2 = np.concatenate([mb[k].reshape(n, -1)[keep].ravel() for k in PARAM_KEYS])
    v2 = np.concatenate([vb[k].reshape(n, -1)[keep].ravel() for k in PARAM_KEYS])
    return p2, m2, v2, keep


def densify_select(sample_err, I, defined, k: int, tau: float = 0.01):
    """Sample-error densification ("new Gaussians with means at the positions of the k highest error
    samples"; "we include false negative positions as the top priority").  Candidates are the samples
    defined in the volume; a false negative is a defined sample the model does not cover (I <= tau, Fig. 6A).  Order:
    false negatives first, then by error, highest first; equal errors by sample index, lowest first.  Returns the
    indices of the first min(k, number of defined samples) samples of that order."""
    err = np.asarray(sample_err, np.float32)
    If = np.asarray(I, np.float32)
    P = len(err)
    d = np.ones(P, bool) if defined is None else (np.asarray(defined) != 0)
    fn = d & ~(If > np.float32(tau))
    cand = np.flatnonzero(d)
    order = sorted(cand.tolist(), key=lambda c: (not fn[c], -float(err[c]), c))
    return np.asarray(order[:min(k, len(order))], np.int64)


def densify(params: dict, m, v, positions, target, sel, raw_scale_init: float, raw_opacity_init: float, clamp: float = 1e-4):
    """Appends one Gaussian per selected sample, "given parameters in the same way as initialization, with values
    corresponding to the ground truth samples" (isotropic, initial weight 0.01, scale by the
    caller): mean = sample position, raw_scale = raw_scale_init on the three axes, identity rotation,
    raw_opacity = raw_opacity_init, raw_scalar = logit(clip(target, clamp, 1 - clamp)) with the float32 bounds clamp and
    1.0f - clamp (the target is float32); zero Adam moments."""
    n, a = len(params["raw_opacity"]), len(sel)
    lo, hi = float(np.float32(clamp)), float(np.float32(1.0) - np.float32(clamp))
    t = np.clip(np.asarray(target, np.float32)[sel].astype(np.float64), lo, hi)
    new = dict(mean=np.asarray(positions, np.float32)[sel].astype(np.float64), raw_scale=np.full((a, 3), np.float32(raw_scale_init), np.float64),
               quat=np.tile(np.array([1.0, 0, 0, 0]), (a, 1)), raw_opacity=np.full(a, np.float32(raw_opacity_init), np.float64),
               raw_scalar=np.log(t / (1 - t)))
    p2 = {k: np.concatenate([np.asarray(params[k], np.float64), new[k]]) for k in PARAM_KEYS}
    mb, vb = _moment_blocks(np.asarray(m), n), _moment_blocks(np.asarray(v), n)
    m2 = np.concatenate([np.concatenate([mb[k], np.zeros(_WIDTH[k] * a)]) for k in PARAM_KEYS])
    v2 = np.concatenate([np.concatenate([vb[k], np.zeros(_WIDTH[k] * a)]) for k in PARAM_KEYS])
    return p2, m2, v2


def backward(g, xyz, phi, I, a, b=None, target=None, tau: float = 0.01, mode: int = 1, hit_mask_in=None,
             covered_in=None):
    """Returns dict(dmean [N,3], dscale [N,3], dquat [N,4], dopacity [N], dscalar [N], err [N]) in f64."""
    s, keep = _gs(g)
    xyz = _f32(xyz)
    P, n = xyz.shape[0], s.n
    phi = np.ascontiguousarray(phi, np.float64)
    I = np.ascontiguousarray(I, np.float64)
    a = np.ascontiguousarray(a, np.float64)
    b = None if b is None else np.ascontiguousarray(b, np.float64)
    target = None if target is None else _f32(target)
    if hit_mask_in is not None:
        hit_mask_in = np.ascontiguousarray(hit_mask_in, np.uint8)
    if covered_in is not None:
        covered_in = np.ascontiguousarray(covered_in, np.uint8)
    out = dict(dmean=np.zeros((n, 3)), dscale=np.zeros((n, 3)), dquat=np.zeros((n, 4)), dopacity=np.zeros(n),
               dscalar=np.zeros(n), err=np.zeros(n))
    rc = lib().wo_backward(C.byref(s), _p(xyz), C.c_int64(P), C.c_float(tau), C.c_int(mode), _p(hit_mask_in),
                           _p(covered_in), _p(phi), _p(I), _p(a), _p(b), _p(target), _p(out["dmean"]), _p(out["dscale"]),
                           _p(out["dquat"]), _p(out["dopacity"]), _p(out["dscalar"]), _p(out["err"]))
    if rc != 0:
        raise RuntimeError("wo_backward failed")
    return out


def brick_ranges(aabb, valid, grid):
    aabb = _f32(aabb)
    valid = np.ascontiguousarray(valid, np.uint8)
    n = aabb.shape[0]
    s = _grid(grid)
    blo = np.zeros((n, 3), np.int32)
    bhi = np.zeros((n, 3), np.int32)
    cnt = np.zeros(n, np.uint32)
    lib().wo_brick_ranges(_p(aabb), _p(valid), C.c_int64(n), C.byref(s), _p(blo), _p(bhi), _p(cnt))
    return blo, bhi, cnt


def brick_keys(blo, bhi, cnt, grid):
    """Sorted (brick<<32 | gaussian) keys u64 [T] and brick_start i64 [nbricks+1]."""
    s = _grid(grid)
    T = int(cnt.astype(np.int64).sum())
    keys = np.zeros(max(T, 1), np.uint64)
    nbricks = int(grid.brick_cnt[0]) * int(grid.brick_cnt[1]) * int(grid.brick_cnt[2])
    start = np.zeros(nbricks + 1, np.int64)
    got = lib().wo_brick_keys(_p(blo), _p(bhi), _p(cnt), C.c_int64(cnt.shape[0]), C.byref(s), _p(keys), _p(start))
    assert got == T
    return keys[:T], start


def morton_codes(xyz, lo, hi, valid=None):
    xyz = _f32(xyz)
    n = xyz.shape[0]
    lo3 = (C.c_float * 3)(*[float(x) for x in lo])
    hi3 = (C.c_float * 3)(*[float(x) for x in hi])
    valid = None if valid is None else np.ascontiguousarray(valid, np.uint8)
    codes = np.zeros(n, np.uint32)
    lib().wo_morton_codes(_p(xyz), _p(valid), C.c_int64(n), lo3, hi3, _p(codes))
    return codes


def morton_order(codes):
    codes = np.ascontiguousarray(codes, np.uint32)
    n = codes.shape[0]
    order = np.zeros(n, np.uint32)
    keys = np.zeros(n, np.uint64)
    lib().wo_morton_order(_p(codes), C.c_int64(n), _p(order), _p(keys))
    return order, keys


def lbvh_build(sorted_keys, leaf_aabb_sorted):
    """Radix tree over sorted unique keys.  Returns dict(left, right, parent, leaf_parent, node_aabb, range_lo, range_hi)."""
    keys = np.ascontiguousarray(sorted_keys, np.uint64)
    bb = _f32(leaf_aabb_sorted)
    n = keys.shape[0]
    m = max(n - 1, 1)
    out = dict(left=np.zeros(m, np.int32), right=np.zeros(m, np.int32), parent=np.zeros(m, np.int32),
               leaf_parent=np.zeros(max(n, 1), np.int32), node_aabb=np.zeros((m, 6), np.float32),
               range_lo=np.zeros(m, np.int32), range_hi=np.zeros(m, np.int32))
    rc = lib().wo_lbvh_build(_p(keys), C.c_int64(n), _p(bb), _p(out["left"]), _p(out["right"]), _p(out["parent"]),
                             _p(out["leaf_parent"]), _p(out["node_aabb"]), _p(out["range_lo"]), _p(out["range_hi"]))
    if rc != 0:
        raise RuntimeError("wo_lbvh_build failed")
    if n < 2:
        for k in ("left", "right", "parent", "node_aabb", "range_lo", "range_hi"):
            out[k] = out[k][:0]
    return out
