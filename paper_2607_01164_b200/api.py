"""Thin Python binding of the C ABI in include/gs.h (argument marshalling only).

Every step of the path runs in the CUDA kernels of ``csrc/``; torch is used for device memory and
the stream handle.  There is no CPU fallback: if ``libgs.so`` is missing or cannot be loaded the
import of the library fails loudly (``GsLibraryError``).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgs.so")

GS_OK, GS_ERR_INVALID_ARG, GS_ERR_STATE, GS_ERR_OOM, GS_ERR_OVERFLOW, GS_ERR_CUDA = range(6)
GS_QUERY_GRID, GS_QUERY_POINTS = 0, 1
_STATUS = {0: "GS_OK", 1: "GS_ERR_INVALID_ARG", 2: "GS_ERR_STATE", 3: "GS_ERR_OOM", 4: "GS_ERR_OVERFLOW", 5: "GS_ERR_CUDA"}

# gs_debug_item
(DBG_RECORDS, DBG_AABB, DBG_BRICK_COUNT, DBG_PAIR_BRICK, DBG_PAIR_GAUSS, DBG_BRICK_START, DBG_LEAF_MORTON, DBG_LEAF_ORDER,
 DBG_NODE_LEFT, DBG_NODE_RIGHT, DBG_NODE_PARENT, DBG_LEAF_PARENT, DBG_NODE_AABB, DBG_POINT_ORDER, DBG_POINT_MORTON) = range(15)

EXPORTS = ["gs_create", "gs_destroy", "gs_last_error", "gs_preprocess", "gs_build_accel", "gs_sample_fwd", "gs_sample_bwd",
           "gs_step_host", "gs_debug_get", "gs_debug_read", "gs_debug_point_sets", "gs_debug_counters",
           "gs_profile_enable", "gs_profile_read", "gs_measure_alu_peaks", "gs_measure_alu_peaks2", "gs_sample_fwd_loss",
           "gs_params_activate", "gs_adam_step", "gs_prune", "gs_densify", "gs_set_sample_count", "gs_status_query", "gs_set_option", "gs_render", "gs_decode_grid",
           "gs_probe_points_static"]
PROF_STAGES = ["preprocess", "build", "fwd", "bwd_pack", "bwd", "finalize", "cull"]


class GsLibraryError(RuntimeError):
    pass


class GsError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{_STATUS.get(status, status)}: {msg}")
        self.status = status


class _Gaussians(C.Structure):
    _fields_ = [("n", C.c_uint32), ("mean", C.c_void_p), ("scale", C.c_void_p), ("quat", C.c_void_p),
                ("opacity", C.c_void_p), ("scalar", C.c_void_p)]


class _Domain(C.Structure):
    _fields_ = [("lo", C.c_float * 3), ("hi", C.c_float * 3)]


class _Query(C.Structure):
    _fields_ = [("kind", C.c_int32), ("dims", C.c_int32 * 3), ("origin", C.c_float * 3), ("spacing", C.c_float * 3),
                ("brick_lo", C.c_int32 * 3), ("brick_cnt", C.c_int32 * 3), ("num_points", C.c_uint64), ("xyz", C.c_void_p),
                ("presorted", C.c_int32), ("jitter", C.c_int32), ("jitter_seed", C.c_uint64)]


class _Grads(C.Structure):
    _fields_ = [("dmean", C.c_void_p), ("dscale", C.c_void_p), ("dquat", C.c_void_p), ("dopacity", C.c_void_p),
                ("dscalar", C.c_void_p), ("err", C.c_void_p)]


class _Loss(C.Structure):
    _fields_ = [("kind", C.c_int32), ("lambda_fn", C.c_float), ("eps_fn", C.c_float), ("lambda_fp", C.c_float),
                ("defined", C.c_void_p), ("num_defined", C.c_uint64)]


class _RawParams(C.Structure):
    _fields_ = [("n", C.c_uint32), ("mean", C.c_void_p), ("raw_scale", C.c_void_p), ("quat", C.c_void_p),
                ("raw_opacity", C.c_void_p), ("raw_scalar", C.c_void_p)]


class _StatusInfo(C.Structure):
    _fields_ = [("num_gaussians", C.c_uint64), ("invalid_gaussians", C.c_uint64), ("grid_pairs", C.c_uint64),
                ("grid_touched", C.c_uint64), ("cull_chunk_capacity", C.c_uint64), ("decode_repeats", C.c_uint64)]


class _AdamCfg(C.Structure):
    _fields_ = [("lr", C.c_float * 5), ("beta1", C.c_float), ("beta2", C.c_float), ("eps", C.c_float), ("step", C.c_int32)]


LOSS_MSE, LOSS_L1 = 0, 1
OPT_POINTS_ACCEL, OPT_ASYNC_BUILD, OPT_BWD_HIT_MASKS = 0, 1, 2
POINTS_GATHER, POINTS_SCATTER = 0, 1
PAPER_LR = (0.00016, 0.001, 0.0001, 0.025, 0.0025)  # mean, scale, quat, opacity (weights), scalar (values): PAPER.md:231

_lib = None


def load_library():
    """dlopen libgs.so and declare the prototypes.  Raises GsLibraryError when it is missing (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise GsLibraryError(f"{LIB_PATH} is missing: build it with `python -m paper_2607_01164_b200.build` "
                             "(there is no CPU fallback)")
    try:
        lib = C.CDLL(LIB_PATH)
    except OSError as e:  # pragma: no cover
        raise GsLibraryError(f"cannot load {LIB_PATH}: {e}") from e
    P = C.c_void_p
    lib.gs_create.argtypes = [C.c_int, P, C.POINTER(P)]
    lib.gs_destroy.argtypes = [P]
    lib.gs_destroy.restype = None
    lib.gs_last_error.argtypes = [P]
    lib.gs_last_error.restype = C.c_char_p
    lib.gs_preprocess.argtypes = [P, C.POINTER(_Gaussians), C.POINTER(_Domain), C.c_float]
    lib.gs_build_accel.argtypes = [P, C.POINTER(_Query)]
    lib.gs_sample_fwd.argtypes = [P, C.POINTER(_Query), P, P, P, P, P, P]
    lib.gs_sample_bwd.argtypes = [P, C.POINTER(_Query), P, P, P, P, P, C.POINTER(_Grads)]
    lib.gs_sample_fwd_loss.argtypes = [P, C.POINTER(_Query), C.POINTER(_Loss), P, P, P, P, P, P, P]
    lib.gs_step_host.argtypes = [P, C.POINTER(_Gaussians), C.POINTER(_Domain), C.c_float, C.POINTER(_Query), P, P, P, P,
                                 C.POINTER(_Grads)]
    lib.gs_debug_get.argtypes = [P, C.c_int32, C.POINTER(P), C.POINTER(C.c_size_t)]
    lib.gs_debug_read.argtypes = [P, C.c_int32, P, C.c_size_t]
    lib.gs_debug_point_sets.argtypes = [P, C.POINTER(_Query), P, P, P]
    lib.gs_debug_counters.argtypes = [P, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
    lib.gs_params_activate.argtypes = [P, C.POINTER(_RawParams), P, P, P]
    lib.gs_adam_step.argtypes = [P, C.POINTER(_RawParams), C.POINTER(_Grads), P, P, C.POINTER(_AdamCfg), P, P, P]
    lib.gs_prune.argtypes = [P, C.POINTER(_RawParams), P, P, P, C.c_float, C.POINTER(C.c_uint32)]
    lib.gs_densify.argtypes = [P, C.POINTER(_RawParams), P, P, C.c_uint32, C.POINTER(_Query), P, P, P, C.c_uint64, P, C.c_uint32,
                               C.c_float, C.c_float, C.POINTER(C.c_uint32)]
    lib.gs_measure_alu_peaks.argtypes = [P, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    lib.gs_measure_alu_peaks2.argtypes = [P, C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_double)]
    lib.gs_set_sample_count.argtypes = [P, C.c_uint64]
    lib.gs_set_option.argtypes = [P, C.c_int32, C.c_int64]
    lib.gs_render.argtypes = [P, C.c_uint32, P, P, P, C.c_uint32, P, C.c_uint32, P]
    lib.gs_decode_grid.argtypes = [P, C.POINTER(_Gaussians), C.c_float, C.POINTER(_Query), C.POINTER(C.c_int32), C.c_int32, P, P]
    lib.gs_status_query.argtypes = [P, C.POINTER(_StatusInfo)]
    lib.gs_probe_points_static.argtypes = [C.c_int, P, C.POINTER(_Gaussians), C.c_float, P, C.c_uint64, P, P, C.c_char_p, C.c_size_t]
    lib.gs_profile_enable.argtypes = [P, C.c_int32]
    lib.gs_profile_read.argtypes = [P, C.POINTER(C.c_float), C.POINTER(C.c_uint32), C.POINTER(C.c_uint64)]
    for name in EXPORTS:
        if name not in ("gs_destroy", "gs_last_error"):
            getattr(lib, name).restype = C.c_int
    _lib = lib
    return lib


def _ptr(t):
    """Device (torch) or host (numpy) array -> address; None -> NULL."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        assert t.flags["C_CONTIGUOUS"]
        return C.c_void_p(t.ctypes.data)
    assert t.is_contiguous()
    return C.c_void_p(t.data_ptr())


def grid_query(grid, jitter_seed=None) -> _Query:
    """``grid``: object with dims, origin, spacing, brick_lo, brick_cnt (e.g. inputs.Grid).  jitter_seed: one random
    sample position inside every voxel's cell instead of its centre (gs.h)."""
    q = _Query()
    q.kind = GS_QUERY_GRID
    if jitter_seed is not None:
        q.jitter = 1
        q.jitter_seed = int(jitter_seed)
    for k in range(3):
        q.dims[k] = int(grid.dims[k])
        q.origin[k] = float(grid.origin[k])
        q.spacing[k] = float(grid.spacing[k])
        q.brick_lo[k] = int(grid.brick_lo[k])
        q.brick_cnt[k] = int(grid.brick_cnt[k])
    return q


def points_query(xyz, presorted: bool = False) -> _Query:
    """``xyz``: [P,3] float32, device tensor (or host array for step_host)."""
    q = _Query()
    q.kind = GS_QUERY_POINTS
    q.num_points = int(xyz.shape[0])
    q.xyz = _ptr(xyz).value if xyz.shape[0] else None
    q.presorted = int(bool(presorted))
    q._keep = xyz
    return q


def query_num_points(q: _Query) -> int:
    if q.kind == GS_QUERY_POINTS:
        return int(q.num_points)
    n = 1
    for k in range(3):
        n *= min(8 * q.brick_cnt[k], q.dims[k] - 8 * q.brick_lo[k])
    return n


def _gaussians(mean, scale, quat, opacity, scalar) -> _Gaussians:
    g = _Gaussians()
    g.n = int(mean.shape[0])
    g.mean, g.scale, g.quat, g.opacity, g.scalar = (_ptr(a).value if g.n else None for a in (mean, scale, quat, opacity, scalar))
    return g


def _domain(dom):
    if dom is None:
        return None
    d = _Domain()
    for k in range(3):
        d.lo[k] = float(dom[0][k])
        d.hi[k] = float(dom[1][k])
    return C.byref(d)


PROBE_MAX_GAUSSIANS = 16384   # GS_PROBE_MAX_GAUSSIANS


def gs_probe_points_static(mean, scale, quat, opacity, scalar, xyz, phi, I, tau: float = 0.01, device: int | None = None, stream=None):
    """gs_probe_points_static (gs.h): Phi and I of a model of at most PROBE_MAX_GAUSSIANS Gaussians at xyz[P,3], written
    into the caller's phi[P] / I[P], without a Context and without any device allocation by the library -- for code
    that runs inside another application's memory pool or a real-time loop and so cannot call cudaMalloc.  All arrays
    are device tensors the caller allocated beforehand.  The scratch is one fixed array shared by all calls on the
    device: do not let two calls overlap on the GPU (use one stream, or order them).  The first call per device does
    a one-time address lookup; make it at start-up."""
    import torch
    lib = load_library()
    if not torch.cuda.is_available():
        raise GsLibraryError("no CUDA device: the W-VEG sampler has no CPU fallback")
    device = torch.cuda.current_device() if device is None else int(device)
    stream = torch.cuda.current_stream(device) if stream is None else stream
    g = _gaussians(mean, scale, quat, opacity, scalar)
    n = int(xyz.shape[0])
    msg = C.create_string_buffer(512)
    st = lib.gs_probe_points_static(device, C.c_void_p(stream.cuda_stream), C.byref(g), C.c_float(tau), _ptr(xyz) if n else None,
                                    C.c_uint64(n), _ptr(phi) if n else None, _ptr(I) if n else None, msg, C.c_size_t(len(msg)))
    if st != GS_OK:
        raise GsError(st, msg.value.decode())


class Context:
    """One gs_ctx bound to the current torch CUDA device and stream."""

    def __init__(self, device: int | None = None, stream=None):
        import torch
        self._torch = torch
        self.lib = load_library()
        if not torch.cuda.is_available():
            raise GsLibraryError("no CUDA device: the W-VEG sampler has no CPU fallback")
        self.device = torch.cuda.current_device() if device is None else int(device)
        self.stream = torch.cuda.current_stream(self.device) if stream is None else stream
        h = C.c_void_p()
        st = self.lib.gs_create(self.device, C.c_void_p(self.stream.cuda_stream), C.byref(h))
        if st != GS_OK:
            raise GsError(st, "gs_create failed")
        self.h = h

    def close(self):
        if getattr(self, "h", None):
            self.lib.gs_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, st):
        if st != GS_OK:
            raise GsError(st, self.lib.gs_last_error(self.h).decode())

    # ---- the four calls of the path ---------------------------------------------------------
    def gs_preprocess(self, mean, scale, quat, opacity, scalar, domain=None, tau: float = 0.01):
        g = _gaussians(mean, scale, quat, opacity, scalar)
        self._check(self.lib.gs_preprocess(self.h, C.byref(g), _domain(domain), C.c_float(tau)))

    def gs_build_accel(self, q: _Query):
        self._check(self.lib.gs_build_accel(self.h, C.byref(q)))

    def gs_sample_fwd(self, q: _Query, phi, I, target=None, loss=None, dL_dphi=None, sample_err=None):
        self._check(self.lib.gs_sample_fwd(self.h, C.byref(q), _ptr(target), _ptr(phi), _ptr(I), _ptr(loss), _ptr(dL_dphi),
                                           _ptr(sample_err)))

    def gs_sample_fwd_loss(self, q: _Query, phi, I, target, kind=LOSS_L1, lambda_fn=0.0, eps_fn=0.0, lambda_fp=0.0, defined=None,
                           num_defined=None, loss_terms=None, dL_dphi=None, dL_dI=None, sample_err=None):
        """Forward with the paper's losses fused (gs.h).  num_defined defaults to P (defined is None)."""
        nd = query_num_points(q) if num_defined is None else int(num_defined)
        d = _ptr(defined)
        spec = _Loss(int(kind), float(lambda_fn), float(eps_fn), float(lambda_fp), d.value if d is not None else None, nd)
        self._check(self.lib.gs_sample_fwd_loss(self.h, C.byref(q), C.byref(spec), _ptr(target), _ptr(phi), _ptr(I), _ptr(loss_terms),
                                                _ptr(dL_dphi), _ptr(dL_dI), _ptr(sample_err)))

    def gs_sample_bwd(self, q: _Query, phi, I, dL_dphi, grads: dict, dL_dI=None, target=None):
        g = _Grads(*[(_ptr(grads.get(k)).value if grads.get(k) is not None else None)
                     for k in ("dmean", "dscale", "dquat", "dopacity", "dscalar", "err")])
        self._check(self.lib.gs_sample_bwd(self.h, C.byref(q), _ptr(phi), _ptr(I), _ptr(dL_dphi), _ptr(dL_dI), _ptr(target),
                                           C.byref(g)))

    def gs_step_host(self, g_host: dict, q_host: _Query, target_host, phi_host, I_host, grads_host: dict | None, domain=None,
                     tau: float = 0.01) -> float:
        """All arrays are numpy (host).  Returns the loss."""
        g = _gaussians(g_host["mean"], g_host["scale"], g_host["quat"], g_host["opacity"], g_host["scalar"])
        loss = C.c_double(0.0)
        gr = None
        if grads_host is not None:
            gr = C.byref(_Grads(*[(_ptr(grads_host.get(k)).value if grads_host.get(k) is not None else None)
                                  for k in ("dmean", "dscale", "dquat", "dopacity", "dscalar", "err")]))
        self._check(self.lib.gs_step_host(self.h, C.byref(g), _domain(domain), C.c_float(tau), C.byref(q_host), _ptr(target_host),
                                          _ptr(phi_host), _ptr(I_host), C.byref(loss), gr))
        return float(loss.value)

    @staticmethod
    def _raw(raw: dict) -> _RawParams:
        n = int(raw["raw_opacity"].shape[0])
        return _RawParams(n, *[_ptr(raw[k]).value for k in ("mean", "raw_scale", "quat", "raw_opacity", "raw_scalar")])

    def gs_params_activate(self, raw: dict, scale, opacity, scalar, n=None):
        """raw: dict of device tensors mean, raw_scale, quat, raw_opacity, raw_scalar (n: Gaussians in use, default all)."""
        r = self._raw(raw)
        if n is not None:
            r.n = int(n)
        self._check(self.lib.gs_params_activate(self.h, C.byref(r), _ptr(scale), _ptr(opacity), _ptr(scalar)))

    def gs_adam_step(self, raw: dict, grads: dict, m, v, step: int, lr=PAPER_LR, beta1=0.9, beta2=0.999, eps=1e-8,
                     scale_out=None, opacity_out=None, scalar_out=None, n=None):
        r = self._raw(raw)
        if n is not None:
            r.n = int(n)
        g = _Grads(*[(_ptr(grads.get(k)).value if grads.get(k) is not None else None)
                     for k in ("dmean", "dscale", "dquat", "dopacity", "dscalar", "err")])
        cfg = _AdamCfg((C.c_float * 5)(*lr), beta1, beta2, eps, int(step))
        self._check(self.lib.gs_adam_step(self.h, C.byref(r), C.byref(g), _ptr(m), _ptr(v), C.byref(cfg), _ptr(scale_out),
                                          _ptr(opacity_out), _ptr(scalar_out)))

    def gs_prune(self, raw: dict, n: int, m, v, opacity, tau2: float = 0.005) -> int:
        """raw: dict of device tensors with room for >= n Gaussians; returns the new count."""
        r = self._raw(raw)
        r.n = int(n)
        out = C.c_uint32()
        self._check(self.lib.gs_prune(self.h, C.byref(r), _ptr(m), _ptr(v), _ptr(opacity), C.c_float(tau2), C.byref(out)))
        return int(out.value)

    def gs_densify(self, raw: dict, n: int, m, v, capacity: int, q: _Query, sample_err, I, target, k: int, raw_scale_init: float,
                   raw_opacity_init: float, defined=None, num_defined=None) -> int:
        r = self._raw(raw)
        r.n = int(n)
        nd = query_num_points(q) if num_defined is None else int(num_defined)
        out = C.c_uint32()
        self._check(self.lib.gs_densify(self.h, C.byref(r), _ptr(m), _ptr(v), int(capacity), C.byref(q), _ptr(sample_err), _ptr(I),
                                        _ptr(defined), nd, _ptr(target), int(k), C.c_float(raw_scale_init),
                                        C.c_float(raw_opacity_init), C.byref(out)))
        return int(out.value)

    def measure_alu_peaks(self):
        """(FP32 FMA lane-instructions per second, MUFU.EX2 per second, FMA lane-operations per second through the packed
        f32x2 form) of this device now; synchronises."""
        a, b, c = C.c_double(), C.c_double(), C.c_double()
        self._check(self.lib.gs_measure_alu_peaks2(self.h, C.byref(a), C.byref(b), C.byref(c)))
        return float(a.value), float(b.value), float(c.value)

    def gs_render(self, origins, dirs, t_range, spp: int, table, rgba):
        """Ray-march the current model (gs.h gs_render): device tensors origins/dirs [n,3], t_range [n,2], table [K,4], rgba [n,4]."""
        self._check(self.lib.gs_render(self.h, C.c_uint32(int(origins.shape[0])), _ptr(origins), _ptr(dirs), _ptr(t_range),
                                       C.c_uint32(int(spp)), _ptr(table), C.c_uint32(int(table.shape[0])), _ptr(rgba)))

    def gs_decode_grid(self, mean, scale, quat, opacity, scalar, region: _Query, batch_bricks, phi, I, streams: int = 0, tau: float = 0.01):
        """Forward-only decode of `region` (a grid query: its brick_lo / brick_cnt give the sub-box) in batches of batch_bricks
        bricks, dealt to `streams` worker contexts (gs.h gs_decode_grid).  phi / I: device tensors, BATCH-MAJOR."""
        g = _gaussians(mean, scale, quat, opacity, scalar)
        bb = (C.c_int32 * 3)(*[int(x) for x in batch_bricks])
        self._check(self.lib.gs_decode_grid(self.h, C.byref(g), C.c_float(tau), C.byref(region), bb, C.c_int32(int(streams)), _ptr(phi), _ptr(I)))

    def gs_set_option(self, key: int, value: int):
        self._check(self.lib.gs_set_option(self.h, C.c_int32(int(key)), C.c_int64(int(value))))

    def gs_set_sample_count(self, total_samples: int):
        self._check(self.lib.gs_set_sample_count(self.h, C.c_uint64(int(total_samples))))

    def gs_status_query(self) -> dict:
        info = _StatusInfo()
        self._check(self.lib.gs_status_query(self.h, C.byref(info)))
        return {k: int(getattr(info, k)) for k, _ in _StatusInfo._fields_}

    def profile_enable(self, on: bool = True):
        self._check(self.lib.gs_profile_enable(self.h, int(on)))

    def profile_read(self):
        """(ms per stage dict, calls per stage dict, kernel launches) since the last read; synchronises."""
        ms = (C.c_float * len(PROF_STAGES))()
        calls = (C.c_uint32 * len(PROF_STAGES))()
        launches = C.c_uint64()
        self._check(self.lib.gs_profile_read(self.h, ms, calls, C.byref(launches)))
        return ({k: float(ms[i]) for i, k in enumerate(PROF_STAGES)}, {k: int(calls[i]) for i, k in enumerate(PROF_STAGES)},
                int(launches.value))

    # ---- helpers -----------------------------------------------------------------------------
    def alloc_grads(self, n: int, with_err: bool = True, flat: bool = False) -> dict:
        """Gradient tensors of n Gaussians.  flat=True: views into ONE contiguous float32 buffer (key "flat"; every section
        starts on a 16-byte boundary), which dist.allreduce_grads sums over the ranks in place with a single collective."""
        t = self._torch
        dev = t.device("cuda", self.device)
        if flat:
            from .dist import flat_layout
            off, total = flat_layout(n)
            buf = t.zeros(total, dtype=t.float32, device=dev)
            out = {k: buf[o:o + n * c].view((n, c) if c > 1 else (n,)) for k, (o, c) in off.items()}
            out["flat"] = buf
            return out
        out = dict(dmean=t.empty((n, 3), dtype=t.float32, device=dev), dscale=t.empty((n, 3), dtype=t.float32, device=dev),
                   dquat=t.empty((n, 4), dtype=t.float32, device=dev), dopacity=t.empty(n, dtype=t.float32, device=dev),
                   dscalar=t.empty(n, dtype=t.float32, device=dev))
        if with_err:
            out["err"] = t.empty(n, dtype=t.float32, device=dev)
        return out

    def debug_get(self, what: int, dtype, cols: int = 1):
        """Copy a context-owned debug buffer to a numpy array (synchronises)."""
        p, n = C.c_void_p(), C.c_size_t()
        self._check(self.lib.gs_debug_get(self.h, what, C.byref(p), C.byref(n)))
        out = np.empty(int(n.value) * cols, dtype)
        self._check(self.lib.gs_debug_read(self.h, what, _ptr(out), out.nbytes))
        return out.reshape(-1, cols) if cols > 1 else out

    def debug_point_sets(self, q: _Query):
        t = self._torch
        dev = t.device("cuda", self.device)
        P = query_num_points(q)
        cnt = t.zeros(max(P, 1), dtype=t.int32, device=dev)
        hs = t.zeros(max(P, 1), dtype=t.int64, device=dev)
        hx = t.zeros(max(P, 1), dtype=t.int64, device=dev)
        self._check(self.lib.gs_debug_point_sets(self.h, C.byref(q), _ptr(cnt), _ptr(hs), _ptr(hx)))
        a, b = C.c_uint64(), C.c_uint64()
        self._check(self.lib.gs_debug_counters(self.h, C.byref(a), C.byref(b)))
        return (cnt.cpu().numpy().view(np.uint32)[:P], hs.cpu().numpy().view(np.uint64)[:P], hx.cpu().numpy().view(np.uint64)[:P],
                int(a.value), int(b.value))
