"""Seeded synthetic inputs for the W-VEG sampling path (shared by oracle tests and GPU tests).

This module holds NO arithmetic of the method (no Gaussian kernel, no aggregation, no
gradients): it only draws model parameters, query positions and target fields with
numpy ``Generator(PCG64(seed))`` and rounds them to fp32.  Both the CPU oracle and the
CUDA path consume exactly these arrays.

The five workloads are the ones BASELINE.json lists (C1..C5); they stand in for the
paper's datasets, which are not available (Open SciVis volumes, Table 4 PAPER.md:385-392;
unstructured meshes, Table 5).  Every generator takes size arguments so
tests can run reduced copies with the same distributions.

Conventions: quaternion order (w, x, y, z); ``scale`` is the linear standard deviation
per principal axis (already activated); ``opacity`` is the paper's weight
w_i in (0, 1); ``scalar`` is v_i.
"""
from __future__ import annotations

import dataclasses
import numpy as np

F32 = np.float32


@dataclasses.dataclass
class Gaussians:
    mean: np.ndarray      # [N,3] f32
    scale: np.ndarray     # [N,3] f32, > 0
    quat: np.ndarray      # [N,4] f32 (w,x,y,z), not necessarily unit
    opacity: np.ndarray   # [N]   f32, the paper's weight w_i
    scalar: np.ndarray    # [N]   f32, the paper's value v_i

    @property
    def n(self) -> int:
        return int(self.mean.shape[0])

    def subset(self, idx) -> "Gaussians":
        return Gaussians(*(np.ascontiguousarray(getattr(self, f.name)[idx]) for f in dataclasses.fields(self)))


@dataclasses.dataclass
class Grid:
    """Structured query: voxel-centre samples p = origin + (i + 0.5) * spacing, x fastest.

    ``brick_lo``/``brick_cnt`` select a brick-aligned (8^3 voxels per brick) sub-box = one batch.
    """
    dims: tuple            # (nx, ny, nz) voxels of the whole grid
    origin: tuple          # (ox, oy, oz)
    spacing: tuple         # (sx, sy, sz)
    brick_lo: tuple = (0, 0, 0)
    brick_cnt: tuple | None = None

    def __post_init__(self):
        if self.brick_cnt is None:
            self.brick_cnt = tuple((d + 7) // 8 - b for d, b in zip(self.dims, self.brick_lo))

    @property
    def batch_dims(self) -> tuple:
        """Voxel extent (bx, by, bz) of this batch, clipped to the grid (ragged last bricks)."""
        return tuple(min(8 * c, d - 8 * lo) for c, d, lo in zip(self.brick_cnt, self.dims, self.brick_lo))

    @property
    def num_points(self) -> int:
        b = self.batch_dims
        return int(b[0]) * int(b[1]) * int(b[2])

    @property
    def domain(self):
        lo = np.asarray(self.origin, F32)
        hi = (lo + np.asarray(self.dims, F32) * np.asarray(self.spacing, F32)).astype(F32)
        return lo, hi

    def batch(self, brick_lo, brick_cnt) -> "Grid":
        return Grid(self.dims, self.origin, self.spacing, tuple(brick_lo), tuple(brick_cnt))


def _unit_grid(n) -> Grid:
    n = (n, n, n) if np.isscalar(n) else tuple(n)
    return Grid(n, (0.0, 0.0, 0.0), tuple(float(F32(1.0) / F32(k)) for k in n))


def voxel_centres(grid: Grid) -> np.ndarray:
    """[P,3] f64 world positions of the batch's samples, for evaluating TARGET fields only.

    (The method's own sample positions are computed inside the oracle / the kernels from the
    grid descriptor; this helper is used to synthesise ground-truth data.)
    """
    bx, by, bz = grid.batch_dims
    ix = np.arange(bx) + 8 * grid.brick_lo[0]
    iy = np.arange(by) + 8 * grid.brick_lo[1]
    iz = np.arange(bz) + 8 * grid.brick_lo[2]
    z, y, x = np.meshgrid(iz, iy, ix, indexing="ij")
    p = np.stack([x.ravel(), y.ravel(), z.ravel()], axis=1).astype(np.float64) + 0.5
    return p * np.asarray(grid.spacing, np.float64) + np.asarray(grid.origin, np.float64)


def _random_quats(rng, n) -> np.ndarray:
    q = rng.standard_normal((n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    return q.astype(F32)


def _sigmoid(x):
    return 1.0 / (1.0 + np.exp(-x))


def _log_uniform(rng, lo, hi, size):
    return np.exp(rng.uniform(np.log(lo), np.log(hi), size))


# ----------------------------------------------------------------------------------------
# C1: tiny structured
# ----------------------------------------------------------------------------------------
def c1_gaussians(seed: int = 0, n: int = 1024) -> Gaussians:
    """BASELINE.json configs[0]: means U[0,1]^3, per-axis scales log-U[0.01,0.05], random unit
    quaternions, opacity = sigmoid(N(0,1)), scalar U[0,1]."""
    rng = np.random.Generator(np.random.PCG64(seed))
    mean = rng.uniform(0.0, 1.0, (n, 3)).astype(F32)
    scale = _log_uniform(rng, 0.01, 0.05, (n, 3)).astype(F32)
    quat = _random_quats(rng, n)
    opacity = _sigmoid(rng.standard_normal(n)).astype(F32)
    scalar = rng.uniform(0.0, 1.0, n).astype(F32)
    return Gaussians(mean, scale, quat, opacity, scalar)


def c1_grid(n: int = 32) -> Grid:
    return _unit_grid(n)


# ----------------------------------------------------------------------------------------
# C2: Marschner-Lobb, 256^3
# ----------------------------------------------------------------------------------------
def marschner_lobb(p: np.ndarray, alpha: float = 0.25, f_m: float = 6.0) -> np.ndarray:
    """Marschner-Lobb test signal on [0,1]^3 (mapped to [-1,1]^3); analytic range is [0,1]."""
    q = 2.0 * np.asarray(p, np.float64) - 1.0
    x, y, z = q[..., 0], q[..., 1], q[..., 2]
    r = np.sqrt(x * x + y * y)
    rho_r = np.cos(2.0 * np.pi * f_m * np.cos(np.pi * r / 2.0))
    return (1.0 - np.sin(np.pi * z / 2.0) + alpha * (1.0 + rho_r)) / (2.0 * (1.0 + alpha))


def c2_grid(n: int = 256) -> Grid:
    return _unit_grid(n)


def c2_gaussians(seed: int = 2, n_grid: int = 256, n: int = 262144, sigma_voxels: float = 1.5) -> Gaussians:
    """configs[1]: Gaussians at distinct random voxel centres, isotropic 1.5-voxel sigma, identity
    rotation, opacity 0.5, scalar = field at the centre."""
    rng = np.random.Generator(np.random.PCG64(seed))
    flat = rng.choice(n_grid ** 3, size=n, replace=False)
    ix, iy, iz = flat % n_grid, (flat // n_grid) % n_grid, flat // (n_grid * n_grid)
    mean64 = (np.stack([ix, iy, iz], axis=1) + 0.5) / n_grid
    mean = mean64.astype(F32)
    scale = np.full((n, 3), sigma_voxels / n_grid, F32)
    quat = np.zeros((n, 4), F32)
    quat[:, 0] = 1.0
    opacity = np.full(n, 0.5, F32)
    scalar = marschner_lobb(mean64).astype(F32)
    return Gaussians(mean, scale, quat, opacity, scalar)


def c2_target(grid: Grid) -> np.ndarray:
    return marschner_lobb(voxel_centres(grid)).astype(F32)


# ----------------------------------------------------------------------------------------
# C3: unstructured mixture
# ----------------------------------------------------------------------------------------
def _rotations(rng, n):
    """n random orthonormal frames (QR of a normal matrix) orienting the mixture components."""
    q, r = np.linalg.qr(rng.standard_normal((n, 3, 3)))
    return q * np.sign(np.diagonal(r, axis1=1, axis2=2))[:, None, :]


def c3_points(seed: int = 3, p: int = 2_000_000, components: int = 16):
    """configs[2]: points from a 16-component anisotropic mixture clipped to [0,1]^3; scalar =
    sum of 8 sinusoids + 1 % Gaussian noise, min-max normalised.  Returns (xyz f32 [P,3], t f32 [P])."""
    rng = np.random.Generator(np.random.PCG64(seed))
    centres = rng.uniform(0.2, 0.8, (components, 3))
    sig = _log_uniform(rng, 0.03, 0.15, (components, 3))
    rot = _rotations(rng, components)
    out = np.empty((p, 3), np.float64)
    filled = 0
    while filled < p:
        m = int((p - filled) * 1.3) + 1024
        k = rng.integers(0, components, m)
        loc = rng.standard_normal((m, 3)) * sig[k]
        pts = centres[k] + np.einsum("mji,mj->mi", rot[k], loc)
        pts = pts[np.all((pts >= 0.0) & (pts < 1.0), axis=1)]
        take = min(len(pts), p - filled)
        out[filled:filled + take] = pts[:take]
        filled += take
    xyz = out.astype(F32)
    freq = rng.uniform(1.0, 8.0, (8, 3)) * 2.0 * np.pi * np.sign(rng.standard_normal((8, 3)))
    phase = rng.uniform(0.0, 2.0 * np.pi, 8)
    t = np.zeros(p, np.float64)
    for f, ph in zip(freq, phase):
        t += np.sin(xyz.astype(np.float64) @ f + ph) / 8.0
    t += 0.01 * rng.standard_normal(p)
    t = (t - t.min()) / (t.max() - t.min())
    return xyz, t.astype(F32)


def c3_gaussians(xyz: np.ndarray, t: np.ndarray, seed: int = 3, n: int = 1_048_576,
                 sigma_lo: float = 0.002, sigma_hi: float = 0.02) -> Gaussians:
    """configs[2] model: means = random subset of the points (the paper initialises from data
    vertices), per-axis scales log-U[0.002,0.02], random rotations."""
    rng = np.random.Generator(np.random.PCG64(seed + 1000))
    idx = rng.choice(len(xyz), size=n, replace=False)
    mean = np.ascontiguousarray(xyz[idx])
    scale = _log_uniform(rng, sigma_lo, sigma_hi, (n, 3)).astype(F32)
    quat = _random_quats(rng, n)
    opacity = _sigmoid(rng.standard_normal(n)).astype(F32)
    scalar = np.ascontiguousarray(t[idx])
    return Gaussians(mean, scale, quat, opacity, scalar)


def batch_indices(seed: int, step: int, total: int, batch: int) -> np.ndarray:
    """A batch of ``batch`` distinct indices in [0,total), fresh per step (sampling w/o replacement)."""
    rng = np.random.Generator(np.random.PCG64([seed, step]))
    if batch >= total:
        return np.arange(total, dtype=np.int64)
    return rng.choice(total, size=batch, replace=False)


# ----------------------------------------------------------------------------------------
# C4: large structured, turbulence-like field
# ----------------------------------------------------------------------------------------
@dataclasses.dataclass
class FourierField:
    """Sum of random Fourier modes with a k^-5/3 energy spectrum (amplitude ~ k^-5/6), affinely
    normalised with analytic bounds so that values lie in [0,1]."""
    k: np.ndarray       # [M,3] wave vectors (cycles per unit length * 2 pi)
    amp: np.ndarray     # [M]
    phase: np.ndarray   # [M]

    def __call__(self, p: np.ndarray) -> np.ndarray:
        p = np.asarray(p, np.float64)
        out = np.zeros(p.shape[:-1], np.float64)
        for k, a, ph in zip(self.k, self.amp, self.phase):
            out += a * np.sin(p @ k + ph)
        s = float(np.sum(np.abs(self.amp)))
        return (out + s) / (2.0 * s)


def c4_field(seed: int = 4, modes: int = 64, kmin: float = 1.0, kmax: float = 32.0) -> FourierField:
    rng = np.random.Generator(np.random.PCG64(seed + 2000))
    kmag = _log_uniform(rng, kmin, kmax, modes)
    d = rng.standard_normal((modes, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    amp = kmag ** (-5.0 / 6.0)
    phase = rng.uniform(0.0, 2.0 * np.pi, modes)
    return FourierField(2.0 * np.pi * kmag[:, None] * d, amp, phase)


def c4_grid(n: int = 1024) -> Grid:
    return _unit_grid(n)


def c4_gaussians(seed: int = 4, n_grid: int = 1024, n: int = 4_194_304, field: FourierField | None = None,
                 elongated_frac: float = 0.05) -> Gaussians:
    """configs[3]: means uniform over the grid; 95 % per-axis scales log-U[0.5,4] voxels; 5 %
    elongated (s, s, 20 s), s log-U[0.5,1] voxels; random rotations."""
    rng = np.random.Generator(np.random.PCG64(seed))
    field = field or c4_field(seed)
    mean64 = rng.uniform(0.0, 1.0, (n, 3))
    scale = _log_uniform(rng, 0.5, 4.0, (n, 3)) / n_grid
    elong = rng.uniform(0.0, 1.0, n) < elongated_frac
    s = _log_uniform(rng, 0.5, 1.0, n) / n_grid
    scale[elong] = np.stack([s, s, 20.0 * s], axis=1)[elong]
    quat = _random_quats(rng, n)
    opacity = _sigmoid(rng.standard_normal(n)).astype(F32)
    mean = mean64.astype(F32)
    scalar = np.empty(n, F32)
    for a in range(0, n, 1 << 18):
        scalar[a:a + (1 << 18)] = field(mean[a:a + (1 << 18)].astype(np.float64)).astype(F32)
    return Gaussians(mean, scale.astype(F32), quat, opacity, scalar)


def c4_target(grid: Grid, field: FourierField) -> np.ndarray:
    """Target of one batch, evaluated on the fly (the whole 1024^3 field is never materialised)."""
    return field(voxel_centres(grid)).astype(F32)


# ----------------------------------------------------------------------------------------
# C5: large unstructured, shell and fragments
# ----------------------------------------------------------------------------------------
def c5_points(seed: int = 5, p: int = 200_000_000, clusters: int = 4096, shell_frac: float = 0.7,
              chunk: int = 1 << 21, workers: int | None = None):
    """configs[4]: 70 % of points in a spherical shell (radius 0.35, thickness 0.05, centre 0.5),
    30 % in ``clusters`` small fragments (sigma 0.004); scalar = radial profile + high-frequency
    noise.  Returns (xyz f32 [P,3], t f32 [P]).

    The full set is 200 M points (3.2 GB with the scalars): it is generated in chunks of 2^21 points, each from a random
    stream of its own (seed, chunk index), so that the chunks can be drawn by a pool of threads and the first k points
    are the same for every p >= k."""
    import concurrent.futures
    import os
    rng = np.random.Generator(np.random.PCG64(seed))
    centres = rng.uniform(0.05, 0.95, (clusters, 3))
    kf = rng.uniform(40.0, 120.0, (4, 3)) * np.sign(rng.standard_normal((4, 3)))
    xyz = np.empty((p, 3), F32)
    t = np.empty(p, F32)

    def draw(a: int):
        n_keep = min(chunk, p - a)
        m = chunk   # a whole chunk is always drawn (and the tail dropped), so that a shorter set is a prefix of a longer one
        r_ = np.random.Generator(np.random.PCG64([seed, 1 + a // chunk]))
        is_shell = r_.uniform(0.0, 1.0, m) < shell_frac
        d = r_.standard_normal((m, 3))
        d /= np.linalg.norm(d, axis=1, keepdims=True)
        rad = 0.35 + 0.05 * (r_.uniform(0.0, 1.0, m) - 0.5)
        pts_shell = 0.5 + d * rad[:, None]
        k = r_.integers(0, clusters, m)
        pts_frag = centres[k] + 0.004 * r_.standard_normal((m, 3))
        pts = np.where(is_shell[:, None], pts_shell, pts_frag)
        pts = np.clip(pts, 0.0, np.nextafter(1.0, 0.0))
        r = np.linalg.norm(pts - 0.5, axis=1)
        val = 0.5 + 0.35 * np.cos(9.0 * r) + 0.0375 * np.sum(np.sin(pts @ kf.T), axis=1)
        xyz[a:a + n_keep] = pts[:n_keep].astype(F32)
        t[a:a + n_keep] = np.clip(val[:n_keep], 0.0, 1.0).astype(F32)

    starts = list(range(0, p, chunk))
    nw = workers if workers else min(len(starts), os.cpu_count() or 1, 32)
    if nw <= 1:
        for a in starts:
            draw(a)
    else:
        with concurrent.futures.ThreadPoolExecutor(max_workers=nw) as ex:
            list(ex.map(draw, starts))
    return xyz, t


def c5_gaussians(xyz: np.ndarray, t: np.ndarray, seed: int = 5, n: int = 8_388_608) -> Gaussians:
    """configs[4] model: means = random subset of the points, per-axis scales log-U[0.0005,0.002]."""
    return c3_gaussians(xyz, t, seed=seed, n=n, sigma_lo=0.0005, sigma_hi=0.002)


def points_domain(xyz: np.ndarray):
    """Axis-aligned box of the data, padded by one ulp so every point quantises inside it."""
    lo = xyz.min(axis=0).astype(F32)
    hi = np.nextafter(xyz.max(axis=0).astype(F32), F32(np.inf))
    return lo, hi


# ----------------------------------------------------------------------------------------
# Rays and transfer functions for the volume-rendering consumer of the sampler
# ----------------------------------------------------------------------------------------
def camera_rays(width: int, height: int, eye, look_at, up=(0.0, 0.0, 1.0), fov_y_deg: float = 40.0,
                box=((0.0, 0.0, 0.0), (1.0, 1.0, 1.0))):
    """Pinhole-camera rays through the pixel centres, clipped to an axis-aligned box (slab test).
    Returns origins [n,3], unit directions [n,3], t_range [n,2] (t_near, t_far; t_far <= t_near for a ray that misses the
    box), all float32, row-major over (y, x).  Input preparation only: the renderer and its oracle both take these arrays."""
    eye = np.asarray(eye, np.float64)
    f = np.asarray(look_at, np.float64) - eye
    f /= np.linalg.norm(f)
    r = np.cross(f, np.asarray(up, np.float64))
    r /= np.linalg.norm(r)
    u = np.cross(r, f)
    ty = np.tan(np.radians(fov_y_deg) / 2.0)
    tx = ty * width / height
    xs = (2.0 * (np.arange(width) + 0.5) / width - 1.0) * tx
    ys = (1.0 - 2.0 * (np.arange(height) + 0.5) / height) * ty
    d = f[None, None, :] + xs[None, :, None] * r[None, None, :] + ys[:, None, None] * u[None, None, :]
    d /= np.linalg.norm(d, axis=2, keepdims=True)
    d = d.reshape(-1, 3)
    o = np.broadcast_to(eye, d.shape)
    lo, hi = np.asarray(box[0], np.float64), np.asarray(box[1], np.float64)
    with np.errstate(divide="ignore", invalid="ignore"):
        t1 = (lo - o) / d
        t2 = (hi - o) / d
    tn = np.nanmax(np.minimum(t1, t2), axis=1)
    tf = np.nanmin(np.maximum(t1, t2), axis=1)
    tn = np.maximum(tn, 0.0)
    return np.ascontiguousarray(o, F32), np.ascontiguousarray(d, F32), np.ascontiguousarray(np.stack([tn, tf], axis=1), F32)


def diverging_transfer(k: int = 256, extinction: float = 40.0) -> np.ndarray:
    """A transfer function table [k,4] float32: a blue-white-red diverging colour ramp (in the spirit of the "coolwarm" map
    the paper renders with) and a LINEAR opacity map (extinction per unit length = extinction * value)."""
    x = np.linspace(0.0, 1.0, k)
    cold, mid, warm = np.array([0.23, 0.30, 0.75]), np.array([0.87, 0.87, 0.87]), np.array([0.71, 0.02, 0.15])
    rgb = np.where(x[:, None] < 0.5, cold + (mid - cold) * (2 * x[:, None]), mid + (warm - mid) * (2 * x[:, None] - 1))
    return np.concatenate([rgb, (extinction * x)[:, None]], axis=1).astype(F32)
