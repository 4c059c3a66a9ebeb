"""CPU ORACLE of the volume-rendering consumer of the sampler.  TEST INFRASTRUCTURE ONLY.

The paper renders its models by ray marching: "each render uses 1,024 samples per pixel ... using the matplotlib
"coolwarm" colormap and linear opacity map" in a NerfAcc-style volume renderer, discarding samples outside the volume's
domain (Fig. 1, Fig. 9).  For a W-VEG model the domain test is the model's own coverage rule
(I_c > tau): an uncovered sample is empty space.  Written out plainly:

    samples      t_k = t_near + (k + 1/2) dt,  dt = (t_far - t_near) / spp,  p_k = o + t_k d            (k = 0 .. spp-1)
    model        (Phi_k, I_k) = W-VEG forward at p_k (Eq. 2/3; oracle/wveg_oracle.c)
    transfer     (r, g, b, sigma)(x) = linear interpolation of a table over x = clamp(Phi, 0, 1)
    emission-absorption, front to back (the standard volume-rendering quadrature [Max 1995], which NerfAcc implements):
                 alpha_k = covered_k ? 1 - exp(-sigma(Phi_k) dt) : 0
                 C = sum_k T_k alpha_k rgb(Phi_k),  T_k = prod_{j<k} (1 - alpha_j),  A = 1 - T_spp

Positions are an integer-deciding quantity (coverage is discontinuous), so they are formed in float32 with ONE fixed
sequence on both sides (DESIGN D27): dt = (t1 - t0) / spp; t_k = fmaf((float)k + 0.5f, dt, t0); p = fmaf(t_k, d, o) per
component -- restated here with numpy float32 operations (fmaf emulated exactly in float64: a product of two float32
values and a float32 addend are exact in float64 up to one rounding, and double rounding cannot occur for 24-bit inputs
... it can: the emulation below therefore rounds the exact rational result, see _fmaf32).  Everything else is float64.
"""
from __future__ import annotations

from fractions import Fraction

import numpy as np

from . import wveg_oracle


def _fmaf32(a, b, c):
    """float32 fma(a, b, c) for arrays of float32, correctly rounded.  a * b is exact in float64 (24 + 24 <= 53 bits); adding
    c in float64 rounds once to 53 bits and the cast to float32 rounds again.  Double rounding can only change the result
    when the float64 sum lies exactly half-way between two float32 values while the exact sum does not; those cases are
    detected and redone in exact rational arithmetic."""
    a = np.asarray(a, np.float32).astype(np.float64)
    b = np.asarray(b, np.float32).astype(np.float64)
    c = np.asarray(c, np.float32).astype(np.float64)
    a, b, c = np.broadcast_arrays(a, b, c)
    s = a * b + c
    out = s.astype(np.float32)
    # candidates for double rounding: the float64 sum is a float32 half-way point (low 29 mantissa bits = 1 followed by zeros)
    bits = s.view(np.uint64) if s.flags["C_CONTIGUOUS"] else np.ascontiguousarray(s).view(np.uint64)
    tie = (bits & np.uint64((1 << 29) - 1)) == np.uint64(1 << 28)
    if np.any(tie):
        flat = out.reshape(-1)
        for i in np.flatnonzero(tie.reshape(-1)):
            exact = Fraction(float(a.reshape(-1)[i])) * Fraction(float(b.reshape(-1)[i])) + Fraction(float(c.reshape(-1)[i]))
            lo = np.float32(float(exact))   # float(Fraction) rounds once to float64; refine around it
            cands = [np.nextafter(lo, np.float32(-np.inf)), lo, np.nextafter(lo, np.float32(np.inf))]
            best = min(cands, key=lambda v: (abs(Fraction(float(v)) - exact), int(np.float32(v).view(np.uint32)) & 1))
            flat[i] = best
    return out


def ray_samples(origins, dirs, t_range, spp: int):
    """Sample positions [n, spp, 3] float32 (the fixed float32 sequence above) and the step dt [n] float32."""
    o = np.asarray(origins, np.float32)
    d = np.asarray(dirs, np.float32)
    t0, t1 = np.asarray(t_range, np.float32)[:, 0], np.asarray(t_range, np.float32)[:, 1]
    dt = ((t1 - t0) / np.float32(spp)).astype(np.float32)
    k = (np.arange(spp, dtype=np.float32) + np.float32(0.5)).astype(np.float32)
    t = _fmaf32(k[None, :], dt[:, None], t0[:, None])                      # [n, spp]
    p = _fmaf32(t[:, :, None], d[:, None, :], o[:, None, :])               # [n, spp, 3]
    return p, dt


def transfer(table, x):
    """Linear interpolation of a [K,4] table (r, g, b, extinction) at x = clamp(value, 0, 1)."""
    tab = np.asarray(table, np.float64)
    K = tab.shape[0]
    u = np.clip(np.asarray(x, np.float64), 0.0, 1.0) * (K - 1)
    i = np.minimum(np.floor(u).astype(np.int64), K - 2)
    f = (u - i)[..., None]
    return tab[i] * (1.0 - f) + tab[i + 1] * f


def render(g, origins, dirs, t_range, spp: int, table, tau: float = 0.01, mode: int = 1):
    """Returns dict(rgba [n,4] float64, phi / I [n,spp] float64 (the model along the rays), covered [n,spp] bool).
    A ray with t_far <= t_near sees nothing (all zeros)."""
    p, dt = ray_samples(origins, dirs, t_range, spp)
    n = p.shape[0]
    valid = np.asarray(t_range, np.float32)[:, 1] > np.asarray(t_range, np.float32)[:, 0]
    fwd = wveg_oracle.forward(g, np.ascontiguousarray(p.reshape(-1, 3)), tau, mode=mode, want_sets=False)
    phi = fwd["phi"].reshape(n, spp)
    I = fwd["I"].reshape(n, spp)
    covered = (I.astype(np.float32) > np.float32(tau)) & valid[:, None]
    tf = transfer(table, phi)
    alpha = np.where(covered, 1.0 - np.exp(-tf[..., 3] * dt.astype(np.float64)[:, None]), 0.0)
    rgba = np.zeros((n, 4))
    T = np.ones(n)
    for k in range(spp):   # front to back
        rgba[:, :3] += (T * alpha[:, k])[:, None] * tf[:, k, :3]
        T = T * (1.0 - alpha[:, k])
    rgba[:, 3] = 1.0 - T
    return dict(rgba=rgba, phi=phi, I=I, covered=covered, dt=dt)
