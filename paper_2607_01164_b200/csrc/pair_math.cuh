// pair_math.cuh -- the per (sample, Gaussian) arithmetic shared by the sm_100a sampling kernels.
// Eq. 3: G = exp(-1/2 d^T R^T S^-2 R d) = exp(-|u|^2 / 2), u = M d, M = S^-1 R, d = p - mu.
// The membership decision qd <= r2 (support G >= tau, D3/D4) is an integer decision:
// its fp32 operation sequence is fixed (round-to-nearest intrinsics are never contracted/reordered).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gs {

struct Rec {          // one Gaussian's record: 4 float4 planes
    float4 a;         // mu.xyz, w
    float4 b;         // M row 0, v
    float4 c;         // M row 1, -
    float4 d;         // M row 2, v w
};

// canonical fp32 sequence (D4): 3 FSUB; u_j = fma(M_j2, dz, fma(M_j1, dy, M_j0 * dx)); qd = fma(u2,u2, fma(u1,u1, u0*u0))
__device__ __forceinline__ float mahalanobis(const Rec &g, float px, float py, float pz, float &u0, float &u1, float &u2) {
    const float dx = __fsub_rn(px, g.a.x), dy = __fsub_rn(py, g.a.y), dz = __fsub_rn(pz, g.a.z);
    u0 = __fmaf_rn(g.b.z, dz, __fmaf_rn(g.b.y, dy, __fmul_rn(g.b.x, dx)));
    u1 = __fmaf_rn(g.c.z, dz, __fmaf_rn(g.c.y, dy, __fmul_rn(g.c.x, dx)));
    u2 = __fmaf_rn(g.d.z, dz, __fmaf_rn(g.d.y, dy, __fmul_rn(g.d.x, dx)));
    return __fmaf_rn(u2, u2, __fmaf_rn(u1, u1, __fmul_rn(u0, u0)));
}

// G = exp(-qd/2) through one MUFU.EX2 (value arithmetic; rel. error ~1e-7)
__device__ __forceinline__ float gauss_weight(float qd) {
    float r;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(qd * -0.72134752044448170368f));
    return r;
}

// grid sample position (D6): p = fmaf((float)i + 0.5f, spacing, origin)
__device__ __forceinline__ float voxel_centre(int i, float spacing, float origin) {
    return __fmaf_rn(__fadd_rn((float)i, 0.5f), spacing, origin);
}

// In-cell jitter of grid samples (DESIGN D26): counter-based, so every kernel (and the oracle) draws the same
// numbers.  The voxel with GLOBAL linear index L draws one 64-bit number h = splitmix64 finaliser of (seed + L); axis a
// takes 21 of its bits, j_a = ((h >> 21 a) & (2^21 - 1)) * 2^-21 - 0.5 in [-0.5, 0.5); the sample sits at
// fmaf(((float)i + 0.5f) + j, spacing, origin).  k_jitter_table writes h once per step (uint2 per voxel of the batch).
__device__ __forceinline__ unsigned long long mix64_u64(unsigned long long z) {
    z += 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}
__device__ __forceinline__ uint2 voxel_hash(unsigned long long seed, unsigned long long L) {
    const unsigned long long h = mix64_u64(seed + L);
    return make_uint2((uint32_t)h, (uint32_t)(h >> 32));
}
__device__ __forceinline__ float jitter_from_bits(uint32_t b21) { return __fmaf_rn((float)b21, 4.76837158203125e-7f, -0.5f); }  // exact
__device__ __forceinline__ void voxel_jitter3(uint2 h, float &jx, float &jy, float &jz) {
    jx = jitter_from_bits(h.x & 0x1FFFFFu);
    jy = jitter_from_bits(((h.x >> 21) | (h.y << 11)) & 0x1FFFFFu);
    jz = jitter_from_bits((h.y >> 10) & 0x1FFFFFu);
}
__device__ __forceinline__ float voxel_sample(int i, float j, float spacing, float origin) {
    return __fmaf_rn(__fadd_rn(__fadd_rn((float)i, 0.5f), j), spacing, origin);
}
// global linear voxel index of the jitter counter
__device__ __forceinline__ unsigned long long voxel_linear(int gx, int gy, int gz, int dimx, int dimy) {
    return ((unsigned long long)gz * (unsigned long long)dimy + (unsigned long long)gy) * (unsigned long long)dimx + (unsigned long long)gx;
}

// Fused-MSE backward coefficients of a GRID batch (written by k_grid_fwd, read by k_grid_bwd): samples are stored in
// aligned pairs, float4 per pair (c even) = (alpha_c, alpha_c+1, beta_c, beta_c+1), so that the two x-neighbours of a
// row arrive as the two halves of packed registers.  Index of alpha_c in floats; beta_c sits 2 floats further.
__device__ __forceinline__ size_t pack2_index(size_t c) { return ((c >> 1) << 2) | (c & 1); }

// id hash for order-free set comparison (splitmix64 finaliser of id + golden gamma)
__device__ __forceinline__ unsigned long long mix64(uint32_t id) {
    unsigned long long z = (unsigned long long)id + 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

// The backward contribution of one hit (S7):  with alpha = a/I, beta = b - alpha Phi (per sample),
//   gamma = alpha v + beta,  t = gamma w G:  dv += alpha w G, dw += gamma G, U += t u, W += t u u^T, E += eps w G
// acc layout: 0 dv | 1 dw | 2..4 U | 5..10 W00 W01 W02 W11 W12 W22 | 11 E
template <int K>
__device__ __forceinline__ void bwd_accumulate(float (&acc)[K], float alpha, float beta, float eps, float w, float v, float G,
                                               float u0, float u1, float u2) {
    const float wG = w * G;
    const float gamma = fmaf(alpha, v, beta);
    const float t = gamma * wG;
    acc[0] = fmaf(alpha, wG, acc[0]);
    acc[1] = fmaf(gamma, G, acc[1]);
    const float t0 = t * u0, t1 = t * u1, t2 = t * u2;
    acc[2] += t0; acc[3] += t1; acc[4] += t2;
    acc[5] = fmaf(t0, u0, acc[5]); acc[6] = fmaf(t0, u1, acc[6]); acc[7] = fmaf(t0, u2, acc[7]);
    acc[8] = fmaf(t1, u1, acc[8]); acc[9] = fmaf(t1, u2, acc[9]); acc[10] = fmaf(t2, u2, acc[10]);
    acc[11] = fmaf(eps, wG, acc[11]);
}

}  // namespace gs
