// preprocess.cu -- S1 (section 4.1.1) and S8 (backward of S1; implied by PAPER.md:140).
//
// S1: one thread per Gaussian.  Everything here feeds integer decisions downstream (brick
// ranges, the hit predicate), so the arithmetic is a fixed sequence of single IEEE operations
// (round-to-nearest intrinsics; the compiler may not contract or reorder them) -- D4/D7.
#include "gs_internal.cuh"

namespace gs {

__device__ __forceinline__ bool finitef(float x) { return fabsf(x) <= 3.402823466e38f; }  // false for NaN/inf

__global__ void __launch_bounds__(256) k_preprocess(const float *__restrict__ mean, const float *__restrict__ scale,
                                                     const float *__restrict__ quat, const float *__restrict__ opacity,
                                                     const float *__restrict__ scalar, uint32_t N, float r,
                                                     float4 *__restrict__ rec, float *__restrict__ aabb,
                                                     float *__restrict__ params, unsigned long long *__restrict__ invalid) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const float mx = mean[3 * i], my = mean[3 * i + 1], mz = mean[3 * i + 2];
    const float s0 = scale[3 * i], s1 = scale[3 * i + 1], s2 = scale[3 * i + 2];
    const float qw = quat[4 * i], qx = quat[4 * i + 1], qy = quat[4 * i + 2], qz = quat[4 * i + 3];
    const float w = opacity[i], v = scalar[i];
    // raw parameters kept for S8 (the caller's arrays are not retained)
    float4 *pp = reinterpret_cast<float4 *>(params) + 2 * (size_t)i;
    pp[0] = make_float4(s0, s1, s2, qw);
    pp[1] = make_float4(qx, qy, qz, 0.f);

    // validity (empty support otherwise): finite parameters, positive scale, non-zero quaternion
    float n2chk = __fmul_rn(qw, qw);
    n2chk = __fadd_rn(n2chk, __fmul_rn(qx, qx));
    n2chk = __fadd_rn(n2chk, __fmul_rn(qy, qy));
    n2chk = __fadd_rn(n2chk, __fmul_rn(qz, qz));
    bool valid = finitef(mx) && finitef(my) && finitef(mz) && (s0 > 0.f) && (s1 > 0.f) && (s2 > 0.f) && finitef(s0) &&
                 finitef(s1) && finitef(s2) && finitef(qw) && finitef(qx) && finitef(qy) && finitef(qz) && (n2chk > 0.f) &&
                 finitef(n2chk) && finitef(w) && finitef(v);
    float4 *r0 = rec + i, *r1 = rec + (size_t)N + i, *r2p = rec + 2 * (size_t)N + i, *r3 = rec + 3 * (size_t)N + i;
    float *bb = aabb + 6 * (size_t)i;
    if (!valid) {
        const float nan = __int_as_float(0x7fc00000);
        const float inf = __int_as_float(0x7f800000);
        *r0 = make_float4(nan, nan, nan, 0.f);  // d = p - NaN makes the predicate false everywhere
        *r1 = make_float4(0.f, 0.f, 0.f, 0.f);
        *r2p = make_float4(0.f, 0.f, 0.f, 0.f);
        *r3 = make_float4(0.f, 0.f, 0.f, 0.f);
        bb[0] = inf; bb[1] = inf; bb[2] = inf; bb[3] = -inf; bb[4] = -inf; bb[5] = -inf;
        atomicAdd(invalid, 1ull);  // surfaced by gs_status_query (D13)
        return;
    }
    // normalisation activation of the rotation
    const float n2 = __fmaf_rn(qz, qz, __fmaf_rn(qy, qy, __fmaf_rn(qx, qx, __fmul_rn(qw, qw))));
    const float nrm = __fsqrt_rn(n2);
    const float a = __fdiv_rn(qw, nrm), x = __fdiv_rn(qx, nrm), y = __fdiv_rn(qy, nrm), z = __fdiv_rn(qz, nrm);
    const float xx = __fmul_rn(x, x), yy = __fmul_rn(y, y), zz = __fmul_rn(z, z);
    const float xy = __fmul_rn(x, y), xz = __fmul_rn(x, z), yz = __fmul_rn(y, z);
    const float ax = __fmul_rn(a, x), ay = __fmul_rn(a, y), az = __fmul_rn(a, z);
    float R[9];
    R[0] = __fsub_rn(1.f, __fmul_rn(2.f, __fadd_rn(yy, zz)));
    R[1] = __fmul_rn(2.f, __fsub_rn(xy, az));
    R[2] = __fmul_rn(2.f, __fadd_rn(xz, ay));
    R[3] = __fmul_rn(2.f, __fadd_rn(xy, az));
    R[4] = __fsub_rn(1.f, __fmul_rn(2.f, __fadd_rn(xx, zz)));
    R[5] = __fmul_rn(2.f, __fsub_rn(yz, ax));
    R[6] = __fmul_rn(2.f, __fsub_rn(xz, ay));
    R[7] = __fmul_rn(2.f, __fadd_rn(yz, ax));
    R[8] = __fsub_rn(1.f, __fmul_rn(2.f, __fadd_rn(xx, yy)));
    const float s[3] = {s0, s1, s2};
    float M[9];
#pragma unroll
    for (int j = 0; j < 3; j++)
#pragma unroll
        for (int k = 0; k < 3; k++) M[3 * j + k] = __fdiv_rn(R[3 * j + k], s[j]);  // M = S^-1 R;  M^T M = R^T S^-2 R (Eq. 3)
    *r0 = make_float4(mx, my, mz, w);
    *r1 = make_float4(M[0], M[1], M[2], v);
    *r2p = make_float4(M[3], M[4], M[5], 0.f);
    *r3 = make_float4(M[6], M[7], M[8], v * w);  // v w: the forward accumulates Nacc += (v w) G with one FMA
    // AABB of the cutoff ellipsoid: half extent along world axis k = r sqrt(sum_j (s_j R_jk)^2), inflated by 1 + 2^-8
    const float mu[3] = {mx, my, mz};
#pragma unroll
    for (int k = 0; k < 3; k++) {
        const float a0 = __fmul_rn(s0, R[k]), a1 = __fmul_rn(s1, R[3 + k]), a2 = __fmul_rn(s2, R[6 + k]);
        const float e = __fmul_rn(r, __fsqrt_rn(__fmaf_rn(a2, a2, __fmaf_rn(a1, a1, __fmul_rn(a0, a0)))));
        const float ei = __fmul_rn(e, 1.00390625f);
        bb[k] = __fsub_rn(mu[k], ei);
        bb[3 + k] = __fadd_rn(mu[k], ei);
    }
}

cudaError_t launch_preprocess(const gs_gaussians &g, float r, float4 *rec, float *aabb, float *params, unsigned long long *invalid,
                              cudaStream_t s) {
    cudaError_t e = cudaMemsetAsync(invalid, 0, sizeof(unsigned long long), s);
    if (e != cudaSuccess || g.n == 0) return e;
    k_preprocess<<<(g.n + 255) / 256, 256, 0, s>>>(g.mean, g.scale, g.quat, g.opacity, g.scalar, g.n, r, rec, aabb, params, invalid); count_launch();
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// S8: from the accumulated (dv, dw, U, W, E) of S7 to gradients of the raw parameters.
//   dmu = M^T U;  ds_j = W_jj / s_j;  dR_jk = -(1/s_j) sum_l W_jl s_l R_lk;
//   dqhat = <dR, dR/dqhat>;  dq = (dqhat - qhat (qhat . dqhat)) / |q|        (chain rule of Eq. 3)
// Values only (no integer decision depends on them), so plain fp32 with FMA contraction.
// ------------------------------------------------------------------------------------------------
// MOMENTS: gacc holds the structured backward's rows of moment sums (layout in sample_grid_bwd.cu) with the
// weight w factored out.  With E_a = column a of M:
//   U = A + sum_a s1_a E_a;   W = Q + sum_a (E_a B_a^T + B_a E_a^T) + sum_{a<=b} s2_ab (E_a E_b^T + E_b E_a^T) / (1 + [a = b])
template <bool MOMENTS>
__device__ __forceinline__ void finalize_one(uint32_t i, const float4 *__restrict__ rec, const float *__restrict__ params,
                                             const float *__restrict__ gacc, uint32_t N, float eps_scale, const gs_grads &out,
                                             const uint32_t *__restrict__ touched) {
    if (touched && touched[i] == 0u) {
#pragma unroll
        for (int k = 0; k < 3; k++) { out.dmean[3 * (size_t)i + k] = 0.f; out.dscale[3 * (size_t)i + k] = 0.f; }
        reinterpret_cast<float4 *>(out.dquat)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        out.dopacity[i] = 0.f;
        out.dscalar[i] = 0.f;
        if (out.err) out.err[i] = 0.f;
        return;
    }
    float dv, dw, E, U[3], W00, W01, W02, W11, W12, W22;
    if (MOMENTS) {
        const float4 *ga = reinterpret_cast<const float4 *>(gacc) + (GACC_GRID / 4) * (size_t)i;
        float m[32];
#pragma unroll
        for (int k = 0; k < 8; k++) {
            const float4 t = ga[k];
            m[4 * k] = t.x; m[4 * k + 1] = t.y; m[4 * k + 2] = t.z; m[4 * k + 3] = t.w;
        }
        const float4 r0 = rec[i], r1 = rec[(size_t)N + i], r2 = rec[2 * (size_t)N + i], r3 = rec[3 * (size_t)N + i];
        const float w = r0.w;
        const float Ec[3][3] = {{r1.x, r2.x, r3.x}, {r1.y, r2.y, r3.y}, {r1.z, r2.z, r3.z}};  // Ec[a] = column a of M
        float Wm[3][3];
#pragma unroll
        for (int j = 0; j < 3; j++) {
            U[j] = m[3 + j] + m[6] * Ec[0][j] + m[7] * Ec[1][j] + m[8] * Ec[2][j];
#pragma unroll
            for (int k = j; k < 3; k++) {
                const int q = j == 0 ? k : (j == 1 ? 2 + k : 5);  // 00 01 02 11 12 22
                float t = m[9 + q];
#pragma unroll
                for (int a = 0; a < 3; a++) t += Ec[a][j] * m[15 + 3 * a + k] + m[15 + 3 * a + j] * Ec[a][k];
                t += m[24] * Ec[0][j] * Ec[0][k] + m[25] * Ec[1][j] * Ec[1][k] + m[26] * Ec[2][j] * Ec[2][k];
                t += m[27] * (Ec[0][j] * Ec[1][k] + Ec[1][j] * Ec[0][k]) + m[28] * (Ec[0][j] * Ec[2][k] + Ec[2][j] * Ec[0][k]) +
                     m[29] * (Ec[1][j] * Ec[2][k] + Ec[2][j] * Ec[1][k]);
                Wm[j][k] = t * w;
            }
            U[j] *= w;
        }
        dv = m[0] * w; dw = m[1]; E = m[2] * w * eps_scale;
        W00 = Wm[0][0]; W01 = Wm[0][1]; W02 = Wm[0][2]; W11 = Wm[1][1]; W12 = Wm[1][2]; W22 = Wm[2][2];
    } else {
        const float4 *ga = reinterpret_cast<const float4 *>(gacc) + 4 * (size_t)i;
        const float4 g0 = ga[0], g1 = ga[1], g2 = ga[2];
        dv = g0.x; dw = g0.y;
        U[0] = g0.z; U[1] = g0.w; U[2] = g1.x;
        W00 = g1.y; W01 = g1.z; W02 = g1.w; W11 = g2.x; W12 = g2.y; W22 = g2.z; E = g2.w;
    }
    const float4 p0 = reinterpret_cast<const float4 *>(params)[2 * (size_t)i];
    const float4 p1 = reinterpret_cast<const float4 *>(params)[2 * (size_t)i + 1];
    const float4 c0 = rec[i];
    const bool valid = (c0.x == c0.x);  // invalid Gaussians carry a NaN mean
    float dmu[3] = {0, 0, 0}, ds[3] = {0, 0, 0}, dq[4] = {0, 0, 0, 0};
    if (valid) {
        const float s[3] = {p0.x, p0.y, p0.z};
        float q[4] = {p0.w, p1.x, p1.y, p1.z};
        const float nrm = sqrtf(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
        const float inv = 1.f / nrm;
        const float a = q[0] * inv, x = q[1] * inv, y = q[2] * inv, z = q[3] * inv;
        float R[9];
        R[0] = 1.f - 2.f * (y * y + z * z); R[1] = 2.f * (x * y - a * z);       R[2] = 2.f * (x * z + a * y);
        R[3] = 2.f * (x * y + a * z);       R[4] = 1.f - 2.f * (x * x + z * z); R[5] = 2.f * (y * z - a * x);
        R[6] = 2.f * (x * z - a * y);       R[7] = 2.f * (y * z + a * x);       R[8] = 1.f - 2.f * (x * x + y * y);
        const float W[9] = {W00, W01, W02, W01, W11, W12, W02, W12, W22};
#pragma unroll
        for (int k = 0; k < 3; k++) dmu[k] = R[k] / s[0] * U[0] + R[3 + k] / s[1] * U[1] + R[6 + k] / s[2] * U[2];
        ds[0] = W00 / s[0]; ds[1] = W11 / s[1]; ds[2] = W22 / s[2];
        float D[9];
#pragma unroll
        for (int j = 0; j < 3; j++)
#pragma unroll
            for (int k = 0; k < 3; k++) {
                float acc = 0.f;
#pragma unroll
                for (int l = 0; l < 3; l++) acc += W[3 * j + l] * s[l] * R[3 * l + k];
                D[3 * j + k] = -acc / s[j];
            }
        float dh[4];
        dh[0] = 2.f * (-z * D[1] + y * D[2] + z * D[3] - x * D[5] - y * D[6] + x * D[7]);
        dh[1] = 2.f * (y * D[1] + z * D[2] + y * D[3] - 2.f * x * D[4] - a * D[5] + z * D[6] + a * D[7] - 2.f * x * D[8]);
        dh[2] = 2.f * (-2.f * y * D[0] + x * D[1] + a * D[2] + x * D[3] + z * D[5] - a * D[6] + z * D[7] - 2.f * y * D[8]);
        dh[3] = 2.f * (-2.f * z * D[0] - a * D[1] + x * D[2] + a * D[3] - 2.f * z * D[4] + y * D[5] + x * D[6] + y * D[7]);
        const float qh[4] = {a, x, y, z};
        const float dot = qh[0] * dh[0] + qh[1] * dh[1] + qh[2] * dh[2] + qh[3] * dh[3];
#pragma unroll
        for (int k = 0; k < 4; k++) dq[k] = (dh[k] - qh[k] * dot) * inv;
    }
#pragma unroll
    for (int k = 0; k < 3; k++) { out.dmean[3 * (size_t)i + k] = dmu[k]; out.dscale[3 * (size_t)i + k] = ds[k]; }
    reinterpret_cast<float4 *>(out.dquat)[i] = make_float4(dq[0], dq[1], dq[2], dq[3]);
    out.dopacity[i] = valid ? dw : 0.f;
    out.dscalar[i] = valid ? dv : 0.f;
    if (out.err) out.err[i] = valid ? E : 0.f;
}

// zero gradients for Gaussian i: an untouched Gaussian, or every Gaussian of a batch whose asynchronous build overflowed
// (its backward did nothing; stale rows of an earlier step must not reach the optimiser)
__device__ __forceinline__ void zero_row(uint32_t i, const gs_grads &out) {
#pragma unroll
    for (int k = 0; k < 3; k++) { out.dmean[3 * (size_t)i + k] = 0.f; out.dscale[3 * (size_t)i + k] = 0.f; }
    reinterpret_cast<float4 *>(out.dquat)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    out.dopacity[i] = 0.f;
    out.dscalar[i] = 0.f;
    if (out.err) out.err[i] = 0.f;
}

template <bool MOMENTS>
__global__ void __launch_bounds__(256) k_finalize(const float4 *__restrict__ rec, const float *__restrict__ params,
                                                   const float *__restrict__ gacc, uint32_t N, float eps_scale, gs_grads out,
                                                   const uint32_t *__restrict__ touched, DevCount dc) {
    // touched != NULL (structured): touched[i] = bricks of the batch Gaussian i overlaps; only those with a non-zero count have
    // an accumulator row, the others get zero gradients right here (no memset pass, no order list)
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    if (dc.total && dc.total[0] > (unsigned long long)dc.cap) { zero_row(i, out); return; }   // asynchronous build whose pair list overflowed
    finalize_one<MOMENTS>(i, rec, params, gacc, N, eps_scale, out, touched);
}

// Structured batches that touch a small part of a large model (configs[3]: 0.3 % of 4.2 M Gaussians): a warp owns 128
// consecutive Gaussians; it reads their touch counts with one 16-byte load per lane and, when none is touched (nearly always),
// zeroes its 128 rows of every gradient tensor with 16-byte stores (13 per lane) -- a write stream instead of ten strided
// 4-byte stores per Gaussian; a warp with a touched Gaussian falls back to the per-Gaussian code.  Needs 16-byte aligned tensors.
template <bool MOMENTS>
__global__ void __launch_bounds__(256) k_finalize_sparse(const float4 *__restrict__ rec, const float *__restrict__ params,
                                                          const float *__restrict__ gacc, uint32_t N, float eps_scale, gs_grads out,
                                                          const uint32_t *__restrict__ touched, DevCount dc) {
    const bool overflowed = dc.total && dc.total[0] > (unsigned long long)dc.cap;   // asynchronous build whose pair list did not fit: all zero
    const int lane = threadIdx.x & 31;
    const uint32_t nwarps = gridDim.x * (blockDim.x >> 5);
    const uint32_t ngroups = (N + 127u) / 128u;
    for (uint32_t grp = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); grp < ngroups; grp += nwarps) {
        const uint32_t i0 = grp * 128u;
        const bool full = i0 + 128u <= N;
        bool any = true;
        if (full) {
            const uint4 t = __ldg(reinterpret_cast<const uint4 *>(touched + i0) + lane);
            any = !overflowed && (t.x | t.y | t.z | t.w) != 0u;
        }
        if (!__any_sync(0xffffffffu, any)) {
            const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
            float4 *dm = reinterpret_cast<float4 *>(out.dmean + 3 * (size_t)i0), *ds = reinterpret_cast<float4 *>(out.dscale + 3 * (size_t)i0);
            float4 *dq = reinterpret_cast<float4 *>(out.dquat) + i0;
#pragma unroll
            for (int k = 0; k < 3; k++) { dm[32 * k + lane] = z; ds[32 * k + lane] = z; }
#pragma unroll
            for (int k = 0; k < 4; k++) dq[32 * k + lane] = z;
            reinterpret_cast<float4 *>(out.dopacity + i0)[lane] = z;
            reinterpret_cast<float4 *>(out.dscalar + i0)[lane] = z;
            if (out.err) reinterpret_cast<float4 *>(out.err + i0)[lane] = z;
        } else {
#pragma unroll 1
            for (int k = 0; k < 4; k++) {
                const uint32_t i = i0 + 32u * k + lane;
                if (i < N) {
                    if (overflowed) zero_row(i, out);
                    else finalize_one<MOMENTS>(i, rec, params, gacc, N, eps_scale, out, touched);
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// second pass of gs_sample_fwd_loss (loss.cuh): the forward wrote dL/dI = -lambda_fn on D- and +lambda_fp on U+;
// Eq. 4 / Eq. 5 divide by |D-| and |U+|, which are complete only now.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_loss_finish(GenLoss L, size_t P, double nd, double *__restrict__ loss_terms) {
    const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const unsigned long long nfn = L.counts[0], nfp = L.counts[1];
    if (c == 0 && loss_terms) {
        loss_terms[0] = nd > 0.0 ? L.sums[0] / nd : 0.0;
        loss_terms[1] = nfn ? (double)L.lam_fn * L.sums[1] / (double)nfn : 0.0;
        loss_terms[2] = nfp ? (double)L.lam_fp * L.sums[2] / (double)nfp : 0.0;
    }
    if (c >= P) return;
    if (L.dL_dI) {
        const float b = L.dL_dI[c];
        if (b < 0.f) L.dL_dI[c] = b / (float)nfn;
        else if (b > 0.f) L.dL_dI[c] = b / (float)nfp;
    }
    if (L.pack4) {  // beta = b - alpha Phi with the normalised b
        const float b = L.pack4[c].w;
        if (b != 0.f) L.pack4[c].y += b / (float)(b < 0.f ? nfn : nfp);
    }
}

cudaError_t launch_loss_finish(const GenLoss &L, size_t P, double nd, double *loss_terms, cudaStream_t s) {
    const bool per_sample = (L.dL_dI || L.pack4) && (L.lam_fn > 0.f || L.lam_fp > 0.f);
    const size_t n = per_sample && P ? P : 1;
    k_loss_finish<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(L, per_sample ? P : 0, nd, loss_terms); count_launch();
    return cudaGetLastError();
}

cudaError_t launch_finalize(const float4 *rec, const float *params, const float *gacc, uint32_t N, bool grid_moments,
                            float eps_scale, const gs_grads &out, const uint32_t *touched, DevCount dc, uint32_t touched_bound, cudaStream_t s) {
    if (N == 0) return cudaSuccess;
    // A 128^3 batch of configs[3] touches 0.3 % of the 4.2 M Gaussians: only those read their 128-byte row.
    // sparse variant: a structured batch with a touch-count array over a large model; it needs 16-byte aligned tensors (the rows
    // of 128 Gaussians then start at multiples of 512 / 1536 bytes of the bases) and the counts 16-byte aligned
    const bool aligned = !(((uintptr_t)out.dmean | (uintptr_t)out.dscale | (uintptr_t)out.dquat | (uintptr_t)out.dopacity | (uintptr_t)out.dscalar |
                            (uintptr_t)out.err | (uintptr_t)touched) & 15);
    if (grid_moments && touched && aligned && N >= (1u << 16) && (uint64_t)touched_bound * 16 <= N) {
        const unsigned blocks = 148 * 8;   // 8 CTAs of 8 warps per SM, each warp striding over groups of 128 Gaussians
        k_finalize_sparse<true><<<blocks, 256, 0, s>>>(rec, params, gacc, N, eps_scale, out, touched, dc);
    } else if (grid_moments) k_finalize<true><<<(N + 255) / 256, 256, 0, s>>>(rec, params, gacc, N, eps_scale, out, touched, dc);
    else k_finalize<false><<<(N + 255) / 256, 256, 0, s>>>(rec, params, gacc, N, 1.f, out, nullptr, DevCount{nullptr, 0});
    count_launch();
    return cudaGetLastError();
}

}  // namespace gs
