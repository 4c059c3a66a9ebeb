// sample_grid_bwd.cu -- structured backward (S7; section 4.1.4, and the warp-per-Gaussian form of
// section 5.1.2 PAPER.md:196 applied to a grid, where the "traversal" is index arithmetic): one warp per
// Gaussian walks the voxels of its AABB, lanes accumulate the 12 partial sums in registers, one
// warp reduction at the end, no atomics.  Weights are recomputed, nothing is stored by the forward.
// Gaussians are processed in the Morton order of their central brick so that the per-sample
// coefficients of neighbouring Gaussians stay in L1/L2.
#include "gs_internal.cuh"
#include "pair_math.cuh"

namespace gs {

// ------------------------------------------------------------------------------------------------
// backward
// ------------------------------------------------------------------------------------------------
// per-sample coefficients (one pass over the batch):  alpha = covered ? a/I : 0,  beta = b - alpha Phi,
// eps = covered ? |Phi - t| / I : 0   (oracle: "per-sample coefficients"; PAPER.md:130 lists the inputs)
__global__ void __launch_bounds__(256) k_pack_samples(const float *__restrict__ phi, const float *__restrict__ I,
                                                       const float *__restrict__ a, const float *__restrict__ b,
                                                       const float *__restrict__ target, size_t P, float tau,
                                                       float4 *__restrict__ pack) {
    const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= P) return;
    const float Ic = I[c], ph = phi[c];
    const bool covered = Ic > tau;
    const float inv = covered ? 1.0f / Ic : 0.f;
    const float alpha = covered ? a[c] * inv : 0.f;
    const float beta = (b ? b[c] : 0.f) - alpha * ph;
    const float eps = (covered && target) ? fabsf(ph - target[c]) * inv : 0.f;
    pack[c] = make_float4(alpha, beta, eps, 0.f);
}

constexpr int BWD_WARPS = 8;

__global__ void __launch_bounds__(BWD_WARPS * 32) k_grid_bwd(const float4 *__restrict__ rec, const float *__restrict__ aabb, uint32_t N,
                                                              GridDesc gd, const float4 *__restrict__ pack, float r2,
                                                              float *__restrict__ gacc, const uint32_t *__restrict__ order,
                                                              uint32_t M) {
    // warp w processes the w-th Gaussian of the brick-ordered list of the M Gaussians that touch the batch
    const uint32_t w = blockIdx.x * BWD_WARPS + (threadIdx.x >> 5);
    if (w >= M) return;
    const uint32_t i = order[w];
    const int lane = threadIdx.x & 31;
    Rec g;
    g.a = rec[i]; g.b = rec[(size_t)N + i]; g.c = rec[2 * (size_t)N + i]; g.d = rec[3 * (size_t)N + i];
    // voxel index box of the AABB inside the batch (conservative; the predicate decides)
    int lo[3], hi[3];
    bool empty = false;
#pragma unroll
    for (int k = 0; k < 3; k++) {
        const float inv_sp = 1.0f / gd.spacing[k];
        const float tl = (aabb[6 * (size_t)i + k] - gd.origin[k]) * inv_sp - 0.5f;
        const float th = (aabb[6 * (size_t)i + 3 + k] - gd.origin[k]) * inv_sp - 0.5f;
        const float first = (float)(BRICK * gd.brick_lo[k]), last = (float)(BRICK * gd.brick_lo[k] + gd.bdim[k] - 1);
        const float fl = fmaxf(ceilf(tl - (1e-3f + 4e-7f * fabsf(tl))), first);
        const float fh = fminf(floorf(th + (1e-3f + 4e-7f * fabsf(th))), last);
        empty |= !(fl <= fh);  // also true for the empty (+inf,-inf) box of an invalid Gaussian
        lo[k] = (int)fl; hi[k] = (int)fh;
    }
    float acc[16];
#pragma unroll
    for (int k = 0; k < 16; k++) acc[k] = 0.f;
    if (!empty) {
        const int nx = hi[0] - lo[0] + 1, ny = hi[1] - lo[1] + 1;
        const int nxy = nx * ny;
        const int step_y = 32 / nx, step_x = 32 - step_y * nx;
        const int x0 = lane % nx, y0 = lane / nx;
        const int ox = BRICK * gd.brick_lo[0], oy = BRICK * gd.brick_lo[1], oz = BRICK * gd.brick_lo[2];
        for (int z = lo[2]; z <= hi[2]; z++) {
            const float pz = voxel_centre(z, gd.spacing[2], gd.origin[2]);
            const size_t zoff = (size_t)(z - oz) * gd.bdim[1];
            int x = x0, y = y0;
            for (int k = lane; k < nxy; k += 32) {
                const int gx = lo[0] + x, gy = lo[1] + y;
                const float px = voxel_centre(gx, gd.spacing[0], gd.origin[0]);
                const float py = voxel_centre(gy, gd.spacing[1], gd.origin[1]);
                float u0, u1, u2;
                const float qd = mahalanobis(g, px, py, pz, u0, u1, u2);
                if (qd <= r2) {
                    const float4 s = __ldg(pack + (zoff + (gy - oy)) * gd.bdim[0] + (gx - ox));
                    bwd_accumulate(acc, s.x, s.y, s.z, g.a.w, g.b.w, gauss_weight(qd), u0, u1, u2);
                }
                x += step_x; y += step_y;
                if (x >= nx) { x -= nx; y++; }
            }
        }
    }
    warp_reduce16(acc, lane);
    // lane 2c holds component c: 16 floats per Gaussian, written as one coalesced 64-byte row
    const float val = __shfl_sync(0xffffffffu, acc[0], (lane & 15) * 2);
    if (lane < 16) gacc[(size_t)i * GACC + lane] = val;
}

cudaError_t launch_pack_samples(const BwdIn &in, size_t P, float tau, float4 *pack, cudaStream_t s) {
    if (P == 0) return cudaSuccess;
    k_pack_samples<<<(unsigned)((P + 255) / 256), 256, 0, s>>>(in.phi, in.I, in.dL_dphi, in.dL_dI, in.target, P, tau, pack); count_launch();
    return cudaGetLastError();
}

cudaError_t launch_grid_bwd(const float4 *rec, const float *aabb, uint32_t N, const GridDesc &gd, const float4 *pack, float r2,
                            float *gacc, const uint32_t *order, uint32_t M, cudaStream_t s) {
    // untouched Gaussians keep a zero accumulator row
    cudaError_t e = cudaMemsetAsync(gacc, 0, (size_t)N * GACC * sizeof(float), s);
    if (e != cudaSuccess || M == 0) return e;
    k_grid_bwd<<<(M + BWD_WARPS - 1) / BWD_WARPS, BWD_WARPS * 32, 0, s>>>(rec, aabb, N, gd, pack, r2, gacc, order, M); count_launch();
    return cudaGetLastError();
}

}  // namespace gs
