// sample_grid_bwd.cu -- structured backward (S7; section 4.1.4, in the warp-per-Gaussian form of
// section 5.1.2 PAPER.md:196 applied to a grid, where the "traversal" is index arithmetic).
//
// One warp per Gaussian, no atomics: the warp enumerates the 2x2x2-voxel CELLS of the Gaussian's
// AABB, culls them with the conservative whitened-space bound (same bound as the forward),
// compacts the surviving cells through a small shared-memory queue so that all 32 lanes stay busy,
// and evaluates 8 voxels per lane with shared canonical sub-expressions.  The weights are
// recomputed (nothing is stored by the forward); each lane keeps the 12 partial sums in registers
// and one transposing-butterfly warp reduction at the end writes the accumulator row.
// Gaussians are processed in the Morton order of their central brick so that the per-sample
// coefficients of neighbouring Gaussians stay in L1/L2.
#include "gs_internal.cuh"
#include "pair_math.cuh"

namespace gs {

// per-sample coefficients (one pass over the batch):  alpha = covered ? a/I : 0,  beta = b - alpha Phi,
// eps = covered ? |Phi - t| / I : 0   (PAPER.md:130 lists the inputs I_c, V_c, dL/dI_c, dL/dV_c)
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

constexpr int BWD_WARPS = 4;
constexpr int GPW = 1;    // Gaussians per warp (consecutive in the order list); 8 measured slower on C2 (0.84 vs 0.73 ms)
constexpr int QCAP = 64;  // per-warp queue of surviving cells (power of two, >= 2 * 32)

__global__ void __launch_bounds__(BWD_WARPS * 32) k_grid_bwd(const float4 *__restrict__ rec, const float *__restrict__ aabb, uint32_t N,
                                                              GridDesc gd, const float4 *__restrict__ pack, float r2,
                                                              float *__restrict__ gacc, const uint32_t *__restrict__ order,
                                                              uint32_t M) {
    __shared__ uint32_t queue[BWD_WARPS][QCAP];
    // warp w processes the w-th Gaussian of the brick-ordered list of the M Gaussians that touch the batch
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // A CTA owns BWD_WARPS * GPW consecutive Gaussians of the order list (one neighbourhood of the grid, so
    // that its per-sample coefficients are shared through this SM's L1); the warps interleave over them.
    for (int rep = 0; rep < GPW; rep++) {
    const uint32_t w = blockIdx.x * (BWD_WARPS * GPW) + rep * BWD_WARPS + warp;
    if (w >= M) return;  // whole warps leave; no block-wide barrier is used below
    const uint32_t i = order[w];
    const float4 ga = __ldg(rec + i), gb = __ldg(rec + (size_t)N + i), gc = __ldg(rec + 2 * (size_t)N + i),
                 gd4 = __ldg(rec + 3 * (size_t)N + i);
    // voxel index box of the AABB inside the batch (conservative; the predicate decides), then its cells
    int clo[3], nc[3], first[3], last[3];
    bool empty = false;
#pragma unroll
    for (int k = 0; k < 3; k++) {
        const float inv_sp = 1.0f / gd.spacing[k];
        const float tl = (aabb[6 * (size_t)i + k] - gd.origin[k]) * inv_sp - 0.5f;
        const float th = (aabb[6 * (size_t)i + 3 + k] - gd.origin[k]) * inv_sp - 0.5f;
        first[k] = BRICK * gd.brick_lo[k];
        last[k] = BRICK * gd.brick_lo[k] + gd.bdim[k] - 1;
        const float fl = fmaxf(ceilf(tl - (1e-3f + 4e-7f * fabsf(tl))), (float)first[k]);
        const float fh = fminf(floorf(th + (1e-3f + 4e-7f * fabsf(th))), (float)last[k]);
        empty |= !(fl <= fh);  // also true for the empty (+inf,-inf) box of an invalid Gaussian
        const int lo = (int)fl, hi = (int)fh;
        clo[k] = lo >> 1;
        nc[k] = (hi >> 1) - clo[k] + 1;
    }
    if (empty) continue;  // the accumulator row stays zero (memset by the launcher)

    // cull bound (not canonical): |M(p - mu)| >= |M(cc - mu)| - rho for every voxel p of a cell with centre cc
    const float hx = 0.5f * gd.spacing[0], hy = 0.5f * gd.spacing[1], hz = 0.5f * gd.spacing[2];
    const float q0 = fabsf(gb.x) * hx + fabsf(gb.y) * hy + fabsf(gb.z) * hz;
    const float q1 = fabsf(gc.x) * hx + fabsf(gc.y) * hy + fabsf(gc.z) * hz;
    const float q2 = fabsf(gd4.x) * hx + fabsf(gd4.y) * hy + fabsf(gd4.z) * hz;
    const float reach = sqrtf(r2) + sqrtf(q0 * q0 + q1 * q1 + q2 * q2);
    const float thr = reach * reach * 1.001953125f;

    float acc[16];
#pragma unroll
    for (int k = 0; k < 16; k++) acc[k] = 0.f;

    // evaluate one cell per lane: (cxi, cyi, czi) = cell coordinates relative to clo
    auto process = [&](uint32_t code, bool on) {
        const int X = 2 * (clo[0] + (int)(code & 1023u)), Y = 2 * (clo[1] + (int)((code >> 10) & 1023u)), Z = 2 * (clo[2] + (int)(code >> 20));
        const float nanv = __int_as_float(0x7fc00000);
        float dx[2], dy[2], dz[2];
        bool okx[2], oky[2], okz[2];
#pragma unroll
        for (int d = 0; d < 2; d++) {  // canonical positions (D6); voxels outside the batch (or an idle lane) become NaN
            okx[d] = on && X + d >= first[0] && X + d <= last[0];
            oky[d] = Y + d >= first[1] && Y + d <= last[1];
            okz[d] = Z + d >= first[2] && Z + d <= last[2];
            dx[d] = __fsub_rn(okx[d] ? voxel_centre(X + d, gd.spacing[0], gd.origin[0]) : nanv, ga.x);
            dy[d] = __fsub_rn(oky[d] ? voxel_centre(Y + d, gd.spacing[1], gd.origin[1]) : nanv, ga.y);
            dz[d] = __fsub_rn(okz[d] ? voxel_centre(Z + d, gd.spacing[2], gd.origin[2]) : nanv, ga.z);
        }
        // canonical sequence (D4) with shared sub-expressions: u_j = fma(M_j2, dz, fma(M_j1, dy, M_j0 * dx))
        float ab[3][4];
#pragma unroll
        for (int row = 0; row < 3; row++) {
            const float4 mr = row == 0 ? gb : row == 1 ? gc : gd4;
            const float a0 = __fmul_rn(mr.x, dx[0]), a1 = __fmul_rn(mr.x, dx[1]);
            ab[row][0] = __fmaf_rn(mr.y, dy[0], a0); ab[row][1] = __fmaf_rn(mr.y, dy[0], a1);
            ab[row][2] = __fmaf_rn(mr.y, dy[1], a0); ab[row][3] = __fmaf_rn(mr.y, dy[1], a1);
        }
        // 32-bit sample index (P < 2^32); wraps for voxels outside the batch, which are never dereferenced
        const uint32_t base = ((uint32_t)(Z - first[2]) * (uint32_t)gd.bdim[1] + (uint32_t)(Y - first[1])) * (uint32_t)gd.bdim[0] + (uint32_t)(X - first[0]);
#pragma unroll
        for (int iz = 0; iz < 2; iz++) {
            // the four coefficient loads of this z-slice are issued up front (no data dependence on the predicate),
            // so their L1/L2 latency overlaps the arithmetic below instead of stalling each hit in turn
            float4 s[4];
#pragma unroll
            for (int v = 0; v < 4; v++) {
                const uint32_t c = base + ((uint32_t)iz * (uint32_t)gd.bdim[1] + (uint32_t)(v >> 1)) * (uint32_t)gd.bdim[0] + (uint32_t)(v & 1);
                s[v] = (okx[v & 1] && oky[v >> 1] && okz[iz]) ? __ldg(pack + c) : make_float4(0.f, 0.f, 0.f, 0.f);
            }
#pragma unroll
            for (int v = 0; v < 4; v++) {
                const float u0 = __fmaf_rn(gb.z, dz[iz], ab[0][v]);
                const float u1 = __fmaf_rn(gc.z, dz[iz], ab[1][v]);
                const float u2 = __fmaf_rn(gd4.z, dz[iz], ab[2][v]);
                const float qd = __fmaf_rn(u2, u2, __fmaf_rn(u1, u1, __fmul_rn(u0, u0)));
                if (qd <= r2) bwd_accumulate(acc, s[v].x, s[v].y, s[v].z, ga.w, gb.w, gauss_weight(qd), u0, u1, u2);
            }
        }
    };

    // enumerate the cells of the AABB, 32 per step; lane-private incremental (x, y, z) decode of the linear index
    const int ncx = nc[0], ncy = nc[1], ncxy = ncx * ncy;
    const int ncells = ncxy * nc[2];
    int z = lane / ncxy, rem = lane - z * ncxy;
    int y = rem / ncx, x = rem - y * ncx;
    const int sz = 32 / ncxy, r32 = 32 - sz * ncxy, sy = r32 / ncx, sx = r32 - sy * ncx;
    uint32_t *q = queue[warp];
    uint32_t head = 0, qn = 0;  // warp-uniform
    for (int basek = 0; basek < ncells; basek += 32) {
        const bool valid = basek + lane < ncells;
        // centre of cell (x, y, z): voxels 2X, 2X+1 -> origin + (2X + 1) spacing
        const float ccx = fmaf((float)(2 * (clo[0] + x) + 1), gd.spacing[0], gd.origin[0]) - ga.x;
        const float ccy = fmaf((float)(2 * (clo[1] + y) + 1), gd.spacing[1], gd.origin[1]) - ga.y;
        const float ccz = fmaf((float)(2 * (clo[2] + z) + 1), gd.spacing[2], gd.origin[2]) - ga.z;
        const float u0 = gb.x * ccx + gb.y * ccy + gb.z * ccz;
        const float u1 = gc.x * ccx + gc.y * ccy + gc.z * ccz;
        const float u2 = gd4.x * ccx + gd4.y * ccy + gd4.z * ccz;
        const bool pass = valid && (u0 * u0 + u1 * u1 + u2 * u2 <= thr);
        const uint32_t bal = __ballot_sync(0xffffffffu, pass);
        if (pass) q[(head + qn + __popc(bal & ((1u << lane) - 1u))) & (QCAP - 1)] = (uint32_t)x | ((uint32_t)y << 10) | ((uint32_t)z << 20);
        qn += __popc(bal);
        __syncwarp();
        if (qn >= 32) {
            process(q[(head + lane) & (QCAP - 1)], true);
            head = (head + 32) & (QCAP - 1);
            qn -= 32;
            __syncwarp();
        }
        x += sx; y += sy; z += sz;
        if (x >= ncx) { x -= ncx; y++; }
        if (y >= ncy) { y -= ncy; z++; }
    }
    if (qn) {
        const bool on = (uint32_t)lane < qn;
        process(on ? q[(head + lane) & (QCAP - 1)] : 0u, on);
    }

    warp_reduce16(acc, lane);
    // lane 2c holds component c: 16 floats per Gaussian, written as one coalesced 64-byte row
    const float val = __shfl_sync(0xffffffffu, acc[0], (lane & 15) * 2);
    if (lane < 16) gacc[(size_t)i * GACC + lane] = val;
    __syncwarp();
    }  // rep
}

cudaError_t launch_pack_samples(const BwdIn &in, size_t P, float tau, float4 *pack, cudaStream_t s) {
    if (P == 0) return cudaSuccess;
    k_pack_samples<<<(unsigned)((P + 255) / 256), 256, 0, s>>>(in.phi, in.I, in.dL_dphi, in.dL_dI, in.target, P, tau, pack);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_grid_bwd(const float4 *rec, const float *aabb, uint32_t N, const GridDesc &gd, const float4 *pack, float r2,
                            float *gacc, const uint32_t *order, uint32_t M, cudaStream_t s) {
    // untouched Gaussians keep a zero accumulator row
    cudaError_t e = cudaMemsetAsync(gacc, 0, (size_t)N * GACC * sizeof(float), s);
    if (e != cudaSuccess || M == 0) return e;
    k_grid_bwd<<<(M + BWD_WARPS * GPW - 1) / (BWD_WARPS * GPW), BWD_WARPS * 32, 0, s>>>(rec, aabb, N, gd, pack, r2, gacc, order, M);
    count_launch();
    return cudaGetLastError();
}

}  // namespace gs
