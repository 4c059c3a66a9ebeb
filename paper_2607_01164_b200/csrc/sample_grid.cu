// sample_grid.cu -- structured sampling kernels.
//   S4 forward (section 4.1.3): one CTA per 8^3 brick, one thread per voxel; the brick's
//     Gaussian list is staged into shared memory in cp.async-fed chunks (double buffered);
//     each voxel accumulates I_c and sum v w G over the Gaussians whose support contains it,
//     then the fused epilogue S6 (normalise, coverage rule, MSE, dL/dPhi, per-sample error).
//   S7 backward (section 4.1.4; the warp-per-Gaussian form of section 5.1.2 PAPER.md:196 applied
//     to a grid, where the "traversal" is index arithmetic): one warp per Gaussian walks the voxels
//     of its AABB, lanes accumulate the 12 partial sums in registers, one warp reduction at the
//     end, no atomics.  Weights are recomputed, nothing is stored by the forward.
#include "gs_internal.cuh"
#include "pair_math.cuh"

namespace gs {

constexpr int FWD_THREADS = 512;
constexpr int CH = 64;   // Gaussians per staged chunk = 2 sub-chunks of 32 (one lane per Gaussian in the cell test)

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N)); }

struct FwdSmem {
    float4 rec[2][4][CH];
    uint32_t id[2][CH];
    double red[FWD_THREADS / 32];
};

__device__ __forceinline__ void stage_chunk(FwdSmem &sm, int buf, const float4 *__restrict__ rec, uint32_t N,
                                            const uint32_t *__restrict__ list, uint32_t n, uint32_t chunk) {
    const int plane = threadIdx.x >> 6, j = threadIdx.x & (CH - 1);
    const uint32_t idx = chunk * CH + j;
    if (plane < 4 && idx < n) {
        const uint32_t id = list[idx];
        cp_async16(&sm.rec[buf][plane][j], rec + (size_t)plane * N + id);
        if (plane == 0) sm.id[buf][j] = id;
    }
    cp_async_commit();
}

template <bool SETS>
__global__ void __launch_bounds__(FWD_THREADS) k_grid_fwd(const float4 *__restrict__ rec, uint32_t N, GridDesc gd,
                                                           const uint32_t *__restrict__ pair_gauss,
                                                           const uint32_t *__restrict__ brick_start, float tau, float r2, FwdOut o,
                                                           double invP) {
    __shared__ FwdSmem sm;
    const uint32_t b = blockIdx.x;
    const uint32_t bx = b % gd.brick_cnt[0], by = (b / gd.brick_cnt[0]) % gd.brick_cnt[1], bz = b / (gd.brick_cnt[0] * gd.brick_cnt[1]);
    const int t = threadIdx.x;
    // A warp owns a row of four 2x2x2-voxel CELLS (8 x 2 x 2 voxels); lanes 8g..8g+7 are cell g.
    const int warp = t >> 5, lane = t & 31, cell = lane >> 3;
    const int vx = 2 * cell + (lane & 1), vy = 2 * (warp & 3) + ((lane >> 1) & 1), vz = 2 * (warp >> 2) + ((lane >> 2) & 1);
    const int lx = bx * BRICK + vx, ly = by * BRICK + vy, lz = bz * BRICK + vz;  // batch-local voxel
    const bool active = lx < gd.bdim[0] && ly < gd.bdim[1] && lz < gd.bdim[2];
    const float nanv = __int_as_float(0x7fc00000);
    // inactive threads (voxels clipped by the grid) carry a NaN position: the predicate is false for them
    const float px = active ? voxel_centre(lx + BRICK * gd.brick_lo[0], gd.spacing[0], gd.origin[0]) : nanv;
    const float py = voxel_centre(ly + BRICK * gd.brick_lo[1], gd.spacing[1], gd.origin[1]);
    const float pz = voxel_centre(lz + BRICK * gd.brick_lo[2], gd.spacing[2], gd.origin[2]);

    const uint32_t start = brick_start[b], n = brick_start[b + 1] - start;
    const uint32_t *list = pair_gauss + start;
    const uint32_t nchunks = (n + CH - 1) / CH;
    float I = 0.f, Nacc = 0.f;
    uint32_t cnt = 0, ntest = 0;
    unsigned long long hsum = 0, hxor = 0;
    // cell geometry of this warp (cull only: not canonical): centre of cell 0, x step = 2 voxels
    const float hx = 0.5f * gd.spacing[0], hy = 0.5f * gd.spacing[1], hz = 0.5f * gd.spacing[2];
    const float ccx0 = fmaf((float)(BRICK * (bx + gd.brick_lo[0]) + 1), gd.spacing[0], gd.origin[0]);
    const float ccy = fmaf((float)(BRICK * (by + gd.brick_lo[1]) + 2 * (warp & 3) + 1), gd.spacing[1], gd.origin[1]);
    const float ccz = fmaf((float)(BRICK * (bz + gd.brick_lo[2]) + 2 * (warp >> 2) + 1), gd.spacing[2], gd.origin[2]);
    const float rcut = sqrtf(r2);

    if (nchunks) stage_chunk(sm, 0, rec, N, list, n, 0);
    for (uint32_t c = 0; c < nchunks; c++) {
        const int buf = c & 1;
        if (c + 1 < nchunks) {
            stage_chunk(sm, buf ^ 1, rec, N, list, n, c + 1);
            cp_async_wait<1>();
        } else {
            cp_async_wait<0>();
        }
        __syncthreads();
        const int m = min((uint32_t)CH, n - c * CH);
        for (int sub = 0; sub < m; sub += 32) {
            // ---- cull below the brick: lane = Gaussian, tested against the warp's four cells.
            // For a cell with centre cc and half extent h (its voxel centres are cc +- h), every voxel p has
            // |M(p - mu)| >= |M(cc - mu)| - rho,  rho = |(sum_k |M_jk| h_k)_j|  =>  no hit unless |M(cc - mu)|^2 <= (r + rho)^2.
            // Conservative (1 + 2^-9 slack covers fp32 rounding); the canonical predicate still decides every pair.
            uint32_t mymask;
            {
                const int j = sub + lane;
                const bool have = j < m;
                Rec g;
                g.a = sm.rec[buf][0][j & (CH - 1)]; g.b = sm.rec[buf][1][j & (CH - 1)];
                g.c = sm.rec[buf][2][j & (CH - 1)]; g.d = sm.rec[buf][3][j & (CH - 1)];
                const float r0 = fabsf(g.b.x) * hx + fabsf(g.b.y) * hy + fabsf(g.b.z) * hz;
                const float r1 = fabsf(g.c.x) * hx + fabsf(g.c.y) * hy + fabsf(g.c.z) * hz;
                const float r2c = fabsf(g.d.x) * hx + fabsf(g.d.y) * hy + fabsf(g.d.z) * hz;
                const float reach = rcut + sqrtf(r0 * r0 + r1 * r1 + r2c * r2c);
                const float thr = reach * reach * 1.001953125f;
                const float dy = ccy - g.a.y, dz = ccz - g.a.z;
                const float e0 = g.b.y * dy + g.b.z * dz, e1 = g.c.y * dy + g.c.z * dz, e2 = g.d.y * dy + g.d.z * dz;
                uint32_t masks[4];
#pragma unroll
                for (int k = 0; k < 4; k++) {
                    const float dx = (ccx0 + (float)(2 * k) * gd.spacing[0]) - g.a.x;
                    const float u0 = fmaf(g.b.x, dx, e0), u1 = fmaf(g.c.x, dx, e1), u2 = fmaf(g.d.x, dx, e2);
                    const float qc = u0 * u0 + u1 * u1 + u2 * u2;
                    masks[k] = __ballot_sync(0xffffffffu, have && qc <= thr);
                }
                mymask = cell == 0 ? masks[0] : cell == 1 ? masks[1] : cell == 2 ? masks[2] : masks[3];
            }
            // ---- each cell (8 lanes) walks its own list; the warp iterates until all four are done
            while (__any_sync(0xffffffffu, mymask != 0u)) {
                if (mymask) {
                    const int j = sub + __ffs(mymask) - 1;
                    mymask &= mymask - 1;
                    Rec g;
                    g.a = sm.rec[buf][0][j]; g.b = sm.rec[buf][1][j]; g.c = sm.rec[buf][2][j]; g.d = sm.rec[buf][3][j];
                    float u0, u1, u2;
                    const float qd = mahalanobis(g, px, py, pz, u0, u1, u2);
                    if (SETS) ntest++;
                    if (qd <= r2) {
                        const float wG = g.a.w * gauss_weight(qd);
                        I += wG;
                        Nacc = fmaf(g.b.w, wG, Nacc);
                        if (SETS) {
                            const unsigned long long h = mix64(sm.id[buf][j]);
                            cnt++; hsum += h; hxor ^= h;
                        }
                    }
                }
            }
        }
        __syncthreads();
    }

    // ---- S6 epilogue: coverage rule I > tau (strict), empty value 0, I always written (D5)
    const bool covered = I > tau;
    const float phi = covered ? __fdividef(Nacc, I) : 0.f;
    float res2 = 0.f;
    if (active) {
        const size_t c = ((size_t)lz * gd.bdim[1] + ly) * gd.bdim[0] + lx;
        o.phi[c] = phi;
        o.I[c] = I;
        if (o.target) {
            const float res = phi - o.target[c];
            res2 = res * res;
            if (o.dL_dphi) o.dL_dphi[c] = covered ? (float)(2.0 * invP) * res : 0.f;
            if (o.sample_err) o.sample_err[c] = fabsf(res);
        }
        if (SETS) {
            if (o.set_count) o.set_count[c] = cnt;
            if (o.set_sum) o.set_sum[c] = hsum;
            if (o.set_xor) o.set_xor[c] = hxor;
        }
    }
    if (o.target && o.loss) {
        double s = (double)res2;
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
        if ((t & 31) == 0) sm.red[t >> 5] = s;
        __syncthreads();
        if (t < 32) {
            double v = t < FWD_THREADS / 32 ? sm.red[t] : 0.0;
#pragma unroll
            for (int d = 8; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
            if (t == 0 && v != 0.0) atomicAdd(o.loss, v * invP);
        }
    }
    if (SETS && o.counters) {
        unsigned long long tested = active ? ntest : 0, hits = cnt;
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            tested += __shfl_xor_sync(0xffffffffu, tested, d);
            hits += __shfl_xor_sync(0xffffffffu, hits, d);
        }
        if ((t & 31) == 0) { atomicAdd(o.counters, tested); atomicAdd(o.counters + 1, hits); }
    }
}

cudaError_t launch_grid_fwd(const float4 *rec, uint32_t N, const GridDesc &gd, const uint32_t *pair_gauss,
                            const uint32_t *brick_start, float tau, float r2, const FwdOut &o, cudaStream_t s) {
    const uint32_t nbricks = (uint32_t)gd.brick_cnt[0] * gd.brick_cnt[1] * gd.brick_cnt[2];
    if (nbricks == 0) return cudaSuccess;
    const double P = (double)gd.bdim[0] * gd.bdim[1] * gd.bdim[2];
    const bool sets = o.set_count || o.set_sum || o.set_xor || o.counters;
    if (sets) k_grid_fwd<true><<<nbricks, FWD_THREADS, 0, s>>>(rec, N, gd, pair_gauss, brick_start, tau, r2, o, 1.0 / P);
    else k_grid_fwd<false><<<nbricks, FWD_THREADS, 0, s>>>(rec, N, gd, pair_gauss, brick_start, tau, r2, o, 1.0 / P);
    count_launch();
    return cudaGetLastError();
}

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
