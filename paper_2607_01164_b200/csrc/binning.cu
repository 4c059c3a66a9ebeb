// binning.cu -- S2: Gaussian -> brick lists for a structured batch (section 4.1.2).
//   k_brick_count : per Gaussian, brick range of its AABB inside the batch and the count n_i
//   (scan)        : offsets = exclusive scan of n_i, T = total
//   k_pair_write  : one thread per PAIR: binary search in the scan for the Gaussian, index
//                   arithmetic for the brick ("parallelizes over total intersections")
//   (radix sort)  : stable sort by brick id => each brick's list is in ascending Gaussian id
//   k_brick_start : start index of every brick's run
// Brick ranges are integer decisions: fixed fp32 sequence (D7).
#include "gs_internal.cuh"

namespace gs {

struct BrickRange { int lo[3], hi[3]; };

// D7: b = floorf((aabb - origin) * inv_brick), clamped in float to [-1, nb], then to the batch
__device__ __forceinline__ uint32_t brick_range(const float *__restrict__ bb, const GridDesc &gd, BrickRange &br) {
    uint32_t cnt = 1;
#pragma unroll
    for (int k = 0; k < 3; k++) {
        const float nb = (float)gd.nb_total[k];
        float fl = floorf(__fmul_rn(__fsub_rn(bb[k], gd.origin[k]), gd.inv_brick[k]));
        float fh = floorf(__fmul_rn(__fsub_rn(bb[3 + k], gd.origin[k]), gd.inv_brick[k]));
        fl = fminf(fmaxf(fl, -1.0f), nb);
        fh = fminf(fmaxf(fh, -1.0f), nb);
        int lo = (int)fl, hi = (int)fh;
        const int first = gd.brick_lo[k], last = gd.brick_lo[k] + gd.brick_cnt[k] - 1;
        lo = max(lo, first);
        hi = min(hi, last);
        br.lo[k] = lo;
        br.hi[k] = hi;
        cnt *= (hi >= lo) ? (uint32_t)(hi - lo + 1) : 0u;
    }
    return cnt;
}

__device__ __forceinline__ uint32_t spread3(uint32_t v) {  // 10 bits -> every third bit
    v &= 0x3ffu;
    v = (v | (v << 16)) & 0x030000FFu;
    v = (v | (v << 8)) & 0x0300F00Fu;
    v = (v | (v << 4)) & 0x030C30C3u;
    v = (v | (v << 2)) & 0x09249249u;
    return v;
}

// Also emits the processing order key of the backward pass: Morton code of the Gaussian's central
// brick (performance only: neighbouring Gaussians are processed together so their voxel data stays
// in L1/L2); Gaussians that touch no brick of the batch get `untouched_key` and sort to the end.
//
// And the per-Gaussian constants of the backward kernel (performance only, nothing canonical): the box of
// 2x2x2-voxel cells that covers the AABB inside the batch, the whitened-space cull threshold of a cell and
// 1 / |e|^2 for the closed-form row intervals (sample_grid_bwd.cu):
//   setup[2 i]     = (clo.x, clo.y, clo.z, flags: 1 = touches no voxel of the batch, 2 = a cell sticks out of the batch)
//   setup[2 i + 1] = (ncx | ncy << 11 | ncz << 22, thr, invA, -)
__global__ void __launch_bounds__(256) k_brick_count(const float *__restrict__ aabb, const float4 *__restrict__ rec, uint32_t N,
                                                      GridDesc gd, float rcut, uint32_t *__restrict__ count,
                                                      unsigned long long *__restrict__ total, uint32_t *__restrict__ okey,
                                                      uint32_t *__restrict__ oval, uint32_t untouched_key,
                                                      float4 *__restrict__ setup) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t c = 0;
    if (i < N) {
        const float *bb = aabb + 6 * (size_t)i;
        // an invalid Gaussian has the empty box (+inf, -inf): fmaxf/fminf clamp it to an empty range.
        // NaN cannot occur here (preprocess writes inf for invalid ones).
        float b6[6];
#pragma unroll
        for (int k = 0; k < 6; k++) b6[k] = bb[k];
        BrickRange br;
        c = brick_range(b6, gd, br);
        count[i] = c;
        uint32_t key = untouched_key;
        if (c) {
            const uint32_t mx = (uint32_t)(((br.lo[0] + br.hi[0]) >> 1) - gd.brick_lo[0]);
            const uint32_t my = (uint32_t)(((br.lo[1] + br.hi[1]) >> 1) - gd.brick_lo[1]);
            const uint32_t mz = (uint32_t)(((br.lo[2] + br.hi[2]) >> 1) - gd.brick_lo[2]);
            key = spread3(mx) | (spread3(my) << 1) | (spread3(mz) << 2);
        }
        okey[i] = key;
        oval[i] = i;
        // ---- backward setup
        int clo[3], nc[3];
        bool empty = false, edge = false;
#pragma unroll
        for (int k = 0; k < 3; k++) {
            const float inv_sp = 1.0f / gd.spacing[k];
            const float tl = (b6[k] - gd.origin[k]) * inv_sp - 0.5f;
            const float th = (b6[3 + k] - gd.origin[k]) * inv_sp - 0.5f;
            const int first = BRICK * gd.brick_lo[k], last = BRICK * gd.brick_lo[k] + gd.bdim[k] - 1;
            const float fl = fmaxf(ceilf(tl - (1e-3f + 4e-7f * fabsf(tl))), (float)first);
            const float fh = fminf(floorf(th + (1e-3f + 4e-7f * fabsf(th))), (float)last);
            empty |= !(fl <= fh);  // also true for the empty (+inf,-inf) box of an invalid Gaussian
            const int lo = empty ? 0 : (int)fl, hi = empty ? 0 : (int)fh;
            clo[k] = lo >> 1;
            nc[k] = (hi >> 1) - clo[k] + 1;
            // `first` is a multiple of 8, so a cell can only stick out of the batch at the upper end (odd extent)
            edge |= 2 * (clo[k] + nc[k]) - 1 > last;
        }
        // cull bound: |M(p - mu)| >= |M(cc - mu)| - rho for every voxel p of a cell with centre cc
        const float4 gb = rec[(size_t)N + i], gc = rec[2 * (size_t)N + i], gd4 = rec[3 * (size_t)N + i];
        const float hx = 0.5f * gd.spacing[0], hy = 0.5f * gd.spacing[1], hz = 0.5f * gd.spacing[2];
        const float q0 = fabsf(gb.x) * hx + fabsf(gb.y) * hy + fabsf(gb.z) * hz;
        const float q1 = fabsf(gc.x) * hx + fabsf(gc.y) * hy + fabsf(gc.z) * hz;
        const float q2 = fabsf(gd4.x) * hx + fabsf(gd4.y) * hy + fabsf(gd4.z) * hz;
        const float reach = rcut + sqrtf(q0 * q0 + q1 * q1 + q2 * q2);
        const float sx2 = 2.f * gd.spacing[0];
        const float e0 = gb.x * sx2, e1 = gc.x * sx2, e2 = gd4.x * sx2;
        setup[2 * (size_t)i] = make_float4(__int_as_float(clo[0]), __int_as_float(clo[1]), __int_as_float(clo[2]),
                                           __uint_as_float((empty ? 1u : 0u) | (edge ? 2u : 0u)));
        setup[2 * (size_t)i + 1] = make_float4(__uint_as_float((uint32_t)nc[0] | ((uint32_t)nc[1] << 11) | ((uint32_t)nc[2] << 22)),
                                               reach * reach * 1.001953125f, 1.0f / (e0 * e0 + e1 * e1 + e2 * e2), 0.f);
    }
    // 64-bit totals: pairs (overflow check) in the low counter, touched Gaussians in the next one
    unsigned long long s = c, m = c ? 1ull : 0ull;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        s += __shfl_xor_sync(0xffffffffu, s, d);
        m += __shfl_xor_sync(0xffffffffu, m, d);
    }
    if ((threadIdx.x & 31) == 0 && s) { atomicAdd(total, s); atomicAdd(total + 1, m); }
}

__global__ void __launch_bounds__(256) k_pair_write(const float *__restrict__ aabb, uint32_t N, GridDesc gd,
                                                     const uint32_t *__restrict__ offset, uint32_t T, uint32_t *__restrict__ key,
                                                     uint32_t *__restrict__ val) {
    const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= T) return;
    // largest i with offset[i] <= t  (offset has N+1 entries, offset[N] = T)
    uint32_t lo = 0, hi = N;  // invariant: offset[lo] <= t < offset[hi]
    while (hi - lo > 1) {
        const uint32_t mid = (lo + hi) >> 1;
        if (offset[mid] <= t) lo = mid; else hi = mid;
    }
    const uint32_t i = lo;
    float b6[6];
#pragma unroll
    for (int k = 0; k < 6; k++) b6[k] = aabb[6 * (size_t)i + k];
    BrickRange br;
    brick_range(b6, gd, br);
    uint32_t local = t - offset[i];
    const uint32_t ex = (uint32_t)(br.hi[0] - br.lo[0] + 1), ey = (uint32_t)(br.hi[1] - br.lo[1] + 1);
    const uint32_t x = local % ex; local /= ex;
    const uint32_t y = local % ey;
    const uint32_t z = local / ey;
    const uint32_t bx = (uint32_t)(br.lo[0] - gd.brick_lo[0]) + x, by = (uint32_t)(br.lo[1] - gd.brick_lo[1]) + y,
                   bz = (uint32_t)(br.lo[2] - gd.brick_lo[2]) + z;
    key[t] = (bz * (uint32_t)gd.brick_cnt[1] + by) * (uint32_t)gd.brick_cnt[0] + bx;
    val[t] = i;
}

__global__ void __launch_bounds__(256) k_brick_start(const uint32_t *__restrict__ key, uint32_t T, uint32_t nbricks,
                                                      uint32_t *__restrict__ start) {
    const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    if (T == 0) {
        for (uint32_t b = t; b <= nbricks; b += gridDim.x * blockDim.x) start[b] = 0;
        return;
    }
    if (t > T) return;
    // thread t closes the gap between key[t-1] and key[t]  (t = 0: from brick 0; t = T: up to nbricks)
    const uint32_t prev = (t == 0) ? 0u : key[t - 1] + 1u;
    const uint32_t cur = (t == T) ? nbricks : key[t];
    for (uint32_t b = prev; b <= cur; b++) start[b] = t;
}

cudaError_t launch_brick_count(const float *aabb, const float4 *rec, uint32_t N, const GridDesc &gd, float rcut, uint32_t *count,
                               unsigned long long *total, uint32_t *okey, uint32_t *oval, uint32_t untouched_key, float4 *setup,
                               cudaStream_t s) {
    cudaError_t e = cudaMemsetAsync(total, 0, 2 * sizeof(unsigned long long), s);
    if (e != cudaSuccess || N == 0) return e;
    k_brick_count<<<(N + 255) / 256, 256, 0, s>>>(aabb, rec, N, gd, rcut, count, total, okey, oval, untouched_key, setup); count_launch();
    return cudaGetLastError();
}

cudaError_t launch_pair_write(const float *aabb, uint32_t N, const GridDesc &gd, const uint32_t *offset, uint32_t T,
                              uint32_t *key, uint32_t *val, cudaStream_t s) {
    if (T == 0) return cudaSuccess;
    k_pair_write<<<(T + 255) / 256, 256, 0, s>>>(aabb, N, gd, offset, T, key, val); count_launch();
    return cudaGetLastError();
}

cudaError_t launch_brick_start(const uint32_t *key, uint32_t T, uint32_t nbricks, uint32_t *start, cudaStream_t s) {
    const uint32_t n = (T == 0) ? nbricks + 1 : T + 1;
    unsigned blocks = (n + 255) / 256;
    if (T == 0 && blocks > 1024) blocks = 1024;
    k_brick_start<<<blocks, 256, 0, s>>>(key, T, nbricks, start); count_launch();
    return cudaGetLastError();
}

}  // namespace gs
