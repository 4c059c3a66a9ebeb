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
__global__ void __launch_bounds__(256) k_brick_count(const float *__restrict__ aabb, uint32_t N, GridDesc gd,
                                                      uint32_t *__restrict__ count, unsigned long long *__restrict__ total,
                                                      uint32_t *__restrict__ okey, uint32_t *__restrict__ oval, uint32_t untouched_key) {
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

cudaError_t launch_brick_count(const float *aabb, uint32_t N, const GridDesc &gd, uint32_t *count, unsigned long long *total,
                               uint32_t *okey, uint32_t *oval, uint32_t untouched_key, cudaStream_t s) {
    cudaError_t e = cudaMemsetAsync(total, 0, 2 * sizeof(unsigned long long), s);
    if (e != cudaSuccess || N == 0) return e;
    k_brick_count<<<(N + 255) / 256, 256, 0, s>>>(aabb, N, gd, count, total, okey, oval, untouched_key); count_launch();
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
