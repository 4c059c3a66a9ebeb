// binning.cu -- S2: Gaussian -> brick lists for a structured batch (section 4.1.2).
// The list of (brick, gaussian) pairs sorted by (brick, gaussian) is produced by an MSD radix sort whose
// first digit is the whole brick id (a counting sort) and whose remaining digits are sorted per bucket:
//   k_brick_count : per Gaussian, brick range of its AABB inside the batch, the count n_i, and one
//                   atomic per overlapped brick into the brick histogram (the (brick, gaussian) pairs
//                   are enumerated by index arithmetic; large Gaussians are spread over the warp:
//                   "parallelizes over total intersections")
//   (scan)        : brick_start = exclusive scan of the histogram, brick_start[nbricks] = T
//   k_pair_fill   : the same enumeration; each pair takes a slot of its brick's run
//   k_bucket_sort : every brick's run is sorted by Gaussian id (bitonic network), so the result is the
//                   unique ascending (brick, gaussian) order whatever order the slots were taken in
// Measured on C2 (T = 2.56 M): the previous pipeline (per-Gaussian scan, pair write with a binary search per
// pair, two 8-bit LSD passes, run boundaries) took 0.25 ms of device time; this one is listed in DESIGN.md.
// Brick ranges are integer decisions: fixed fp32 sequence (D7).
#include "gs_internal.cuh"
#include "pair_math.cuh"
#include <algorithm>
using std::max;

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

// ---- enumeration of the bricks of a range ("parallelizes over total intersections").  The ranges of the
// 32 Gaussians of a warp are laid end to end (warp scan of their sizes) and the pairs are dealt to the lanes 32 at a
// time: a lane finds the Gaussian of its pair by a binary search in the scan (5 shuffles) and the brick by index
// arithmetic.  Ranges of more than COOP_MAX bricks are spread over the warp one Gaussian after the other.
// f(brick_id, gaussian_id) is called exactly once per (brick, gaussian) pair.  All 32 lanes must call this.
constexpr uint32_t COOP_MAX = 1024;

template <class F>
__device__ __forceinline__ void for_each_pair(const BrickRange &br, uint32_t c, uint32_t i, const GridDesc &gd, int lane, F f) {
    const uint32_t nbx = (uint32_t)gd.brick_cnt[0], nby = (uint32_t)gd.brick_cnt[1];
    const uint32_t ex = c ? (uint32_t)(br.hi[0] - br.lo[0] + 1) : 1u, ey = c ? (uint32_t)(br.hi[1] - br.lo[1] + 1) : 1u;
    // batch-local id of the range's first brick
    const uint32_t b0 = c ? (((uint32_t)(br.lo[2] - gd.brick_lo[2]) * nby + (uint32_t)(br.lo[1] - gd.brick_lo[1])) * nbx +
                             (uint32_t)(br.lo[0] - gd.brick_lo[0]))
                          : 0u;
    const bool big = c > COOP_MAX;
    const uint32_t cs = big ? 0u : c;
    uint32_t incl = cs;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t up = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += up;
    }
    const uint32_t total = __shfl_sync(0xffffffffu, incl, 31), excl = incl - cs;
    const float rex = 1.0f / (float)ex, rey = 1.0f / (float)ey;
    for (uint32_t t0 = 0; t0 < total; t0 += 32) {
        const uint32_t t = t0 + (uint32_t)lane;
        int src = 0;  // smallest lane whose inclusive count exceeds t
#pragma unroll
        for (int step = 16; step > 0; step >>= 1) {
            const uint32_t v = __shfl_sync(0xffffffffu, incl, src + step - 1);
            if (v <= t) src += step;
        }
        const uint32_t sexcl = __shfl_sync(0xffffffffu, excl, src), sex = __shfl_sync(0xffffffffu, ex, src),
                       sey = __shfl_sync(0xffffffffu, ey, src), sb0 = __shfl_sync(0xffffffffu, b0, src),
                       si = __shfl_sync(0xffffffffu, i, src);
        const float srex = __shfl_sync(0xffffffffu, rex, src), srey = __shfl_sync(0xffffffffu, rey, src);
        if (t < total) {
            // local < 1024: (local + 0.5) / e is at least 0.5 / 1024 away from an integer, far more than fp32 rounding
            const uint32_t local = t - sexcl;
            const uint32_t r = (uint32_t)(((float)local + 0.5f) * srex);
            const uint32_t x = local - r * sex;
            const uint32_t z = (uint32_t)(((float)r + 0.5f) * srey);
            const uint32_t y = r - z * sey;
            f(sb0 + (z * nby + y) * nbx + x, si);
        }
    }
    uint32_t todo = __ballot_sync(0xffffffffu, big);
    while (todo) {
        const int src = __ffs(todo) - 1;
        todo &= todo - 1;
        const uint32_t sc = __shfl_sync(0xffffffffu, c, src), sex = __shfl_sync(0xffffffffu, ex, src),
                       sey = __shfl_sync(0xffffffffu, ey, src), sb0 = __shfl_sync(0xffffffffu, b0, src),
                       si = __shfl_sync(0xffffffffu, i, src);
        for (uint32_t t = lane; t < sc; t += 32) {
            const uint32_t x = t % sex, r = t / sex;
            const uint32_t y = r % sey, z = r / sey;
            f(sb0 + (z * nby + y) * nbx + x, si);
        }
    }
}

// ---- coarse index (small batches of a large grid).  A batch looks only at the Gaussians listed in the coarse cells it
// overlaps; a Gaussian listed in several of them is handled in the FIRST one (lowest coordinates) of the batch it overlaps.
__device__ __forceinline__ void coarse_range(const float *__restrict__ bb, const GridDesc &gd, int (&lo)[3], int (&hi)[3], bool &empty) {
    empty = false;
#pragma unroll
    for (int k = 0; k < 3; k++) {
        const float nb = (float)gd.nb_total[k];
        float fl = floorf(__fmul_rn(__fsub_rn(bb[k], gd.origin[k]), gd.inv_brick[k]));
        float fh = floorf(__fmul_rn(__fsub_rn(bb[3 + k], gd.origin[k]), gd.inv_brick[k]));
        fl = fminf(fmaxf(fl, -1.0f), nb);
        fh = fminf(fmaxf(fh, -1.0f), nb);
        const int l = max((int)fl, 0), h = min((int)fh, gd.nb_total[k] - 1);
        empty |= h < l;   // also the (+inf, -inf) box of an invalid Gaussian
        lo[k] = l / COARSE_B;
        hi[k] = h / COARSE_B;
    }
}

// which Gaussian does thread t of a count / fill pass look at?  Returns false for a thread without one.
__device__ __forceinline__ bool pick_gaussian(const CandSegs &cs, const float *__restrict__ aabb, const GridDesc &gd, uint32_t N, uint32_t t,
                                              uint32_t &i) {
    if (!cs.ids) { i = t; return t < N; }
    // With an index the candidates are few (a batch touches a sliver of the model): ONE candidate per warp, held by lane 0, so
    // that for_each_pair deals its bricks to the 32 lanes at once (32 candidates per warp made every warp walk a chain of
    // dependent atomic round trips: 30 us for 12,600 candidates)
    if (t & 31u) return false;
    t >>= 5;
    if (t >= cs.total) return false;
    int sg = 0;
    while (t >= cs.prefix[sg + 1]) sg++;
    i = cs.ids[cs.start[sg] + (t - cs.prefix[sg])];
    int lo[3], hi[3];
    bool empty;
    float b6[6];
#pragma unroll
    for (int k = 0; k < 6; k++) b6[k] = aabb[6 * (size_t)i + k];
    coarse_range(b6, gd, lo, hi, empty);
    // owner = the first coarse cell of (Gaussian's cells) intersected with (batch's cells)
    return !empty && max(lo[0], cs.clo[0]) == cs.cell[sg][0] && max(lo[1], cs.clo[1]) == cs.cell[sg][1] && max(lo[2], cs.clo[2]) == cs.cell[sg][2];
}

__global__ void __launch_bounds__(256) k_coarse_index(const float *__restrict__ aabb, uint32_t N, GridDesc gd, int ncx, int ncy,
                                                       uint32_t *__restrict__ hist, const uint32_t *__restrict__ start, uint32_t *__restrict__ ids) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    float b6[6];
#pragma unroll
    for (int k = 0; k < 6; k++) b6[k] = aabb[6 * (size_t)i + k];
    int lo[3], hi[3];
    bool empty;
    coarse_range(b6, gd, lo, hi, empty);
    if (empty) return;
    for (int z = lo[2]; z <= hi[2]; z++)
        for (int y = lo[1]; y <= hi[1]; y++)
            for (int x = lo[0]; x <= hi[0]; x++) {
                const uint32_t c = ((uint32_t)z * ncy + y) * ncx + x;
                if (ids) ids[start[c] + (atomicSub(hist + c, 1u) - 1u)] = i;   // second pass: take a slot (counts the cell down to zero)
                else atomicAdd(hist + c, 1u);
            }
}

// Morton code of the Gaussian's central brick, coarsened to at most ORDER_BITS bits per axis: the processing
// order of the backward pass (performance only: neighbouring Gaussians are processed together so that their
// voxel data stays in L1/L2).
__device__ __forceinline__ uint32_t order_key(const BrickRange &br, const GridDesc &gd, int order_shift) {
    const uint32_t mx = (uint32_t)(((br.lo[0] + br.hi[0]) >> 1) - gd.brick_lo[0]) >> order_shift;
    const uint32_t my = (uint32_t)(((br.lo[1] + br.hi[1]) >> 1) - gd.brick_lo[1]) >> order_shift;
    const uint32_t mz = (uint32_t)(((br.lo[2] + br.hi[2]) >> 1) - gd.brick_lo[2]) >> order_shift;
    return spread3(mx) | (spread3(my) << 1) | (spread3(mz) << 2);
}

// hist = [nbricks brick counters | order-bucket counters].  Also writes the per-Gaussian constants of the
// backward kernel (performance only, nothing canonical): the box of 2x2x2-voxel cells that covers the AABB
// inside the batch, the whitened-space cull threshold of a cell and 1 / |e|^2 for the closed-form row
// intervals (sample_grid_bwd.cu):
//   setup[2 i]     = (clo.x, clo.y, clo.z, flags: 1 = touches no voxel of the batch, 2 = a cell sticks out of the batch)
//   setup[2 i + 1] = ((ncx - 1) | (ncy - 1) << 10 | (ncz - 1) << 20, thr, invA, -)   (a batch spans <= 2048 voxels = 1024 cells per axis)
__global__ void __launch_bounds__(256) k_brick_count(const float *__restrict__ aabb, const float4 *__restrict__ rec, uint32_t N,
                                                      GridDesc gd, float rcut, uint32_t *__restrict__ count,
                                                      unsigned long long *__restrict__ total, uint32_t *__restrict__ hist,
                                                      uint32_t nbricks, int order_shift, float4 *__restrict__ setup,
                                                      const __grid_constant__ CandSegs cs) {
    uint32_t i = 0;
    const bool mine = pick_gaussian(cs, aabb, gd, N, blockIdx.x * blockDim.x + threadIdx.x, i);
    const int lane = threadIdx.x & 31;
    uint32_t c = 0;
    BrickRange br{};
    if (mine) {
        const float *bb = aabb + 6 * (size_t)i;
        // an invalid Gaussian has the empty box (+inf, -inf): fmaxf/fminf clamp it to an empty range.
        // NaN cannot occur here (preprocess writes inf for invalid ones).
        float b6[6];
#pragma unroll
        for (int k = 0; k < 6; k++) b6[k] = bb[k];
        c = brick_range(b6, gd, br);
        count[i] = c;
        if (c) atomicAdd(hist + nbricks + order_key(br, gd, order_shift), 1u);
      if (c) {  // a Gaussian that touches no brick of the batch is never looked at again (no record read, no setup row)
        // ---- backward setup
        int clo[3], nc[3];
        bool empty = false, edge = false;
#pragma unroll
        for (int k = 0; k < 3; k++) {
            const float inv_sp = 1.0f / gd.spacing[k];
            // voxel i is sampled at its centre i + 0.5, or with jitter anywhere in [i, i + 1) (in units of the spacing)
            const float tl = (b6[k] - gd.origin[k]) * inv_sp - (gd.jitter ? 1.0f : 0.5f);
            const float th = (b6[3 + k] - gd.origin[k]) * inv_sp - (gd.jitter ? 0.0f : 0.5f);
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
        const float hh = gd.jitter ? 1.0f : 0.5f;  // half extent of a cell's samples around the cell centre, in voxels
        const float hx = hh * gd.spacing[0], hy = hh * gd.spacing[1], hz = hh * gd.spacing[2];
        const float q0 = fabsf(gb.x) * hx + fabsf(gb.y) * hy + fabsf(gb.z) * hz;
        const float q1 = fabsf(gc.x) * hx + fabsf(gc.y) * hy + fabsf(gc.z) * hz;
        const float q2 = fabsf(gd4.x) * hx + fabsf(gd4.y) * hy + fabsf(gd4.z) * hz;
        const float reach = rcut + sqrtf(q0 * q0 + q1 * q1 + q2 * q2);
        const float sx2 = 2.f * gd.spacing[0];
        const float e0 = gb.x * sx2, e1 = gc.x * sx2, e2 = gd4.x * sx2;
        setup[2 * (size_t)i] = make_float4(__int_as_float(clo[0]), __int_as_float(clo[1]), __int_as_float(clo[2]),
                                           __uint_as_float((empty ? 1u : 0u) | (edge ? 2u : 0u)));
        setup[2 * (size_t)i + 1] = make_float4(__uint_as_float((uint32_t)(nc[0] - 1) | ((uint32_t)(nc[1] - 1) << 10) | ((uint32_t)(nc[2] - 1) << 20)),
                                               reach * reach * 1.001953125f, 1.0f / (e0 * e0 + e1 * e1 + e2 * e2), 0.f);
      }
    }
    if (!cs.ids && !__any_sync(0xffffffffu, c != 0u)) return;  // a warp whose 32 Gaussians all miss the batch (most warps of a small batch)
    for_each_pair(br, c, i, gd, lane, [&](uint32_t b, uint32_t) { atomicAdd(hist + b, 1u); });
    // 64-bit totals: pairs (overflow check) in the low counter, touched Gaussians in the next one
    unsigned long long s = c, m = c ? 1ull : 0ull;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        s += __shfl_xor_sync(0xffffffffu, s, d);
        m += __shfl_xor_sync(0xffffffffu, m, d);
    }
    if (cs.ids) {   // a warp per candidate: thousands of warps would queue up on the two counters; add them per CTA
        __shared__ unsigned long long red[2];
        if (threadIdx.x == 0) { red[0] = 0ull; red[1] = 0ull; }
        __syncthreads();
        if (lane == 0 && s) { atomicAdd(&red[0], s); atomicAdd(&red[1], m); }
        __syncthreads();
        if (threadIdx.x == 0 && red[0]) { atomicAdd(total, red[0]); atomicAdd(total + 1, red[1]); }
        return;
    }
    if (lane == 0 && s) { atomicAdd(total, s); atomicAdd(total + 1, m); }
}

// Every pair takes a slot of its brick's run by counting the brick's histogram entry DOWN (so the histogram is
// all zero again afterwards); the order list of the backward is filled the same way.  Nothing is written when
// the pair list does not fit `cap` entries: the host then grows the buffer and repeats this kernel.
__global__ void __launch_bounds__(256) k_pair_fill(const float *__restrict__ aabb, const uint32_t *__restrict__ count, uint32_t N, GridDesc gd,
                                                    const unsigned long long *__restrict__ total, uint32_t cap,
                                                    uint32_t *__restrict__ hist, const uint32_t *__restrict__ start, uint32_t nbricks,
                                                    int order_shift, uint32_t *__restrict__ pair_gauss, uint32_t *__restrict__ order,
                                                    const __grid_constant__ CandSegs cs) {
    if (total[0] > (unsigned long long)cap) {   // the list does not fit: write nothing; total[3] remembers it for the host (sticky)
        if (blockIdx.x == 0 && threadIdx.x == 0) const_cast<unsigned long long *>(total)[3] = 1ull;
        return;
    }
    const uint32_t T = (uint32_t)total[0];
    uint32_t i = 0;
    const bool mine = pick_gaussian(cs, aabb, gd, N, blockIdx.x * blockDim.x + threadIdx.x, i);
    const int lane = threadIdx.x & 31;
    uint32_t c = 0;
    BrickRange br{};
    if (mine && count[i]) {  // the count pass left n_i: untouched Gaussians cost 4 bytes here
        float b6[6];
#pragma unroll
        for (int k = 0; k < 6; k++) b6[k] = aabb[6 * (size_t)i + k];
        c = brick_range(b6, gd, br);
        if (c) {
            const uint32_t m = nbricks + order_key(br, gd, order_shift);
            order[start[m] - T + (atomicSub(hist + m, 1u) - 1u)] = i;
        }
    }
    if (!__any_sync(0xffffffffu, c != 0u)) return;
    for_each_pair(br, c, i, gd, lane, [&](uint32_t b, uint32_t id) { pair_gauss[start[b] + (atomicSub(hist + b, 1u) - 1u)] = id; });
}

// ---- per-brick sort of the Gaussian ids.  Bitonic network in its all-ascending form (the first step of every
// merge compares mirror positions), so that a run of any length n is sorted as if padded with +inf to a power of
// two: a comparator whose upper index is >= n does nothing.
template <class SYNC>
__device__ __forceinline__ void bitonic_ascending(uint32_t *a, uint32_t n, uint32_t tid, uint32_t nthreads, SYNC sync) {
    uint32_t n2 = 1;
    while (n2 < n) n2 <<= 1;
    for (uint32_t k = 2; k <= n2; k <<= 1) {
        for (uint32_t j = k >> 1; j > 0; j >>= 1) {
            const bool flip = (j == (k >> 1));
            for (uint32_t t = tid; t < (n2 >> 1); t += nthreads) {
                // t-th comparator of this step: lower index lo has bit j clear
                const uint32_t lo = ((t & ~(j - 1)) << 1) | (t & (j - 1));
                const uint32_t hi = flip ? (lo ^ (k - 1)) : (lo | j);
                if (hi < n) {
                    const uint32_t x = a[lo], y = a[hi];
                    if (x > y) { a[lo] = y; a[hi] = x; }
                }
            }
            sync();
        }
    }
}

constexpr int BS_WARPS = 4;
constexpr uint32_t BS_SMEM = 1024;  // entries a warp sorts in shared memory

__global__ void __launch_bounds__(BS_WARPS * 32) k_bucket_sort(const unsigned long long *__restrict__ total, uint32_t cap,
                                                                const uint32_t *__restrict__ start, uint32_t nbricks,
                                                                uint32_t *__restrict__ pair_gauss) {
    __shared__ __align__(16) uint32_t sm[BS_WARPS][BS_SMEM];
    if (total[0] > (unsigned long long)cap) return;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t b = blockIdx.x * BS_WARPS + warp;
    uint32_t s = 0, n = 0;
    if (b < nbricks) { s = start[b]; n = start[b + 1] - s; }
    uint32_t *run = pair_gauss + s;
    if (n > 1 && n <= 32) {  // one id per lane: compare-exchange through shuffles
        uint32_t v = (uint32_t)lane < n ? run[lane] : 0xffffffffu;
#pragma unroll
        for (int k = 2; k <= 32; k <<= 1) {
#pragma unroll
            for (int j = k >> 1; j > 0; j >>= 1) {
                const int partner = (j == (k >> 1)) ? (lane ^ (k - 1)) : (lane ^ j);
                const uint32_t o = __shfl_sync(0xffffffffu, v, partner);
                v = (lane < partner) ? min(v, o) : max(v, o);
            }
        }
        if ((uint32_t)lane < n) run[lane] = v;
    } else if (n > 32 && n <= 128) {
        // four ids per lane (element e = 32 r + lane), the same all-ascending bitonic network: partners in other lanes
        // come through shuffles, partners in the same lane (e ^ 32) are a register compare-exchange
        uint32_t v[4];
#pragma unroll
        for (int r = 0; r < 4; r++) v[r] = (uint32_t)lane + 32u * r < n ? run[lane + 32 * r] : 0xffffffffu;
        auto cmpex = [&](uint32_t mine, uint32_t other, bool lower) { return lower ? min(mine, other) : max(mine, other); };
#pragma unroll
        for (int k = 2; k <= 32; k <<= 1) {
#pragma unroll
            for (int j = k >> 1; j > 0; j >>= 1) {
                const int x = (j == (k >> 1)) ? (k - 1) : j;      // lane ^ x is the partner; the lower index has bit j clear
                const bool lower = (lane & j) == 0;
#pragma unroll
                for (int r = 0; r < 4; r++) v[r] = cmpex(v[r], __shfl_xor_sync(0xffffffffu, v[r], x), lower);
            }
        }
        {   // k = 64: flip e ^ 63 = (lane ^ 31, r ^ 1); the lower index has r even
            uint32_t o[4];
#pragma unroll
            for (int r = 0; r < 4; r++) o[r] = __shfl_xor_sync(0xffffffffu, v[r ^ 1], 31);
#pragma unroll
            for (int r = 0; r < 4; r++) v[r] = cmpex(v[r], o[r], (r & 1) == 0);
#pragma unroll
            for (int j = 16; j > 0; j >>= 1) {
                const bool lower = (lane & j) == 0;
#pragma unroll
                for (int r = 0; r < 4; r++) v[r] = cmpex(v[r], __shfl_xor_sync(0xffffffffu, v[r], j), lower);
            }
        }
        if (n > 64) {  // k = 128: flip e ^ 127 = (lane ^ 31, r ^ 3), lower index has r < 2; then e ^ 32 = (lane, r ^ 1)
            uint32_t o[4];
#pragma unroll
            for (int r = 0; r < 4; r++) o[r] = __shfl_xor_sync(0xffffffffu, v[r ^ 3], 31);
#pragma unroll
            for (int r = 0; r < 4; r++) v[r] = cmpex(v[r], o[r], (r & 2) == 0);
            const uint32_t a0 = min(v[0], v[1]), a1 = max(v[0], v[1]), a2 = min(v[2], v[3]), a3 = max(v[2], v[3]);
            v[0] = a0; v[1] = a1; v[2] = a2; v[3] = a3;
#pragma unroll
            for (int j = 16; j > 0; j >>= 1) {
                const bool lower = (lane & j) == 0;
#pragma unroll
                for (int r = 0; r < 4; r++) v[r] = cmpex(v[r], __shfl_xor_sync(0xffffffffu, v[r], j), lower);
            }
        }
#pragma unroll
        for (int r = 0; r < 4; r++)
            if ((uint32_t)lane + 32u * r < n) run[lane + 32 * r] = v[r];
    } else if (n > 128 && n <= BS_SMEM) {
        uint32_t *a = sm[warp];
        for (uint32_t t = lane; t < n; t += 32) a[t] = run[t];
        __syncwarp();
        bitonic_ascending(a, n, (uint32_t)lane, 32u, [] { __syncwarp(); });
        for (uint32_t t = lane; t < n; t += 32) run[t] = a[t];
    }
    // runs longer than a warp's shared memory: the whole CTA sorts them in place in global memory, one after the other
    __syncthreads();
    for (int w = 0; w < BS_WARPS; w++) {
        const uint32_t bw = blockIdx.x * BS_WARPS + w;
        if (bw >= nbricks) break;
        const uint32_t sw = start[bw], nw = start[bw + 1] - sw;
        if (nw <= BS_SMEM) continue;  // block-uniform
        bitonic_ascending(pair_gauss + sw, nw, threadIdx.x, (uint32_t)(BS_WARPS * 32), [] { __syncthreads(); });
    }
}

// debug view: the brick id of every entry of the sorted pair list (gs_debug_get(GS_DBG_PAIR_BRICK))
__global__ void __launch_bounds__(256) k_expand_bricks(const uint32_t *__restrict__ start, uint32_t nbricks, uint32_t *__restrict__ key) {
    const uint32_t b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nbricks) return;
    for (uint32_t t = start[b]; t < start[b + 1]; t++) key[t] = b;
}

cudaError_t launch_brick_count(const float *aabb, const float4 *rec, uint32_t N, const GridDesc &gd, float rcut, uint32_t *count,
                               unsigned long long *total, uint32_t *hist, uint32_t nbricks, uint32_t norder, int order_shift,
                               float4 *setup, const CandSegs &cs, cudaStream_t s) {
    // (total, hist and -- with an index -- the stale counts were reset by launch_build_reset)
    if (N == 0) return cudaSuccess;
    const uint64_t work64 = cs.ids ? (uint64_t)cs.total * 32 : N;   // with an index: a warp per candidate (pick_gaussian)
    if (work64 == 0 || work64 > 0xffffff00ull) return work64 ? cudaErrorInvalidValue : cudaSuccess;
    const uint32_t work = (uint32_t)work64;
    k_brick_count<<<(work + 255) / 256, 256, 0, s>>>(aabb, rec, N, gd, rcut, count, total, hist, nbricks, order_shift, setup, cs); count_launch();
    return cudaGetLastError();
}

cudaError_t launch_pair_fill(const float *aabb, const uint32_t *count, uint32_t N, const GridDesc &gd, const unsigned long long *total, uint32_t cap,
                             uint32_t *hist, const uint32_t *start, uint32_t nbricks, int order_shift, uint32_t *pair_gauss,
                             uint32_t *order, const CandSegs &cs, cudaStream_t s) {
    if (N == 0) return cudaSuccess;
    const uint32_t work = cs.ids ? cs.total * 32u : N;
    if (work) { k_pair_fill<<<(work + 255) / 256, 256, 0, s>>>(aabb, count, N, gd, total, cap, hist, start, nbricks, order_shift, pair_gauss, order, cs); count_launch(); }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    k_bucket_sort<<<(nbricks + BS_WARPS - 1) / BS_WARPS, BS_WARPS * 32, 0, s>>>(total, cap, start, nbricks, pair_gauss); count_launch();
    return cudaGetLastError();
}

// One launch instead of three memsets in front of every build (small batches are bound by the host's launch rate): zero the
// pair / touched totals and the brick + order histogram, and -- when the previous batch came from the coarse index -- put the
// counts of ITS candidates back to zero (the other Gaussians already read "touches nothing").
__global__ void __launch_bounds__(256) k_build_reset(unsigned long long *__restrict__ total, uint32_t *__restrict__ hist, uint32_t nh,
                                                      uint32_t *__restrict__ count, const __grid_constant__ CandSegs prev) {
    const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t < 2) total[t] = 0ull;
    if (t < nh) hist[t] = 0u;
    if (prev.ids && t < prev.total) {
        int sg = 0;
        while (t >= prev.prefix[sg + 1]) sg++;
        count[prev.ids[prev.start[sg] + (t - prev.prefix[sg])]] = 0u;
    }
}

cudaError_t launch_build_reset(unsigned long long *total, uint32_t *hist, uint32_t nh, uint32_t *count, const CandSegs &prev, cudaStream_t s) {
    const uint32_t work = max(max(nh, prev.ids ? prev.total : 0u), 2u);
    k_build_reset<<<(work + 255) / 256, 256, 0, s>>>(total, hist, nh, count, prev); count_launch();
    return cudaGetLastError();
}

cudaError_t launch_coarse_count(const float *aabb, uint32_t N, const GridDesc &full, const int nc[3], uint32_t *hist, cudaStream_t s) {
    cudaError_t e = cudaMemsetAsync(hist, 0, (size_t)nc[0] * nc[1] * nc[2] * sizeof(uint32_t), s);
    if (e != cudaSuccess || N == 0) return e;
    k_coarse_index<<<(N + 255) / 256, 256, 0, s>>>(aabb, N, full, nc[0], nc[1], hist, nullptr, nullptr); count_launch();
    return cudaGetLastError();
}

cudaError_t launch_coarse_fill(const float *aabb, uint32_t N, const GridDesc &full, const int nc[3], uint32_t *hist, const uint32_t *start,
                               uint32_t *ids, cudaStream_t s) {
    if (N == 0) return cudaSuccess;
    k_coarse_index<<<(N + 255) / 256, 256, 0, s>>>(aabb, N, full, nc[0], nc[1], hist, start, ids); count_launch();
    return cudaGetLastError();
}

// sample positions of a jittered batch (D26): one hash per voxel, three 21-bit offsets, the canonical
// position fmaf(((float)i + 0.5f) + j, spacing, origin) per axis; written once per step and read by the forward, the
// backward and the densification (16 B per voxel)
__global__ void __launch_bounds__(256) k_jitter_table(GridDesc gd, float4 *__restrict__ jit) {
    const uint32_t x = blockIdx.x * blockDim.x + threadIdx.x, y = blockIdx.y, z = blockIdx.z;
    if (x >= (uint32_t)gd.bdim[0]) return;
    const int gx = (int)x + BRICK * gd.brick_lo[0], gy = (int)y + BRICK * gd.brick_lo[1], gz = (int)z + BRICK * gd.brick_lo[2];
    float jx, jy, jz;
    voxel_jitter3(voxel_hash(gd.jitter_seed, voxel_linear(gx, gy, gz, gd.dims[0], gd.dims[1])), jx, jy, jz);
    jit[((size_t)z * gd.bdim[1] + y) * gd.bdim[0] + x] =
        make_float4(voxel_sample(gx, jx, gd.spacing[0], gd.origin[0]), voxel_sample(gy, jy, gd.spacing[1], gd.origin[1]),
                    voxel_sample(gz, jz, gd.spacing[2], gd.origin[2]), 0.f);
}

cudaError_t launch_jitter_table(const GridDesc &gd, float4 *jit, cudaStream_t s) {
    const dim3 grid((unsigned)((gd.bdim[0] + 255) / 256), (unsigned)gd.bdim[1], (unsigned)gd.bdim[2]);
    k_jitter_table<<<grid, 256, 0, s>>>(gd, jit); count_launch();
    return cudaGetLastError();
}

cudaError_t launch_expand_bricks(const uint32_t *start, uint32_t nbricks, uint32_t *key, cudaStream_t s) {
    if (nbricks == 0) return cudaSuccess;
    k_expand_bricks<<<(nbricks + 255) / 256, 256, 0, s>>>(start, nbricks, key); count_launch();
    return cudaGetLastError();
}

}  // namespace gs
