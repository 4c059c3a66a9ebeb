// scan_sort.cu -- device-wide exclusive scan and a stable LSD radix sort of (u32 key, u32 value) pairs.
// Used for the prefix sum over per-Gaussian brick counts, the sort of the
// (brick, gaussian) pairs by brick and the Morton sorts of the LBVH (north_star (2)).
// Hand-written (no CUB): reduce-then-scan with a recursive scan of the tile sums; the sort is
// 8 bits per pass, per-tile digit histograms -> global scan -> stable per-warp ranked scatter.
#include "gs_internal.cuh"

namespace gs {

// ------------------------------------------------------------------------------------------------
// exclusive scan
// ------------------------------------------------------------------------------------------------
constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ITEMS = 8;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;  // 2048

__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v, int lane) {
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        uint32_t t = __shfl_up_sync(0xffffffffu, v, d);
        if (lane >= d) v += t;
    }
    return v;
}

// exclusive scan of one value per thread over the block; returns the exclusive prefix, *total = block sum
__device__ __forceinline__ uint32_t block_excl_scan(uint32_t v, uint32_t *total, uint32_t *smem /*>= 33*/) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    uint32_t incl = warp_incl_scan(v, lane);
    if (lane == 31) smem[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        uint32_t w = lane < nwarp ? smem[lane] : 0u;
        uint32_t wi = warp_incl_scan(w, lane);
        smem[lane] = wi - w;
        if (lane == 31) smem[32] = wi;
    }
    __syncthreads();
    uint32_t r = incl - v + smem[warp];
    *total = smem[32];
    __syncthreads();
    return r;
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_reduce(const uint32_t *__restrict__ in, size_t n, uint32_t *__restrict__ sums) {
    __shared__ uint32_t sm[40];
    const size_t base = (size_t)blockIdx.x * SCAN_TILE + (size_t)threadIdx.x * SCAN_ITEMS;
    uint32_t s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; k++)
        if (base + k < n) s += in[base + k];
    uint32_t total;
    block_excl_scan(s, &total, sm);
    if (threadIdx.x == 0) sums[blockIdx.x] = total;
}

// scans one tile; offsets (nullable) = exclusive scan of the tile sums; writes out[n] = grand total when last tile
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_tile(const uint32_t *__restrict__ in, uint32_t *__restrict__ out, size_t n,
                                                             const uint32_t *__restrict__ offsets, int write_total) {
    __shared__ uint32_t sm[40];
    const size_t base = (size_t)blockIdx.x * SCAN_TILE + (size_t)threadIdx.x * SCAN_ITEMS;
    uint32_t v[SCAN_ITEMS], s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; k++) {
        v[k] = (base + k < n) ? in[base + k] : 0u;
        s += v[k];
    }
    uint32_t total;
    uint32_t pre = block_excl_scan(s, &total, sm) + (offsets ? offsets[blockIdx.x] : 0u);
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; k++) {
        if (base + k < n) out[base + k] = pre;
        pre += v[k];
    }
    if (write_total && blockIdx.x == gridDim.x - 1 && threadIdx.x == SCAN_THREADS - 1) out[n] = pre;
}

// small inputs (a grid batch's brick histogram): ONE launch, one CTA walking the tiles with a running carry
constexpr int SCAN_SMALL_THREADS = 1024;
__global__ void __launch_bounds__(SCAN_SMALL_THREADS) k_scan_small(const uint32_t *__restrict__ in, uint32_t *__restrict__ out, size_t n) {
    __shared__ uint32_t sm[40];
    uint32_t carry = 0;
    for (size_t tile = 0; tile < n; tile += (size_t)SCAN_SMALL_THREADS * SCAN_ITEMS) {
        const size_t base = tile + (size_t)threadIdx.x * SCAN_ITEMS;
        uint32_t v[SCAN_ITEMS], s = 0;
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; k++) {
            v[k] = (base + k < n) ? in[base + k] : 0u;
            s += v[k];
        }
        uint32_t total;
        uint32_t pre = block_excl_scan(s, &total, sm) + carry;
#pragma unroll
        for (int k = 0; k < SCAN_ITEMS; k++) {
            if (base + k < n) out[base + k] = pre;
            pre += v[k];
        }
        carry += total;
    }
    if (threadIdx.x == 0) out[n] = carry;
}

static cudaError_t scan_rec(const uint32_t *in, uint32_t *out, size_t n, uint32_t *tmp, int write_total, cudaStream_t s) {
    const size_t tiles = (n + SCAN_TILE - 1) / SCAN_TILE;
    if (tiles <= 1) {
        k_scan_tile<<<1, SCAN_THREADS, 0, s>>>(in, out, n, nullptr, write_total); count_launch();
        return cudaGetLastError();
    }
    uint32_t *sums = tmp;                  // [tiles]
    uint32_t *next = tmp + ((tiles + 63) & ~size_t(63));
    k_scan_reduce<<<(unsigned)tiles, SCAN_THREADS, 0, s>>>(in, n, sums); count_launch();
    cudaError_t e = scan_rec(sums, sums, tiles, next, 0, s);
    if (e != cudaSuccess) return e;
    k_scan_tile<<<(unsigned)tiles, SCAN_THREADS, 0, s>>>(in, out, n, sums, write_total); count_launch();
    return cudaGetLastError();
}

cudaError_t exclusive_scan_u32(const uint32_t *in, uint32_t *out, size_t n, DevBuf &tmp, cudaStream_t s) {
    if (n == 0) return cudaMemsetAsync(out, 0, sizeof(uint32_t), s);
    if (n <= 16 * SCAN_TILE) {
        k_scan_small<<<1, SCAN_SMALL_THREADS, 0, s>>>(in, out, n); count_launch();
        return cudaGetLastError();
    }
    const size_t tiles = (n + SCAN_TILE - 1) / SCAN_TILE;
    cudaError_t e = tmp.reserve((tiles + 64 + tiles / 1024 + 128) * 2 * sizeof(uint32_t));
    if (e != cudaSuccess) return e;
    return scan_rec(in, out, n, tmp.as<uint32_t>(), 1, s);
}

// ------------------------------------------------------------------------------------------------
// radix sort: 8 bits per pass.  A tile is SORT_WARPS contiguous warp segments of SORT_SEG items;
// stable order inside a tile = (warp, round, lane).
// ------------------------------------------------------------------------------------------------
constexpr int SORT_WARPS = 8;
constexpr int SORT_ROUNDS = 16;
constexpr int SORT_SEG = 32 * SORT_ROUNDS;            // 512 items per warp
constexpr int SORT_TILE = SORT_WARPS * SORT_SEG;      // 4096 items per block
constexpr int RADIX = 256;
static_assert(SORT_WARPS * 32 == RADIX, "k_sort_scatter: one thread per digit");

// lanes holding the same 8-bit digit as this one (inactive lanes pass d = 0xffffffff and are excluded by `ok`): eight ballots,
// one per digit bit -- a fixed 16 instructions where match.any.sync iterates over the distinct values of the warp
__device__ __forceinline__ uint32_t digit_peers(uint32_t d, bool ok) {
    uint32_t peers = __ballot_sync(0xffffffffu, ok);
#pragma unroll
    for (int b = 0; b < 8; b++) {
        const uint32_t bal = __ballot_sync(0xffffffffu, (d >> b) & 1u);
        peers &= ((d >> b) & 1u) ? bal : ~bal;
    }
    return peers;
}

// per-warp digit histogram of its segment into smem wh[warp][256] (no atomics: one warp owns a row)
__device__ __forceinline__ void warp_histogram(const uint32_t *__restrict__ keys, size_t n, size_t seg_base, int shift, uint32_t mask,
                                               uint32_t *wh, int lane) {
    for (int d = lane; d < RADIX; d += 32) wh[d] = 0;
    __syncwarp();
#pragma unroll 4
    for (int r = 0; r < SORT_ROUNDS; r++) {
        const size_t idx = seg_base + (size_t)r * 32 + lane;
        const bool ok = idx < n;
        const uint32_t d = ok ? ((keys[idx] >> shift) & mask) : 0xffffffffu;
        const uint32_t peers = digit_peers(d, ok);
        if (ok && (int)(__ffs(peers) - 1) == lane) wh[d] += __popc(peers);
        __syncwarp();
    }
}

// per-tile digit counts: shared-memory atomics (a count needs no order)
__global__ void __launch_bounds__(SORT_WARPS * 32) k_sort_hist(const uint32_t *__restrict__ keys, size_t n, int shift, uint32_t mask,
                                                                uint32_t *__restrict__ hist /*[256][ntiles]*/, uint32_t ntiles) {
    __shared__ uint32_t sh[RADIX];
    for (int d = threadIdx.x; d < RADIX; d += blockDim.x) sh[d] = 0;
    __syncthreads();
    const size_t base = (size_t)blockIdx.x * SORT_TILE;
#pragma unroll 4
    for (int r = 0; r < SORT_TILE / (SORT_WARPS * 32); r++) {
        const size_t idx = base + (size_t)r * (SORT_WARPS * 32) + threadIdx.x;
        if (idx < n) atomicAdd(&sh[(keys[idx] >> shift) & mask], 1u);
    }
    __syncthreads();
    for (int d = threadIdx.x; d < RADIX; d += blockDim.x) hist[(size_t)d * ntiles + blockIdx.x] = sh[d];
}

// Stable scatter of one tile.  The rank of an item inside the tile is (items of smaller digits) + (items of its digit in
// earlier warps) + (earlier items of its digit in its own warp: __match_any_sync ranking, order (round, lane)).  The tile is
// first permuted into that order in shared memory and then written out slot by slot, so that consecutive threads write
// consecutive addresses of a digit's run (a direct scatter wrote 4 bytes per 32-byte sector).
__global__ void __launch_bounds__(SORT_WARPS * 32) k_sort_scatter(const uint32_t *__restrict__ keys, const uint32_t *__restrict__ vals,
                                                                   uint32_t *__restrict__ keys_out, uint32_t *__restrict__ vals_out,
                                                                   size_t n, int shift, uint32_t mask,
                                                                   const uint32_t *__restrict__ hist_scanned, uint32_t ntiles) {
    __shared__ uint32_t wh[SORT_WARPS][RADIX];
    __shared__ uint32_t tstart[RADIX];   // first slot of the digit's run inside the tile
    __shared__ uint32_t gbase[RADIX];    // global position of that slot
    __shared__ uint32_t skey[SORT_TILE], sval[SORT_TILE];
    __shared__ uint32_t scan_sm[40];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const size_t tile_base = (size_t)blockIdx.x * SORT_TILE;
    const size_t seg_base = tile_base + (size_t)warp * SORT_SEG;
    warp_histogram(keys, n, seg_base, shift, mask, wh[warp], lane);
    __syncthreads();
    // per digit (thread d, RADIX == blockDim): tile count -> exclusive scan over the digits = run starts; per-warp offsets
    {
        const int d = threadIdx.x;
        uint32_t cnt = 0;
#pragma unroll
        for (int w = 0; w < SORT_WARPS; w++) cnt += wh[w][d];
        uint32_t total;
        const uint32_t start = block_excl_scan(cnt, &total, scan_sm);
        tstart[d] = start;
        gbase[d] = hist_scanned[(size_t)d * ntiles + blockIdx.x];
        uint32_t run = start;
#pragma unroll
        for (int w = 0; w < SORT_WARPS; w++) {
            const uint32_t c = wh[w][d];
            wh[w][d] = run;
            run += c;
        }
    }
    __syncthreads();
    uint32_t *base = wh[warp];
#pragma unroll 4
    for (int r = 0; r < SORT_ROUNDS; r++) {
        const size_t idx = seg_base + (size_t)r * 32 + lane;
        const bool ok = idx < n;
        const uint32_t k = ok ? keys[idx] : 0u;
        const uint32_t d = ok ? ((k >> shift) & mask) : 0xffffffffu;
        const uint32_t peers = digit_peers(d, ok);
        uint32_t slot = 0;
        if (ok) slot = base[d] + __popc(peers & ((1u << lane) - 1u));
        __syncwarp();
        if (ok && (int)(__ffs(peers) - 1) == lane) base[d] += __popc(peers);
        __syncwarp();
        if (ok) {
            skey[slot] = k;
            sval[slot] = vals[idx];
        }
    }
    __syncthreads();
    const uint32_t count = (uint32_t)(n - tile_base < (size_t)SORT_TILE ? n - tile_base : (size_t)SORT_TILE);
    for (uint32_t i = threadIdx.x; i < count; i += SORT_WARPS * 32) {
        const uint32_t k = skey[i];
        const uint32_t d = (k >> shift) & mask;
        const uint32_t dst = gbase[d] + (i - tstart[d]);
        keys_out[dst] = k;
        vals_out[dst] = sval[i];
    }
}

cudaError_t radix_sort_pairs(uint32_t *keys[2], uint32_t *vals[2], size_t n, int bits, DevBuf &hist, DevBuf &tmp,
                             cudaStream_t s, int *result_sel) {
    *result_sel = 0;
    if (n <= 1 || bits <= 0) return cudaSuccess;
    const uint32_t ntiles = (uint32_t)((n + SORT_TILE - 1) / SORT_TILE);
    const size_t hn = (size_t)RADIX * ntiles;
    cudaError_t e = hist.reserve((hn + 1) * sizeof(uint32_t));
    if (e != cudaSuccess) return e;
    int sel = 0;
    for (int shift = 0; shift < bits; shift += 8) {
        const int nb = (bits - shift) < 8 ? (bits - shift) : 8;
        const uint32_t mask = (1u << nb) - 1u;
        k_sort_hist<<<ntiles, SORT_WARPS * 32, 0, s>>>(keys[sel], n, shift, mask, hist.as<uint32_t>(), ntiles); count_launch();
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        e = exclusive_scan_u32(hist.as<uint32_t>(), hist.as<uint32_t>(), hn, tmp, s);
        if (e != cudaSuccess) return e;
        k_sort_scatter<<<ntiles, SORT_WARPS * 32, 0, s>>>(keys[sel], vals[sel], keys[sel ^ 1], vals[sel ^ 1], n, shift, mask,
                                                         hist.as<uint32_t>(), ntiles); count_launch();
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        sel ^= 1;
    }
    *result_sel = sel;
    return cudaSuccess;
}

}  // namespace gs
