// lbvh.cu -- S3: LBVH over the Gaussians' cutoff AABBs, rebuilt every step (north_star (2)).
// The paper builds a BVH over the sample positions with cuBQL and queries it per Gaussian
// (PAPER.md:184-190); north_star fixes the opposite direction (per-point traversal), see DESIGN.md.
//   k_morton      : 30-bit Morton code of a position inside the domain box (D8), x in the low bit
//   (radix sort)  : stable sort of (code, id) => order by the unique 64-bit key (code << 32 | id)
//   k_karras      : binary radix tree, one thread per internal node (Karras 2012)
//   k_refit       : bottom-up exact min/max boxes with per-node arrival counters; the thread that completes a node also
//                   writes its 64-byte traversal record (both children's boxes and links)
//   k_sort_records: the Gaussian records in leaf order, 64 contiguous bytes each (neighbouring leaves are
//                   neighbouring in memory; a record is two full 32-byte sectors)
#include "gs_internal.cuh"

namespace gs {

__global__ void __launch_bounds__(256) k_morton(const float *__restrict__ xyz, int stride, int nan_is_invalid, size_t n, MortonParams mp,
                                                 uint32_t *__restrict__ codes, uint32_t *__restrict__ ids) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float x = xyz[i * stride], y = xyz[i * stride + 1], z = xyz[i * stride + 2];
    uint32_t code;
    if (nan_is_invalid && x != x) {
        code = 1u << 30;  // invalid Gaussians sort to the end
    } else {
        // D8: q = (int) min(max((x - lo) * scale, 0), 1023), truncation
        code = morton30(x, y, z, mp);
    }
    codes[i] = code;
    ids[i] = (uint32_t)i;
}

cudaError_t launch_morton(const float *xyz, size_t stride_floats, const float *nan_invalid, size_t n, const gs_domain &dom,
                          uint32_t *codes, uint32_t *ids, cudaStream_t s) {
    if (n == 0) return cudaSuccess;
    const MortonParams mp = morton_params(dom);
    k_morton<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(xyz, (int)stride_floats, nan_invalid != nullptr, n, mp, codes, ids); count_launch();
    return cudaGetLastError();
}

// common-prefix length of the 64-bit keys at sorted positions i and j; -1 outside [0, n)
__device__ __forceinline__ int delta(const uint32_t *__restrict__ codes, const uint32_t *__restrict__ ids, int n, int i, int j) {
    if (j < 0 || j >= n) return -1;
    const unsigned long long a = ((unsigned long long)codes[i] << 32) | ids[i];
    const unsigned long long b = ((unsigned long long)codes[j] << 32) | ids[j];
    return __clzll((long long)(a ^ b));  // keys are unique, so a ^ b != 0
}

__global__ void __launch_bounds__(256) k_karras(const uint32_t *__restrict__ codes, const uint32_t *__restrict__ ids, int n,
                                                 int32_t *__restrict__ left, int32_t *__restrict__ right, int32_t *__restrict__ parent,
                                                 int32_t *__restrict__ leaf_parent) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n - 1) return;
    const int d = (delta(codes, ids, n, i, i + 1) - delta(codes, ids, n, i, i - 1)) >= 0 ? 1 : -1;
    const int dmin = delta(codes, ids, n, i, i - d);
    int lmax = 2;
    while (delta(codes, ids, n, i, i + lmax * d) > dmin) lmax <<= 1;
    int l = 0;
    for (int t = lmax >> 1; t >= 1; t >>= 1)
        if (delta(codes, ids, n, i, i + (l + t) * d) > dmin) l += t;
    const int j = i + l * d;
    const int dnode = delta(codes, ids, n, i, j);
    int s = 0;
    for (int t = (l + 1) >> 1;; t = (t + 1) >> 1) {
        if (delta(codes, ids, n, i, i + (s + t) * d) > dnode) s += t;
        if (t == 1) break;
    }
    const int gamma = i + s * d + min(d, 0);
    const int lo = min(i, j), hi = max(i, j);
    if (lo == gamma) { left[i] = ~gamma; leaf_parent[gamma] = i; }
    else { left[i] = gamma; parent[gamma] = i; }
    if (hi == gamma + 1) { right[i] = ~(gamma + 1); leaf_parent[gamma + 1] = i; }
    else { right[i] = gamma + 1; parent[gamma + 1] = i; }
    if (i == 0) parent[0] = -1;
}

// a 24-byte box is 8-byte aligned: three 8-byte loads / stores (L2: written by other threads of this launch)
__device__ __forceinline__ void load_box(const float *p, float (&b)[6]) {
    const float2 *q = reinterpret_cast<const float2 *>(p);
    const float2 a0 = __ldcg(q), a1 = __ldcg(q + 1), a2 = __ldcg(q + 2);
    b[0] = a0.x; b[1] = a0.y; b[2] = a1.x; b[3] = a1.y; b[4] = a2.x; b[5] = a2.y;
}

// Bottom-up refit: the thread that arrives second at a node has both children complete; it unites their boxes, writes the
// node's box (read by the parent and by the debug view) AND the node's 64-byte traversal record:
//   [0] l.lo.xyz l.hi.x | [1] l.hi.yz r.lo.xy | [2] r.lo.z r.hi.xyz | [3] left, right (bits), -, -
// child link >= 0: internal node; < 0: ~(sorted position of the leaf), which indexes the sorted records directly
__global__ void __launch_bounds__(256) k_refit(const uint32_t *__restrict__ ids, const float *__restrict__ aabb, int n,
                                                const int32_t *__restrict__ left, const int32_t *__restrict__ right,
                                                const int32_t *__restrict__ parent, const int32_t *__restrict__ leaf_parent,
                                                float *__restrict__ node_aabb, uint32_t *__restrict__ flags, float4 *__restrict__ packed) {
    const int leaf = blockIdx.x * blockDim.x + threadIdx.x;
    if (leaf >= n) return;
    int node = leaf_parent[leaf];
    // the thread carries the box of the subtree it has finished in registers: at a node only the SIBLING's box is loaded
    float mine[6];
    load_box(aabb + 6 * (size_t)ids[leaf], mine);
    int from = ~leaf;   // the child link under which the parent knows this subtree
    while (node >= 0) {
        if (atomicAdd(&flags[node], 1u) == 0u) return;  // first arrival: the sibling subtree is not done yet
        __threadfence();
        const int l = left[node], r = right[node];
        const bool am_left = l == from;
        const int sib = am_left ? r : l;
        float other[6], a[6], b[6];
        load_box(sib < 0 ? aabb + 6 * (size_t)ids[~sib] : node_aabb + 6 * (size_t)sib, other);
#pragma unroll
        for (int k = 0; k < 6; k++) { a[k] = am_left ? mine[k] : other[k]; b[k] = am_left ? other[k] : mine[k]; }
#pragma unroll
        for (int k = 0; k < 3; k++) { mine[k] = fminf(a[k], b[k]); mine[3 + k] = fmaxf(a[3 + k], b[3 + k]); }
        float2 *out = reinterpret_cast<float2 *>(node_aabb + 6 * (size_t)node);
        __stcg(out, make_float2(mine[0], mine[1]));
        __stcg(out + 1, make_float2(mine[2], mine[3]));
        __stcg(out + 2, make_float2(mine[4], mine[5]));
        packed[4 * (size_t)node + 0] = make_float4(a[0], a[1], a[2], a[3]);
        packed[4 * (size_t)node + 1] = make_float4(a[4], a[5], b[0], b[1]);
        packed[4 * (size_t)node + 2] = make_float4(b[2], b[3], b[4], b[5]);
        packed[4 * (size_t)node + 3] = make_float4(__int_as_float(l), __int_as_float(r), 0.f, 0.f);
        __threadfence();
        from = node;
        node = parent[node];
    }
}

// records in leaf order: sorted[4 k .. 4 k + 3] = planes a, b, c, d of Gaussian ids[k], with the id in c.w
__global__ void __launch_bounds__(256) k_sort_records(const uint32_t *__restrict__ ids, const float4 *__restrict__ rec, uint32_t N,
                                                       float4 *__restrict__ sorted) {
    const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;   // one thread per (leaf, plane): coalesced 16-byte stores
    const uint32_t k = t >> 2, plane = t & 3u;
    if (k >= N) return;
    const uint32_t id = ids[k];
    float4 v = __ldg(rec + (size_t)plane * N + id);
    if (plane == 2u) v.w = __uint_as_float(id);
    sorted[t] = v;
}

cudaError_t launch_lbvh(const uint32_t *codes, const uint32_t *ids, const float *aabb, const float4 *rec, uint32_t N, int32_t *left,
                        int32_t *right, int32_t *parent, int32_t *leaf_parent, float *node_aabb, uint32_t *flags, float4 *packed,
                        float4 *sorted_rec, cudaStream_t s) {
    if (N >= 1) { k_sort_records<<<(unsigned)(((size_t)N * 4 + 255) / 256), 256, 0, s>>>(ids, rec, N, sorted_rec); count_launch(); }
    if (N < 2) {
        if (N == 1) return cudaMemsetAsync(leaf_parent, 0xff, sizeof(int32_t), s);
        return cudaSuccess;
    }
    const int n = (int)N;
    cudaError_t e = cudaMemsetAsync(flags, 0, sizeof(uint32_t) * (N - 1), s);
    if (e != cudaSuccess) return e;
    k_karras<<<(n - 1 + 255) / 256, 256, 0, s>>>(codes, ids, n, left, right, parent, leaf_parent); count_launch();
    k_refit<<<(n + 255) / 256, 256, 0, s>>>(ids, aabb, n, left, right, parent, leaf_parent, node_aabb, flags, packed); count_launch();
    return cudaGetLastError();
}

}  // namespace gs
