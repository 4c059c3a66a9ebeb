// sample_points.cu -- unstructured sampling kernels (S5 forward, S7 backward; section 5.1.2).
// A warp is a packet of 32 consecutive points of the coherence-sorted order.  The packet walks the
// LBVH over the Gaussians with one shared short stack (shared memory): a child is entered when ANY
// lane's point lies in its box; at a leaf every lane evaluates the canonical predicate for its own
// point.  Forward: per-lane accumulation of I and sum v w G, fused epilogue S6.  Backward: the
// weights are recomputed, per-lane partial sums are reduced across the packet with the
// transposing butterfly and added to the Gaussian's accumulator with one reduction instruction
// per warp (the paper's unstructured backward also ends in a warp-wide reduction).
#include "gs_internal.cuh"
#include "pair_math.cuh"

namespace gs {

constexpr int PT_WARPS = 8;
constexpr int STACK = 64;

__device__ __forceinline__ bool in_box(float px, float py, float pz, float lx, float ly, float lz, float hx, float hy, float hz) {
    return px >= lx && px <= hx && py >= ly && py <= hy && pz >= lz && pz <= hz;
}

__device__ __forceinline__ Rec load_rec(const float4 *__restrict__ rec, uint32_t N, uint32_t id) {
    Rec g;
    g.a = __ldg(rec + id); g.b = __ldg(rec + (size_t)N + id); g.c = __ldg(rec + 2 * (size_t)N + id); g.d = __ldg(rec + 3 * (size_t)N + id);
    return g;
}

// Generic packet traversal: calls leaf(gaussian_id) warp-uniformly for every leaf whose box holds a lane's point.
template <class LeafFn>
__device__ __forceinline__ void traverse(const float4 *__restrict__ nodes, uint32_t N, float px, float py, float pz, int32_t *stack,
                                         uint32_t *overflow, LeafFn leaf) {
    if (N == 0) return;
    if (N == 1) { leaf(0u); return; }
    int sp = 0;
    int32_t node = 0;
    while (true) {
        const float4 n0 = __ldg(nodes + 4 * (size_t)node), n1 = __ldg(nodes + 4 * (size_t)node + 1),
                     n2 = __ldg(nodes + 4 * (size_t)node + 2), n3 = __ldg(nodes + 4 * (size_t)node + 3);
        const bool inl = in_box(px, py, pz, n0.x, n0.y, n0.z, n0.w, n1.x, n1.y);
        const bool inr = in_box(px, py, pz, n1.z, n1.w, n2.x, n2.y, n2.z, n2.w);
        const bool gol = __any_sync(0xffffffffu, inl), gor = __any_sync(0xffffffffu, inr);
        const int32_t lc = __float_as_int(n3.x), rc = __float_as_int(n3.y);
        int32_t next = -1;
        bool have_next = false;
        if (gol) {
            if (lc < 0) leaf((uint32_t)~lc);
            else { next = lc; have_next = true; }
        }
        if (gor) {
            if (rc < 0) leaf((uint32_t)~rc);
            else if (have_next) {
                if (sp < STACK) { if ((threadIdx.x & 31) == 0) stack[sp] = rc; sp++; }
                else if ((threadIdx.x & 31) == 0) *overflow = 1u;
            } else { next = rc; have_next = true; }
        }
        if (!have_next) {
            if (sp == 0) break;
            sp--;
            __syncwarp();
            next = stack[sp];
        }
        __syncwarp();
        node = next;
    }
}

template <bool SETS>
__global__ void __launch_bounds__(PT_WARPS * 32) k_points_fwd(const float4 *__restrict__ rec, uint32_t N, const float4 *__restrict__ nodes,
                                                               const float *__restrict__ xyz, const uint32_t *__restrict__ pt_order,
                                                               uint64_t P, float tau, float r2, FwdOut o, double invP,
                                                               uint32_t *__restrict__ overflow) {
    __shared__ int32_t stacks[PT_WARPS][STACK];
    __shared__ double red[PT_WARPS];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint64_t k = ((uint64_t)blockIdx.x * PT_WARPS + warp) * 32 + lane;
    const bool active = k < P;
    const uint64_t c = active ? (pt_order ? (uint64_t)pt_order[k] : k) : 0;
    const float nanv = __int_as_float(0x7fc00000);
    const float px = active ? xyz[3 * c] : nanv, py = active ? xyz[3 * c + 1] : nanv, pz = active ? xyz[3 * c + 2] : nanv;
    float I = 0.f, Nacc = 0.f;
    uint32_t cnt = 0, tested = 0;
    unsigned long long hsum = 0, hxor = 0;
    traverse(nodes, N, px, py, pz, stacks[warp], overflow, [&](uint32_t id) {
        const Rec g = load_rec(rec, N, id);
        float u0, u1, u2;
        const float qd = mahalanobis(g, px, py, pz, u0, u1, u2);
        if (SETS) tested++;
        if (qd <= r2) {
            const float wG = g.a.w * gauss_weight(qd);
            I += wG;
            Nacc = fmaf(g.b.w, wG, Nacc);
            if (SETS) { const unsigned long long h = mix64(id); cnt++; hsum += h; hxor ^= h; }
        }
    });
    const bool covered = I > tau;
    const float phi = covered ? __fdividef(Nacc, I) : 0.f;
    float res2 = 0.f;
    if (active) {
        o.phi[c] = phi;
        o.I[c] = I;
        if (o.target) {
            const float res = phi - o.target[c];
            res2 = res * res;
            if (o.dL_dphi) o.dL_dphi[c] = covered ? (float)(2.0 * invP) * res : 0.f;
            if (o.sample_err) o.sample_err[c] = fabsf(res);
            if (o.pack2) {
                const float al = covered ? __fdividef((float)(2.0 * invP) * res, I) : 0.f;
                o.pack2[c] = make_float2(al, -al * phi);
            }
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
        if (lane == 0) red[warp] = s;
        __syncthreads();
        if (threadIdx.x == 0) {
            double v = 0.0;
            for (int w = 0; w < PT_WARPS; w++) v += red[w];
            if (v != 0.0) atomicAdd(o.loss, v * invP);
        }
    }
    if (SETS && o.counters) {
        unsigned long long t = active ? tested : 0, h = cnt;
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) { t += __shfl_xor_sync(0xffffffffu, t, d); h += __shfl_xor_sync(0xffffffffu, h, d); }
        if (lane == 0) { atomicAdd(o.counters, t); atomicAdd(o.counters + 1, h); }
    }
}

__global__ void __launch_bounds__(PT_WARPS * 32) k_points_bwd(const float4 *__restrict__ rec, uint32_t N, const float4 *__restrict__ nodes,
                                                               const float *__restrict__ xyz, const uint32_t *__restrict__ pt_order,
                                                               uint64_t P, float tau, float r2, BwdIn in, float *__restrict__ gacc,
                                                               uint32_t *__restrict__ overflow) {
    __shared__ int32_t stacks[PT_WARPS][STACK];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint64_t k = ((uint64_t)blockIdx.x * PT_WARPS + warp) * 32 + lane;
    const bool active = k < P;
    const uint64_t c = active ? (pt_order ? (uint64_t)pt_order[k] : k) : 0;
    const float nanv = __int_as_float(0x7fc00000);
    const float px = active ? xyz[3 * c] : nanv, py = active ? xyz[3 * c + 1] : nanv, pz = active ? xyz[3 * c + 2] : nanv;
    // per-sample coefficients: alpha = covered ? a/I : 0, beta = b - alpha Phi, eps = covered ? |Phi - t|/I : 0
    float alpha = 0.f, beta = 0.f, eps = 0.f;
    if (active && in.pack2) {  // fused MSE: eps = |res| / I = |alpha| * P / 2
        const float2 s = __ldg(in.pack2 + c);
        alpha = s.x; beta = s.y; eps = fabsf(s.x) * in.eps_scale;
    } else if (active) {
        const float Ic = in.I[c], ph = in.phi[c];
        const bool covered = Ic > tau;
        const float inv = covered ? 1.0f / Ic : 0.f;
        alpha = covered ? in.dL_dphi[c] * inv : 0.f;
        beta = (in.dL_dI ? in.dL_dI[c] : 0.f) - alpha * ph;
        eps = (covered && in.target) ? fabsf(ph - in.target[c]) * inv : 0.f;
    }
    traverse(nodes, N, px, py, pz, stacks[warp], overflow, [&](uint32_t id) {
        const Rec g = load_rec(rec, N, id);
        float u0, u1, u2;
        const float qd = mahalanobis(g, px, py, pz, u0, u1, u2);
        const bool hit = qd <= r2;
        if (!__any_sync(0xffffffffu, hit)) return;
        float acc[16];
#pragma unroll
        for (int q = 0; q < 16; q++) acc[q] = 0.f;
        if (hit) bwd_accumulate(acc, alpha, beta, eps, g.a.w, g.b.w, gauss_weight(qd), u0, u1, u2);
        warp_reduce16(acc, lane);
        const float val = __shfl_sync(0xffffffffu, acc[0], (lane & 15) * 2);
        if (lane < 12) atomicAdd(gacc + (size_t)id * GACC + lane, val);
    });
}

cudaError_t launch_points_fwd(const float4 *rec, uint32_t N, const float4 *nodes, const uint32_t *leaf_order, const float *xyz,
                              const uint32_t *pt_order, uint64_t P, float tau, float r2, const FwdOut &o, uint32_t *overflow,
                              cudaStream_t s) {
    (void)leaf_order;
    if (P == 0) return cudaSuccess;
    const unsigned blocks = (unsigned)((P + PT_WARPS * 32 - 1) / (PT_WARPS * 32));
    const bool sets = o.set_count || o.set_sum || o.set_xor || o.counters;
    if (sets) k_points_fwd<true><<<blocks, PT_WARPS * 32, 0, s>>>(rec, N, nodes, xyz, pt_order, P, tau, r2, o, 1.0 / (double)P, overflow);
    else k_points_fwd<false><<<blocks, PT_WARPS * 32, 0, s>>>(rec, N, nodes, xyz, pt_order, P, tau, r2, o, 1.0 / (double)P, overflow);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_points_bwd(const float4 *rec, uint32_t N, const float4 *nodes, const uint32_t *leaf_order, const float *xyz,
                              const uint32_t *pt_order, uint64_t P, float tau, float r2, const BwdIn &in, float *gacc,
                              uint32_t *overflow, cudaStream_t s) {
    (void)leaf_order;
    if (P == 0) return cudaSuccess;
    const unsigned blocks = (unsigned)((P + PT_WARPS * 32 - 1) / (PT_WARPS * 32));
    k_points_bwd<<<blocks, PT_WARPS * 32, 0, s>>>(rec, N, nodes, xyz, pt_order, P, tau, r2, in, gacc, overflow); count_launch();
    return cudaGetLastError();
}

}  // namespace gs
