// sample_scatter.cu -- the PAPER'S OWN unstructured formulation (section 5.1, Fig. 7), as the second
// mode of a point query (gs_set_option(GS_OPT_POINTS_ACCEL, GS_POINTS_SCATTER)):
//   * the acceleration structure is built over the SAMPLE POSITIONS ("we construct a BVH over the sample positions", wide
//     leaves): the query points are Morton-sorted and an implicit 32-ary tree is laid over the sorted array --
//     leaf = SC_LEAF consecutive points, an inner node = 32 consecutive children -- with exact min/max boxes per level;
//   * forward: one WARP PER GAUSSIAN walks the tree with the Gaussian's cutoff AABB (Fig. 7B); the 32 children
//     of a node are tested by the 32 lanes at once; at a leaf every lane evaluates its points and adds (w G, v w G) to the
//     sample's accumulators with one vector atomic (red.global.add.v2.f32); a separate kernel normalises
//     and runs the fused loss epilogue S6;
//   * backward: the same walk, "each thread accumulates partial gradients locally before performing a warp-wide
//     reduction": 12 sums per lane, one transposing butterfly, one row written per Gaussian -- no atomics.
// Membership is decided by the canonical predicate (D4), so the ID sets are the ones of the gather mode, bit for bit.
// What differs from the paper: the tree is implicit over a Morton sort (no cuBQL), children are tested lane-parallel, and
// the ellipsoid is tested against a child's box in whitened space before descending (the Gaussian's AABB alone is loose
// for rotated needles).
#include "gs_internal.cuh"
#include "pair_math.cuh"
#include "f32x2.cuh"

namespace gs {

#ifndef GS_SCATTER_PPL
#define GS_SCATTER_PPL 2   // points per lane at a leaf (2: the pair rides in packed f32x2 registers)
#endif
constexpr int SC_PPL = GS_SCATTER_PPL;
constexpr int SC_WARPS = 4;
constexpr int SC_STACK = 7 * 32;   // entries per warp: at most 32 pushed per level, <= 7 levels

// sorted positions (float4: x y z 0; points past the end are NaN) -------------------------------------------------------
__global__ void __launch_bounds__(256) k_sc_sorted(const float *__restrict__ xyz, const uint32_t *__restrict__ order, uint64_t P,
                                                    uint64_t Ppad, float4 *__restrict__ spt) {
    const uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= Ppad) return;
    const float nanv = __int_as_float(0x7fc00000);
    float4 v = make_float4(nanv, nanv, nanv, 0.f);
    if (k < P) {
        const uint64_t c = order ? order[k] : k;
        v = make_float4(xyz[3 * c], xyz[3 * c + 1], xyz[3 * c + 2], 0.f);
    }
    spt[k] = v;
}

// boxes of one tree level, SoA: box[k * n + i], k = lo.xyz hi.xyz.  Level 0: warp per leaf over its points; level l > 0:
// warp per node over its <= 32 children.  fminf / fmaxf drop NaN (a leaf without real points keeps the empty box).
__global__ void __launch_bounds__(256) k_sc_level(const float4 *__restrict__ spt, const float *__restrict__ child, uint32_t nchild,
                                                   float *__restrict__ box, uint32_t n) {
    const uint32_t node = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (node >= n) return;
    const float inf = __int_as_float(0x7f800000);
    float lo[3] = {inf, inf, inf}, hi[3] = {-inf, -inf, -inf};
    if (spt) {
#pragma unroll
        for (int s = 0; s < SC_PPL; s++) {
            const float4 p = spt[(size_t)node * (32 * SC_PPL) + s * 32 + lane];
            lo[0] = fminf(lo[0], p.x); lo[1] = fminf(lo[1], p.y); lo[2] = fminf(lo[2], p.z);
            hi[0] = fmaxf(hi[0], p.x); hi[1] = fmaxf(hi[1], p.y); hi[2] = fmaxf(hi[2], p.z);
        }
    } else {
        const uint32_t c = node * 32u + lane;
        if (c < nchild) {
#pragma unroll
            for (int k = 0; k < 3; k++) { lo[k] = child[(size_t)k * nchild + c]; hi[k] = child[(size_t)(3 + k) * nchild + c]; }
        }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
#pragma unroll
        for (int k = 0; k < 3; k++) {
            lo[k] = fminf(lo[k], __shfl_xor_sync(0xffffffffu, lo[k], d));
            hi[k] = fmaxf(hi[k], __shfl_xor_sync(0xffffffffu, hi[k], d));
        }
    }
    if (lane < 3) box[(size_t)lane * n + node] = lo[lane];
    else if (lane < 6) box[(size_t)lane * n + node] = hi[lane - 3];
}

// Can the cutoff ellipsoid of the Gaussian reach the box [lo, hi]?  Conservative (the bound of the structured kernels and of
// k_points_cull): distance, in whitened space, to the box that bounds the whitened image of [lo, hi].
__device__ __forceinline__ bool sc_reaches(const float4 &ga, const float4 &gb, const float4 &gc, const float4 &gd, const float (&b)[6],
                                           float r2s) {
    const float cx = 0.5f * b[0] + 0.5f * b[3], cy = 0.5f * b[1] + 0.5f * b[4], cz = 0.5f * b[2] + 0.5f * b[5];
    const float hx = fmaxf(b[3] - cx, cx - b[0]) * 1.000001f, hy = fmaxf(b[4] - cy, cy - b[1]) * 1.000001f,
                hz = fmaxf(b[5] - cz, cz - b[2]) * 1.000001f;
    const float dx = cx - ga.x, dy = cy - ga.y, dz = cz - ga.z;
    const float u0 = fmaf(gb.z, dz, fmaf(gb.y, dy, gb.x * dx)), u1 = fmaf(gc.z, dz, fmaf(gc.y, dy, gc.x * dx)),
                u2 = fmaf(gd.z, dz, fmaf(gd.y, dy, gd.x * dx));
    const float e0 = fmaf(fabsf(gb.z), hz, fmaf(fabsf(gb.y), hy, fabsf(gb.x) * hx)), e1 = fmaf(fabsf(gc.z), hz, fmaf(fabsf(gc.y), hy, fabsf(gc.x) * hx)),
                e2 = fmaf(fabsf(gd.z), hz, fmaf(fabsf(gd.y), hy, fabsf(gd.x) * hx));
    const float v0 = fmaxf(fabsf(u0) - e0, 0.f), v1 = fmaxf(fabsf(u1) - e1, 0.f), v2 = fmaxf(fabsf(u2) - e2, 0.f);
    // an infinite box (a point at infinity) gives NaN / inf here: !(x > r2s) keeps it (conservative)
    return !(fmaf(v2, v2, fmaf(v1, v1, v0 * v0)) > r2s);
}

// The walk shared by forward and backward: calls leaf_fn(leaf index) for every leaf the Gaussian can reach.  All 32 lanes
// take part; `stack` is this warp's shared-memory stack.
template <class F>
__device__ __forceinline__ void sc_walk(const PtTree &T, const float4 &ga, const float4 &gb, const float4 &gc, const float4 &gd,
                                        const float (&bb)[6], float r2s, uint32_t *stack, int lane, F leaf_fn) {
    int sp = 0;
    int cl = T.levels - 1;            // level of the children tested next
    uint32_t cbase = 0, cnt = T.n[cl];   // the top level has <= 32 nodes: they are the children of a virtual root
    const uint32_t lt = (1u << lane) - 1u;
    while (true) {
        bool ov = false;
        const uint32_t c = cbase + lane;
        if ((uint32_t)lane < cnt) {
            const float *bx = T.box + T.off[cl];
            const uint32_t n = T.n[cl];
            float b[6];
#pragma unroll
            for (int k = 0; k < 6; k++) b[k] = __ldg(bx + (size_t)k * n + c);
            ov = (b[0] <= bb[3]) & (b[3] >= bb[0]) & (b[1] <= bb[4]) & (b[4] >= bb[1]) & (b[2] <= bb[5]) & (b[5] >= bb[2]);
            if (ov) ov = sc_reaches(ga, gb, gc, gd, b, r2s);
        }
        uint32_t m = __ballot_sync(0xffffffffu, ov);
        if (cl == 0) {
            while (m) {
                const int bit = __ffs((int)m) - 1;
                m &= m - 1u;
                leaf_fn(cbase + (uint32_t)bit);
            }
        } else if (m) {
            if (ov) stack[sp + __popc(m & lt)] = ((uint32_t)cl << 27) | c;
            sp += __popc(m);
            __syncwarp();
        }
        if (sp == 0) break;
        const uint32_t e = stack[--sp];
        __syncwarp();
        cl = (int)(e >> 27) - 1;
        cbase = (e & 0x07ffffffu) * 32u;
        cnt = min(32u, T.n[cl] - cbase);
    }
}

__device__ __forceinline__ void red_add_v2(float *addr, float a, float b) {
    asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(addr), "f"(a), "f"(b) : "memory");
}

// ---- forward: warp per Gaussian, atomics into the samples ------------------------------------------------
template <bool SETS>
__global__ void __launch_bounds__(SC_WARPS * 32) k_sc_fwd(const float4 *__restrict__ rec, const float *__restrict__ aabb,
                                                          const uint32_t *__restrict__ gorder, uint32_t N, const __grid_constant__ PtTree T,
                                                          const float4 *__restrict__ spt, float2 *__restrict__ acc, float r2, float r2s,
                                                          const uint32_t *__restrict__ pt_order, uint64_t P, FwdOut o) {
    __shared__ uint32_t stack_all[SC_WARPS][SC_STACK];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    uint32_t *stack = stack_all[warp];
    const uint32_t nw = gridDim.x * SC_WARPS;
    for (uint32_t g = blockIdx.x * SC_WARPS + warp; g < N; g += nw) {
        const uint32_t i = gorder[g];
        const float4 ga = __ldg(rec + i), gb = __ldg(rec + (size_t)N + i), gc = __ldg(rec + 2 * (size_t)N + i), gd = __ldg(rec + 3 * (size_t)N + i);
        if (ga.x != ga.x) continue;   // invalid Gaussian (NaN mean): empty support
        float bb[6];
#pragma unroll
        for (int k = 0; k < 6; k++) bb[k] = __ldg(aabb + 6 * (size_t)i + k);
        unsigned long long hid = 0;
        if (SETS) hid = mix64(i);
        sc_walk(T, ga, gb, gc, gd, bb, r2s, stack, lane, [&](uint32_t leaf) {
            const size_t k0 = (size_t)leaf * (32 * SC_PPL) + (size_t)lane * SC_PPL;   // this lane's points are neighbours in memory
            bool hit[SC_PPL];
            float G[SC_PPL];
            if constexpr (SC_PPL == 2) {
                const float4 p0 = __ldg(spt + k0), p1 = __ldg(spt + k0 + 1);
                f2 u0, u1, u2;
                const f2 qd = mahalanobis2(ga.x, ga.y, ga.z, gb.x, gb.y, gb.z, gc.x, gc.y, gc.z, gd.x, gd.y, gd.z, pk(p0.x, p1.x), pk(p0.y, p1.y),
                                           pk(p0.z, p1.z), u0, u1, u2);
                upk(gauss_weight2(qd, r2, hit[0], hit[SC_PPL - 1]), G[0], G[SC_PPL - 1]);
            } else {
                const float4 p0 = __ldg(spt + k0);
                Rec q{ga, gb, gc, gd};
                float u0, u1, u2;
                const float qd = mahalanobis(q, p0.x, p0.y, p0.z, u0, u1, u2);
                hit[0] = qd <= r2;
                G[0] = gauss_weight(qd);
            }
#pragma unroll
            for (int s = 0; s < SC_PPL; s++) {
                if (hit[s]) {
                    red_add_v2(reinterpret_cast<float *>(acc + k0 + s), ga.w * G[s], gd.w * G[s]);   // gd.w = v w
                    if (SETS) {
                        const uint64_t c = pt_order ? pt_order[k0 + s] : k0 + s;
                        if (o.set_count) atomicAdd(o.set_count + c, 1u);
                        if (o.set_sum) atomicAdd(o.set_sum + c, hid);
                        if (o.set_xor) atomicXor(o.set_xor + c, hid);
                    }
                }
            }
            if (SETS && o.counters && lane == 0) atomicAdd(o.counters, 32ull * SC_PPL);   // pairs tested (padding included)
        });
    }
}

// ---- normalise + S6 epilogue ("a separate kernel to normalize the samples") -------------------------------
__global__ void __launch_bounds__(256) k_sc_norm(const float2 *__restrict__ acc, const uint32_t *__restrict__ pt_order, uint64_t P, float tau,
                                                  FwdOut o, double invP, const uint32_t *__restrict__ set_count_for_hits) {
    const uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    const bool active = k < P;
    float res2 = 0.f;
    LossPartial lp;
    unsigned long long hits = 0;
    if (active) {
        const uint64_t c = pt_order ? pt_order[k] : k;
        const float2 a = acc[k];
        const float I = a.x;
        const bool covered = I > tau;
        const float phi = covered ? __fdividef(a.y, I) : 0.f;
        o.phi[c] = phi;
        o.I[c] = I;
        if (o.gen.on) {
            loss_sample(o.gen, c, phi, I, covered, tau, o.target, o.dL_dphi, o.sample_err, lp);
        } else if (o.target) {
            const float res = phi - o.target[c];
            res2 = res * res;
            if (o.dL_dphi) o.dL_dphi[c] = covered ? (float)(2.0 * invP) * res : 0.f;
            if (o.sample_err) o.sample_err[c] = fabsf(res);
            if (o.pack2) {
                const float al = covered ? __fdividef((float)(2.0 * invP) * res, I) : 0.f;
                o.pack2[k] = make_float2(al, -al * phi);   // sorted order, as in gather mode
            }
        }
        if (set_count_for_hits) hits = set_count_for_hits[c];
    }
    if (o.gen.on) loss_flush(o.gen, lp, lane);
    if (!o.gen.on && o.target && o.loss) {
        double s = (double)res2;
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
        if (lane == 0 && s != 0.0) atomicAdd(o.loss, s * invP);
    }
    if (set_count_for_hits && o.counters) {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) hits += __shfl_xor_sync(0xffffffffu, hits, d);
        if (lane == 0 && hits) atomicAdd(o.counters + 1, hits);
    }
}

// ---- backward ------------------------------------------------------------------------------------------------------------
// per sorted point: position and the backward coefficients (alpha, beta, eps), 32 bytes.  A point that lies in no support
// (past the end, NaN / infinite) gets a harmless finite position and zero coefficients (the packed accumulation is unconditional).
__global__ void __launch_bounds__(256) k_sc_coef(const float4 *__restrict__ spt, const uint32_t *__restrict__ pt_order, uint64_t P,
                                                  uint64_t Ppad, float tau, BwdIn in, float4 *__restrict__ coef) {
    const uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= Ppad) return;
    float4 p = spt[k];
    float alpha = 0.f, beta = 0.f, eps = 0.f;
    const bool ok = k < P && fabsf(p.x) <= 3.402823466e38f && fabsf(p.y) <= 3.402823466e38f && fabsf(p.z) <= 3.402823466e38f;
    if (ok) {
        const uint64_t c = pt_order ? pt_order[k] : k;
        if (in.pack2) {  // fused MSE: eps = |res| / I = |alpha| * P / 2
            const float2 s = __ldg(in.pack2 + k);
            alpha = s.x; beta = s.y; eps = fabsf(s.x) * in.eps_scale;
        } else {
            const float Ic = in.I[c], ph = in.phi[c];
            const bool covered = Ic > tau;
            const float inv = covered ? 1.0f / Ic : 0.f;
            alpha = covered ? in.dL_dphi[c] * inv : 0.f;
            beta = (in.dL_dI ? in.dL_dI[c] : 0.f) - alpha * ph;
            eps = (covered && in.target) ? fabsf(ph - in.target[c]) * inv : 0.f;
        }
    } else {
        p = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    coef[2 * k] = make_float4(p.x, p.y, p.z, alpha);
    coef[2 * k + 1] = make_float4(beta, eps, 0.f, 0.f);
}

// warp-wide sums of 16 values: afterwards lane L (and L + 16) holds the sum of component L & 15 in v[0] (16 SHFL)
__device__ __forceinline__ void warp_reduce16(float (&v)[16], int lane) {
#pragma unroll
    for (int h = 8; h >= 1; h >>= 1) {
        const bool up = lane & h;
#pragma unroll
        for (int k = 0; k < h; k++) {
            const float send = up ? v[k] : v[k + h];
            const float keep = up ? v[k + h] : v[k];
            v[k] = keep + __shfl_xor_sync(0xffffffffu, send, h);
        }
    }
    v[0] += __shfl_xor_sync(0xffffffffu, v[0], 16);
}

__global__ void __launch_bounds__(SC_WARPS * 32) k_sc_bwd(const float4 *__restrict__ rec, const float *__restrict__ aabb,
                                                          const uint32_t *__restrict__ gorder, uint32_t N, const __grid_constant__ PtTree T,
                                                          const float4 *__restrict__ coef, float r2, float r2s, float *__restrict__ gacc) {
    __shared__ uint32_t stack_all[SC_WARPS][SC_STACK];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    uint32_t *stack = stack_all[warp];
    const uint32_t nw = gridDim.x * SC_WARPS;
    for (uint32_t g = blockIdx.x * SC_WARPS + warp; g < N; g += nw) {
        const uint32_t i = gorder[g];
        const float4 ga = __ldg(rec + i), gb = __ldg(rec + (size_t)N + i), gc = __ldg(rec + 2 * (size_t)N + i), gd = __ldg(rec + 3 * (size_t)N + i);
        if (ga.x != ga.x) {   // invalid Gaussian: zero row (rows are not pre-zeroed)
            if (lane < GACC) gacc[(size_t)i * GACC + lane] = 0.f;
            continue;
        }
        float bb[6];
#pragma unroll
        for (int k = 0; k < 6; k++) bb[k] = __ldg(aabb + 6 * (size_t)i + k);
        f2 acc[12];
#pragma unroll
        for (int q = 0; q < 12; q++) acc[q] = pk(0.f, 0.f);
        const f2 w2 = bc(ga.w), v2 = bc(gb.w);
        sc_walk(T, ga, gb, gc, gd, bb, r2s, stack, lane, [&](uint32_t leaf) {
            const size_t k0 = (size_t)leaf * (32 * SC_PPL) + (size_t)lane * SC_PPL;
            const float4 a0 = __ldg(coef + 2 * k0), b0 = __ldg(coef + 2 * k0 + 1);
            const float4 a1 = SC_PPL == 2 ? __ldg(coef + 2 * k0 + 2) : make_float4(0.f, 0.f, 0.f, 0.f);
            const float4 b1 = SC_PPL == 2 ? __ldg(coef + 2 * k0 + 3) : make_float4(0.f, 0.f, 0.f, 0.f);
            f2 u0, u1, u2;
            const f2 qd = mahalanobis2(ga.x, ga.y, ga.z, gb.x, gb.y, gb.z, gc.x, gc.y, gc.z, gd.x, gd.y, gd.z, pk(a0.x, a1.x), pk(a0.y, a1.y),
                                       pk(a0.z, a1.z), u0, u1, u2);
            bool h0, h1;
            const f2 G = gauss_weight2(qd, r2, h0, h1);
            const f2 alpha = pk(a0.w, a1.w), beta = pk(b0.x, b1.x), eps = pk(b0.y, b1.y);
            const f2 wG = mul2(w2, G);
            const f2 gamma = fma2(alpha, v2, beta);
            const f2 t = mul2(gamma, wG);
            acc[0] = fma2(alpha, wG, acc[0]);
            acc[1] = fma2(gamma, G, acc[1]);
            const f2 t0 = mul2(t, u0), t1 = mul2(t, u1), t2 = mul2(t, u2);
            acc[2] = add2(acc[2], t0); acc[3] = add2(acc[3], t1); acc[4] = add2(acc[4], t2);
            acc[5] = fma2(t0, u0, acc[5]); acc[6] = fma2(t0, u1, acc[6]); acc[7] = fma2(t0, u2, acc[7]);
            acc[8] = fma2(t1, u1, acc[8]); acc[9] = fma2(t1, u2, acc[9]); acc[10] = fma2(t2, u2, acc[10]);
            acc[11] = fma2(eps, wG, acc[11]);
        });
        float s[16];
#pragma unroll
        for (int q = 0; q < 12; q++) s[q] = lo(acc[q]) + hi(acc[q]);
#pragma unroll
        for (int q = 12; q < 16; q++) s[q] = 0.f;
        warp_reduce16(s, lane);
        if (lane < GACC) gacc[(size_t)i * GACC + lane] = s[0];   // one row per Gaussian, written once: no atomics
        __syncwarp();
    }
}

// ---- launchers -----------------------------------------------------------------------------------------------------------
uint64_t scatter_padded_points(uint64_t P) { return (P + 63) / 64 * 64; }   // whole leaves (32 * SC_PPL <= 64) and whole packets
static_assert(64 % (32 * SC_PPL) == 0, "leaf size");

// number of tree levels and nodes per level for P points; returns the total node count
uint32_t scatter_tree_shape(uint64_t P, PtTree *T) {
    uint64_t n = scatter_padded_points(P) / (32 * SC_PPL);
    if (n == 0) n = 1;
    uint32_t off = 0;
    int l = 0;
    for (;; l++) {
        T->n[l] = (uint32_t)n;
        T->off[l] = off * 6;
        off += (uint32_t)n;
        if (n <= 32) break;
        n = (n + 31) / 32;
    }
    T->levels = l + 1;
    return off;
}

cudaError_t launch_sorted_points(const float *xyz, const uint32_t *pt_order, uint64_t P, float4 *spt, cudaStream_t s) {
    const uint64_t Ppad = scatter_padded_points(P ? P : 1);
    k_sc_sorted<<<(unsigned)((Ppad + 255) / 256), 256, 0, s>>>(xyz, pt_order, P, Ppad, spt); count_launch();
    return cudaGetLastError();
}

cudaError_t launch_scatter_build(uint64_t P, PtTree T, const float4 *spt, float *box, cudaStream_t s) {
    for (int l = 0; l < T.levels; l++) {
        const uint32_t n = T.n[l];
        k_sc_level<<<(unsigned)(((size_t)n * 32 + 255) / 256), 256, 0, s>>>(l == 0 ? spt : nullptr, l ? box + T.off[l - 1] : nullptr, l ? T.n[l - 1] : 0u,
                                                                            box + T.off[l], n);
        count_launch();
    }
    return cudaGetLastError();
}

static unsigned sc_blocks(uint32_t N) {
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const unsigned want = (N + SC_WARPS - 1) / SC_WARPS;
    const unsigned cap = (unsigned)sms * 64;   // grid-stride: the resident warps take the Gaussians in Morton order
    return want < cap ? (want ? want : 1u) : cap;
}

cudaError_t launch_scatter_fwd(const float4 *rec, const float *aabb, const uint32_t *gorder, uint32_t N, const PtTree &T, const float4 *spt,
                               float2 *acc, const uint32_t *pt_order, uint64_t P, float tau, float r2, const FwdOut &o, cudaStream_t s) {
    if (P == 0) return cudaSuccess;
    const uint64_t Ppad = scatter_padded_points(P);
    cudaError_t e = cudaMemsetAsync(acc, 0, Ppad * sizeof(float2), s);
    if (e != cudaSuccess) return e;
    const bool sets = o.set_count || o.set_sum || o.set_xor || o.counters;
    const float r2s = r2 * 1.001953125f;
    if (sets) {   // the debug sets are accumulated with atomics on the caller's arrays
        if (o.set_count && (e = cudaMemsetAsync(o.set_count, 0, P * 4, s)) != cudaSuccess) return e;
        if (o.set_sum && (e = cudaMemsetAsync(o.set_sum, 0, P * 8, s)) != cudaSuccess) return e;
        if (o.set_xor && (e = cudaMemsetAsync(o.set_xor, 0, P * 8, s)) != cudaSuccess) return e;
    }
    if (N) {
        if (sets) k_sc_fwd<true><<<sc_blocks(N), SC_WARPS * 32, 0, s>>>(rec, aabb, gorder, N, T, spt, acc, r2, r2s, pt_order, P, o);
        else k_sc_fwd<false><<<sc_blocks(N), SC_WARPS * 32, 0, s>>>(rec, aabb, gorder, N, T, spt, acc, r2, r2s, pt_order, P, o);
        count_launch();
    }
    const double invP = o.inv_count > 0.0 ? o.inv_count : 1.0 / (double)P;
    k_sc_norm<<<(unsigned)((P + 255) / 256), 256, 0, s>>>(acc, pt_order, P, tau, o, invP, sets ? o.set_count : nullptr); count_launch();
    return cudaGetLastError();
}

cudaError_t launch_scatter_bwd(const float4 *rec, const float *aabb, const uint32_t *gorder, uint32_t N, const PtTree &T, const float4 *spt,
                               float4 *coef, const uint32_t *pt_order, uint64_t P, float tau, float r2, const BwdIn &in, float *gacc,
                               cudaStream_t s) {
    if (N == 0) return cudaSuccess;
    const uint64_t Ppad = scatter_padded_points(P ? P : 1);
    k_sc_coef<<<(unsigned)((Ppad + 255) / 256), 256, 0, s>>>(spt, pt_order, P, Ppad, tau, in, coef); count_launch();
    k_sc_bwd<<<sc_blocks(N), SC_WARPS * 32, 0, s>>>(rec, aabb, gorder, N, T, coef, r2, r2 * 1.001953125f, gacc); count_launch();
    return cudaGetLastError();
}

}  // namespace gs
