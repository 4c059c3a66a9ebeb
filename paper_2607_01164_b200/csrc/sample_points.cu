// sample_points.cu -- unstructured sampling kernels (S5 forward, S7 backward; section 5.1.2).
// A warp is a packet of 32 consecutive points of the coherence-sorted order and walks the LBVH
// over the Gaussians with one short stack in shared memory.  Three stages, each with its own
// lane mapping, connected by small shared-memory queues (so that no stage waits on a memory
// round trip per pair):
//   1. traverse  lane = tree node.  Up to 32 nodes are popped per step; both children's boxes
//                (one 64-byte node) are tested against the packet's bounding box; internal
//                children go back on the stack, leaf children (Gaussian ids) to the candidate queue.
//   2. refine    lane = candidate Gaussian.  Its record is fetched and the cutoff ellipsoid is
//                tested against the packet box in whitened space (|M (c - mu)| <= r + rho, the
//                bound the structured kernels use per cell); survivors are compacted.
//   3. evaluate  forward: lane = point, the staged survivor records are read from shared memory
//                (broadcast) and every pair runs the canonical predicate (D4) + Eq. 3.
//                backward: lane = Gaussian, loop over the packet's 32 points (broadcast from
//                shared memory): the 12 per-Gaussian sums stay in registers -- the reduction over
//                the packet costs no shuffles -- and leave with three 16-byte vector reductions
//                (RED.ADD.F32x4) per (packet, Gaussian); the paper's backward is the same
//                "per Gaussian, loop over the leaf's positions" shape.
// Stages 1 and 2 are conservative culls only; membership is decided by the canonical predicate.
#include "gs_internal.cuh"
#include "pair_math.cuh"

namespace gs {

constexpr int PT_WARPS = 8;
constexpr int STK_CAP = 256;             // stack entries per packet
constexpr int STK_WIDE = STK_CAP - 66;   // above this fill level one node is popped per step (pure DFS: growth <= tree height <= 64)
constexpr int CQ_CAP = 96;               // candidate queue: < 32 before a step, a step adds <= 64
constexpr int SV_CAP = 64;               // survivor buffer: < 32 before a refine round, a round adds <= 32

struct PacketBox { float lx, ly, lz, hx, hy, hz; };

__device__ __forceinline__ float warp_min(float v) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v = fminf(v, __shfl_xor_sync(0xffffffffu, v, d));
    return v;
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, d));
    return v;
}

// Stage 1: one traversal step.  sp, cn are warp-uniform.
__device__ __forceinline__ bool boxes_overlap(const PacketBox &b, float lx, float ly, float lz, float hx, float hy, float hz) {
    return lx <= b.hx && hx >= b.lx && ly <= b.hy && hy >= b.ly && lz <= b.hz && hz >= b.lz;
}

__device__ __forceinline__ void traverse_step(const float4 *__restrict__ nodes, const PacketBox &b, const PacketBox &b2, int32_t *stack, int &sp,
                                              uint32_t *cand, int &cn, int lane, uint32_t *overflow) {
    int k = min(min(32, sp), max(1, STK_WIDE - sp));
    const bool act = lane < k;
    bool il = false, ir = false, ll = false, lr = false;
    int32_t lc = 0, rc = 0;
    if (act) {
        const int32_t node = stack[sp - 1 - lane];
        const float4 *np = nodes + 4 * (size_t)node;
        const float4 n0 = __ldg(np), n1 = __ldg(np + 1), n2 = __ldg(np + 2), n3 = __ldg(np + 3);
        const bool ol = boxes_overlap(b, n0.x, n0.y, n0.z, n0.w, n1.x, n1.y) || boxes_overlap(b2, n0.x, n0.y, n0.z, n0.w, n1.x, n1.y);
        const bool orr = boxes_overlap(b, n1.z, n1.w, n2.x, n2.y, n2.z, n2.w) || boxes_overlap(b2, n1.z, n1.w, n2.x, n2.y, n2.z, n2.w);
        lc = __float_as_int(n3.x); rc = __float_as_int(n3.y);
        il = ol && lc >= 0; ll = ol && lc < 0;
        ir = orr && rc >= 0; lr = orr && rc < 0;
    }
    __syncwarp();
    sp -= k;
    const uint32_t lt = (1u << lane) - 1u;
    const uint32_t bil = __ballot_sync(0xffffffffu, il), bir = __ballot_sync(0xffffffffu, ir);
    const uint32_t bll = __ballot_sync(0xffffffffu, ll), blr = __ballot_sync(0xffffffffu, lr);
    const int nil = __popc(bil), nir = __popc(bir), nll = __popc(bll), nlr = __popc(blr);
    if (sp + nil + nir > STK_CAP) {  // cannot happen for trees of height <= 64 (see STK_WIDE); never write out of bounds
        if (lane == 0) *overflow = 1u;
        sp = 0;
        return;
    }
    if (il) stack[sp + __popc(bil & lt)] = lc;
    if (ir) stack[sp + nil + __popc(bir & lt)] = rc;
    sp += nil + nir;
    if (ll) cand[cn + __popc(bll & lt)] = (uint32_t)~lc;
    if (lr) cand[cn + nll + __popc(blr & lt)] = (uint32_t)~rc;
    cn += nll + nlr;
    __syncwarp();
}

// Stage 2 test: can the cutoff ellipsoid of `g` reach the box (centre c, half extent h)?  For every p in the box
// |M (p - mu)| >= |M (c - mu)| - rho with rho = |(sum_k |M_jk| h_k)_j|, so the Gaussian is dropped when
// |M (c - mu)|^2 > (r + rho)^2 (1 + 2^-9) (the slack covers fp32 rounding of this bound and of the canonical sequence).
__device__ __forceinline__ bool ellipsoid_reaches(const Rec &g, float cx, float cy, float cz, float hx, float hy, float hz, float rcut) {
    const float dx = cx - g.a.x, dy = cy - g.a.y, dz = cz - g.a.z;
    const float u0 = fmaf(g.b.z, dz, fmaf(g.b.y, dy, g.b.x * dx));
    const float u1 = fmaf(g.c.z, dz, fmaf(g.c.y, dy, g.c.x * dx));
    const float u2 = fmaf(g.d.z, dz, fmaf(g.d.y, dy, g.d.x * dx));
    const float e0 = fmaf(fabsf(g.b.z), hz, fmaf(fabsf(g.b.y), hy, fabsf(g.b.x) * hx));
    const float e1 = fmaf(fabsf(g.c.z), hz, fmaf(fabsf(g.c.y), hy, fabsf(g.c.x) * hx));
    const float e2 = fmaf(fabsf(g.d.z), hz, fmaf(fabsf(g.d.y), hy, fabsf(g.d.x) * hx));
    const float qc = fmaf(u2, u2, fmaf(u1, u1, u0 * u0));
    const float reach = rcut + sqrtf(fmaf(e2, e2, fmaf(e1, e1, e0 * e0)));
    // false for NaN records (invalid Gaussians, D13) and for a NaN box (empty part); true for an infinite box (see segment_box)
    return qc <= reach * reach * 1.001953125f;
}

__device__ __forceinline__ Rec load_rec(const float4 *__restrict__ rec, uint32_t N, uint32_t id) {
    Rec g;
    g.a = __ldg(rec + id); g.b = __ldg(rec + (size_t)N + id); g.c = __ldg(rec + 2 * (size_t)N + id); g.d = __ldg(rec + 3 * (size_t)N + id);
    return g;
}

struct PacketState {      // per-warp shared memory of stage 1
    int32_t stack[STK_CAP];
    uint32_t cand[CQ_CAP];
};

// Packet set-up shared by both kernels: the point of this lane, the packet's boxes and the root of the traversal.
// A packet of 32 consecutive Morton-sorted points can straddle a jump of the Z curve (its box then spans a large
// part of the domain).  The packet is therefore cut once, at its highest-level jump (largest code[i] ^ code[i+1]):
// each part lies inside one Morton cell and gets its own box; a Gaussian is kept when it reaches either.
struct CullBox { float cx, cy, cz, hx, hy, hz; };
struct Packet {
    uint64_t c; bool active; float px, py, pz;
    PacketBox box[2]; CullBox cb[2];
    int sp, cn;
};

__device__ __forceinline__ void segment_box(float px, float py, float pz, bool in_seg, PacketBox &b, CullBox &cb) {
    const float nanv = __int_as_float(0x7fc00000);
    const float x = in_seg ? px : nanv, y = in_seg ? py : nanv, z = in_seg ? pz : nanv;
    // fminf/fmaxf drop NaN operands: the box spans the segment's real points (none => NaN box, nothing overlaps it)
    b.lx = warp_min(x); b.ly = warp_min(y); b.lz = warp_min(z);
    b.hx = warp_max(x); b.hy = warp_max(y); b.hz = warp_max(z);
    cb.cx = 0.5f * b.lx + 0.5f * b.hx; cb.cy = 0.5f * b.ly + 0.5f * b.hy; cb.cz = 0.5f * b.lz + 0.5f * b.hz;
    // half extents measured from the rounded centre, so the box [c - h, c + h] certainly holds every point
    cb.hx = fmaxf(b.hx - cb.cx, cb.cx - b.lx) * 1.000001f; cb.hy = fmaxf(b.hy - cb.cy, cb.cy - b.ly) * 1.000001f;
    cb.hz = fmaxf(b.hz - cb.cz, cb.cz - b.lz) * 1.000001f;
    const float big = 3.0e38f;   // infinite coordinates: a box that culls nothing
    if (b.lx < -big || b.ly < -big || b.lz < -big || b.hx > big || b.hy > big || b.hz > big) {
        cb.cx = cb.cy = cb.cz = 0.f;
        cb.hx = cb.hy = cb.hz = 1.0e30f;   // finite, so that 0 * h stays 0; the reach overflows to +inf
    }
}

__device__ __forceinline__ void packet_init(Packet &pk, PacketState &st, const float *__restrict__ xyz, const uint32_t *__restrict__ pt_order,
                                            uint64_t P, uint32_t N, const MortonParams &mp, int warp, int lane) {
    const uint64_t k = ((uint64_t)blockIdx.x * PT_WARPS + warp) * 32 + lane;
    pk.active = k < P;
    pk.c = pk.active ? (pt_order ? (uint64_t)pt_order[k] : k) : 0;
    const float nanv = __int_as_float(0x7fc00000);
    pk.px = pk.active ? xyz[3 * pk.c] : nanv; pk.py = pk.active ? xyz[3 * pk.c + 1] : nanv; pk.pz = pk.active ? xyz[3 * pk.c + 2] : nanv;
    const uint32_t code = morton30(pk.px, pk.py, pk.pz, mp);
    const uint32_t next = __shfl_down_sync(0xffffffffu, code, 1);
    const uint32_t jump = lane < 31 ? (code ^ next) : 0u;
    const uint32_t top = __reduce_max_sync(0xffffffffu, jump);
    const int cut = top ? __ffs(__ballot_sync(0xffffffffu, jump == top)) - 1 : 31;   // part 0 = lanes [0, cut], part 1 = the rest
    segment_box(pk.px, pk.py, pk.pz, lane <= cut, pk.box[0], pk.cb[0]);
    segment_box(pk.px, pk.py, pk.pz, lane > cut, pk.box[1], pk.cb[1]);
    pk.sp = 0; pk.cn = 0;
    if (N >= 2) { if (lane == 0) st.stack[0] = 0; pk.sp = 1; }
    else if (N == 1) { if (lane == 0) st.cand[0] = 0u; pk.cn = 1; }
    __syncwarp();
}

__device__ __forceinline__ bool reaches_packet(const Rec &g, const Packet &pk, float rcut) {
    return ellipsoid_reaches(g, pk.cb[0].cx, pk.cb[0].cy, pk.cb[0].cz, pk.cb[0].hx, pk.cb[0].hy, pk.cb[0].hz, rcut) ||
           ellipsoid_reaches(g, pk.cb[1].cx, pk.cb[1].cy, pk.cb[1].cz, pk.cb[1].hx, pk.cb[1].hy, pk.cb[1].hz, rcut);
}

template <bool SETS>
__global__ void __launch_bounds__(PT_WARPS * 32) k_points_fwd(const float4 *__restrict__ rec, uint32_t N, const float4 *__restrict__ nodes,
                                                               const float *__restrict__ xyz, const uint32_t *__restrict__ pt_order,
                                                               uint64_t P, MortonParams mp, float tau, float r2, float rcut, FwdOut o, double invP,
                                                               uint32_t *__restrict__ overflow) {
    __shared__ PacketState pstate[PT_WARPS];
    __shared__ float4 srec_all[PT_WARPS][4][SV_CAP];   // staged survivor records (plane c's .w carries the Gaussian id)
    __shared__ double red[PT_WARPS];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    PacketState &st = pstate[warp];
    float4 (*srec)[SV_CAP] = srec_all[warp];
    Packet pk;
    packet_init(pk, st, xyz, pt_order, P, N, mp, warp, lane);
    const float px = pk.px, py = pk.py, pz = pk.pz;
    float I = 0.f, Nacc = 0.f;
    uint32_t cnt = 0, tested = 0;
    unsigned long long hsum = 0, hxor = 0;
    int sp = pk.sp, cn = pk.cn, sn = 0;
    const uint32_t lt = (1u << lane) - 1u;
    while (true) {
        while (cn < 32 && sp > 0) traverse_step(nodes, pk.box[0], pk.box[1], st.stack, sp, st.cand, cn, lane, overflow);
        if (cn > 0) {   // stage 2: refine up to 32 candidates
            const int k = min(cn, 32);
            bool keep = false;
            Rec g;
            uint32_t id = 0;
            if (lane < k) {
                id = st.cand[cn - 1 - lane];
                g = load_rec(rec, N, id);
                keep = reaches_packet(g, pk, rcut);
            }
            cn -= k;
            const uint32_t bk = __ballot_sync(0xffffffffu, keep);
            if (keep) {
                const int slot = sn + __popc(bk & lt);
                g.c.w = __uint_as_float(id);
                srec[0][slot] = g.a; srec[1][slot] = g.b; srec[2][slot] = g.c; srec[3][slot] = g.d;
            }
            sn += __popc(bk);
            __syncwarp();
        }
        const bool done = cn == 0 && sp == 0;
        if (sn >= 32 || (done && sn > 0)) {   // stage 3: every lane evaluates its point against the staged records
#pragma unroll 2
            for (int j = 0; j < sn; j++) {
                Rec g;
                g.a = srec[0][j]; g.b = srec[1][j]; g.c = srec[2][j]; g.d = srec[3][j];
                float u0, u1, u2;
                const float qd = mahalanobis(g, px, py, pz, u0, u1, u2);
                const bool hit = qd <= r2;
                const float wG = hit ? g.a.w * gauss_weight(qd) : 0.f;
                I += wG;
                Nacc = fmaf(g.b.w, wG, Nacc);
                if (SETS && hit) { const unsigned long long h = mix64(__float_as_uint(g.c.w)); cnt++; hsum += h; hxor ^= h; }
            }
            if (SETS) tested += (uint32_t)sn;
            sn = 0;
            __syncwarp();
        }
        if (done) break;
    }
    const bool active = pk.active;
    const uint64_t c = pk.c;
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

__device__ __forceinline__ void red_add_v4(float *addr, float a, float b, float c, float d) {
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}

__global__ void __launch_bounds__(PT_WARPS * 32) k_points_bwd(const float4 *__restrict__ rec, uint32_t N, const float4 *__restrict__ nodes,
                                                               const float *__restrict__ xyz, const uint32_t *__restrict__ pt_order,
                                                               uint64_t P, MortonParams mp, float tau, float r2, float rcut, BwdIn in,
                                                               float *__restrict__ gacc, uint32_t *__restrict__ overflow) {
    __shared__ PacketState pstate[PT_WARPS];
    __shared__ uint32_t surv_all[PT_WARPS][SV_CAP];
    __shared__ float4 pts_all[PT_WARPS][2][32];   // [0] x y z alpha   [1] beta eps - -
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    PacketState &st = pstate[warp];
    uint32_t *surv = surv_all[warp];
    float4 (*pts)[32] = pts_all[warp];
    Packet pk;
    packet_init(pk, st, xyz, pt_order, P, N, mp, warp, lane);
    {
        // per-sample coefficients: alpha = covered ? a/I : 0, beta = b - alpha Phi, eps = covered ? |Phi - t|/I : 0
        const bool active = pk.active;
        const uint64_t c = pk.c;
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
        pts[0][lane] = make_float4(pk.px, pk.py, pk.pz, alpha);   // inactive lanes hold NaN positions: never a hit
        pts[1][lane] = make_float4(beta, eps, 0.f, 0.f);
        __syncwarp();
    }
    int sp = pk.sp, cn = pk.cn, sn = 0;
    const uint32_t lt = (1u << lane) - 1u;
    while (true) {
        while (cn < 32 && sp > 0) traverse_step(nodes, pk.box[0], pk.box[1], st.stack, sp, st.cand, cn, lane, overflow);
        if (cn > 0) {   // stage 2
            const int k = min(cn, 32);
            bool keep = false;
            uint32_t id = 0;
            if (lane < k) {
                id = st.cand[cn - 1 - lane];
                const Rec g = load_rec(rec, N, id);
                keep = reaches_packet(g, pk, rcut);
            }
            cn -= k;
            const uint32_t bk = __ballot_sync(0xffffffffu, keep);
            if (keep) surv[sn + __popc(bk & lt)] = id;
            sn += __popc(bk);
            __syncwarp();
        }
        const bool done = cn == 0 && sp == 0;
        if (sn >= 32 || (done && sn > 0)) {   // stage 3: lane = Gaussian, loop over the packet's points
            const int k = min(sn, 32);
            if (lane < k) {
                const uint32_t id = surv[sn - 1 - lane];
                const Rec g = load_rec(rec, N, id);
                float acc[16];
#pragma unroll
                for (int q = 0; q < 16; q++) acc[q] = 0.f;
                bool any = false;
#pragma unroll 4
                for (int p = 0; p < 32; p++) {
                    const float4 pa = pts[0][p], pb = pts[1][p];
                    float u0, u1, u2;
                    const float qd = mahalanobis(g, pa.x, pa.y, pa.z, u0, u1, u2);
                    if (qd <= r2) {
                        any = true;
                        bwd_accumulate(acc, pa.w, pb.x, pb.y, g.a.w, g.b.w, gauss_weight(qd), u0, u1, u2);
                    }
                }
                if (any) {
                    float *row = gacc + (size_t)id * GACC;
                    red_add_v4(row, acc[0], acc[1], acc[2], acc[3]);
                    red_add_v4(row + 4, acc[4], acc[5], acc[6], acc[7]);
                    red_add_v4(row + 8, acc[8], acc[9], acc[10], acc[11]);
                }
            }
            sn -= k;
            __syncwarp();
        }
        if (done && sn == 0) break;
    }
}

cudaError_t launch_points_fwd(const float4 *rec, uint32_t N, const float4 *nodes, const uint32_t *leaf_order, const float *xyz,
                              const uint32_t *pt_order, uint64_t P, const gs_domain &dom, float tau, float r2, float rcut, const FwdOut &o,
                              uint32_t *overflow, cudaStream_t s) {
    (void)leaf_order;
    if (P == 0) return cudaSuccess;
    const unsigned blocks = (unsigned)((P + PT_WARPS * 32 - 1) / (PT_WARPS * 32));
    const bool sets = o.set_count || o.set_sum || o.set_xor || o.counters;
    if (sets) k_points_fwd<true><<<blocks, PT_WARPS * 32, 0, s>>>(rec, N, nodes, xyz, pt_order, P, morton_params(dom), tau, r2, rcut, o, 1.0 / (double)P, overflow);
    else k_points_fwd<false><<<blocks, PT_WARPS * 32, 0, s>>>(rec, N, nodes, xyz, pt_order, P, morton_params(dom), tau, r2, rcut, o, 1.0 / (double)P, overflow);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_points_bwd(const float4 *rec, uint32_t N, const float4 *nodes, const uint32_t *leaf_order, const float *xyz,
                              const uint32_t *pt_order, uint64_t P, const gs_domain &dom, float tau, float r2, float rcut, const BwdIn &in, float *gacc,
                              uint32_t *overflow, cudaStream_t s) {
    (void)leaf_order;
    if (P == 0) return cudaSuccess;
    const unsigned blocks = (unsigned)((P + PT_WARPS * 32 - 1) / (PT_WARPS * 32));
    k_points_bwd<<<blocks, PT_WARPS * 32, 0, s>>>(rec, N, nodes, xyz, pt_order, P, morton_params(dom), tau, r2, rcut, in, gacc, overflow); count_launch();
    return cudaGetLastError();
}

}  // namespace gs
