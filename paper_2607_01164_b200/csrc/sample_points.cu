// sample_points.cu -- unstructured sampling kernels (S5 forward, S7 backward; section 5.1.2).
// A warp is a packet of 32 consecutive points of the coherence-sorted order.
//
//   k_points_cull  (part of gs_build_accel)  The packet walks the LBVH over the Gaussians with one short stack in
//       shared memory and writes the list of Gaussians that can reach it.  Two stages with their own lane mapping:
//         traverse  lane = tree node.  Up to 32 nodes are popped per step; both children's boxes (one 64-byte
//                   node) are tested against the packet's boxes; internal children go back on the stack, leaf
//                   children (sorted positions of Gaussians) to the candidate queue.
//         refine    lane = candidate Gaussian.  Its record is fetched and the cutoff ellipsoid is tested against
//                   the packet's boxes in whitened space (|M (c - mu)| <= r + rho, the bound the structured
//                   kernels use per cell); survivors are appended to the packet's list.
//       Both are conservative culls only; membership is decided by the canonical predicate in the kernels below.
//       The node loads of the next step and the record loads of the next refine round are issued before the
//       previous ones are consumed.  The list is a chain of 32-entry chunks taken from a pool with one atomic
//       per chunk; forward and backward both read it (the traversal runs once per step, not twice).
//   k_points_fwd   lane = point: the chunk's 32 records are staged in shared memory (broadcast reads) and every
//       pair runs the canonical predicate (D4) + Eq. 3; fused epilogue S6.
//   k_points_bwd   lane = Gaussian, loop over the packet's 32 points (broadcast from shared memory): the 12
//       per-Gaussian sums stay in registers -- the reduction over the packet costs no shuffles -- and leave with
//       three 16-byte vector reductions (RED.ADD.F32x4) per (packet, Gaussian).  The paper's backward has the same
//       "per Gaussian, loop over the leaf's positions" shape.
#include "gs_internal.cuh"
#include "pair_math.cuh"
#include "f32x2.cuh"

namespace gs {

#ifndef GS_CULL_WARPS
#define GS_CULL_WARPS 4
#endif
#ifndef GS_EVAL_WARPS
#define GS_EVAL_WARPS 4
#endif
constexpr int CULL_WARPS = GS_CULL_WARPS;  // packets per CTA of k_points_cull
constexpr int EVAL_WARPS = GS_EVAL_WARPS;  // packets per CTA of k_points_fwd / k_points_bwd
constexpr int STK_CAP = 256;             // stack entries per packet
constexpr int STK_WIDE = STK_CAP - 66;   // above this fill level one node is popped per step (pure DFS: growth <= tree height <= 64)
constexpr int CQ_CAP = 128;              // candidate queue: a step runs only with <= 64 queued and adds <= 64
constexpr uint32_t NO_CHUNK = 0xffffffffu;

struct PacketBox { float lx, ly, lz, hx, hy, hz; };
struct CullBox { float cx, cy, cz, hx, hy, hz; };

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

__device__ __forceinline__ bool boxes_overlap(const PacketBox &b, float lx, float ly, float lz, float hx, float hy, float hz) {
    return (lx <= b.hx) & (hx >= b.lx) & (ly <= b.hy) & (hy >= b.ly) & (lz <= b.hz) & (hz >= b.lz);
}

// Refine test: can the cutoff ellipsoid of `g` reach the box (centre c, half extent h)?  For every p in the box
// |M (p - mu)| >= |M (c - mu)| - rho with rho = |(sum_k |M_jk| h_k)_j|, so the Gaussian is dropped when
// |M (c - mu)|^2 > (r + rho)^2 (1 + 2^-9) (the slack covers fp32 rounding of this bound and of the canonical sequence).
__device__ __forceinline__ bool ellipsoid_reaches(const Rec &g, const CullBox &c, float rcut) {
    const float dx = c.cx - g.a.x, dy = c.cy - g.a.y, dz = c.cz - g.a.z;
    const float u0 = fmaf(g.b.z, dz, fmaf(g.b.y, dy, g.b.x * dx));
    const float u1 = fmaf(g.c.z, dz, fmaf(g.c.y, dy, g.c.x * dx));
    const float u2 = fmaf(g.d.z, dz, fmaf(g.d.y, dy, g.d.x * dx));
    const float e0 = fmaf(fabsf(g.b.z), c.hz, fmaf(fabsf(g.b.y), c.hy, fabsf(g.b.x) * c.hx));
    const float e1 = fmaf(fabsf(g.c.z), c.hz, fmaf(fabsf(g.c.y), c.hy, fabsf(g.c.x) * c.hx));
    const float e2 = fmaf(fabsf(g.d.z), c.hz, fmaf(fabsf(g.d.y), c.hy, fabsf(g.d.x) * c.hx));
    const float qc = fmaf(u2, u2, fmaf(u1, u1, u0 * u0));
    const float reach = rcut + sqrtf(fmaf(e2, e2, fmaf(e1, e1, e0 * e0)));
    // Tighter: component j of M (p - mu) stays within [u_j - e_j, u_j + e_j] over the box, so its magnitude is at least
    // max(0, |u_j| - e_j) and |M (p - mu)|^2 >= sum_j max(0, |u_j| - e_j)^2 (the distance to the box that bounds the
    // whitened image of the packet box).  It implies the spherical bound; for a Gaussian that is thin along one axis and
    // lies beside the packet along another it is much smaller than r + rho.
    const float v0 = fmaxf(fabsf(u0) - e0, 0.f), v1 = fmaxf(fabsf(u1) - e1, 0.f), v2 = fmaxf(fabsf(u2) - e2, 0.f);
    const float dmin2 = fmaf(v2, v2, fmaf(v1, v1, v0 * v0));
    const float r2s = rcut * rcut * 1.001953125f;
    // the spherical test stays: it is false for NaN records (invalid Gaussians, D13) and for a NaN box (empty part),
    // where fmaxf would drop the NaN; both are true for an infinite box (see segment_box)
    return (qc <= reach * reach * 1.001953125f) & (dmin2 <= r2s);
}

// A packet of 32 consecutive Morton-sorted points can straddle a jump of the Z curve (its box then spans a large
// part of the domain).  The packet is therefore cut once, at its highest-level jump (largest code[i] ^ code[i+1]):
// each part lies inside one Morton cell and gets its own box; a Gaussian is kept when it reaches either.
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

// The point of lane `lane` of packet `packet` (NaN for lanes past the end: never inside anything).
struct PacketPoint { uint64_t c; bool active; float px, py, pz; };
// Positions come from the SORTED copy of the query points (float4 per point, written once per gs_build_accel; the slots past
// the end hold NaN): one coalesced 16-byte load per lane instead of three scattered 4-byte gathers through the order array in
// each of the cull, forward and backward kernels.
__device__ __forceinline__ PacketPoint load_point(const float4 *__restrict__ spt, const uint32_t *__restrict__ pt_order, uint64_t P,
                                                  uint64_t packet, int lane) {
    PacketPoint pp;
    const uint64_t k = packet * 32 + lane;
    pp.active = k < P;
    pp.c = pp.active ? (pt_order ? (uint64_t)pt_order[k] : k) : 0;
    // the copy is NaN-padded to a multiple of 64 points (scatter_padded_points); a cull group of 4 packets can reach past
    // that, where nothing was allocated: those lanes get NaN without a load
    const float nan = __int_as_float(0x7fc00000);
    const float4 v = k < ((P + 63) & ~(uint64_t)63) ? __ldg(spt + k) : make_float4(nan, nan, nan, nan);
    pp.px = v.x; pp.py = v.y; pp.pz = v.z;
    return pp;
}

// Warp-cooperative gather of `count` (<= 32) 64-byte objects base[4 * index .. 4 * index + 3] into shared memory: lane l
// copies the 16-byte piece l & 3 of four objects, so one copy instruction touches 8 cache lines instead of 32 (a
// lane-per-object LDG.128 x 4 spends four times the L1 tag cycles).  Object j lands at dst[4 j + (piece ^ ((j >> 1) & 3))]:
// the swizzle makes the later lane-per-object 16-byte reads bank-conflict free (SWIZZLE = false: plain layout, for
// readers that broadcast one object to all lanes).  Completed by cp.async.wait_all.
template <bool SWIZZLE = true>
__device__ __forceinline__ void gather64(const float4 *__restrict__ base, uint32_t index_of_lane, int count, float4 *dst, int lane) {
    const int piece = lane & 3;
#pragma unroll
    for (int i = 0; i < 4; i++) {
        const int j = i * 8 + (lane >> 2);
        const uint32_t idx = __shfl_sync(0xffffffffu, index_of_lane, j);
        if (i * 8 < count && j < count) {
            const unsigned sdst = (unsigned)__cvta_generic_to_shared(dst + 4 * j + (SWIZZLE ? (piece ^ ((j >> 1) & 3)) : piece));
            asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(sdst), "l"(base + 4 * (size_t)idx + piece) : "memory");
        }
    }
}

// ---------------------------------------------------------------------------------------------------------
// k_points_cull: per-packet list of the Gaussians (sorted positions) whose cutoff ellipsoid can reach the packet.
// List = chain of chunks: head[packet] = (first chunk, entries in it); every further chunk (link[chunk]) is full.
// One warp serves a GROUP of CULL_GP consecutive packets (128 Morton-adjacent points): the tree is walked ONCE per group
// with the group's two boxes -- the upper levels of the walk, a chain of dependent L2 round trips with a handful of busy
// lanes, were half the kernel when every packet walked alone (configs[4]: 12 of 32 lanes busy per step) -- and the refine
// stage tests every candidate against the boxes of each of the group's packets and feeds one survivor queue per packet.
// ---------------------------------------------------------------------------------------------------------
#ifndef GS_CULL_MINB
#define GS_CULL_MINB 6
#endif
// CULL_GP = packets per group (per warp): 4 when the lists are short (the walk dominates), 2 when they are long (the refine
// stage, which tests every candidate against every packet of the group, dominates); chosen per build from the list sizes
// of the previous step (launch_points_cull)
template <int CULL_GP>
__global__ void __launch_bounds__(CULL_WARPS * 32, GS_CULL_MINB) k_points_cull(const float4 *__restrict__ srt, uint32_t N, const float4 *__restrict__ nodes,
                                                                  const float4 *__restrict__ xyz /*sorted copy*/, const uint32_t *__restrict__ pt_order,
                                                                  uint64_t P, MortonParams mp, float rcut, CullLists o,
                                                                  uint32_t *__restrict__ overflow) {
    __shared__ int32_t stack_all[CULL_WARPS][STK_CAP];
    __shared__ uint32_t cand_all[CULL_WARPS][CQ_CAP];
    __shared__ uint32_t surv_all[CULL_WARPS][CULL_GP][64];
    __shared__ CullBox cbox_all[CULL_WARPS][CULL_GP][2];                      // the two segment boxes of every packet of the group
    __shared__ float4 nbuf_all[CULL_WARPS][128], rbuf_all[CULL_WARPS][128];   // 32 nodes / 32 records of 64 B, swizzled
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint64_t npackets = (P + 31) / 32;
    const uint64_t packet0 = ((uint64_t)blockIdx.x * CULL_WARPS + warp) * CULL_GP;   // first packet of this warp's group
    if (packet0 >= npackets) return;
    int32_t *stack = stack_all[warp];
    uint32_t *cand = cand_all[warp];
    uint32_t (*surv)[64] = surv_all[warp];
    CullBox (*cbox)[2] = cbox_all[warp];
    float4 *nbuf = nbuf_all[warp], *rbuf = rbuf_all[warp];
    PacketBox box0, box1;   // the group's two boxes (the node tests of the walk)
    {
        // Packets and the group are cut at their highest-level jump of the Z curve (largest code[i] ^ code[i + 1]): each part
        // lies inside one Morton cell and gets its own box.
        PacketPoint pp[CULL_GP];
        uint32_t code[CULL_GP], gjump[CULL_GP];
#pragma unroll
        for (int g = 0; g < CULL_GP; g++) {
            pp[g] = load_point(xyz, pt_order, P, packet0 + g, lane);
            code[g] = morton30(pp[g].px, pp[g].py, pp[g].pz, mp);
        }
        uint32_t gtop = 0;
#pragma unroll
        for (int g = 0; g < CULL_GP; g++) {
            const uint32_t next = __shfl_down_sync(0xffffffffu, code[g], 1);
            const uint32_t jump = (lane < 31 && ((packet0 + g) * 32 + lane + 1) < P) ? (code[g] ^ next) : 0u;
            const uint32_t top = __reduce_max_sync(0xffffffffu, jump);
            const int cut = top ? __ffs(__ballot_sync(0xffffffffu, jump == top)) - 1 : 31;   // part 0 = lanes [0, cut], part 1 = the rest
            PacketBox b;
            CullBox c0, c1;
            segment_box(pp[g].px, pp[g].py, pp[g].pz, lane <= cut, b, c0);
            segment_box(pp[g].px, pp[g].py, pp[g].pz, lane > cut, b, c1);
            if (lane == 0) { cbox[g][0] = c0; cbox[g][1] = c1; }
            // jump to the first point of the next packet of the group (lane 31 only)
            uint32_t across = 0u;
            if (g + 1 < CULL_GP) {
                const uint32_t first_next = __shfl_sync(0xffffffffu, code[g + 1 < CULL_GP ? g + 1 : g], 0);
                if (lane == 31 && (packet0 + g + 1) * 32 < P) across = code[g] ^ first_next;
            }
            gjump[g] = lane == 31 ? across : jump;
            gtop = max(gtop, __reduce_max_sync(0xffffffffu, gjump[g]));
        }
        // position (packet, lane) of the group's cut: the first occurrence of the largest jump
        int cut_g = CULL_GP, cut_l = 31;
#pragma unroll
        for (int g = CULL_GP - 1; g >= 0; g--) {
            const uint32_t hitm = __ballot_sync(0xffffffffu, gtop != 0u && gjump[g] == gtop);
            if (hitm) { cut_g = g; cut_l = __ffs((int)hitm) - 1; }
        }
        const float nanv = __int_as_float(0x7fc00000);
        float lo0[3] = {nanv, nanv, nanv}, hi0[3] = {nanv, nanv, nanv}, lo1[3] = {nanv, nanv, nanv}, hi1[3] = {nanv, nanv, nanv};
#pragma unroll
        for (int g = 0; g < CULL_GP; g++) {   // fminf / fmaxf drop NaN operands (inactive lanes, the other part)
            const bool first = g < cut_g || (g == cut_g && lane <= cut_l);
            const float p3[3] = {pp[g].px, pp[g].py, pp[g].pz};
#pragma unroll
            for (int k = 0; k < 3; k++) {
                lo0[k] = fminf(lo0[k], first ? p3[k] : nanv); hi0[k] = fmaxf(hi0[k], first ? p3[k] : nanv);
                lo1[k] = fminf(lo1[k], first ? nanv : p3[k]); hi1[k] = fmaxf(hi1[k], first ? nanv : p3[k]);
            }
        }
        box0.lx = warp_min(lo0[0]); box0.ly = warp_min(lo0[1]); box0.lz = warp_min(lo0[2]);
        box0.hx = warp_max(hi0[0]); box0.hy = warp_max(hi0[1]); box0.hz = warp_max(hi0[2]);
        box1.lx = warp_min(lo1[0]); box1.ly = warp_min(lo1[1]); box1.lz = warp_min(lo1[2]);
        box1.hx = warp_max(hi1[0]); box1.hy = warp_max(hi1[1]); box1.hz = warp_max(hi1[2]);
    }
    int sp = 0, cn = 0;   // stack entries, queued candidates (warp-uniform)
    int sn[CULL_GP];      // survivors of every packet not yet written
    uint32_t prev[CULL_GP];
#pragma unroll
    for (int g = 0; g < CULL_GP; g++) { sn[g] = 0; prev[g] = NO_CHUNK; }
    if (N >= 2) { if (lane == 0) stack[0] = 0; sp = 1; }
    else if (N == 1) { if (lane == 0) cand[0] = 0u; cn = 1; }
    __syncwarp();
    const uint32_t lt = (1u << lane) - 1u;
    while (true) {
        // ---- issue: nodes of the next traversal step (one node per step when the stack is nearly full: pure DFS grows
        //      the stack by at most the tree height <= 64, so STK_CAP cannot be exceeded)
        const int kA = (sp > 0 && cn <= CQ_CAP - 64) ? min(min(32, sp), max(1, STK_WIDE - sp)) : 0;
        if (kA > 0) gather64(nodes, lane < kA ? (uint32_t)stack[sp - 1 - lane] : 0u, kA, nbuf, lane);
        sp -= kA;
        // ---- issue: records of the next refine round (full rounds while the traversal is running)
        const int kB = (cn >= 32 || (sp == 0 && kA == 0)) ? min(cn, 32) : 0;
        const uint32_t pos = lane < kB ? cand[cn - 1 - lane] : 0u;
        if (kB > 0) gather64(srt, pos, kB, rbuf, lane);
        cn -= kB;
        const bool drain = kA == 0 && kB == 0;   // => stack and queue are empty
        // ---- write full chunks of survivors while the loads are in flight
#pragma unroll
        for (int g = 0; g < CULL_GP; g++) {
            if (sn[g] >= 32) {
                uint32_t c = 0;
                if (lane == 0) c = atomicAdd(o.top, 1u);
                c = __shfl_sync(0xffffffffu, c, 0);
                if (c < o.cap) {
                    o.ids[(size_t)c * 32 + lane] = surv[g][sn[g] - 32 + lane];
                    if (lane == 0) o.link[c] = prev[g];
                }
                prev[g] = c;
                sn[g] -= 32;
            }
        }
        asm volatile("cp.async.wait_all;" ::: "memory");
        __syncwarp();
        // ---- traverse: consume the nodes
        if (kA > 0) {
            bool il = false, ir = false, ll = false, lr = false;
            int32_t lc = 0, rc = 0;
            if (lane < kA) {
                const int f = (lane >> 1) & 3;
                const float4 n0 = nbuf[4 * lane + f], n1 = nbuf[4 * lane + (1 ^ f)], n2 = nbuf[4 * lane + (2 ^ f)], n3 = nbuf[4 * lane + (3 ^ f)];
                const bool ol = boxes_overlap(box0, n0.x, n0.y, n0.z, n0.w, n1.x, n1.y) | boxes_overlap(box1, n0.x, n0.y, n0.z, n0.w, n1.x, n1.y);
                const bool orr = boxes_overlap(box0, n1.z, n1.w, n2.x, n2.y, n2.z, n2.w) | boxes_overlap(box1, n1.z, n1.w, n2.x, n2.y, n2.z, n2.w);
                lc = __float_as_int(n3.x); rc = __float_as_int(n3.y);
                il = ol & (lc >= 0); ll = ol & (lc < 0);
                ir = orr & (rc >= 0); lr = orr & (rc < 0);
            }
            const uint32_t bil = __ballot_sync(0xffffffffu, il), bir = __ballot_sync(0xffffffffu, ir);
            const uint32_t bll = __ballot_sync(0xffffffffu, ll), blr = __ballot_sync(0xffffffffu, lr);
            const int nil = __popc(bil), nll = __popc(bll);
            const int sp2 = sp + nil + __popc(bir);
            if (sp2 > STK_CAP) {   // unreachable for trees of height <= 64; never write out of bounds
                if (lane == 0) *overflow = 1u;
            } else {
                if (il) stack[sp + __popc(bil & lt)] = lc;
                if (ir) stack[sp + nil + __popc(bir & lt)] = rc;
                sp = sp2;
            }
            if (ll) cand[cn + __popc(bll & lt)] = (uint32_t)~lc;
            if (lr) cand[cn + nll + __popc(blr & lt)] = (uint32_t)~rc;
            cn += nll + __popc(blr);
        }
        // ---- refine: consume the records; every packet of the group keeps the candidates that reach one of its two boxes
        if (kB > 0) {
            Rec g;
            if (lane < kB) {
                const int f = (lane >> 1) & 3;
                g.a = rbuf[4 * lane + f]; g.b = rbuf[4 * lane + (1 ^ f)]; g.c = rbuf[4 * lane + (2 ^ f)]; g.d = rbuf[4 * lane + (3 ^ f)];
            } else {
                const float nanv = __int_as_float(0x7fc00000);
                g.a = g.b = g.c = g.d = make_float4(nanv, nanv, nanv, nanv);   // never reaches anything
            }
            // world half extents of the cutoff ellipsoid from the whitening matrix alone (rows m_j = R_j / s_j):
            // e_k^2 = r^2 sum_j s_j^2 R_jk^2 = r^2 sum_j M_jk^2 / |m_j|^4, inflated (a cull only; the walk tested this box against
            // the GROUP's boxes, here it is tested against each packet's own)
            float ex, ey, ez;
            {
                const float n0 = fmaf(g.b.z, g.b.z, fmaf(g.b.y, g.b.y, g.b.x * g.b.x)), n1 = fmaf(g.c.z, g.c.z, fmaf(g.c.y, g.c.y, g.c.x * g.c.x)),
                            n2 = fmaf(g.d.z, g.d.z, fmaf(g.d.y, g.d.y, g.d.x * g.d.x));
                const float i0 = __frcp_rn(n0 * n0), i1 = __frcp_rn(n1 * n1), i2 = __frcp_rn(n2 * n2);
                const float rr = rcut * 1.004f;
                ex = rr * sqrtf(fmaf(g.d.x * g.d.x, i2, fmaf(g.c.x * g.c.x, i1, g.b.x * g.b.x * i0)));
                ey = rr * sqrtf(fmaf(g.d.y * g.d.y, i2, fmaf(g.c.y * g.c.y, i1, g.b.y * g.b.y * i0)));
                ez = rr * sqrtf(fmaf(g.d.z * g.d.z, i2, fmaf(g.c.z * g.c.z, i1, g.b.z * g.b.z * i0)));
            }
#pragma unroll
            for (int q = 0; q < CULL_GP; q++) {
                if (packet0 + q >= npackets) continue;   // warp-uniform
                bool keep = false;
#pragma unroll
                for (int sgm = 0; sgm < 2; sgm++) {
                    const CullBox cb = cbox[q][sgm];
                    // !(x > y) keeps NaN (an infinite box / an overflowing extent culls nothing); a NaN box (empty part) fails the ellipsoid test
                    const bool near = !(fabsf(cb.cx - g.a.x) > cb.hx + ex) & !(fabsf(cb.cy - g.a.y) > cb.hy + ey) & !(fabsf(cb.cz - g.a.z) > cb.hz + ez);
                    keep |= near & ellipsoid_reaches(g, cb, rcut);
                }
                const uint32_t bk = __ballot_sync(0xffffffffu, keep);
                if (keep) surv[q][sn[q] + __popc(bk & lt)] = pos;
                sn[q] += __popc(bk);
            }
        }
        __syncwarp();
        if (drain) break;
    }
    // the remaining (< 32 ... or exactly 32 from the last round) survivors: at most two more chunks per packet; the last one
    // written is the head
#pragma unroll
    for (int g = 0; g < CULL_GP; g++) {
        if (packet0 + g >= npackets) continue;
        uint32_t head_cnt = prev[g] == NO_CHUNK ? 0u : 32u;
        int n = sn[g];
        while (n > 0) {
            const int k = min(n, 32);
            uint32_t c = 0;
            if (lane == 0) c = atomicAdd(o.top, 1u);
            c = __shfl_sync(0xffffffffu, c, 0);
            if (c < o.cap) {
                // a partial chunk must be the head (every linked chunk is full): write the full one first
                if (lane < k) o.ids[(size_t)c * 32 + lane] = surv[g][(n > 32 ? 0 : n - k) + lane];
                if (lane == 0) o.link[c] = prev[g];
            }
            prev[g] = c;
            head_cnt = (uint32_t)k;
            if (n > 32) {   // 32 < n < 64: entries [0, 32) went out as a full chunk, move the tail down
                const uint32_t t = lane < n - 32 ? surv[g][32 + lane] : 0u;
                __syncwarp();
                if (lane < n - 32) surv[g][lane] = t;
                __syncwarp();
            }
            n -= k;
        }
        if (lane == 0) o.head[packet0 + g] = make_uint2(prev[g], head_cnt);
    }
}

// ---------------------------------------------------------------------------------------------------------
// k_points_fwd: the packet's list is consumed chunk by chunk (32 records staged in shared memory).
// Lane = (half h = lane >> 4, point pair q = lane & 15): the lane evaluates the packet's points 2q and 2q + 1, packed
// in the two halves of f32x2 registers, against the entries j = h, h + 2, ... of the chunk (the record is a scalar
// broadcast to both halves).  One warp-iteration therefore tests 2 Gaussians x 32 points in ~28 issue slots
// (15 packed instructions for the canonical sequence) where the scalar form needed 27 slots per Gaussian.
// ---------------------------------------------------------------------------------------------------------
template <bool SETS, bool MASKS>
__global__ void __launch_bounds__(EVAL_WARPS * 32) k_points_fwd(const float4 *__restrict__ srt, const float4 *__restrict__ xyz /*sorted copy*/,
                                                                 const uint32_t *__restrict__ pt_order, uint64_t P, CullLists L, float tau,
                                                                 float r2, FwdOut o, double invP) {
    __shared__ float4 buf_all[EVAL_WARPS][2][128];   // two chunks of 32 records of 64 B (plane c's .w carries the Gaussian id)
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint64_t packet = (uint64_t)blockIdx.x * EVAL_WARPS + warp;
    if (packet * 32 >= P) return;
    float4 (*buf)[128] = buf_all[warp];
    const PacketPoint pp = load_point(xyz, pt_order, P, packet, lane);   // lane's own point (epilogue); NaN when past the end
    const int half = lane >> 4, q2 = 2 * (lane & 15);
    const f2 px = pk(__shfl_sync(0xffffffffu, pp.px, q2), __shfl_sync(0xffffffffu, pp.px, q2 + 1));
    const f2 py = pk(__shfl_sync(0xffffffffu, pp.py, q2), __shfl_sync(0xffffffffu, pp.py, q2 + 1));
    const f2 pz = pk(__shfl_sync(0xffffffffu, pp.pz, q2), __shfl_sync(0xffffffffu, pp.pz, q2 + 1));
    f2 I2 = pk(0.f, 0.f), N2 = pk(0.f, 0.f);
    uint32_t cnt[2] = {0, 0}, tested = 0;
    unsigned long long hsum[2] = {0, 0}, hxor[2] = {0, 0};
    // Software pipeline over the chain of chunks: while chunk k is evaluated, the records of chunk k+1 are being
    // copied into the other buffer and the ids of chunk k+2 are being loaded.
    const uint2 head = __ldg(L.head + packet);
    uint32_t c0 = head.x, c1 = NO_CHUNK, c2 = NO_CHUNK, pos1 = 0u;
    int n0 = (int)head.y, b = 0;
    if (c0 != NO_CHUNK) {
        const uint32_t pos0 = lane < n0 ? __ldg(L.ids + (size_t)c0 * 32 + lane) : 0u;
        c1 = __ldg(L.link + c0);
        gather64<false>(srt, pos0, n0, buf[0], lane);
        if (c1 != NO_CHUNK) { pos1 = __ldg(L.ids + (size_t)c1 * 32 + lane); c2 = __ldg(L.link + c1); }   // linked chunks are full
    }
    while (c0 != NO_CHUNK) {
        asm volatile("cp.async.wait_all;" ::: "memory");
        __syncwarp();
        uint32_t pos2 = 0u, c3 = NO_CHUNK;
        if (c1 != NO_CHUNK) gather64<false>(srt, pos1, 32, buf[b ^ 1], lane);
        if (c2 != NO_CHUNK) { pos2 = __ldg(L.ids + (size_t)c2 * 32 + lane); c3 = __ldg(L.link + c2); }
        const float4 *rb = buf[b];
        // bit j: entry j of this chunk hits one of THIS LANE's two points (the halves hold the even / odd entries); one OR-reduction
        // over the warp per chunk then gives the chunk's mask (a vote per entry cost the forward 50 %: measured)
        uint32_t emask = 0, ebit = 1u << half;
#pragma unroll 4
        for (int j = half; j < n0; j += 2) {
            const float4 ga = rb[4 * j], gb = rb[4 * j + 1], gc = rb[4 * j + 2], gd = rb[4 * j + 3];
            f2 u0, u1, u2;
            const f2 qd = mahalanobis2(ga.x, ga.y, ga.z, gb.x, gb.y, gb.z, gc.x, gc.y, gc.z, gd.x, gd.y, gd.z, px, py, pz, u0, u1, u2);
            bool h0, h1;
            const f2 G = gauss_weight2(qd, r2, h0, h1);
            if (MASKS) {
                if (h0 | h1) emask |= ebit;
                ebit <<= 2;
            }
            I2 = fma2(bc(ga.w), G, I2);
            N2 = fma2(bc(gd.w), G, N2);   // d.w = v w
            if (SETS) {
                const unsigned long long h = mix64(__float_as_uint(gc.w));
                if (h0) { cnt[0]++; hsum[0] += h; hxor[0] ^= h; }
                if (h1) { cnt[1]++; hsum[1] += h; hxor[1] ^= h; }
            }
        }
        if (SETS) tested += (uint32_t)n0;
        __syncwarp();
        if (MASKS) {   // the backward drops the entries that hit nothing (44 % of configs[4]'s, 33 % of configs[2]'s) before it gathers their records
            emask = __reduce_or_sync(0xffffffffu, emask);
            if (lane == 0) L.mask[c0] = make_uint2(emask, c2);   // c2: the chunk two links on, already in a register here
        }
        c0 = c1; n0 = 32; c1 = c2; pos1 = pos2; c2 = c3; b ^= 1;
    }
    // the two halves hold the sums over the even / odd entries: add them, then hand point `lane` its own result
    float Il, Ih, Nl, Nh;
    upk(I2, Il, Ih);
    upk(N2, Nl, Nh);
    Il += __shfl_xor_sync(0xffffffffu, Il, 16); Ih += __shfl_xor_sync(0xffffffffu, Ih, 16);
    Nl += __shfl_xor_sync(0xffffffffu, Nl, 16); Nh += __shfl_xor_sync(0xffffffffu, Nh, 16);
    const int src = lane >> 1;
    const bool odd = lane & 1;
    const float Ia = __shfl_sync(0xffffffffu, Il, src), Ib = __shfl_sync(0xffffffffu, Ih, src);
    const float Na = __shfl_sync(0xffffffffu, Nl, src), Nb = __shfl_sync(0xffffffffu, Nh, src);
    const float I = odd ? Ib : Ia, Nacc = odd ? Nb : Na;
    uint32_t mycnt = 0;
    unsigned long long mysum = 0, myxor = 0;
    if (SETS) {
#pragma unroll
        for (int d = 0; d < 2; d++) {
            cnt[d] += __shfl_xor_sync(0xffffffffu, cnt[d], 16);
            hsum[d] += __shfl_xor_sync(0xffffffffu, hsum[d], 16);
            hxor[d] ^= __shfl_xor_sync(0xffffffffu, hxor[d], 16);
        }
        const uint32_t ca = __shfl_sync(0xffffffffu, cnt[0], src), cb = __shfl_sync(0xffffffffu, cnt[1], src);
        const unsigned long long sa = __shfl_sync(0xffffffffu, hsum[0], src), sb = __shfl_sync(0xffffffffu, hsum[1], src);
        const unsigned long long xa = __shfl_sync(0xffffffffu, hxor[0], src), xb = __shfl_sync(0xffffffffu, hxor[1], src);
        mycnt = odd ? cb : ca; mysum = odd ? sb : sa; myxor = odd ? xb : xa;
    }
    const bool active = pp.active;
    const uint64_t c = pp.c;
    const bool covered = I > tau;
    const float phi = covered ? __fdividef(Nacc, I) : 0.f;
    float res2 = 0.f;
    LossPartial lp;
    if (active) {
        o.phi[c] = phi;
        o.I[c] = I;
        if (o.gen.on) {
            loss_sample(o.gen, c, phi, I, covered, tau, o.target, o.dL_dphi, o.sample_err, lp);
        } else if (o.target) {
            const float res = phi - o.target[c];
            res2 = res * res;
            if (o.dL_dphi) o.dL_dphi[c] = covered ? (float)(2.0 * invP) * res : 0.f;
            if (o.sample_err) o.sample_err[c] = fabsf(res);
            if (o.pack2) {   // kept in SORTED order (position packet * 32 + lane): the backward reads it back coalesced
                const float al = covered ? __fdividef((float)(2.0 * invP) * res, I) : 0.f;
                o.pack2[packet * 32 + lane] = make_float2(al, -al * phi);
            }
        }
        if (SETS) {
            if (o.set_count) o.set_count[c] = mycnt;
            if (o.set_sum) o.set_sum[c] = mysum;
            if (o.set_xor) o.set_xor[c] = myxor;
        }
    }
    if (o.gen.on) loss_flush(o.gen, lp, lane);
    if (!o.gen.on && o.target && o.loss) {   // one reduction per packet (no CTA barrier: a warp's slot frees as soon as its packet is done)
        double s = (double)res2;
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
        if (lane == 0 && s != 0.0) atomicAdd(o.loss, s * invP);
    }
    if (SETS && o.counters) {
        unsigned long long t = active ? tested : 0, h = active ? mycnt : 0;
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) { t += __shfl_xor_sync(0xffffffffu, t, d); h += __shfl_xor_sync(0xffffffffu, h, d); }
        if (lane == 0) { atomicAdd(o.counters, t); atomicAdd(o.counters + 1, h); }
    }
}

// ---------------------------------------------------------------------------------------------------------
// k_points_bwd: lane = Gaussian of the chunk, loop over the packet's 32 points.
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void red_add_v4(float *addr, float a, float b, float c, float d) {
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}

__global__ void __launch_bounds__(EVAL_WARPS * 32) k_points_bwd(const float4 *__restrict__ srt, const float4 *__restrict__ xyz /*sorted copy*/,
                                                                 const uint32_t *__restrict__ pt_order, uint64_t P, CullLists L, float tau,
                                                                 float r2, BwdIn in, float *__restrict__ gacc) {
    // the packet's points as PAIRS (2i, 2i + 1) for the packed arithmetic: [i][0] = x0 x1 y0 y1, [i][1] = z0 z1 alpha0 alpha1,
    // [i][2] = beta0 beta1 eps0 eps1
    __shared__ __align__(16) float pts_all[EVAL_WARPS][16][12];
    __shared__ float4 buf_all[EVAL_WARPS][2][128];  // two chunks of 32 records of 64 B, swizzled (see gather64)
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint64_t packet = (uint64_t)blockIdx.x * EVAL_WARPS + warp;
    if (packet * 32 >= P) return;
    float (*pts)[12] = pts_all[warp];
    float4 (*buf)[128] = buf_all[warp];
    {
        const PacketPoint pp = load_point(xyz, pt_order, P, packet, lane);
        // per-sample coefficients: alpha = covered ? a/I : 0, beta = b - alpha Phi, eps = covered ? |Phi - t|/I : 0
        const bool active = pp.active;
        const uint64_t c = pp.c;
        float alpha = 0.f, beta = 0.f, eps = 0.f;
        if (active && in.pack2) {  // fused MSE: eps = |res| / I = |alpha| * P / 2
            const float2 s = __ldg(in.pack2 + packet * 32 + lane);   // sorted order, see k_points_fwd
            alpha = s.x; beta = s.y; eps = fabsf(s.x) * in.eps_scale;
        } else if (active) {
            const float Ic = in.I[c], ph = in.phi[c];
            const bool covered = Ic > tau;
            const float inv = covered ? 1.0f / Ic : 0.f;
            alpha = covered ? in.dL_dphi[c] * inv : 0.f;
            beta = (in.dL_dI ? in.dL_dI[c] : 0.f) - alpha * ph;
            eps = (covered && in.target) ? fabsf(ph - in.target[c]) * inv : 0.f;
        }
        // The sums below are accumulated without a branch (a miss has G = 0), so a NaN / infinite position would turn
        // 0 * u into NaN for every Gaussian of the list.  Such a point (a lane past the end, or a non-finite query) lies
        // in no support: it takes part with zero coefficients at a harmless finite position.
        float x = pp.px, y = pp.py, z = pp.pz;
        if (!(fabsf(x) <= 3.402823466e38f && fabsf(y) <= 3.402823466e38f && fabsf(z) <= 3.402823466e38f)) {
            x = y = z = 0.f;
            alpha = beta = eps = 0.f;
        }
        float *row = pts[lane >> 1] + (lane & 1);
        row[0] = x; row[2] = y; row[4] = z; row[6] = alpha; row[8] = beta; row[10] = eps;
        __syncwarp();
    }
    // same software pipeline as the forward: records of chunk k+1 and ids of chunk k+2 are in flight during chunk k
    const uint2 head = __ldg(L.head + packet);
    uint32_t c0 = head.x, c1 = NO_CHUNK, c2 = NO_CHUNK, pos1 = 0u;
    int n0 = (int)head.y, b = 0;
    if (c0 != NO_CHUNK) {
        const uint32_t pos0 = lane < n0 ? __ldg(L.ids + (size_t)c0 * 32 + lane) : 0u;
        c1 = __ldg(L.link + c0);
        gather64<true>(srt, pos0, n0, buf[0], lane);
        if (c1 != NO_CHUNK) { pos1 = __ldg(L.ids + (size_t)c1 * 32 + lane); c2 = __ldg(L.link + c1); }   // linked chunks are full
    }
    while (c0 != NO_CHUNK) {
        asm volatile("cp.async.wait_all;" ::: "memory");
        __syncwarp();
        uint32_t pos2 = 0u, c3 = NO_CHUNK;
        if (c1 != NO_CHUNK) gather64<true>(srt, pos1, 32, buf[b ^ 1], lane);
        if (c2 != NO_CHUNK) { pos2 = __ldg(L.ids + (size_t)c2 * 32 + lane); c3 = __ldg(L.link + c2); }
        if (lane < n0) {
            const float4 *rb = buf[b] + 4 * lane;
            const int f = (lane >> 1) & 3;
            Rec g;
            g.a = rb[f]; g.b = rb[1 ^ f]; g.c = rb[2 ^ f]; g.d = rb[3 ^ f];
            // lane = Gaussian (scalars, broadcast to both halves); two points per iteration ride in the halves.  A miss has
            // G = 0 and adds nothing, so the 12 sums are accumulated unconditionally (no divergent branch).
            f2 acc[12];
#pragma unroll
            for (int q = 0; q < 12; q++) acc[q] = pk(0.f, 0.f);
            bool any = false;
            const f2 w2 = bc(g.a.w), v2 = bc(g.b.w);
#pragma unroll 4
            for (int i = 0; i < 16; i++) {
                const ulonglong2 A = *reinterpret_cast<const ulonglong2 *>(pts[i]), B = *reinterpret_cast<const ulonglong2 *>(pts[i] + 4),
                                 C = *reinterpret_cast<const ulonglong2 *>(pts[i] + 8);
                f2 u0, u1, u2;
                const f2 qd = mahalanobis2(g.a.x, g.a.y, g.a.z, g.b.x, g.b.y, g.b.z, g.c.x, g.c.y, g.c.z, g.d.x, g.d.y, g.d.z, A.x, A.y, B.x, u0, u1, u2);
                bool h0, h1;
                const f2 G = gauss_weight2(qd, r2, h0, h1);
                any |= h0 | h1;
                const f2 alpha = B.y, beta = C.x, eps = C.y;
                // S7: gamma = alpha v + beta, t = gamma w G: dv += alpha w G, dw += gamma G, U += t u, W += t u u^T, E += eps w G
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
            }
            if (any) {
                float s[12];
#pragma unroll
                for (int q = 0; q < 12; q++) s[q] = lo(acc[q]) + hi(acc[q]);
                float *row = gacc + (size_t)__float_as_uint(g.c.w) * GACC;
                red_add_v4(row, s[0], s[1], s[2], s[3]);
                red_add_v4(row + 4, s[4], s[5], s[6], s[7]);
                red_add_v4(row + 8, s[8], s[9], s[10], s[11]);
            }
        }
        __syncwarp();
        c0 = c1; n0 = 32; c1 = c2; pos1 = pos2; c2 = c3; b ^= 1;
    }
}

// ---------------------------------------------------------------------------------------------------------
// k_points_bwd_masked: the same sums as k_points_bwd over the entries that HIT.  The forward left one bit per list entry
// (CullLists::mask); here a warp walks its packet's chain, keeps the ids whose bit is set in a 64-slot ring, and as soon as 32
// have come together gathers their records and evaluates them, lane = Gaussian -- so every lane holds a Gaussian that reaches
// the packet, whatever chunk it came from, and the records of the others are never read.  One batch's gather is in flight
// while the previous batch is evaluated.  Per entry the arithmetic and its order are those of k_points_bwd.
// ---------------------------------------------------------------------------------------------------------
#ifndef GS_BWDM_MINB
#define GS_BWDM_MINB 4   // measured: 5 resident CTAs (96 registers, a few spills) is slower (configs[4] 3.34 vs 3.18 ms)
#endif
__global__ void __launch_bounds__(EVAL_WARPS * 32, GS_BWDM_MINB) k_points_bwd_masked(const float4 *__restrict__ srt, const float4 *__restrict__ xyz /*sorted copy*/,
                                                                        const uint32_t *__restrict__ pt_order, uint64_t P, CullLists L, float tau,
                                                                        float r2, BwdIn in, float *__restrict__ gacc) {
    __shared__ __align__(16) float pts_all[EVAL_WARPS][16][12];   // as in k_points_bwd
    __shared__ float4 buf_all[EVAL_WARPS][2][128];
    __shared__ uint32_t ring_all[EVAL_WARPS][64];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint64_t packet = (uint64_t)blockIdx.x * EVAL_WARPS + warp;
    if (packet * 32 >= P) return;
    float (*pts)[12] = pts_all[warp];
    float4 (*buf)[128] = buf_all[warp];
    uint32_t *ring = ring_all[warp];
    {
        const PacketPoint pp = load_point(xyz, pt_order, P, packet, lane);
        const bool active = pp.active;
        const uint64_t c = pp.c;
        float alpha = 0.f, beta = 0.f, eps = 0.f;
        if (active && in.pack2) {
            const float2 s = __ldg(in.pack2 + packet * 32 + lane);
            alpha = s.x; beta = s.y; eps = fabsf(s.x) * in.eps_scale;
        } else if (active) {
            const float Ic = in.I[c], ph = in.phi[c];
            const bool covered = Ic > tau;
            const float inv = covered ? 1.0f / Ic : 0.f;
            alpha = covered ? in.dL_dphi[c] * inv : 0.f;
            beta = (in.dL_dI ? in.dL_dI[c] : 0.f) - alpha * ph;
            eps = (covered && in.target) ? fabsf(ph - in.target[c]) * inv : 0.f;
        }
        float x = pp.px, y = pp.py, z = pp.pz;
        if (!(fabsf(x) <= 3.402823466e38f && fabsf(y) <= 3.402823466e38f && fabsf(z) <= 3.402823466e38f)) {   // see k_points_bwd
            x = y = z = 0.f;
            alpha = beta = eps = 0.f;
        }
        float *row = pts[lane >> 1] + (lane & 1);
        row[0] = x; row[2] = y; row[4] = z; row[6] = alpha; row[8] = beta; row[10] = eps;
        __syncwarp();
    }
    // The chain is read two chunks ahead: A is the chunk being appended, B the next one (its loads in flight), and as soon as A's
    // mask word is here its skip link names the chunk after B, whose loads are issued before A is used.
    const uint2 head = __ldg(L.head + packet);
    uint32_t cA = head.x, cB = NO_CHUNK, idA = 0u, idB = 0u;
    uint2 wA = make_uint2(0u, NO_CHUNK), wB = make_uint2(0u, NO_CHUNK);
    if (cA != NO_CHUNK) {   // the head chunk holds head.y entries, every linked chunk 32
        const int n = (int)head.y;
        idA = lane < n ? __ldg(L.ids + (size_t)cA * 32 + lane) : 0u;
        wA = __ldg(L.mask + cA);
        if (n < 32) wA.x &= (1u << n) - 1u;
        cB = __ldg(L.link + cA);
        if (cB != NO_CHUNK) { idB = __ldg(L.ids + (size_t)cB * 32 + lane); wB = __ldg(L.mask + cB); }
    }
    uint32_t cnt = 0, done = 0;   // ids appended to the ring / ids handed to a gather so far
    int pend = 0, slot = 0;        // entries of the batch whose records are on their way into buf[slot]
    while (true) {
        while (cA != NO_CHUNK && cnt - done < 32u) {
            const uint32_t cC = cB != NO_CHUNK ? wA.y : NO_CHUNK;
            uint32_t idC = 0u;
            uint2 wC = make_uint2(0u, NO_CHUNK);
            if (cC != NO_CHUNK) { idC = __ldg(L.ids + (size_t)cC * 32 + lane); wC = __ldg(L.mask + cC); }
            const uint32_t m = wA.x;
            if ((m >> lane) & 1u) ring[(cnt + __popc(m & ((1u << lane) - 1u))) & 63u] = idA;
            cnt += __popc(m);
            cA = cB; idA = idB; wA = wB;
            cB = cC; idB = idC; wB = wC;
        }
        __syncwarp();
        const int nb = (int)(cnt - done < 32u ? cnt - done : 32u);
        if (pend) {
            asm volatile("cp.async.wait_all;" ::: "memory");
            __syncwarp();
        }
        if (nb) {
            const uint32_t pos = lane < nb ? ring[(done + lane) & 63u] : 0u;
            gather64<true>(srt, pos, nb, buf[slot ^ 1], lane);
            done += (uint32_t)nb;
        }
        if (lane < pend) {
            const float4 *rb = buf[slot] + 4 * lane;
            const int f = (lane >> 1) & 3;
            Rec g;
            g.a = rb[f]; g.b = rb[1 ^ f]; g.c = rb[2 ^ f]; g.d = rb[3 ^ f];
            f2 acc[12];
#pragma unroll
            for (int q = 0; q < 12; q++) acc[q] = pk(0.f, 0.f);
            bool any = false;
            const f2 w2 = bc(g.a.w), v2 = bc(g.b.w);
#pragma unroll 4
            for (int i = 0; i < 16; i++) {
                const ulonglong2 A = *reinterpret_cast<const ulonglong2 *>(pts[i]), B = *reinterpret_cast<const ulonglong2 *>(pts[i] + 4),
                                 C = *reinterpret_cast<const ulonglong2 *>(pts[i] + 8);
                f2 u0, u1, u2;
                const f2 qd = mahalanobis2(g.a.x, g.a.y, g.a.z, g.b.x, g.b.y, g.b.z, g.c.x, g.c.y, g.c.z, g.d.x, g.d.y, g.d.z, A.x, A.y, B.x, u0, u1, u2);
                bool h0, h1;
                const f2 G = gauss_weight2(qd, r2, h0, h1);
                any |= h0 | h1;
                const f2 alpha = B.y, beta = C.x, eps = C.y;
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
            }
            if (any) {
                float s[12];
#pragma unroll
                for (int q = 0; q < 12; q++) s[q] = lo(acc[q]) + hi(acc[q]);
                float *row = gacc + (size_t)__float_as_uint(g.c.w) * GACC;
                red_add_v4(row, s[0], s[1], s[2], s[3]);
                red_add_v4(row + 4, s[4], s[5], s[6], s[7]);
                red_add_v4(row + 8, s[8], s[9], s[10], s[11]);
            }
        }
        __syncwarp();
        if (!nb) break;
        pend = nb;
        slot ^= 1;
    }
}

cudaError_t launch_points_cull(const float4 *sorted_rec, uint32_t N, const float4 *nodes, const float4 *xyz, const uint32_t *pt_order,
                               uint64_t P, const gs_domain &dom, float rcut, const CullLists &lists, uint32_t *overflow, int group,
                               cudaStream_t s) {
    if (P == 0) return cudaSuccess;
    cudaError_t e = cudaMemsetAsync(lists.top, 0, sizeof(uint32_t), s);
    if (e != cudaSuccess) return e;
    const uint64_t packets = (P + 31) / 32, groups = (packets + group - 1) / group;
    const unsigned blocks = (unsigned)((groups + CULL_WARPS - 1) / CULL_WARPS);
    if (group == 2) k_points_cull<2><<<blocks, CULL_WARPS * 32, 0, s>>>(sorted_rec, N, nodes, xyz, pt_order, P, morton_params(dom), rcut, lists, overflow);
    else k_points_cull<4><<<blocks, CULL_WARPS * 32, 0, s>>>(sorted_rec, N, nodes, xyz, pt_order, P, morton_params(dom), rcut, lists, overflow);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_points_fwd(const float4 *sorted_rec, const float4 *xyz, const uint32_t *pt_order, uint64_t P, const CullLists &lists,
                              float tau, float r2, const FwdOut &o, cudaStream_t s) {
    if (P == 0) return cudaSuccess;
    const uint64_t packets = (P + 31) / 32;
    const unsigned blocks = (unsigned)((packets + EVAL_WARPS - 1) / EVAL_WARPS);
    const bool sets = o.set_count || o.set_sum || o.set_xor || o.counters;
    const double invP = o.inv_count > 0.0 ? o.inv_count : 1.0 / (double)P;
    if (sets) k_points_fwd<true, false><<<blocks, EVAL_WARPS * 32, 0, s>>>(sorted_rec, xyz, pt_order, P, lists, tau, r2, o, invP);
    else if (lists.mask) k_points_fwd<false, true><<<blocks, EVAL_WARPS * 32, 0, s>>>(sorted_rec, xyz, pt_order, P, lists, tau, r2, o, invP);
    else k_points_fwd<false, false><<<blocks, EVAL_WARPS * 32, 0, s>>>(sorted_rec, xyz, pt_order, P, lists, tau, r2, o, invP);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_points_bwd(const float4 *sorted_rec, const float4 *xyz, const uint32_t *pt_order, uint64_t P, const CullLists &lists,
                              float tau, float r2, const BwdIn &in, float *gacc, bool use_masks, cudaStream_t s) {
    if (P == 0) return cudaSuccess;
    const uint64_t packets = (P + 31) / 32;
    const unsigned blocks = (unsigned)((packets + EVAL_WARPS - 1) / EVAL_WARPS);
    if (use_masks && lists.mask) k_points_bwd_masked<<<blocks, EVAL_WARPS * 32, 0, s>>>(sorted_rec, xyz, pt_order, P, lists, tau, r2, in, gacc);
    else k_points_bwd<<<blocks, EVAL_WARPS * 32, 0, s>>>(sorted_rec, xyz, pt_order, P, lists, tau, r2, in, gacc);
    count_launch();
    return cudaGetLastError();
}

}  // namespace gs
