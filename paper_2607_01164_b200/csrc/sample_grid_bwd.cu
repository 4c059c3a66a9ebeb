// sample_grid_bwd.cu -- structured backward (S7; section 4.1.4, in the warp-per-Gaussian form of
// section 5.1.2 PAPER.md:196 applied to a grid, where the "traversal" is index arithmetic).
//
// One warp per Gaussian, no atomics.  The warp
//   1. enumerates the ROWS (y, z) of 2x2x2-voxel cells of the Gaussian's AABB, one row per lane, and
//      solves the conservative whitened-space cull bound for the row in closed form: the cells of a
//      row that can hold a hit form an interval [lo, hi] around the row's closest approach;
//   2. pushes the surviving cells through a shared-memory ring (warp scan of the interval lengths)
//      so that every evaluation round has 32 busy lanes;
//   3. evaluates one cell (8 voxels) per lane with the canonical predicate (shared sub-expressions),
//      recomputing the weights (nothing is stored by the forward).  Inside a cell the whitened
//      coordinate is affine in the voxel index, u(v) = u(0) + ix dx E_x + iy dy E_y + iz dz E_z (E_a = column a
//      of M, dx/dy/dz the cell's exact position steps), so the sums U = sum g u and W = sum g u u^T are
//      accumulated through the cell's index moments of g (sum g, sum g ix, sum g ix iy, ...) instead of
//      per voxel: 59 instructions per cell instead of 96, no branches (a miss has G = 0);
//   4. finishes with one transposing butterfly and writes the 128-byte row of moment sums, which
//      k_finalize turns into (dv, dw, U, W, E).
// Gaussians are processed in the Morton order of their central brick so that the per-sample
// coefficients of neighbouring Gaussians stay in L1/L2.
//
// Per-sample coefficients: PACK2 = float2 (alpha, beta) written by the fused-MSE forward, where the error
// share is eps = |alpha| * eps_scale; otherwise float4 (alpha, beta, eps, -) written by k_pack_samples.
#include <type_traits>

#include "gs_internal.cuh"
#include "pair_math.cuh"
#include "f32x2.cuh"

namespace gs {

// per-sample coefficients (one pass over the batch):  alpha = covered ? a/I : 0,  beta = b - alpha Phi,
// eps = covered ? |Phi - t| / I : 0   (PAPER.md:130 lists the inputs I_c, V_c, dL/dI_c, dL/dV_c)
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

#ifndef GS_BWD_WARPS
#define GS_BWD_WARPS 4
#define GS_BWD_MINB 4
#define GS_BWD_GPW 8
#define GS_BWD_INTERLEAVE 1
#endif
constexpr int BWD_WARPS = GS_BWD_WARPS;
constexpr int BWD_MINB = GS_BWD_MINB;  // resident CTAs per SM the register allocation must allow
constexpr int GPW_MANY = GS_BWD_GPW;   // Gaussians per warp when the batch touches many Gaussians (launch sized by Gaussians / (warps x GPW))
constexpr int GPW_FEW = 1;             // ... when it touches few (configs[3] batches: ~10 k): one Gaussian per warp keeps every SM busy
constexpr bool INTERLEAVE = GS_BWD_INTERLEAVE;  // the warps of a CTA take neighbouring Gaussians of the order list at the same time
constexpr int QCAP = 512;  // per-warp ring of surviving cells (power of two, >= 31 + 32 * SLICE)
constexpr int SLICE = 8;   // cells of its interval a lane pushes per pass

// Row of moment sums of one Gaussian (GACC_GRID floats; the weight w is factored out of all of them and applied by
// k_finalize).  With g = gamma G, gamma = alpha v + beta, per cell m000 = sum g, a100 = dx sum_{ix=1} g, a200 = dx a100,
// a110 = dx dy sum_{ix=iy=1} g, ... and u0 = u(voxel 0 of the cell):
//   0 sum alpha G | 1 sum g | 2 sum eps G | 3..5 sum m000 u0 | 6..8 sum (a100, a010, a001) | 9..14 sum m000 u0 u0^T (00 01 02 11 12 22)
//   15..17 sum a100 u0 | 18..20 sum a010 u0 | 21..23 sum a001 u0 | 24..29 sum (a200, a020, a002, a110, a101, a011) | 30, 31 unused
// Transposing butterfly over 32 values: afterwards lane L holds in v[0] the warp-wide sum of component L (31 SHFL).
__device__ __forceinline__ void warp_reduce32(float (&v)[32], int lane) {
#pragma unroll
    for (int h = 16; h >= 1; h >>= 1) {
        const bool up = lane & h;
#pragma unroll
        for (int k = 0; k < h; k++) {
            const float send = up ? v[k] : v[k + h];
            const float keep = up ? v[k + h] : v[k];
            v[k] = keep + __shfl_xor_sync(0xffffffffu, send, h);
        }
    }
}

template <bool PACK2, bool JIT, bool ASYNC, int GPW>
__global__ void __launch_bounds__(BWD_WARPS * 32, BWD_MINB) k_grid_bwd(const float4 *__restrict__ rec, const float4 *__restrict__ setup, uint32_t N,
                                                              GridDesc gd, const void *__restrict__ pack_, float r2,
                                                              float *__restrict__ gacc, const uint32_t *__restrict__ order,
                                                              uint32_t M, const float4 *__restrict__ jit /*JIT: per-voxel sample positions*/, DevCount dc) {
    __shared__ uint32_t queue[BWD_WARPS][QCAP];
    // records (4 planes) + setup rows (2) of the Gaussian being processed and of the next one: copied asynchronously one
    // Gaussian ahead, so that a Gaussian starts from shared memory instead of six dependent L2 round trips
    __shared__ float4 gstage[BWD_WARPS][2][8];
    __shared__ __align__(16) float red[BWD_WARPS][32][32];   // the 32 x 32 transpose of the final reduction
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // a warp processes GPW consecutive Gaussians of the brick-ordered list of the M Gaussians that touch the batch
    // slot `rep` of this warp is entry w0 + rep * wstride of the order list
    if (ASYNC) {   // asynchronous build: M lives on the device; nothing to do if the pair list overflowed its buffer
        if (dc.total[0] > (unsigned long long)dc.cap) return;
        M = (uint32_t)dc.total[1];
    }
    const uint32_t wstride = INTERLEAVE ? BWD_WARPS : 1;
    // the launch covers every entry of the order list when the host knew M; with a device-side M the CTAs stride over it
    for (uint32_t cta = blockIdx.x; ASYNC ? (uint64_t)cta * (BWD_WARPS * GPW) < M : cta == blockIdx.x; cta += gridDim.x) {
    const uint32_t w0 = INTERLEAVE ? cta * (BWD_WARPS * GPW) + warp : (cta * BWD_WARPS + warp) * GPW;
    if (w0 >= M) return;  // whole warps leave; no block-wide barrier is used below (later CTA slots start beyond this one)
    const uint32_t my_id = (lane < GPW && w0 + lane * wstride < M) ? order[w0 + lane * wstride] : 0u;
    const uint32_t bdx = (uint32_t)gd.bdim[0], bdy = (uint32_t)gd.bdim[1];
    int first[3], last[3];
#pragma unroll
    for (int k = 0; k < 3; k++) {
        first[k] = BRICK * gd.brick_lo[k];
        last[k] = BRICK * gd.brick_lo[k] + gd.bdim[k] - 1;
    }
    const bool odd_x = (gd.bdim[0] & 1) != 0;  // x-pairs of coefficients are 16-byte aligned only for an even x extent
    uint32_t *q = queue[warp];

    // lane l < 6 copies piece l of Gaussian `id` (planes a..d, setup rows 0..1) into stage buffer `buf`
    auto fetch = [&](uint32_t id, int buf) {
        if (lane < 6) {
            const float4 *src = lane < 4 ? rec + (size_t)lane * N + id : setup + 2 * (size_t)id + (lane - 4);
            const unsigned dst = (unsigned)__cvta_generic_to_shared(&gstage[warp][buf][lane]);
            asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    fetch(__shfl_sync(0xffffffffu, my_id, 0), 0);
    for (int rep = 0; rep < GPW && w0 + rep * wstride < M; rep++) {
    const uint32_t i = __shfl_sync(0xffffffffu, my_id, rep);
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncwarp();
    const float4 *gs_ = gstage[warp][rep & 1];
    const float4 ga = gs_[0], gb = gs_[1], gc = gs_[2], gd4 = gs_[3];
    // cell box of the AABB inside the batch, cull threshold and 1 / |e|^2: precomputed per Gaussian (k_brick_count)
    const float4 s0 = gs_[4], s1 = gs_[5];
    if (rep + 1 < GPW && w0 + (rep + 1) * wstride < M) fetch(__shfl_sync(0xffffffffu, my_id, rep + 1), (rep + 1) & 1);
    const int clo[3] = {__float_as_int(s0.x), __float_as_int(s0.y), __float_as_int(s0.z)};
    const uint32_t flags = __float_as_uint(s0.w), ncp = __float_as_uint(s1.x);
    if (flags & 1u) {  // touches a brick of the batch but none of its voxels: a zero row (rows are not pre-zeroed)
        gacc[(size_t)i * GACC_GRID + lane] = 0.f;
        continue;
    }
    const bool edge = (flags & 2u) || odd_x;
    const int ncx = (int)(ncp & 1023u) + 1, ncy = (int)((ncp >> 10) & 1023u) + 1, ncz = (int)((ncp >> 20) & 1023u) + 1;
    const float thr = s1.y, invA = s1.z;

    float acc[32];
#pragma unroll
    for (int k = 0; k < 32; k++) acc[k] = 0.f;

    // evaluate one cell per lane: code = cell coordinates relative to clo (x | y << 10 | z << 20).
    // EDGE = some cell of this Gaussian may stick out of the batch.  Voxels outside the batch and idle lanes (which
    // re-evaluate cell 0) get zero coefficients, so whatever their G is, they add nothing.
    auto process = [&](uint32_t code, bool on, auto edge_tag) {
        constexpr bool EDGE = decltype(edge_tag)::value;
        const int X = 2 * (clo[0] + (int)(code & 1023u)), Y = 2 * (clo[1] + (int)((code >> 10) & 1023u)), Z = 2 * (clo[2] + (int)(code >> 20));
        // 32-bit sample index (P < 2^32) of the cell's first voxel
        const uint32_t base = ((uint32_t)(Z - first[2]) * bdy + (uint32_t)(Y - first[1])) * bdx + (uint32_t)(X - first[0]);
        // per-sample coefficients of the 8 voxels: issued up front (no data dependence on the predicate), so their
        // L1/L2 latency overlaps the arithmetic below
        // PACK2: al2[r] / be2[r] = (alpha, beta) of the row's two x-neighbours in packed halves (pair layout of pack2_index)
        f2 al2[4], be2[4];
        float ep[8];
        if (!EDGE && PACK2) {
            const float4 *p4 = reinterpret_cast<const float4 *>(pack_);
#pragma unroll
            for (int r = 0; r < 4; r++) {  // (y, z) rows of the cell: one 16-byte load per x-pair
                const uint32_t c = base + ((uint32_t)(r >> 1) * bdy + (uint32_t)(r & 1)) * bdx;
                const float4 s = on ? __ldg(p4 + (c >> 1)) : make_float4(0.f, 0.f, 0.f, 0.f);
                al2[r] = pk(s.x, s.y); be2[r] = pk(s.z, s.w);
            }
        } else {
            bool okx[2], oky[2], okz[2];
#pragma unroll
            for (int d = 0; d < 2; d++) {
                okx[d] = !EDGE || X + d <= last[0];
                oky[d] = !EDGE || Y + d <= last[1];
                okz[d] = !EDGE || Z + d <= last[2];
            }
            float al[8], be[8];
#pragma unroll
            for (int v = 0; v < 8; v++) {
                const uint32_t c = base + ((uint32_t)(v >> 2) * bdy + (uint32_t)((v >> 1) & 1)) * bdx + (uint32_t)(v & 1);
                const bool ok = on && okx[v & 1] && oky[(v >> 1) & 1] && okz[v >> 2];
                if (PACK2) {
                    const float *pf = reinterpret_cast<const float *>(pack_) + pack2_index(c);
                    al[v] = ok ? __ldg(pf) : 0.f; be[v] = ok ? __ldg(pf + 2) : 0.f;
                } else {
                    const float4 s = ok ? __ldg(reinterpret_cast<const float4 *>(pack_) + c) : make_float4(0.f, 0.f, 0.f, 0.f);
                    al[v] = s.x; be[v] = s.y; ep[v] = s.z;
                }
            }
#pragma unroll
            for (int r = 0; r < 4; r++) { al2[r] = pk(al[2 * r], al[2 * r + 1]); be2[r] = pk(be[2 * r], be[2 * r + 1]); }
        }
        if (JIT) {
            // jittered samples (D26): no two voxels of the cell share a coordinate and u is not affine in the
            // voxel index, so every voxel is its own "cell" of the moment sums: m000 = g, u0 = u(voxel), no index moments
#pragma unroll
            for (int v = 0; v < 8; v++) {
                const int gx = X + (v & 1), gy = Y + ((v >> 1) & 1), gz = Z + (v >> 2);
                // the voxel's sample position from the per-step table (a voxel outside the batch has zero coefficients: any
                // finite position will do)
                const bool inb = gx <= last[0] && gy <= last[1] && gz <= last[2];
                const uint32_t cv = base + ((uint32_t)(v >> 2) * bdy + (uint32_t)((v >> 1) & 1)) * bdx + (uint32_t)(v & 1);
                const float4 sp = (on && inb) ? __ldg(jit + cv) : make_float4(0.f, 0.f, 0.f, 0.f);
                const float dxv = __fsub_rn(sp.x, ga.x), dyv = __fsub_rn(sp.y, ga.y), dzv = __fsub_rn(sp.z, ga.z);
                const float u0 = __fmaf_rn(gb.z, dzv, __fmaf_rn(gb.y, dyv, __fmul_rn(gb.x, dxv)));
                const float u1 = __fmaf_rn(gc.z, dzv, __fmaf_rn(gc.y, dyv, __fmul_rn(gc.x, dxv)));
                const float u2 = __fmaf_rn(gd4.z, dzv, __fmaf_rn(gd4.y, dyv, __fmul_rn(gd4.x, dxv)));
                const float qd = __fmaf_rn(u2, u2, __fmaf_rn(u1, u1, __fmul_rn(u0, u0)));
                const float G = qd <= r2 ? gauss_weight(qd) : 0.f;
                const float alv = (v & 1) ? hi(al2[v >> 1]) : lo(al2[v >> 1]), bev = (v & 1) ? hi(be2[v >> 1]) : lo(be2[v >> 1]);
                const float gg = fmaf(alv, gb.w, bev) * G;
                acc[0] = fmaf(alv, G, acc[0]);
                acc[2] = fmaf(PACK2 ? fabsf(alv) : ep[v], G, acc[2]);
                acc[1] += gg;
                const float t0 = gg * u0, t1 = gg * u1, t2 = gg * u2;
                acc[3] += t0; acc[4] += t1; acc[5] += t2;
                acc[9] = fmaf(t0, u0, acc[9]); acc[10] = fmaf(t0, u1, acc[10]); acc[11] = fmaf(t0, u2, acc[11]);
                acc[12] = fmaf(t1, u1, acc[12]); acc[13] = fmaf(t1, u2, acc[13]); acc[14] = fmaf(t2, u2, acc[14]);
            }
            return;
        }
        // canonical positions (D6) and sequence (D4), packed over the x-neighbours (f32x2.cuh) with the sub-expressions
        // shared between voxels of equal x / equal (x, y): u_j = fma(M_j2, dz, fma(M_j1, dy, M_j0 * dx))
        float dx[2], dy[2], dz[2];
        const f2 dx2 = sub2(pk(voxel_centre(X, gd.spacing[0], gd.origin[0]), voxel_centre(X + 1, gd.spacing[0], gd.origin[0])), bc(ga.x));
        upk(dx2, dx[0], dx[1]);
        upk(sub2(pk(voxel_centre(Y, gd.spacing[1], gd.origin[1]), voxel_centre(Y + 1, gd.spacing[1], gd.origin[1])), bc(ga.y)), dy[0], dy[1]);
        upk(sub2(pk(voxel_centre(Z, gd.spacing[2], gd.origin[2]), voxel_centre(Z + 1, gd.spacing[2], gd.origin[2])), bc(ga.z)), dz[0], dz[1]);
        f2 qd[4];   // pair r = (y, z) row of the cell: voxels 2r, 2r + 1
        float c0 = 0.f, c1 = 0.f, c2 = 0.f;  // c = u(voxel 0)
#pragma unroll
        for (int row = 0; row < 3; row++) {
            const float4 mr = row == 0 ? gb : row == 1 ? gc : gd4;
            const f2 a2 = mul2(bc(mr.x), dx2);
            f2 ab[2];
#pragma unroll
            for (int iy = 0; iy < 2; iy++) ab[iy] = fma2(bc(mr.y), bc(dy[iy]), a2);
#pragma unroll
            for (int r = 0; r < 4; r++) {  // r = y | z << 1
                const f2 u = fma2(bc(mr.z), bc(dz[r >> 1]), ab[r & 1]);
                if (r == 0) { if (row == 0) c0 = lo(u); else if (row == 1) c1 = lo(u); else c2 = lo(u); }
                qd[r] = row == 0 ? mul2(u, u) : fma2(u, u, qd[r]);
            }
        }
        // g = gamma G per voxel (G = 0 for a miss: the canonical predicate decides membership); the coefficients are first
        // needed here, a whole cell's worth of arithmetic after their loads were issued
        f2 g2[4], a0 = pk(0.f, 0.f);
        float g[8];
#pragma unroll
        for (int r = 0; r < 4; r++) {
            bool h0, h1;
            const f2 G = gauss_weight2(qd[r], r2, h0, h1);
            g2[r] = mul2(fma2(al2[r], bc(gb.w), be2[r]), G);
            a0 = fma2(al2[r], G, a0);
            float G0, G1;
            upk(G, G0, G1);
            acc[2] = fmaf(PACK2 ? fabsf(lo(al2[r])) : ep[2 * r], G0, acc[2]);
            acc[2] = fmaf(PACK2 ? fabsf(hi(al2[r])) : ep[2 * r + 1], G1, acc[2]);
            upk(g2[r], g[2 * r], g[2 * r + 1]);
        }
        acc[0] += lo(a0) + hi(a0);
        // index moments of g over the cell
        const f2 sA = add2(g2[0], g2[1]), sB = add2(g2[2], g2[3]), sS = add2(sA, sB), sT = add2(g2[1], g2[3]);
        const float m100 = hi(sS), m000 = lo(sS) + m100, m110 = hi(sT), m010 = lo(sT) + m110, m101 = hi(sB), m001 = lo(sB) + m101,
                    m011 = g[6] + g[7];
        // exact position steps of this cell (the canonical positions are rounded, so they differ from the spacing by an ulp)
        const float ex = dx[1] - dx[0], ey = dy[1] - dy[0], ez = dz[1] - dz[0];
        const float a100 = m100 * ex, a010 = m010 * ey, a001 = m001 * ez;
        acc[1] += m000;
        const float t0 = m000 * c0, t1 = m000 * c1, t2 = m000 * c2;
        acc[3] += t0; acc[4] += t1; acc[5] += t2;
        acc[6] += a100; acc[7] += a010; acc[8] += a001;
        acc[9] = fmaf(t0, c0, acc[9]); acc[10] = fmaf(t0, c1, acc[10]); acc[11] = fmaf(t0, c2, acc[11]);
        acc[12] = fmaf(t1, c1, acc[12]); acc[13] = fmaf(t1, c2, acc[13]); acc[14] = fmaf(t2, c2, acc[14]);
        acc[15] = fmaf(a100, c0, acc[15]); acc[16] = fmaf(a100, c1, acc[16]); acc[17] = fmaf(a100, c2, acc[17]);
        acc[18] = fmaf(a010, c0, acc[18]); acc[19] = fmaf(a010, c1, acc[19]); acc[20] = fmaf(a010, c2, acc[20]);
        acc[21] = fmaf(a001, c0, acc[21]); acc[22] = fmaf(a001, c1, acc[22]); acc[23] = fmaf(a001, c2, acc[23]);
        acc[24] = fmaf(a100, ex, acc[24]); acc[25] = fmaf(a010, ey, acc[25]); acc[26] = fmaf(a001, ez, acc[26]);
        acc[27] = fmaf(m110 * ex, ey, acc[27]); acc[28] = fmaf(m101 * ex, ez, acc[28]); acc[29] = fmaf(m011 * ey, ez, acc[29]);
    };

    // ---- enumeration: lane = row (y, z) of cells.  Along the row the cell centre moves by 2 voxels in x:
    // u(cx) = u_row + cx * e, e = M[:,0] * 2 sx.  |u(cx)|^2 <= thr  <=>  |cx - cx*| <= sqrt((thr - Dmin) / |e|^2),
    // cx* = -(u_row . e) / |e|^2 the closest approach and Dmin = |u(cx*)|^2 (evaluated from the vector: no cancellation).
    const int nrows = ncy * ncz;
    const float sx2 = 2.f * gd.spacing[0];
    const float e0 = gb.x * sx2, e1 = gc.x * sx2, e2 = gd4.x * sx2;
    const float ccx0 = fmaf((float)(2 * clo[0] + 1), gd.spacing[0], gd.origin[0]) - ga.x;
    uint32_t head = 0, qn = 0;  // warp-uniform
    auto drain = [&](uint32_t keep) {
        while (qn > keep) {
            const bool on = (uint32_t)lane < qn;
            const uint32_t code = on ? q[(head + lane) & (QCAP - 1)] : 0u;
            __syncwarp();
            if (edge) process(code, on, std::true_type{});
            else process(code, on, std::false_type{});
            const uint32_t used = qn < 32u ? qn : 32u;
            head = (head + used) & (QCAP - 1);
            qn -= used;
        }
    };
    for (int rbase = 0; rbase < nrows; rbase += 32) {
        const int r = rbase + lane;
        const int z = r / ncy, y = r - z * ncy;
        const float ccy = fmaf((float)(2 * (clo[1] + y) + 1), gd.spacing[1], gd.origin[1]) - ga.y;
        const float ccz = fmaf((float)(2 * (clo[2] + z) + 1), gd.spacing[2], gd.origin[2]) - ga.z;
        const float u0 = gb.x * ccx0 + gb.y * ccy + gb.z * ccz;
        const float u1 = gc.x * ccx0 + gc.y * ccy + gc.z * ccz;
        const float u2 = gd4.x * ccx0 + gd4.y * ccy + gd4.z * ccz;
        const float cs = -(u0 * e0 + u1 * e1 + u2 * e2) * invA;
        const float v0 = fmaf(cs, e0, u0), v1 = fmaf(cs, e1, u1), v2 = fmaf(cs, e2, u2);
        const float room = thr - (v0 * v0 + v1 * v1 + v2 * v2);
        int x = 0, remaining = 0;
        if (r < nrows && room >= 0.f) {
            const float hw = sqrtf(room * invA) + 2e-3f + 1e-6f * fabsf(cs);
            const float flo = fmaxf(ceilf(cs - hw), 0.f), fhi = fminf(floorf(cs + hw), (float)(ncx - 1));
            if (flo <= fhi) { x = (int)flo; remaining = (int)fhi - x + 1; }
        }
        while (__any_sync(0xffffffffu, remaining > 0)) {
            const int take = remaining < SLICE ? remaining : SLICE;
            int incl = take;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, incl, d);
                if (lane >= d) incl += t;
            }
            const uint32_t total = (uint32_t)__shfl_sync(0xffffffffu, incl, 31);
            const uint32_t pos = head + qn + (uint32_t)(incl - take);
            const uint32_t code0 = (uint32_t)x | ((uint32_t)y << 10) | ((uint32_t)z << 20);
#pragma unroll
            for (int j = 0; j < SLICE; j++)
                if (j < take) q[(pos + j) & (QCAP - 1)] = code0 + j;
            qn += total;
            x += take;
            remaining -= take;
            __syncwarp();
            drain(31u);
        }
    }
    drain(0u);

    // Reduction over the lanes through a 32 x 32 transpose in shared memory: lane L stores its 32 partial sums as row L
    // (16-byte chunks swizzled by L & 7: conflict-free per quarter warp), then sums column L (for a fixed row the 32 lanes read
    // the 32 distinct words of one 128-byte row).  8 STS.128 + 32 LDS + 32 FADD instead of the 31-shuffle butterfly with its
    // 62 selects; the summation order is fixed, so the result stays bit-deterministic.
    {
        float4 *row = reinterpret_cast<float4 *>(red[warp][lane]);
#pragma unroll
        for (int k = 0; k < 8; k++) row[k ^ (lane & 7)] = make_float4(acc[4 * k], acc[4 * k + 1], acc[4 * k + 2], acc[4 * k + 3]);
        __syncwarp();
        const int kc = lane >> 2, e = lane & 3;
        float s4[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int r = 0; r < 32; r++) s4[r & 3] += red[warp][r][((kc ^ (r & 7)) << 2) | e];
        // lane c holds component c: one coalesced 128-byte row per Gaussian
        gacc[(size_t)i * GACC_GRID + lane] = (s4[0] + s4[1]) + (s4[2] + s4[3]);
        __syncwarp();
    }
    }  // rep
    }  // cta slot
}

cudaError_t launch_pack_samples(const BwdIn &in, size_t P, float tau, float4 *pack, cudaStream_t s) {
    if (P == 0) return cudaSuccess;
    k_pack_samples<<<(unsigned)((P + 255) / 256), 256, 0, s>>>(in.phi, in.I, in.dL_dphi, in.dL_dI, in.target, P, tau, pack);
    count_launch();
    return cudaGetLastError();
}

cudaError_t launch_grid_bwd(const float4 *rec, const float4 *setup, uint32_t N, const GridDesc &gd, const void *pack, bool pack2,
                            float r2, float *gacc, const uint32_t *order, uint32_t M, const float4 *jit, DevCount dc, cudaStream_t s) {
    // only the M Gaussians of the order list get (and need) an accumulator row: k_finalize reads those alone
    if (M == 0) return cudaSuccess;
    // few Gaussians (the launch bound M of a small batch): one per warp, so that the launch has enough CTAs for every SM
    const bool few = M < 148u * BWD_MINB * BWD_WARPS * GPW_MANY;
    const int gpw = few ? GPW_FEW : GPW_MANY;
    const unsigned blocks = (M + BWD_WARPS * gpw - 1) / (BWD_WARPS * gpw);
#define GS_BWD_LAUNCH(P2_, JIT_, ASYNC_) \
    do { if (few) k_grid_bwd<P2_, JIT_, ASYNC_, GPW_FEW><<<blocks, BWD_WARPS * 32, 0, s>>>(rec, setup, N, gd, pack, r2, gacc, order, M, jit, dc); \
         else k_grid_bwd<P2_, JIT_, ASYNC_, GPW_MANY><<<blocks, BWD_WARPS * 32, 0, s>>>(rec, setup, N, gd, pack, r2, gacc, order, M, jit, dc); } while (0)
    const bool as = dc.total != nullptr;
    if (gd.jitter) {
        if (pack2) { if (as) GS_BWD_LAUNCH(true, true, true); else GS_BWD_LAUNCH(true, true, false); }
        else { if (as) GS_BWD_LAUNCH(false, true, true); else GS_BWD_LAUNCH(false, true, false); }
    } else {
        if (pack2) { if (as) GS_BWD_LAUNCH(true, false, true); else GS_BWD_LAUNCH(true, false, false); }
        else { if (as) GS_BWD_LAUNCH(false, false, true); else GS_BWD_LAUNCH(false, false, false); }
    }
#undef GS_BWD_LAUNCH
    count_launch();
    return cudaGetLastError();
}

}  // namespace gs
