// sample_grid_fwd.cu -- structured forward (S4 + S6; section 4.1.3).
//
// One CTA (2 warps) per 8^3 brick.  The brick's Gaussian list (S2) is staged into shared memory with
// cp.async ("each thread block cooperatively loads a batch of Gaussians ... into shared memory").
// Below the brick the kernel culls per CELL of 2x2x2 voxels:
//   * list building: lane = Gaussian; it tests its Gaussian against the warp's 32 cells with a
//     conservative whitened-space bound and a ballot per cell produces the cell's bit mask
//     (|u0 + ix ex|^2 is expanded per cell row, so a cell costs ~2 FFMA + compare + vote);
//   * evaluation: lane = cell; the lane walks its own masks and evaluates its 8 voxels against each
//     listed Gaussian.  The canonical fp32 predicate sequence (D4) shares sub-expressions between
//     voxels with equal x / y coordinates, so 8 voxel tests cost 72 FP32 instructions instead of 136
//     with bit-identical results.
// Epilogue S6 is fused: coverage rule, normalisation, MSE partial sums, dL/dPhi, per-sample error.
#include "gs_internal.cuh"
#include "pair_math.cuh"
#include "f32x2.cuh"

namespace gs {

#ifndef GS_FWD_MINB
#define GS_FWD_MINB 12  // resident CTAs per SM the register allocation must allow (swept 10, 12, 14, 16 with the packed list building)
#endif
constexpr int FWD_THREADS = 64;
constexpr int CAP = 128;  // Gaussians staged per round (4 sub-chunks of 32)

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;" ::: "memory"); }

template <bool SETS, bool JIT, bool ASYNC>
__global__ void __launch_bounds__(FWD_THREADS, GS_FWD_MINB) k_grid_fwd(const float4 *__restrict__ rec, uint32_t N, GridDesc gd,
                                                           const uint32_t *__restrict__ pair_gauss,
                                                           const uint32_t *__restrict__ brick_start, float tau, float r2, FwdOut o,
                                                           double invP, const float4 *__restrict__ jit /*JIT: per-voxel sample positions*/, DevCount dc) {
    __shared__ float4 srec[4][CAP];
    __shared__ uint32_t sid[CAP];
    __shared__ uint4 smask[FWD_THREADS / 32][32];  // [warp][cell] -> masks of the 4 sub-chunks
    if (ASYNC && dc.total[0] > (unsigned long long)dc.cap) {   // the speculative pair list did not fit: nothing valid to read
        // the status only reaches the host with a later call; a NaN loss tells the caller in band that this batch did not happen
        if (blockIdx.x == 0 && threadIdx.x == 0) {
            const double nan = __longlong_as_double(0x7ff8000000000000ll);
            if (o.gen.on) atomicAdd(o.gen.sums, nan);
            else if (o.target && o.loss) atomicAdd(o.loss, nan);
        }
        return;
    }
    const uint32_t b = blockIdx.x;
    const int bx = b % gd.brick_cnt[0], by = (b / gd.brick_cnt[0]) % gd.brick_cnt[1], bz = b / (gd.brick_cnt[0] * gd.brick_cnt[1]);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // lane = cell (cx, cy, cz) of the warp's 4 x 4 x 2 cell block; cell = 2 x 2 x 2 voxels
    const int cx = lane & 3, cy = (lane >> 2) & 3, cz = 2 * warp + (lane >> 4);
    const int lx = bx * BRICK + 2 * cx, ly = by * BRICK + 2 * cy, lz = bz * BRICK + 2 * cz;  // batch-local first voxel
    const float nanv = __int_as_float(0x7fc00000);
    // canonical sample positions (D6); voxels clipped by the grid get NaN, which fails every predicate
    float px[2], py[2], pz[2];
#pragma unroll
    for (int d = 0; d < 2; d++) {
        px[d] = (lx + d < gd.bdim[0]) ? voxel_centre(lx + d + BRICK * gd.brick_lo[0], gd.spacing[0], gd.origin[0]) : nanv;
        py[d] = (ly + d < gd.bdim[1]) ? voxel_centre(ly + d + BRICK * gd.brick_lo[1], gd.spacing[1], gd.origin[1]) : nanv;
        pz[d] = (lz + d < gd.bdim[2]) ? voxel_centre(lz + d + BRICK * gd.brick_lo[2], gd.spacing[2], gd.origin[2]) : nanv;
    }
    // the two x-neighbours of a row ride in the halves of one packed register (f32x2.cuh)
    const f2 px2 = pk(px[0], px[1]), py2 = pk(py[0], py[1]), pz2 = pk(pz[0], pz[1]);
    // JIT: every voxel has its own position inside its cell (D26); pair r = voxels (2r, 2r + 1), v = x | y << 1 | z << 2
    f2 jp[JIT ? 4 : 1][3];
    if (JIT) {
#pragma unroll
        for (int r = 0; r < 4; r++) {
            float c[2][3];
#pragma unroll
            for (int d = 0; d < 2; d++) {
                const int x = lx + d, y = ly + (r & 1), z = lz + (r >> 1);
                const bool in = x < gd.bdim[0] && y < gd.bdim[1] && z < gd.bdim[2];
                float4 sp = make_float4(nanv, nanv, nanv, 0.f);
                if (in) sp = jit[((uint32_t)z * (uint32_t)gd.bdim[1] + (uint32_t)y) * (uint32_t)gd.bdim[0] + (uint32_t)x];
                c[d][0] = sp.x; c[d][1] = sp.y; c[d][2] = sp.z;
            }
            jp[r][0] = pk(c[0][0], c[1][0]); jp[r][1] = pk(c[0][1], c[1][1]); jp[r][2] = pk(c[0][2], c[1][2]);
        }
    }
    // cull geometry (not canonical): centre of the warp's cell (0,0,0), cell pitch = 2 voxels, half extent = half a voxel
    const float c0x = fmaf((float)(BRICK * (bx + gd.brick_lo[0]) + 1), gd.spacing[0], gd.origin[0]);
    const float c0y = fmaf((float)(BRICK * (by + gd.brick_lo[1]) + 1), gd.spacing[1], gd.origin[1]);
    const float c0z = fmaf((float)(BRICK * (bz + gd.brick_lo[2]) + 4 * warp + 1), gd.spacing[2], gd.origin[2]);
    // half extent of a cell's samples around the cell centre: half a voxel, a whole one when they are jittered
    const float hh = JIT ? 1.0f : 0.5f;
    const float hx = hh * gd.spacing[0], hy = hh * gd.spacing[1], hz = hh * gd.spacing[2];
    const float rcut = sqrtf(r2);

    f2 I2[4], N2[4];   // pair r = voxels (2r, 2r + 1) of the cell
    uint32_t cnt[SETS ? 8 : 1], ntest = 0;
    unsigned long long hsum[SETS ? 8 : 1], hxor[SETS ? 8 : 1];
#pragma unroll
    for (int r = 0; r < 4; r++) { I2[r] = pk(0.f, 0.f); N2[r] = pk(0.f, 0.f); }
    if (SETS) {
#pragma unroll
        for (int v = 0; v < 8; v++) { cnt[v] = 0; hsum[v] = 0; hxor[v] = 0; }
    }

    const uint32_t start = brick_start[b], n = brick_start[b + 1] - start;
    const uint32_t *list = pair_gauss + start;
    uint32_t *mywords = reinterpret_cast<uint32_t *>(&smask[warp][0]);
    for (uint32_t round = 0; round < n; round += CAP) {
        const int m = min((uint32_t)CAP, n - round);
        if (round) __syncthreads();  // everyone is done with the previous round's records
        for (int j = threadIdx.x; j < m; j += FWD_THREADS) {
            const uint32_t id = list[round + j];
            cp_async16(&srec[0][j], rec + id);
            cp_async16(&srec[1][j], rec + (size_t)N + id);
            cp_async16(&srec[2][j], rec + 2 * (size_t)N + id);
            cp_async16(&srec[3][j], rec + 3 * (size_t)N + id);
            if (SETS) sid[j] = id;
        }
        smask[warp][lane] = make_uint4(0u, 0u, 0u, 0u);
        cp_async_wait_all();
        __syncthreads();
        // ---- list building: lane = Gaussian sub + lane, against the warp's 32 cells.
        // For a cell with centre cc and half extent h (its voxel centres are cc +- h) every voxel p obeys
        // |M(p - mu)| >= |M(cc - mu)| - rho, rho = |(sum_k |M_jk| h_k)_j|, so the cell holds no hit unless
        // |M(cc - mu)|^2 <= (r + rho)^2.  2^-9 slack covers fp32 rounding; the canonical predicate decides.
        for (int sub = 0; sub < m; sub += 32) {
            const int j = sub + lane;
            const bool have = j < m;
            const int js = have ? j : 0;
            const float4 ga = srec[0][js], gb = srec[1][js], gc = srec[2][js], gd4 = srec[3][js];
            const float q0 = fabsf(gb.x) * hx + fabsf(gb.y) * hy + fabsf(gb.z) * hz;
            const float q1 = fabsf(gc.x) * hx + fabsf(gc.y) * hy + fabsf(gc.z) * hz;
            const float q2 = fabsf(gd4.x) * hx + fabsf(gd4.y) * hy + fabsf(gd4.z) * hz;
            const float reach = rcut + sqrtf(q0 * q0 + q1 * q1 + q2 * q2);
            const float thr = have ? reach * reach * 1.001953125f : -1.f;
            const float dx0 = c0x - ga.x, dy0 = c0y - ga.y, dz0 = c0z - ga.z;
            const float ub0 = gb.x * dx0 + gb.y * dy0 + gb.z * dz0;
            const float ub1 = gc.x * dx0 + gc.y * dy0 + gc.z * dz0;
            const float ub2 = gd4.x * dx0 + gd4.y * dy0 + gd4.z * dz0;
            const float sx2 = 2.f * gd.spacing[0], sy2 = 2.f * gd.spacing[1], sz2 = 2.f * gd.spacing[2];
            const float ex0 = gb.x * sx2, ex1 = gc.x * sx2, ex2 = gd4.x * sx2;
            const float ey0 = gb.y * sy2, ey1 = gc.y * sy2, ey2 = gd4.y * sy2;
            const float ez0 = gb.z * sz2, ez1 = gc.z * sz2, ez2 = gd4.z * sz2;
            const float exx = ex0 * ex0 + ex1 * ex1 + ex2 * ex2;  // |ex|^2
            const int word = sub >> 5;
            // two y-rows of cells per packed instruction (f32x2.cuh; a cull bound, not the canonical sequence):
            // y = z + iy ey for iy = (0, 1) and (2, 3) in the halves; |y + ix ex|^2 = |y|^2 + ix (2 y.ex) + ix^2 |ex|^2
            const f2 ex0d = bc(2.f * ex0), ex1d = bc(2.f * ex1), ex2d = bc(2.f * ex2);
#pragma unroll
            for (int iz = 0; iz < 2; iz++) {
                const float z0 = fmaf((float)iz, ez0, ub0), z1 = fmaf((float)iz, ez1, ub1), z2 = fmaf((float)iz, ez2, ub2);
#pragma unroll
                for (int ip = 0; ip < 2; ip++) {   // row pair: iy = 2 ip, 2 ip + 1
                    const f2 iy2 = pk((float)(2 * ip), (float)(2 * ip + 1));
                    const f2 y0 = fma2(iy2, bc(ey0), bc(z0)), y1 = fma2(iy2, bc(ey1), bc(z1)), y2 = fma2(iy2, bc(ey2), bc(z2));
                    const f2 yy = fma2(y2, y2, fma2(y1, y1, mul2(y0, y0)));
                    const f2 ye = fma2(y2, ex2d, fma2(y1, ex1d, mul2(y0, ex0d)));
#pragma unroll
                    for (int ix = 0; ix < 4; ix++) {
                        float qa, qb;
                        upk(ix == 0 ? yy : fma2(bc((float)(ix * ix)), bc(exx), fma2(bc((float)ix), ye, yy)), qa, qb);
                        const uint32_t bala = __ballot_sync(0xffffffffu, qa <= thr), balb = __ballot_sync(0xffffffffu, qb <= thr);
                        if (lane == 0) {
                            mywords[4 * (iz * 16 + (2 * ip) * 4 + ix) + word] = bala;
                            mywords[4 * (iz * 16 + (2 * ip + 1) * 4 + ix) + word] = balb;
                        }
                    }
                }
            }
        }
        __syncwarp();
        // ---- evaluation: lane = cell, walking its own masks over the whole round; 8 voxels per listed Gaussian.
        // The 128-bit mask is walked as 32-bit words.  Empty words are squeezed out first (once per round), so that inside
        // the loop ONE predicated refill is enough whenever the current word runs dry (left > 0 => the next word has a bit).
        const uint4 mk = smask[warp][lane];
        uint32_t w0 = mk.x, w1 = mk.y, w2 = mk.z, w3 = mk.w;
        int b0 = 0, b1 = 32, b2 = 64, b3 = 96;
        if (w2 == 0u) { w2 = w3; b2 = b3; w3 = 0u; }
        if (w1 == 0u) { w1 = w2; b1 = b2; w2 = w3; b2 = b3; w3 = 0u; }
        if (w0 == 0u) { w0 = w1; b0 = b1; w1 = w2; b1 = b2; w2 = w3; b2 = b3; w3 = 0u; }
        for (int left = __popc(w0) + __popc(w1) + __popc(w2) + __popc(w3); left > 0; left--) {
            if (w0 == 0u) { w0 = w1; b0 = b1; w1 = w2; b1 = b2; w2 = w3; b2 = b3; }
            const int j = b0 + __ffs((int)w0) - 1;
            w0 &= w0 - 1u;
            const float4 ga = srec[0][j], gb = srec[1][j], gc = srec[2][j], gd4 = srec[3][j];
            // canonical sequence (D4): d = p - mu; u_j = fma(M_j2, dz, fma(M_j1, dy, M_j0 * dx)); qd = fma(u2, u2, fma(u1, u1, u0 * u0)),
            // packed over the x-neighbours (every packed instruction is the scalar one on both halves) and shared between the
            // voxels of equal x / equal (x, y): 36 packed instructions for the 8 voxels of the cell
            f2 qd[4];
            if (JIT) {  // no two voxels share a coordinate: the plain canonical sequence per pair
#pragma unroll
                for (int r = 0; r < 4; r++) {
                    f2 u0, u1, u2;
                    qd[r] = mahalanobis2(ga.x, ga.y, ga.z, gb.x, gb.y, gb.z, gc.x, gc.y, gc.z, gd4.x, gd4.y, gd4.z, jp[r][0], jp[r][1], jp[r][2], u0, u1, u2);
                }
            } else {
                const f2 dx2 = sub2(px2, bc(ga.x));
                float dy[2], dz[2];
                upk(sub2(py2, bc(ga.y)), dy[0], dy[1]);
                upk(sub2(pz2, bc(ga.z)), dz[0], dz[1]);
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
                        qd[r] = row == 0 ? mul2(u, u) : fma2(u, u, qd[r]);
                    }
                }
            }
            if (SETS) ntest += 8;
#pragma unroll
            for (int r = 0; r < 4; r++) {
                bool h0, h1;
                const f2 G = gauss_weight2(qd[r], r2, h0, h1);   // G = 0 for a miss
                I2[r] = fma2(bc(ga.w), G, I2[r]);
                N2[r] = fma2(bc(gd4.w), G, N2[r]);  // gd4.w = v w
                if (SETS) {
                    const unsigned long long h = mix64(sid[j]);
                    if (h0) { cnt[2 * r]++; hsum[2 * r] += h; hxor[2 * r] ^= h; }
                    if (h1) { cnt[2 * r + 1]++; hsum[2 * r + 1] += h; hxor[2 * r + 1] ^= h; }
                }
            }
        }
    }

    // ---- S6 epilogue: coverage rule I > tau (strict), empty value 0, I always written (D5)
    float res2 = 0.f;
    unsigned long long tested = 0, hits = 0;
    const float dscale = (float)(2.0 * invP);
    const uint32_t bdx = (uint32_t)gd.bdim[0], bdy = (uint32_t)gd.bdim[1];
    const bool vec2 = !SETS && !(bdx & 1u) && !o.gen.on && o.vec_ok;  // x-pairs are 8-byte aligned when the batch's x extent is even
    LossPartial lp;
    float I[8], Nacc[8];
#pragma unroll
    for (int r = 0; r < 4; r++) { upk(I2[r], I[2 * r], I[2 * r + 1]); upk(N2[r], Nacc[2 * r], Nacc[2 * r + 1]); }
#pragma unroll
    for (int r = 0; r < 4; r++) {  // the cell's four x-rows: (y, z) = (ly + (r & 1), lz + (r >> 1))
        const uint32_t y = (uint32_t)ly + (r & 1), z = (uint32_t)lz + (r >> 1);
        if (y >= bdy || z >= (uint32_t)gd.bdim[2] || (uint32_t)lx >= bdx) continue;
        const uint32_t c = (z * bdy + y) * bdx + (uint32_t)lx;  // P < 2^32
        float ph[2], Iv[2];
        bool cov[2];
#pragma unroll
        for (int d = 0; d < 2; d++) {
            const int v = r * 2 + d;
            cov[d] = I[v] > tau;
            ph[d] = cov[d] ? __fdividef(Nacc[v], I[v]) : 0.f;
            Iv[d] = I[v];
        }
        if (vec2) {
            *reinterpret_cast<float2 *>(o.phi + c) = make_float2(ph[0], ph[1]);
            *reinterpret_cast<float2 *>(o.I + c) = make_float2(Iv[0], Iv[1]);
            if (o.target) {
                const float2 t = *reinterpret_cast<const float2 *>(o.target + c);
                const float r0 = ph[0] - t.x, r1 = ph[1] - t.y;
                res2 = fmaf(r0, r0, fmaf(r1, r1, res2));
                if (o.dL_dphi) *reinterpret_cast<float2 *>(o.dL_dphi + c) = make_float2(cov[0] ? dscale * r0 : 0.f, cov[1] ? dscale * r1 : 0.f);
                if (o.sample_err) *reinterpret_cast<float2 *>(o.sample_err + c) = make_float2(fabsf(r0), fabsf(r1));
                if (o.pack2) {  // backward coefficients of the fused MSE: alpha = a / I, beta = -alpha Phi (eps = |alpha| P / 2)
                    const float a0 = cov[0] ? __fdividef(dscale * r0, Iv[0]) : 0.f, a1 = cov[1] ? __fdividef(dscale * r1, Iv[1]) : 0.f;
                    *reinterpret_cast<float4 *>(o.pack2 + c) = make_float4(a0, a1, -a0 * ph[0], -a1 * ph[1]);   // pair layout, see pack2_index
                }
            }
        } else {
#pragma unroll
            for (int d = 0; d < 2; d++) {
                if ((uint32_t)lx + d >= bdx) continue;
                const int v = r * 2 + d;
                o.phi[c + d] = ph[d];
                o.I[c + d] = Iv[d];
                if (o.gen.on) {
                    loss_sample(o.gen, c + d, ph[d], Iv[d], cov[d], tau, o.target, o.dL_dphi, o.sample_err, lp);
                } else if (o.target) {
                    const float res = ph[d] - o.target[c + d];
                    res2 = fmaf(res, res, res2);
                    if (o.dL_dphi) o.dL_dphi[c + d] = cov[d] ? dscale * res : 0.f;
                    if (o.sample_err) o.sample_err[c + d] = fabsf(res);
                    if (o.pack2) {
                        const float al = cov[d] ? __fdividef(dscale * res, Iv[d]) : 0.f;
                        float *pk2 = reinterpret_cast<float *>(o.pack2) + pack2_index(c + d);
                        pk2[0] = al; pk2[2] = -al * ph[d];
                    }
                }
                if (SETS) {
                    if (o.set_count) o.set_count[c + d] = cnt[v];
                    if (o.set_sum) o.set_sum[c + d] = hsum[v];
                    if (o.set_xor) o.set_xor[c + d] = hxor[v];
                    tested += ntest / 8;
                    hits += cnt[v];
                }
            }
        }
    }
    if (o.gen.on) loss_flush(o.gen, lp, lane);
    if (!o.gen.on && o.target && o.loss) {
        double s = (double)res2;
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
        if (lane == 0 && s != 0.0) atomicAdd(o.loss, s * invP);
    }
    if (SETS && o.counters) {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            tested += __shfl_xor_sync(0xffffffffu, tested, d);
            hits += __shfl_xor_sync(0xffffffffu, hits, d);
        }
        if (lane == 0) { atomicAdd(o.counters, tested); atomicAdd(o.counters + 1, hits); }
    }
}

cudaError_t launch_grid_fwd(const float4 *rec, uint32_t N, const GridDesc &gd, const uint32_t *pair_gauss,
                            const uint32_t *brick_start, float tau, float r2, const FwdOut &o, const float4 *jit, DevCount dc, cudaStream_t s) {
    const uint32_t nbricks = (uint32_t)gd.brick_cnt[0] * gd.brick_cnt[1] * gd.brick_cnt[2];
    if (nbricks == 0) return cudaSuccess;
    const double P = o.inv_count > 0.0 ? 1.0 / o.inv_count : (double)gd.bdim[0] * gd.bdim[1] * gd.bdim[2];
    const bool sets = o.set_count || o.set_sum || o.set_xor || o.counters;
#define GS_FWD_LAUNCH(SETS_, JIT_, ASYNC_) \
    k_grid_fwd<SETS_, JIT_, ASYNC_><<<nbricks, FWD_THREADS, 0, s>>>(rec, N, gd, pair_gauss, brick_start, tau, r2, o, 1.0 / P, jit, dc)
    const bool as = dc.total != nullptr;
    if (gd.jitter) {
        if (sets) { if (as) GS_FWD_LAUNCH(true, true, true); else GS_FWD_LAUNCH(true, true, false); }
        else { if (as) GS_FWD_LAUNCH(false, true, true); else GS_FWD_LAUNCH(false, true, false); }
    } else {
        if (sets) { if (as) GS_FWD_LAUNCH(true, false, true); else GS_FWD_LAUNCH(true, false, false); }
        else { if (as) GS_FWD_LAUNCH(false, false, true); else GS_FWD_LAUNCH(false, false, false); }
    }
#undef GS_FWD_LAUNCH
    count_launch();
    return cudaGetLastError();
}

}  // namespace gs
