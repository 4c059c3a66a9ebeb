// loss.cuh -- the paper's training losses in the forward epilogue (S6; gs_sample_fwd_loss in include/gs.h):
// L1 / MSE reconstruction over the defined samples, false-negative term Eq. 4,
// false-positive term Eq. 5.  The counts |D-| and |U+| that normalise Eq. 4 / Eq. 5 are only known
// after the last sample, so the epilogue writes dL/dI un-normalised (-lambda_fn on D-, +lambda_fp on U+: the sign
// names the class) and k_loss_finish divides by the counts.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gs {

struct GenLoss {
    int on;                      // 0: the fused-MSE epilogue of gs_sample_fwd
    int kind;                    // gs_loss_kind
    const uint8_t *defined;      // nullable
    float *dL_dI;                // nullable
    float4 *pack4;               // nullable (grid): backward coefficients (alpha, beta, eps, -) for gs_sample_bwd(dL_dphi = NULL)
    float lam_fn, thr_fn, lam_fp;
    float inv_nd;                // 1 / |D|
    double *sums;                // [3] sum_D rho(res) | sum_{D-} (thr - I) | sum_{U+} I
    unsigned long long *counts;  // [2] |D-| | |U+|
};

struct LossPartial {  // per-thread partial sums of the epilogue
    float rec = 0.f, fn = 0.f, fp = 0.f;
    uint32_t nfn = 0, nfp = 0;
};

// one sample: writes dL_dphi / dL_dI / sample_err (each nullable) and adds to the partial sums
__device__ __forceinline__ void loss_sample(const GenLoss &L, size_t c, float phi, float I, bool covered, float tau, const float *target,
                                            float *dL_dphi, float *sample_err, LossPartial &acc) {
    const bool def = L.defined ? L.defined[c] != 0 : true;
    float a = 0.f, b = 0.f, e = 0.f;
    if (def) {
        const float res = phi - target[c];
        e = fabsf(res);
        if (L.kind == GS_LOSS_L1) {
            acc.rec += e;
            if (covered) a = res > 0.f ? L.inv_nd : (res < 0.f ? -L.inv_nd : 0.f);
        } else {
            acc.rec = fmaf(res, res, acc.rec);
            if (covered) a = 2.f * res * L.inv_nd;
        }
        if (L.lam_fn > 0.f && I < L.thr_fn) {
            acc.fn += L.thr_fn - I;
            acc.nfn++;
            b = -L.lam_fn;
        }
    } else if (L.lam_fp > 0.f && I >= tau) {
        acc.fp += I;
        acc.nfp++;
        b = L.lam_fp;
    }
    if (dL_dphi) dL_dphi[c] = a;
    if (L.dL_dI) L.dL_dI[c] = b;
    if (sample_err) sample_err[c] = e;
    if (L.pack4) {  // alpha = a / I, beta = b - alpha Phi (b still un-normalised: kept in .w for k_loss_finish), eps = |res| / I
        const float inv = covered ? __fdividef(1.0f, I) : 0.f;
        const float alpha = a * inv;
        L.pack4[c] = make_float4(alpha, -alpha * phi, e * inv, b);
    }
}

// warp reduction of the partial sums, one atomic per non-zero term and warp
__device__ __forceinline__ void loss_flush(const GenLoss &L, const LossPartial &acc, int lane) {
    double r = (double)acc.rec, f = (double)acc.fn, p = (double)acc.fp;
    uint32_t n = acc.nfn | (acc.nfp << 16);  // at most 8 samples per thread
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        r += __shfl_xor_sync(0xffffffffu, r, d);
        f += __shfl_xor_sync(0xffffffffu, f, d);
        p += __shfl_xor_sync(0xffffffffu, p, d);
        n += __shfl_xor_sync(0xffffffffu, n, d);
    }
    if (lane == 0) {
        if (r != 0.0) atomicAdd(L.sums, r);
        if (f != 0.0) atomicAdd(L.sums + 1, f);
        if (p != 0.0) atomicAdd(L.sums + 2, p);
        if (n & 0xffffu) atomicAdd(L.counts, (unsigned long long)(n & 0xffffu));
        if (n >> 16) atomicAdd(L.counts + 1, (unsigned long long)(n >> 16));
    }
}

}  // namespace gs
