// optim.cu -- training-step completion: the activations of the raw parameters (PAPER.md:140:
// sigmoid for v_i and w_i, exponential for S_i; R_i is normalised inside k_preprocess) and one Adam step
// (Kingma & Ba, the paper's [20]; learning rates of PAPER.md:231) on the raw parameters, fed with the gradients
// w.r.t. the ACTIVATED values that gs_sample_bwd returns.  One thread per parameter element; HBM-bound
// (13 parameters + 13 gradients + 2 x 12 moments read, 12 + 24 + 5 written: 340 B per Gaussian).
#include <math.h>

#include "gs_internal.cuh"

namespace gs {

__global__ void __launch_bounds__(256) k_activate(uint32_t n, const float *__restrict__ raw_scale, const float *__restrict__ raw_opacity,
                                                   const float *__restrict__ raw_scalar, float *__restrict__ scale,
                                                   float *__restrict__ opacity, float *__restrict__ scalar) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
#pragma unroll
    for (int k = 0; k < 3; k++) scale[3 * (size_t)i + k] = expf(raw_scale[3 * (size_t)i + k]);
    opacity[i] = 1.0f / (1.0f + expf(-raw_opacity[i]));
    scalar[i] = 1.0f / (1.0f + expf(-raw_scalar[i]));
}

// sigmoid'(x) = s (1 - s) = e / (1 + e)^2 with e = exp(-|x|): no cancellation where s is close to 1
__device__ __forceinline__ float sigmoid_deriv(float x) {
    const float e = expf(-fabsf(x)), d = 1.0f + e;
    return e / (d * d);
}

struct AdamK {
    float lr[5], b1, b2, eps, c1inv, c2inv;  // c1inv = 1 / (1 - b1^t), c2inv = 1 / (1 - b2^t)
};

// m = b1 m + (1 - b1) g;  v = b2 v + (1 - b2) g^2;  p -= lr (m c1inv) / (sqrt(v c2inv) + eps)
__device__ __forceinline__ float adam1(float p, float g, float *__restrict__ m, float *__restrict__ v, size_t k, float lr, const AdamK &a) {
    const float mk = fmaf(a.b1, m[k], (1.0f - a.b1) * g);
    const float vk = fmaf(a.b2, v[k], (1.0f - a.b2) * g * g);
    m[k] = mk;
    v[k] = vk;
    return p - lr * (mk * a.c1inv) / (sqrtf(vk * a.c2inv) + a.eps);
}

// moments: one block of 12 n floats each, mean 3n | scale 3n | quat 4n | opacity n | scalar n -- the same order and
// widths as the parameter tensors, so element e of the concatenated parameters has its moments at m[e], v[e].
// One thread per ELEMENT (not per Gaussian): every load and store of a warp is one contiguous 128-byte run.
__global__ void __launch_bounds__(256) k_adam_step(gs_raw_params p, gs_grads g, float *__restrict__ m, float *__restrict__ v, AdamK a,
                                                    float *__restrict__ scale_out, float *__restrict__ opacity_out,
                                                    float *__restrict__ scalar_out) {
    const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const size_t n = p.n;
    if (e >= 12 * n) return;
    if (e < 3 * n) {
        p.mean[e] = adam1(p.mean[e], g.dmean[e], m, v, e, a.lr[0], a);
    } else if (e < 6 * n) {
        const size_t k = e - 3 * n;
        const float rs = p.raw_scale[k];
        const float rs_new = adam1(rs, g.dscale[k] * expf(rs), m, v, e, a.lr[1], a);  // d exp(x) / dx = exp(x)
        p.raw_scale[k] = rs_new;
        if (scale_out) scale_out[k] = expf(rs_new);
    } else if (e < 10 * n) {
        const size_t k = e - 6 * n;
        p.quat[k] = adam1(p.quat[k], g.dquat[k], m, v, e, a.lr[2], a);
    } else if (e < 11 * n) {
        const size_t k = e - 10 * n;
        const float rw = p.raw_opacity[k];
        const float rw_new = adam1(rw, g.dopacity[k] * sigmoid_deriv(rw), m, v, e, a.lr[3], a);  // sigmoid' = s (1 - s)
        p.raw_opacity[k] = rw_new;
        if (opacity_out) opacity_out[k] = 1.0f / (1.0f + expf(-rw_new));
    } else {
        const size_t k = e - 11 * n;
        const float rv = p.raw_scalar[k];
        const float rv_new = adam1(rv, g.dscalar[k] * sigmoid_deriv(rv), m, v, e, a.lr[4], a);
        p.raw_scalar[k] = rv_new;
        if (scalar_out) scalar_out[k] = 1.0f / (1.0f + expf(-rv_new));
    }
}

cudaError_t launch_activate(const gs_raw_params &p, float *scale, float *opacity, float *scalar, cudaStream_t s) {
    if (p.n == 0) return cudaSuccess;
    k_activate<<<(p.n + 255) / 256, 256, 0, s>>>(p.n, p.raw_scale, p.raw_opacity, p.raw_scalar, scale, opacity, scalar); count_launch();
    return cudaGetLastError();
}

cudaError_t launch_adam_step(const gs_raw_params &p, const gs_grads &g, float *m, float *v, const gs_adam_cfg &cfg, float *scale_out,
                             float *opacity_out, float *scalar_out, cudaStream_t s) {
    if (p.n == 0) return cudaSuccess;
    AdamK a;
    for (int k = 0; k < 5; k++) a.lr[k] = cfg.lr[k];
    a.b1 = cfg.beta1; a.b2 = cfg.beta2; a.eps = cfg.eps;
    a.c1inv = (float)(1.0 / (1.0 - pow((double)cfg.beta1, (double)cfg.step)));
    a.c2inv = (float)(1.0 / (1.0 - pow((double)cfg.beta2, (double)cfg.step)));
    const size_t elems = 12 * (size_t)p.n;
    k_adam_step<<<(unsigned)((elems + 255) / 256), 256, 0, s>>>(p, g, m, v, a, scale_out, opacity_out, scalar_out); count_launch();
    return cudaGetLastError();
}

}  // namespace gs
