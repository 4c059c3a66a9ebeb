// densify.cu -- density control on the device: pruning by the weight threshold
// and sample-error densification (new Gaussians "with means at the positions of the k highest error
// samples", "given parameters in the same way as initialization, with values corresponding to the ground truth
// samples"; false negatives first).  All integer work is deterministic:
//   prune   : flags -> exclusive scan -> kept indices in their order -> gather of the 12 parameters and 2 x 12 moments
//   densify : key = (false negative << 31 | float bits of the error + 1) for defined samples, 0 otherwise; stable
//             LSD radix sort on ~key (descending key, ascending sample index inside equal keys); one new Gaussian per
//             selected sample; re-layout of the moment blocks for the new count.
// Moment blocks are [12 n]: mean 3n | scale 3n | quat 4n | opacity n | scalar n, so a change of n moves the blocks:
// everything is gathered into scratch arrays first and copied back.
#include <math.h>

#include "gs_internal.cuh"
#include "pair_math.cuh"

namespace gs {

__global__ void __launch_bounds__(256) k_prune_flags(const float *__restrict__ opacity, uint32_t n, float tau2, uint32_t *__restrict__ flag) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) flag[i] = opacity[i] >= tau2 ? 1u : 0u;   // "removes Gaussians below a chosen threshold"
}

__global__ void __launch_bounds__(256) k_kept_indices(const uint32_t *__restrict__ flag, const uint32_t *__restrict__ pos, uint32_t n,
                                                       uint32_t *__restrict__ src) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n && flag[i]) src[pos[i]] = i;
}

struct ParamSet { float *mean, *raw_scale, *quat, *raw_opacity, *raw_scalar, *m, *v; };

// new[j] = old[src[j]] (src = NULL: identity) for the parameters and both moment blocks; j < n_copy
__global__ void __launch_bounds__(256) k_regather(ParamSet o, uint32_t n_old, ParamSet d, uint32_t n_new, const uint32_t *__restrict__ src,
                                                   uint32_t n_copy) {
    const uint32_t j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_copy) return;
    const size_t i = src ? src[j] : j, no = n_old, nn = n_new;
#pragma unroll
    for (int k = 0; k < 3; k++) {
        d.mean[3 * (size_t)j + k] = o.mean[3 * i + k];
        d.raw_scale[3 * (size_t)j + k] = o.raw_scale[3 * i + k];
        d.m[3 * (size_t)j + k] = o.m[3 * i + k];
        d.v[3 * (size_t)j + k] = o.v[3 * i + k];
        d.m[3 * nn + 3 * (size_t)j + k] = o.m[3 * no + 3 * i + k];
        d.v[3 * nn + 3 * (size_t)j + k] = o.v[3 * no + 3 * i + k];
    }
#pragma unroll
    for (int k = 0; k < 4; k++) {
        d.quat[4 * (size_t)j + k] = o.quat[4 * i + k];
        d.m[6 * nn + 4 * (size_t)j + k] = o.m[6 * no + 4 * i + k];
        d.v[6 * nn + 4 * (size_t)j + k] = o.v[6 * no + 4 * i + k];
    }
    d.raw_opacity[j] = o.raw_opacity[i];
    d.raw_scalar[j] = o.raw_scalar[i];
    d.m[10 * nn + j] = o.m[10 * no + i];
    d.v[10 * nn + j] = o.v[10 * no + i];
    d.m[11 * nn + j] = o.m[11 * no + i];
    d.v[11 * nn + j] = o.v[11 * no + i];
}

// sort key of a sample: ascending ~key = false negatives first, then highest error first
__global__ void __launch_bounds__(256) k_select_keys(const float *__restrict__ err, const float *__restrict__ I,
                                                      const uint8_t *__restrict__ defined, size_t P, float tau, uint32_t *__restrict__ key,
                                                      uint32_t *__restrict__ val) {
    const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= P) return;
    uint32_t k = 0;
    if (!defined || defined[c]) {
        const uint32_t fn = I[c] > tau ? 0u : 1u;                 // defined but not covered (Fig. 6A)
        k = (fn << 31) | (__float_as_uint(fabsf(err[c])) + 1u);   // err >= 0: its bit pattern orders like its value
    }
    key[c] = ~k;
    val[c] = (uint32_t)c;
}

// Gaussian n_old + j from the j-th selected sample
__global__ void __launch_bounds__(256) k_new_gaussians(ParamSet d, uint32_t n_old, uint32_t n_new, const uint32_t *__restrict__ sel,
                                                        GridDesc gd, const float4 *__restrict__ jit, const float *__restrict__ xyz /*NULL: grid*/,
                                                        const float *__restrict__ target, float raw_scale_init, float raw_opacity_init,
                                                        float clamp) {
    const uint32_t j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_new - n_old) return;
    const uint32_t c = sel[j];
    float px, py, pz;
    if (xyz) {
        px = xyz[3 * (size_t)c]; py = xyz[3 * (size_t)c + 1]; pz = xyz[3 * (size_t)c + 2];
    } else {  // batch-local sample index, x fastest (D6)
        const uint32_t bdx = (uint32_t)gd.bdim[0], bdy = (uint32_t)gd.bdim[1];
        const uint32_t x = c % bdx, y = (c / bdx) % bdy, z = c / (bdx * bdy);
        const int gx = (int)x + BRICK * gd.brick_lo[0], gy = (int)y + BRICK * gd.brick_lo[1], gz = (int)z + BRICK * gd.brick_lo[2];
        if (gd.jitter) {  // the sample the error was measured at (D26)
            const float4 sp = jit[c];
            px = sp.x; py = sp.y; pz = sp.z;
        } else {
            px = voxel_centre(gx, gd.spacing[0], gd.origin[0]);
            py = voxel_centre(gy, gd.spacing[1], gd.origin[1]);
            pz = voxel_centre(gz, gd.spacing[2], gd.origin[2]);
        }
    }
    const size_t g = (size_t)n_old + j, nn = n_new;
    d.mean[3 * g] = px; d.mean[3 * g + 1] = py; d.mean[3 * g + 2] = pz;
#pragma unroll
    for (int k = 0; k < 3; k++) {
        d.raw_scale[3 * g + k] = raw_scale_init;
        d.m[3 * g + k] = 0.f; d.v[3 * g + k] = 0.f;
        d.m[3 * nn + 3 * g + k] = 0.f; d.v[3 * nn + 3 * g + k] = 0.f;
    }
    d.quat[4 * g] = 1.f; d.quat[4 * g + 1] = 0.f; d.quat[4 * g + 2] = 0.f; d.quat[4 * g + 3] = 0.f;
#pragma unroll
    for (int k = 0; k < 4; k++) { d.m[6 * nn + 4 * g + k] = 0.f; d.v[6 * nn + 4 * g + k] = 0.f; }
    d.raw_opacity[g] = raw_opacity_init;
    const float t = fminf(fmaxf(target[c], clamp), 1.0f - clamp);
    d.raw_scalar[g] = logf(t / (1.0f - t));   // sigmoid(raw_scalar) = the ground-truth value
    d.m[10 * nn + g] = 0.f; d.v[10 * nn + g] = 0.f;
    d.m[11 * nn + g] = 0.f; d.v[11 * nn + g] = 0.f;
}

static ParamSet carve(float *base, size_t n) {  // scratch: 13 n parameters, then 12 n + 12 n moments
    ParamSet s;
    s.mean = base; s.raw_scale = base + 3 * n; s.quat = base + 6 * n; s.raw_opacity = base + 10 * n; s.raw_scalar = base + 11 * n;
    s.m = base + 12 * n; s.v = base + 24 * n;
    return s;
}

static cudaError_t copy_back(const ParamSet &tmp, const ParamSet &dst, size_t n, cudaStream_t s) {
    const struct { float *d; const float *t; size_t cnt; } job[] = {
        {dst.mean, tmp.mean, 3 * n}, {dst.raw_scale, tmp.raw_scale, 3 * n}, {dst.quat, tmp.quat, 4 * n}, {dst.raw_opacity, tmp.raw_opacity, n},
        {dst.raw_scalar, tmp.raw_scalar, n}, {dst.m, tmp.m, 12 * n}, {dst.v, tmp.v, 12 * n}};
    for (const auto &j : job) {
        if (!j.cnt) continue;
        cudaError_t e = cudaMemcpyAsync(j.d, j.t, j.cnt * sizeof(float), cudaMemcpyDeviceToDevice, s);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

// flags / positions / kept indices live in `work` (3 n uint32); returns with the kept count at pos[n] (device)
cudaError_t launch_prune_index(const float *opacity, uint32_t n, float tau2, uint32_t *work, DevBuf &scan_tmp, cudaStream_t s) {
    if (n == 0) return cudaMemsetAsync(work, 0, 4, s);   // pos[0] = count = 0
    uint32_t *flag = work, *pos = work + n, *src = work + 2 * (size_t)n + 1;
    k_prune_flags<<<(n + 255) / 256, 256, 0, s>>>(opacity, n, tau2, flag); count_launch();
    cudaError_t e = exclusive_scan_u32(flag, pos, n, scan_tmp, s);
    if (e != cudaSuccess) return e;
    k_kept_indices<<<(n + 255) / 256, 256, 0, s>>>(flag, pos, n, src); count_launch();
    return cudaGetLastError();
}

cudaError_t launch_regather(const gs_raw_params &p, float *m, float *v, uint32_t n_new, const uint32_t *src, uint32_t n_copy, float *scratch,
                            bool back, cudaStream_t s) {
    const ParamSet o{p.mean, p.raw_scale, p.quat, p.raw_opacity, p.raw_scalar, m, v};
    const ParamSet d = carve(scratch, n_new);
    if (n_copy) { k_regather<<<(n_copy + 255) / 256, 256, 0, s>>>(o, p.n, d, n_new, src, n_copy); count_launch(); }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess || !back) return e;
    return copy_back(d, o, n_new, s);
}

cudaError_t launch_select_keys(const float *err, const float *I, const uint8_t *defined, size_t P, float tau, uint32_t *key, uint32_t *val,
                               cudaStream_t s) {
    if (P == 0) return cudaSuccess;
    k_select_keys<<<(unsigned)((P + 255) / 256), 256, 0, s>>>(err, I, defined, P, tau, key, val); count_launch();
    return cudaGetLastError();
}

cudaError_t launch_new_gaussians(const gs_raw_params &p, float *m, float *v, uint32_t n_new, const uint32_t *sel, const GridDesc &gd,
                                 const float4 *jit, const float *xyz, const float *target, float raw_scale_init, float raw_opacity_init, float clamp,
                                 float *scratch, cudaStream_t s) {
    const ParamSet o{p.mean, p.raw_scale, p.quat, p.raw_opacity, p.raw_scalar, m, v};
    const ParamSet d = carve(scratch, n_new);
    const uint32_t add = n_new - p.n;
    if (add) {
        k_new_gaussians<<<(add + 255) / 256, 256, 0, s>>>(d, p.n, n_new, sel, gd, jit, xyz, target, raw_scale_init, raw_opacity_init, clamp);
        count_launch();
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    return copy_back(d, o, n_new, s);
}

}  // namespace gs
