// peaks.cu -- measured denominators of the plain-ALU roofline:
// how many FP32 FMA lane-instructions and how many MUFU.EX2 the chip retires per second at the clock it
// runs at now.  Two dependency-free-enough loops (8 independent chains per thread, all warps resident),
// timed with CUDA events on the context's stream.  Not part of the sampling path.
#include "gs_internal.cuh"

namespace gs {

constexpr int PK_THREADS = 256;
constexpr int PK_CHAINS = 8;
constexpr int PK_ITERS = 4096;

__global__ void __launch_bounds__(PK_THREADS) k_peak_ffma(float *__restrict__ sink, float a, float b) {
    float x[PK_CHAINS];
#pragma unroll
    for (int k = 0; k < PK_CHAINS; k++) x[k] = (float)(threadIdx.x + k);
    for (int it = 0; it < PK_ITERS; it++) {
#pragma unroll
        for (int k = 0; k < PK_CHAINS; k++) x[k] = __fmaf_rn(x[k], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < PK_CHAINS; k++) s += x[k];
    if (s == 123.456f) sink[0] = s;  // keeps the loop alive; never true for the constants used
}

// packed FP32 (sm_100: fma.rn.f32x2 = FFMA2, two FMAs per lane-instruction); rate counted in FMA lane-OPERATIONS
__global__ void __launch_bounds__(PK_THREADS) k_peak_ffma2(float *__restrict__ sink, float a, float b) {
    unsigned long long x[PK_CHAINS], pa, pb;
    asm("mov.b64 %0, {%1, %1};" : "=l"(pa) : "f"(a));
    asm("mov.b64 %0, {%1, %1};" : "=l"(pb) : "f"(b));
#pragma unroll
    for (int k = 0; k < PK_CHAINS; k++) asm("mov.b64 %0, {%1, %2};" : "=l"(x[k]) : "f"((float)(threadIdx.x + k)), "f"((float)(threadIdx.x + k + 1)));
    for (int it = 0; it < PK_ITERS; it++) {
#pragma unroll
        for (int k = 0; k < PK_CHAINS; k++) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(x[k]) : "l"(pa), "l"(pb));
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < PK_CHAINS; k++) {
        float lo, hi;
        asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(x[k]));
        s += lo + hi;
    }
    if (s == 123.456f) sink[0] = s;
}

__global__ void __launch_bounds__(PK_THREADS) k_peak_ex2(float *__restrict__ sink, float a) {
    float x[PK_CHAINS];
#pragma unroll
    for (int k = 0; k < PK_CHAINS; k++) x[k] = -(float)(threadIdx.x + k) * a;
    for (int it = 0; it < PK_ITERS; it++) {
#pragma unroll
        for (int k = 0; k < PK_CHAINS; k++) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(x[k]));
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < PK_CHAINS; k++) s += x[k];
    if (s == 123.456f) sink[0] = s;
}

// rates in lane-instructions per second (one FMA / one EX2 of one thread = one lane-instruction)
cudaError_t measure_alu_peaks(float *sink, cudaStream_t s, double *ffma_per_s, double *ex2_per_s, double *ffma2_per_s) {
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    const unsigned blocks = (unsigned)sms * 8;  // 2048 threads per SM: every warp slot busy
    cudaEvent_t ev[4];
    for (auto &x : ev)
        if ((e = cudaEventCreate(&x)) != cudaSuccess) return e;
    double best[3] = {0.0, 0.0, 0.0};
    for (int rep = 0; rep < 4; rep++) {  // first repetition warms the clocks up
        cudaEventRecord(ev[0], s);
        k_peak_ffma<<<blocks, PK_THREADS, 0, s>>>(sink, 0.999f, 0.001f); count_launch();
        cudaEventRecord(ev[1], s);
        k_peak_ex2<<<blocks, PK_THREADS, 0, s>>>(sink, 1e-3f); count_launch();
        cudaEventRecord(ev[2], s);
        k_peak_ffma2<<<blocks, PK_THREADS, 0, s>>>(sink, 0.999f, 0.001f); count_launch();
        cudaEventRecord(ev[3], s);
        if ((e = cudaEventSynchronize(ev[3])) != cudaSuccess) break;
        float ms0 = 0.f, ms1 = 0.f, ms2 = 0.f;
        cudaEventElapsedTime(&ms0, ev[0], ev[1]);
        cudaEventElapsedTime(&ms1, ev[1], ev[2]);
        cudaEventElapsedTime(&ms2, ev[2], ev[3]);
        const double n = (double)blocks * PK_THREADS * PK_CHAINS * PK_ITERS;
        if (rep && ms0 > 0.f && n / (ms0 * 1e-3) > best[0]) best[0] = n / (ms0 * 1e-3);
        if (rep && ms1 > 0.f && n / (ms1 * 1e-3) > best[1]) best[1] = n / (ms1 * 1e-3);
        if (rep && ms2 > 0.f && 2.0 * n / (ms2 * 1e-3) > best[2]) best[2] = 2.0 * n / (ms2 * 1e-3);
    }
    for (auto &x : ev) cudaEventDestroy(x);
    if (e != cudaSuccess) return e;
    *ffma_per_s = best[0];
    *ex2_per_s = best[1];
    if (ffma2_per_s) *ffma2_per_s = best[2];
    return cudaGetLastError();
}

}  // namespace gs
