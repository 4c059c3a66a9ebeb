// probe_static.cu -- gs_probe_points_static: Eq. 2 / Eq. 3 (cutoff PAPER.md:116, coverage rule
// PAPER.md:126) of a SMALL model at a list of points, for callers that must not allocate device memory.
//
// Who that is: code running inside somebody else's memory budget.  A renderer or an inference server that claimed
// the whole GPU for its own pool at start-up (a later cudaMalloc fails, or steals from the pool's head-room); a
// real-time loop, where cudaMalloc / cudaFree stall every stream of the device for an unpredictable time; a plug-in
// that is only allowed to touch the buffers its host hands it.  Every other entry point of this library goes through
// a gs_ctx whose grow-only arenas come from cudaMalloc, starting in gs_create.  This one needs no context.
//
// What stands in for the arenas: the per-Gaussian records that S1 (k_preprocess, unchanged) writes before anything can
// be sampled -- 64 B of (mu, w, M = S^-1 R, v) + 24 B cutoff AABB + 32 B raw parameters per Gaussian + one counter --
// live in ONE file-scope device array of fixed size, sized for GS_PROBE_MAX_GAUSSIANS.  The array is part of the
// library's device image: every GPU that loads libgs.so carries its 1.9 MiB until the process exits, used or not.
//
// Host code cannot use the array's name as an address (on the host the name is only a handle of the runtime; a kernel
// given it would fault or scribble over unrelated memory).  The device address is looked up with cudaGetSymbolAddress,
// once per device, with that device current (probe_scratch_of below), and handed to the kernels as a plain pointer.
#include <mutex>
#include <stdarg.h>
#include <stdio.h>
#include <math.h>

#include "gs_internal.cuh"
#include "pair_math.cuh"

namespace {

constexpr size_t PROBE_MAX = GS_PROBE_MAX_GAUSSIANS;
constexpr size_t PROBE_OFF_REC = 0;                        // float4 [4][n]   (plane stride = the call's n, not PROBE_MAX)
constexpr size_t PROBE_OFF_AABB = 64 * PROBE_MAX;          // float  [n][6]
constexpr size_t PROBE_OFF_PARAMS = 88 * PROBE_MAX;        // float4 [n][2]
constexpr size_t PROBE_OFF_INVALID = 120 * PROBE_MAX;      // unsigned long long: Gaussians with empty support (cleared by every call)
constexpr size_t PROBE_BYTES = 120 * PROBE_MAX + 256;
static_assert(PROBE_OFF_AABB % 256 == 0 && PROBE_OFF_PARAMS % 256 == 0 && PROBE_OFF_INVALID % 256 == 0, "sub-buffers stay 256-byte aligned");

// The scratch.  Shared by every call on a device; it keeps whatever the last call left in it.
static __device__ __align__(256) unsigned char g_probe_scratch[PROBE_BYTES];

constexpr int PROBE_MAX_DEVICES = 64;
std::mutex g_probe_mu;
unsigned char *g_probe_ptr[PROBE_MAX_DEVICES];   // device address of g_probe_scratch on device d (NULL: not looked up yet)

// Set-up, once per device; the caller has made `device` current.  No allocation: the array already exists on the device.
cudaError_t probe_scratch_of(int device, unsigned char **out) {
    std::lock_guard<std::mutex> lock(g_probe_mu);
    if (!g_probe_ptr[device]) {
        unsigned char *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void **)&p, g_probe_scratch);
        if (e != cudaSuccess) return e;
        g_probe_ptr[device] = p;
    }
    *out = g_probe_ptr[device];
    return cudaSuccess;
}

}  // namespace

namespace gs {
constexpr int PROBE_THREADS = 256;
constexpr int PROBE_TILE = 128;   // Gaussians staged per round: 8 KiB of shared memory

// One thread per point, every Gaussian of the model tested against it (no acceleration structure: at <= 16,384
// Gaussians the records are 1 MiB and stay in L2).  Membership is the library's canonical fp32 predicate (pair_math.cuh,
// DESIGN D4), so a point's set of contributing Gaussians is the one gs_sample_fwd finds; the sums run in ascending
// Gaussian index, so values agree with gs_sample_fwd up to fp32 summation order.
__global__ void __launch_bounds__(PROBE_THREADS) k_probe_points(const float4 *__restrict__ rec, uint32_t N, const float *__restrict__ xyz,
                                                                 uint64_t P, float tau, float r2, float *__restrict__ phi,
                                                                 float *__restrict__ I) {
    __shared__ float4 sm[4][PROBE_TILE];
    const uint64_t c = (uint64_t)blockIdx.x * PROBE_THREADS + threadIdx.x;
    const bool active = c < P;
    const float nan = __int_as_float(0x7fc00000);
    const float px = active ? xyz[3 * c] : nan, py = active ? xyz[3 * c + 1] : nan, pz = active ? xyz[3 * c + 2] : nan;
    float Iacc = 0.f, Nacc = 0.f;
    for (uint32_t base = 0; base < N; base += PROBE_TILE) {
        const uint32_t n = N - base < (uint32_t)PROBE_TILE ? N - base : (uint32_t)PROBE_TILE;
        for (uint32_t k = threadIdx.x; k < 4u * PROBE_TILE; k += PROBE_THREADS) {
            const uint32_t plane = k / PROBE_TILE, j = k % PROBE_TILE;
            if (j < n) sm[plane][j] = rec[(size_t)plane * N + base + j];
        }
        __syncthreads();
        for (uint32_t j = 0; j < n; j++) {
            gs::Rec g;
            g.a = sm[0][j]; g.b = sm[1][j]; g.c = sm[2][j]; g.d = sm[3][j];
            float u0, u1, u2;
            const float qd = gs::mahalanobis(g, px, py, pz, u0, u1, u2);
            if (qd <= r2) {   // false for a NaN point and for an invalid Gaussian (mu = NaN)
                const float G = gs::gauss_weight(qd);
                Iacc = fmaf(g.a.w, G, Iacc);
                Nacc = fmaf(g.d.w, G, Nacc);   // d.w = v w
            }
        }
        __syncthreads();
    }
    if (active) {
        I[c] = Iacc;
        phi[c] = Iacc > tau ? __fdividef(Nacc, Iacc) : 0.f;   // below the threshold the sample is empty
    }
}

}  // namespace gs

namespace {

gs_status probe_fail(gs_status st, char *err_host, size_t err_cap, const char *fmt, ...) {
    if (err_host && err_cap) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(err_host, err_cap, fmt, ap);
        va_end(ap);
    }
    return st;
}

struct DeviceGuard {   // the call leaves the thread's current device as it found it
    int prev = -1;
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

}  // namespace

extern "C" gs_status gs_probe_points_static(int device, void *cuda_stream, const gs_gaussians *g, float tau, const float *xyz,
                                            uint64_t num_points, float *phi, float *I, char *err_host, size_t err_cap) {
    if (err_host && err_cap) err_host[0] = 0;
    if (!g) return probe_fail(GS_ERR_INVALID_ARG, err_host, err_cap, "gaussians is NULL");
    if (g->n > GS_PROBE_MAX_GAUSSIANS)
        return probe_fail(GS_ERR_INVALID_ARG, err_host, err_cap,
                          "gs_probe_points_static: %u Gaussians exceed GS_PROBE_MAX_GAUSSIANS = %u, the size of the library's fixed "
                          "scratch; use gs_preprocess / gs_build_accel / gs_sample_fwd (which allocate) for larger models",
                          g->n, (unsigned)GS_PROBE_MAX_GAUSSIANS);
    if (g->n > 0 && (!g->mean || !g->scale || !g->quat || !g->opacity || !g->scalar))
        return probe_fail(GS_ERR_INVALID_ARG, err_host, err_cap, "gaussians: NULL parameter array");
    if (!(tau > 0.f && tau < 1.f)) return probe_fail(GS_ERR_INVALID_ARG, err_host, err_cap, "tau must lie in (0,1)");
    if (num_points > GS_PROBE_MAX_POINTS)
        return probe_fail(GS_ERR_INVALID_ARG, err_host, err_cap, "gs_probe_points_static: %llu points exceed GS_PROBE_MAX_POINTS = %llu per call",
                          (unsigned long long)num_points, (unsigned long long)GS_PROBE_MAX_POINTS);
    if (num_points > 0 && (!xyz || !phi || !I)) return probe_fail(GS_ERR_INVALID_ARG, err_host, err_cap, "xyz / phi / I is NULL");
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count || device >= PROBE_MAX_DEVICES) {
        cudaGetLastError();
        return probe_fail(GS_ERR_CUDA, err_host, err_cap, "no CUDA device %d", device);
    }
    DeviceGuard guard;
    int cur = -1;
    cudaError_t e = cudaGetDevice(&cur);
    if (e == cudaSuccess && cur != device) {
        e = cudaSetDevice(device);
        if (e == cudaSuccess) guard.prev = cur;
    }
    unsigned char *scratch = nullptr;
    if (e == cudaSuccess) e = probe_scratch_of(device, &scratch);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return probe_fail(GS_ERR_CUDA, err_host, err_cap, "set-up of the static scratch on device %d: %s", device, cudaGetErrorString(e));
    }
    if (num_points == 0) return GS_OK;
    cudaStream_t s = reinterpret_cast<cudaStream_t>(cuda_stream);
    float4 *rec = reinterpret_cast<float4 *>(scratch + PROBE_OFF_REC);
    // support G >= tau  <=>  |u|^2 <= r2 = -2 ln tau, both rounded to fp32 once (as gs_preprocess does, DESIGN D3)
    const float r2 = (float)(-2.0 * log((double)tau));
    const float r = (float)sqrt((double)r2);
    // S1 into the static scratch: the library's own k_preprocess, given the looked-up address.  It overwrites rows
    // [0, n) of every sub-buffer and clears the invalid-Gaussian counter itself; rows beyond n keep older contents
    // and are never read (k_probe_points is bounded by this call's n).
    e = gs::launch_preprocess(*g, r, rec, reinterpret_cast<float *>(scratch + PROBE_OFF_AABB), reinterpret_cast<float *>(scratch + PROBE_OFF_PARAMS),
                              reinterpret_cast<unsigned long long *>(scratch + PROBE_OFF_INVALID), s);
    if (e == cudaSuccess) {
        gs::k_probe_points<<<(unsigned)((num_points + gs::PROBE_THREADS - 1) / gs::PROBE_THREADS), gs::PROBE_THREADS, 0, s>>>(rec, g->n, xyz, num_points, tau, r2, phi, I);
        gs::count_launch();
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        cudaGetLastError();
        return probe_fail(GS_ERR_CUDA, err_host, err_cap, "gs_probe_points_static: %s", cudaGetErrorString(e));
    }
    return GS_OK;
}
