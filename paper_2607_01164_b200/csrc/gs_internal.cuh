// gs_internal.cuh -- shared declarations of the sm_100a W-VEG sampler (not part of the C ABI).
// Citations: PAPER.md:<line> of arxiv/paper_2607_01164; "D<n>" = the numbered readings in DESIGN.md.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include <string>
#include <vector>

#include "../../include/gs.h"
#include "loss.cuh"

namespace gs {

constexpr int BRICK = 8;            // bricks of 8^3 voxels (north_star (3))
constexpr int BRICK_VOX = 512;
constexpr int GACC = 16;            // floats per Gaussian in the gradient accumulator (13 used)
// gacc layout: 0 dv | 1 dw | 2..4 U | 5..10 W00 W01 W02 W11 W12 W22 | 11 E | 12..15 unused
constexpr int GACC_GRID = 32;       // the structured backward writes a row of moment sums instead (sample_grid_bwd.cu)

// Grow-only device buffer owned by the context.
struct DevBuf {
    void *p = nullptr;
    size_t cap = 0;
    cudaError_t reserve(size_t bytes) {
        if (bytes <= cap) return cudaSuccess;
        if (p) { cudaFree(p); p = nullptr; cap = 0; }
        size_t want = bytes + bytes / 8 + 256;
        cudaError_t e = cudaMalloc(&p, want);
        if (e != cudaSuccess) { p = nullptr; cap = 0; return e; }
        cap = want;
        return cudaSuccess;
    }
    // grow to at least `bytes`, keeping the first `keep` bytes of the contents (waits for stream s)
    cudaError_t reserve_keep(size_t bytes, size_t keep, cudaStream_t s) {
        if (bytes <= cap) return cudaSuccess;
        const size_t want = bytes + bytes / 8 + 256;
        void *np = nullptr;
        cudaError_t e = cudaMalloc(&np, want);
        if (e != cudaSuccess) return e;
        if (p && keep) e = cudaMemcpyAsync(np, p, keep < cap ? keep : cap, cudaMemcpyDeviceToDevice, s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        if (e != cudaSuccess) { cudaFree(np); return e; }
        if (p) cudaFree(p);
        p = np;
        cap = want;
        return cudaSuccess;
    }
    void release() { if (p) cudaFree(p); p = nullptr; cap = 0; }
    template <class T> T *as() const { return reinterpret_cast<T *>(p); }
};

struct GridDesc {          // one batch of a structured grid (gs_query, GS_QUERY_GRID)
    int dims[3];
    float origin[3], spacing[3];
    int brick_lo[3], brick_cnt[3];
    int bdim[3];           // clipped voxel extent of the batch
    float inv_brick[3];    // 1.0f / (8.0f * spacing)  (D7)
    int nb_total[3];       // bricks of the whole grid per axis
    int jitter;            // samples at a random position of their cell (D26) instead of its centre
    unsigned long long jitter_seed;
};

// Candidate Gaussians of a grid batch from the coarse index (binning.cu): up to 8 coarse cells, each a slice of the index's
// id list.  ids == NULL: no index, every Gaussian of the model is looked at.
constexpr int COARSE_B = 16;   // bricks per coarse cell and axis (128 voxels: the batch size of configs[3])
struct CandSegs {
    const uint32_t *ids;
    uint32_t n, total;          // segments, candidates (with duplicates: a Gaussian is listed in every coarse cell it overlaps)
    uint32_t start[8], prefix[9];
    int cell[8][3];             // coarse coordinates of the segment's cell
    int clo[3];                 // first coarse cell of the batch per axis
};

// scatter mode of a point query (sample_scatter.cu): implicit 32-ary tree over the Morton-sorted query points
struct PtTree {
    const float *box;   // per level SoA boxes: box[off[l] + k * n[l] + i], k = lo.xyz hi.xyz
    uint32_t off[8];    // in floats
    uint32_t n[8];      // nodes per level (level 0 = leaves)
    int levels;
};

// 30-bit Morton code of a position inside the domain box (D8): 10 bits per axis, x in the low bit,
// q = (int) min(max((x - lo) * (1024 / (hi - lo)), 0), 1023) with the scale computed once on the host in fp32.
struct MortonParams { float lo[3], scale[3]; };
inline MortonParams morton_params(const gs_domain &dom) {
    MortonParams mp;
    for (int k = 0; k < 3; k++) {
        mp.lo[k] = dom.lo[k];
        mp.scale[k] = 1024.0f / (dom.hi[k] - dom.lo[k]);
    }
    return mp;
}
#ifdef __CUDACC__
__device__ __forceinline__ uint32_t expand10(uint32_t v) {  // 10 bits -> every third bit
    v &= 0x3ffu;
    v = (v | (v << 16)) & 0x030000FFu;
    v = (v | (v << 8)) & 0x0300F00Fu;
    v = (v | (v << 4)) & 0x030C30C3u;
    v = (v | (v << 2)) & 0x09249249u;
    return v;
}
__device__ __forceinline__ uint32_t morton30(float x, float y, float z, const MortonParams &mp) {
    const float tx = __fmul_rn(__fsub_rn(x, mp.lo[0]), mp.scale[0]);
    const float ty = __fmul_rn(__fsub_rn(y, mp.lo[1]), mp.scale[1]);
    const float tz = __fmul_rn(__fsub_rn(z, mp.lo[2]), mp.scale[2]);
    const uint32_t qx = (uint32_t)(int)fminf(fmaxf(tx, 0.0f), 1023.0f);
    const uint32_t qy = (uint32_t)(int)fminf(fmaxf(ty, 0.0f), 1023.0f);
    const uint32_t qz = (uint32_t)(int)fminf(fmaxf(tz, 0.0f), 1023.0f);
    return expand10(qx) | (expand10(qy) << 1) | (expand10(qz) << 2);
}
#endif

}  // namespace gs

struct gs_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    std::string err;
    // ---- S1 state
    bool have_pre = false;
    uint32_t N = 0;
    float tau = 0.f, r2 = 0.f, r = 0.f;
    bool have_dom = false;
    gs_domain dom{};
    const float *scale_in = nullptr;  // NOT retained beyond gs_preprocess; see params copy below
    gs::DevBuf rec;      // float4 [4][N]
    gs::DevBuf aabb;     // float [N][6]
    gs::DevBuf params;   // float [N][8]: scale.xyz, quat (raw) wxyz, pad  (needed by S8)
    // ---- accel (grid)
    int accel_kind = -1;  // -1 none, else gs_query_kind
    gs_query accel_q{};
    gs::GridDesc grid{};
    uint32_t T = 0, nbricks = 0;
    bool have_pair_brick = false;
    uint32_t M = 0;       // Gaussians that touch the current batch (grid): length of the backward's order list
    gs::DevBuf bcount;    // uint32 [N]: bricks overlapped by each Gaussian
    gs::DevBuf bhist;     // uint32 [nbricks + norder]: pairs per brick | Gaussians per order bucket
    gs::DevBuf pair_gauss;   // uint32 [T]: Gaussian ids, ascending inside every brick's run
    gs::DevBuf pair_brick;   // uint32 [T]: debug view only (gs_debug_get)
    gs::DevBuf grid_order;   // uint32 [M]: processing order of the backward
    gs::DevBuf brick_start;  // uint32 [nbricks + norder + 1]: runs of the bricks, then of the order buckets (offset by T)
    // coarse index over the Gaussians (built when small batches of a large grid follow one another without a gs_preprocess)
    gs::DevBuf cidx_hist, cidx_start, cidx_ids;
    std::vector<uint32_t> cidx_start_host;
    bool cidx_valid = false;
    int cidx_nc[3] = {0, 0, 0};
    gs::GridDesc cidx_geom{};
    uint32_t builds_since_pre = 0;   // grid builds since the last gs_preprocess
    gs::CandSegs prev_cand{};        // candidates of the previous build (their counts are cleared by the next one); ids == NULL: none
    bool bcount_exact = false;       // bcount holds 0 for every Gaussian outside prev_cand (false: unknown, clear everything)
    gs::DevBuf jit;          // float4 [P]: sample positions of a jittered grid batch (D26)
    gs::DevBuf bwd_setup;    // float4 [N][2]: per-Gaussian constants of the structured backward (k_brick_count)
    // ---- accel (points)
    uint64_t P = 0;
    gs::DevBuf leaf_key[2], leaf_val[2];
    int leaf_sel = 0;
    gs::DevBuf node_left, node_right, node_parent, leaf_parent, node_aabb, node_flag;
    gs::DevBuf bvh_nodes;  // packed traversal nodes
    gs::DevBuf sorted_rec; // float4 [N][4]: records in leaf order (id in plane c's .w)
    gs::DevBuf cull_ids, cull_link, cull_head;  // per-packet survivor lists (see CullLists)
    gs::DevBuf cull_mask;      // uint2 [cull_cap]: per-chunk hit bits (+ skip link) of the last forward on the current lists
    bool have_hit_masks = false;   // cull_mask is valid for the current point accel (a gather-mode forward ran since its build)
    int opt_bwd_hit_masks = 1;     // gs_set_option(GS_OPT_BWD_HIT_MASKS)
    uint32_t cull_cap = 0;   // chunks the pool holds
    double cull_per_packet = 0.0;   // list entries per packet of the last build (picks the cull kernel's group size)
    gs::DevBuf pt_key[2], pt_val[2];
    int pt_sel = 0;
    bool have_pt_order = false;
    // ---- scratch
    gs::DevBuf scan_tmp, sort_hist, gacc, misc, counters, dbg;
    gs::DevBuf dens_work, dens_scratch, sel_key[2], sel_val[2];  // gs_prune / gs_densify
    int fused_pack = 0;  // misc holds backward coefficients written by the last forward: 1 = float2 (alpha, beta) of gs_sample_fwd's
                         // fused MSE, 2 = float4 (alpha, beta, eps, -) of gs_sample_fwd_loss on a grid; 0 = none
    gs::DevBuf rn_xyz, rn_phi, rn_I;   // gs_render: samples of a chunk of rays
    gs::DevBuf h2d[16];  // staging for gs_step_host
    cudaStream_t aux_stream = nullptr;  // gs_step_host: the target's H2D copy overlaps preprocess + build
    cudaEvent_t aux_event = nullptr, aux_event2 = nullptr;
    int lbvh_state = 0;   // Gaussian side of a point accel since the last gs_preprocess: 0 = not built, 1 = Morton order (scatter mode), 2 = + LBVH
    cudaEvent_t points_ready = nullptr;   // set by gs_step_host: gs_build_accel waits for it before it touches the query points
    // gs_decode_grid: worker contexts on streams of their own (created on first use, destroyed with this context)
    std::vector<gs_ctx *> decode_workers;
    std::vector<cudaStream_t> decode_streams;
    cudaEvent_t decode_event = nullptr;
    uint64_t decode_repeats = 0;   // batches gs_decode_grid had to repeat (asynchronous build overflow)
    int opt_async_build = 0;    // gs_set_option(GS_OPT_ASYNC_BUILD)
    bool grid_pending = false;  // T / M of the current grid accel are still on their way to grid_host (grid_event)
    unsigned long long *grid_host = nullptr;   // pinned [2]: T, M
    cudaEvent_t grid_event = nullptr;
    uint32_t grid_warm_N = 0xffffffffu;        // N of the last synchronously built grid accel (async needs a known capacity)
    uint32_t M_hint = 0;                       // M of the last resolved build: sizes the backward's grid while M is pending
    int opt_points_accel = 0;   // gs_set_option(GS_OPT_POINTS_ACCEL): mode the NEXT point accel is built in
    int points_mode = 0;        // mode of the current point accel (gs_points_accel)
    gs::DevBuf sc_spt, sc_box, sc_acc, sc_coef;  // scatter mode: sorted positions, tree boxes, (I, Nacc) accumulators, backward coefficients
    gs::PtTree sc_tree{};
    uint64_t sample_count = 0;  // gs_set_sample_count: samples the fused loss mean runs over (0 = the query's own P)
    // ---- measurement (gs_profile_*)
    unsigned long long launches = 0;  // kernels launched for this context since the last gs_profile_read
    bool prof = false;
    struct ProfPair { cudaEvent_t a, b; int stage; };
    std::vector<ProfPair> prof_pending, prof_free;
};

namespace gs {
// kernels launched by this library, counted per context: every C-ABI entry point binds the calling thread to its
// context's counter (LaunchScope in gs_api.cu); the launchers below bump it through this thread-local pointer
extern thread_local unsigned long long *tl_launches;
inline void count_launch(int n = 1) { if (tl_launches) *tl_launches += (unsigned long long)n; }
}  // namespace gs

namespace gs {

// ---- launchers (each enqueues on `s`, returns the launch error) ---------------------------------
cudaError_t launch_preprocess(const gs_gaussians &g, float r, float4 *rec, float *aabb, float *params, unsigned long long *invalid, cudaStream_t s);

// exclusive prefix sum of n uint32 (out may alias in); out[n] = total is written too (out has n+1 slots)
cudaError_t exclusive_scan_u32(const uint32_t *in, uint32_t *out, size_t n, DevBuf &tmp, cudaStream_t s);
// stable LSD radix sort of (key, val) pairs on key bits [0, bits); returns the index (0/1) of the
// buffer pair holding the result.  keys[0]/vals[0] hold the input.
cudaError_t radix_sort_pairs(uint32_t *keys[2], uint32_t *vals[2], size_t n, int bits, DevBuf &hist, DevBuf &tmp,
                             cudaStream_t s, int *result_sel);

// S2 (binning.cu).  hist = [nbricks | norder] counters (zeroed here, counted down to zero again by launch_pair_fill);
// start = exclusive scan of hist (nbricks + norder + 1 entries).  launch_pair_fill writes nothing when *total > cap.
cudaError_t launch_brick_count(const float *aabb, const float4 *rec, uint32_t N, const GridDesc &gd, float rcut, uint32_t *count,
                               unsigned long long *total, uint32_t *hist, uint32_t nbricks, uint32_t norder, int order_shift,
                               float4 *setup, const CandSegs &cs, cudaStream_t s);
cudaError_t launch_pair_fill(const float *aabb, const uint32_t *count, uint32_t N, const GridDesc &gd, const unsigned long long *total, uint32_t cap,
                             uint32_t *hist, const uint32_t *start, uint32_t nbricks, int order_shift, uint32_t *pair_gauss,
                             uint32_t *order, const CandSegs &cs, cudaStream_t s);
cudaError_t launch_build_reset(unsigned long long *total, uint32_t *hist, uint32_t nh, uint32_t *count, const CandSegs &prev, cudaStream_t s);
// coarse index over the Gaussians for small batches of a large grid: cell = COARSE_B^3 bricks; CSR (start[ncells + 1], ids)
cudaError_t launch_coarse_count(const float *aabb, uint32_t N, const GridDesc &full, const int nc[3], uint32_t *hist, cudaStream_t s);
cudaError_t launch_coarse_fill(const float *aabb, uint32_t N, const GridDesc &full, const int nc[3], uint32_t *hist, const uint32_t *start,
                               uint32_t *ids, cudaStream_t s);
cudaError_t launch_expand_bricks(const uint32_t *start, uint32_t nbricks, uint32_t *key, cudaStream_t s);

// GS_OPT_ASYNC_BUILD: the pair count T and the touched-Gaussian count M of a grid batch stay on the device (total[0],
// total[1]); kernels read M there and return at once when T outgrew the speculative pair buffer (total == NULL: the
// host knows both, the synchronous build)
struct DevCount {
    const unsigned long long *total;
    uint32_t cap;
};

struct FwdOut {
    const float *target; float *phi; float *I; double *loss; float *dL_dphi; float *sample_err;
    uint32_t *set_count; unsigned long long *set_sum; unsigned long long *set_xor;   // debug sets (nullable)
    unsigned long long *counters;                                                   // [2] tested, hits (nullable)
    float2 *pack2;  // nullable: per-sample backward coefficients (alpha, beta) of the fused MSE loss; eps = |alpha| P / 2
    GenLoss gen;    // gen.on: the epilogue of gs_sample_fwd_loss (loss.cuh) instead of the fused MSE
    double inv_count;  // 1 / (samples of the MSE mean); 0 = 1 / (this query's P)  (gs_set_sample_count: sample-sharded ranks)
    int vec_ok;        // the caller's per-sample arrays are all 8-byte aligned: x-pairs may be moved as float2
};
struct BwdIn {
    const float *phi; const float *I; const float *dL_dphi; const float *dL_dI; const float *target;
    const float2 *pack2;  // non-null: (alpha, beta) already written by the forward (fused MSE); the other fields are unused
    float eps_scale;      // with pack2: eps = |alpha| * eps_scale  (= P / 2 for the mean-squared error)
};

cudaError_t launch_grid_fwd(const float4 *rec, uint32_t N, const GridDesc &gd, const uint32_t *pair_gauss,
                            const uint32_t *brick_start, float tau, float r2, const FwdOut &o, const float4 *jit, DevCount dc, cudaStream_t s);
// per-voxel sample positions of a jittered batch (gd.jitter; D26), batch-local sample order, written once per gs_build_accel
cudaError_t launch_jitter_table(const GridDesc &gd, float4 *jit, cudaStream_t s);
// second pass of gs_sample_fwd_loss: dL_dI[c] /= |D-| or |U+| (by sign), loss_terms = (L_rec, L_FN, L_FP)
cudaError_t launch_loss_finish(const GenLoss &L, size_t P, double nd, double *loss_terms, cudaStream_t s);
cudaError_t launch_pack_samples(const BwdIn &in, size_t P, float tau, float4 *pack, cudaStream_t s);
cudaError_t launch_grid_bwd(const float4 *rec, const float4 *setup, uint32_t N, const GridDesc &gd, const void *pack, bool pack2,
                            float r2, float *gacc, const uint32_t *order, uint32_t M, const float4 *jit, DevCount dc, cudaStream_t s);

// grid_moments: gacc holds the structured backward's rows of moment sums (GACC_GRID floats, spacing-free: the cell steps are
// folded in), only for the Gaussians with touched[i] != 0 (the others get zero gradients); eps_scale multiplies the error share
// (fused MSE: eps = |alpha| * eps_scale, else 1); touched_bound: an upper bound of the number of touched Gaussians (picks the kernel)
cudaError_t launch_finalize(const float4 *rec, const float *params, const float *gacc, uint32_t N, bool grid_moments,
                            float eps_scale, const gs_grads &out, const uint32_t *touched, DevCount dc, uint32_t touched_bound, cudaStream_t s);

// optim.cu: activations of the raw parameters and one Adam step on them
cudaError_t launch_activate(const gs_raw_params &p, float *scale, float *opacity, float *scalar, cudaStream_t s);
cudaError_t launch_adam_step(const gs_raw_params &p, const gs_grads &g, float *m, float *v, const gs_adam_cfg &cfg, float *scale_out,
                             float *opacity_out, float *scalar_out, cudaStream_t s);

// densify.cu: pruning and sample-error densification (all on `s`; `work` = 3 n + 1 uint32: flags | positions (n + 1) | kept indices)
cudaError_t launch_prune_index(const float *opacity, uint32_t n, float tau2, uint32_t *work, DevBuf &scan_tmp, cudaStream_t s);
// gathers the parameters and moments of the first n_copy Gaussians of the new set (src = NULL: identity) into `scratch`
// (37 n_new floats, laid out for n_new) and, with back = true, copies all of it back over the caller's arrays
cudaError_t launch_regather(const gs_raw_params &p, float *m, float *v, uint32_t n_new, const uint32_t *src, uint32_t n_copy, float *scratch,
                            bool back, cudaStream_t s);
cudaError_t launch_select_keys(const float *err, const float *I, const uint8_t *defined, size_t P, float tau, uint32_t *key, uint32_t *val,
                               cudaStream_t s);
cudaError_t launch_new_gaussians(const gs_raw_params &p, float *m, float *v, uint32_t n_new, const uint32_t *sel, const GridDesc &gd,
                                 const float4 *jit, const float *xyz, const float *target, float raw_scale_init, float raw_opacity_init, float clamp,
                                 float *scratch, cudaStream_t s);

// render.cu: samples of a chunk of rays (sample-major: sample k of ray r at k * nrays + r) and their compositing
cudaError_t launch_ray_samples(const float *org, const float *dir, const float *trange, uint32_t nrays, uint32_t spp, float *xyz,
                               cudaStream_t s);
cudaError_t launch_composite(const float *phi, const float *I, const float *trange, uint32_t nrays, uint32_t spp, float tau,
                             const float4 *table, uint32_t K, float4 *rgba, cudaStream_t s);

// peaks.cu: FP32 FMA and MUFU.EX2 lane-instructions per second (register-only loops, CUDA events on `s`; synchronises)
cudaError_t measure_alu_peaks(float *sink, cudaStream_t s, double *ffma_per_s, double *ex2_per_s, double *ffma2_per_s);

// LBVH
cudaError_t launch_morton(const float *xyz, size_t stride_floats, const float *aabb_valid /*nullable: aabb[N][6]*/, size_t n,
                          const gs_domain &dom, uint32_t *codes, uint32_t *ids, cudaStream_t s);
cudaError_t launch_lbvh(const uint32_t *codes, const uint32_t *ids, const float *aabb, const float4 *rec, uint32_t N, int32_t *left,
                        int32_t *right, int32_t *parent, int32_t *leaf_parent, float *node_aabb, uint32_t *flags, float4 *packed,
                        float4 *sorted_rec, cudaStream_t s);
// per-packet (32 sorted points) lists of the Gaussians that can reach the packet: chains of 32-entry chunks
struct CullLists {
    uint32_t *ids;    // [cap][32] sorted positions of Gaussians
    uint32_t *link;   // [cap] next chunk of the chain (0xffffffff = end); every linked chunk is full
    uint2 *head;      // [packets] (first chunk, entries in it)
    uint32_t *top;    // chunks requested so far (may exceed cap: the host then grows the pool and repeats)
    uint32_t cap;
    uint2 *mask;      // [cap] nullable: .x bit j = entry j of chunk c hits at least one point of its packet; .y = the chunk TWO links
                      // further down the chain (what link[link[c]] would give, 0xffffffff = none), so that a reader can have the loads
                      // of two chunks in flight instead of chasing one link at a time.  Written by k_points_fwd (which evaluates every
                      // (entry, point) predicate and walks the chain anyway), read by k_points_bwd_masked
};
cudaError_t launch_points_cull(const float4 *sorted_rec, uint32_t N, const float4 *nodes, const float4 *xyz /*sorted copy*/, const uint32_t *pt_order,
                               uint64_t P, const gs_domain &dom, float rcut, const CullLists &lists, uint32_t *overflow, int group /*2 or 4 packets per warp*/,
                               cudaStream_t s);
cudaError_t launch_points_fwd(const float4 *sorted_rec, const float4 *xyz /*sorted copy*/, const uint32_t *pt_order, uint64_t P, const CullLists &lists,
                              float tau, float r2, const FwdOut &o, cudaStream_t s);
// scatter mode (the paper's formulation): see sample_scatter.cu
uint64_t scatter_padded_points(uint64_t P);
uint32_t scatter_tree_shape(uint64_t P, PtTree *T);
// sorted copy of the query points (float4, padded with NaN to a multiple of 64): read by every point kernel of both modes
cudaError_t launch_sorted_points(const float *xyz, const uint32_t *pt_order, uint64_t P, float4 *spt, cudaStream_t s);
cudaError_t launch_scatter_build(uint64_t P, PtTree T, const float4 *spt, float *box, cudaStream_t s);
cudaError_t launch_scatter_fwd(const float4 *rec, const float *aabb, const uint32_t *gorder, uint32_t N, const PtTree &T, const float4 *spt,
                               float2 *acc, const uint32_t *pt_order, uint64_t P, float tau, float r2, const FwdOut &o, cudaStream_t s);
cudaError_t launch_scatter_bwd(const float4 *rec, const float *aabb, const uint32_t *gorder, uint32_t N, const PtTree &T, const float4 *spt,
                               float4 *coef, const uint32_t *pt_order, uint64_t P, float tau, float r2, const BwdIn &in, float *gacc,
                               cudaStream_t s);
// use_masks: lists.mask holds the hit bits of a forward on these lists (k_points_bwd_masked: entries without a hit are dropped and
// the surviving ones compacted across chunks before their records are gathered); false: every entry is evaluated (k_points_bwd)
cudaError_t launch_points_bwd(const float4 *sorted_rec, const float4 *xyz /*sorted copy*/, const uint32_t *pt_order, uint64_t P, const CullLists &lists,
                              float tau, float r2, const BwdIn &in, float *gacc, bool use_masks, cudaStream_t s);

}  // namespace gs
