/*
 * gs.h -- C ABI of the B200-native W-VEG sampler (world-space volume-encoding Gaussians).
 *
 * The library evaluates, at 3D query positions, the normalised Gaussian kernel regression of
 * arxiv/paper_2607_01164 (PAPER.md = /root/reference/PAPER.md):
 *
 *     Phi(p) = sum_i w_i v_i G_i(p) / sum_i w_i G_i(p)                      (Eq. 2)
 *     G_i(p) = exp(-1/2 (p-mu_i)^T R_i^T S_i^-2 R_i (p-mu_i))               (Eq. 3)
 *
 * over the Gaussians whose cutoff support {G_i >= tau} contains p (tau_1 = 0.01),
 * and the analytic gradients of a loss L(Phi, I) w.r.t. every Gaussian parameter
 * (PAPER.md:130, :140), for a structured grid (section 4.1) or an unstructured point
 * list (section 5.1).  DESIGN.md lists the readings D1..D14 taken where the paper is
 * silent; the ones a caller must know are repeated at the entry points below.
 *
 * Conventions
 *   - Every pointer is DEVICE memory on the context's GPU unless its name ends in _host
 *     (gs_step_host takes host memory only).  The caller owns every buffer it passes; the library never
 *     frees or retains them beyond the call's enqueued work (gs_preprocess retains NOTHING: it copies
 *     what it needs into context-owned records).  The context owns all scratch (grow-only) and
 *     frees it in gs_destroy.
 *   - All work is enqueued on the stream given to gs_create.  Calls return after enqueueing,
 *     except that gs_build_accel synchronises once (grid: to read the pair count T; points: to read
 *     the size of the per-packet cull lists and grow their pool if needed; GS_OPT_ASYNC_BUILD removes the grid's), and
 *     gs_step_host, gs_decode_grid, gs_status_query and the gs_debug_* calls synchronise before returning.  Outputs are
 *     valid once the caller synchronises the stream.
 *   - Every call returns a gs_status; no exception or abort crosses the ABI.  Arguments are
 *     validated before any launch.  gs_last_error gives a human-readable message for the last
 *     non-OK status of that context.
 *   - Call order: gs_preprocess -> gs_build_accel -> gs_sample_fwd -> gs_sample_bwd.  A call made
 *     out of order returns GS_ERR_STATE.  gs_build_accel may be repeated with a new query (a new
 *     batch) without repeating gs_preprocess as long as the Gaussians are unchanged.
 *   - Layouts are dense, row-major, fp32: mean[N,3], scale[N,3], quat[N,4] in (w,x,y,z) order,
 *     opacity[N], scalar[N]; per-sample arrays are [P].
 *   - Alignment: every array must be aligned to its element type (4 bytes; 8 for double / uint64 arrays);
 *     gs_grads.dquat must be 16-byte aligned (INVALID_ARG otherwise).  The per-sample arrays of gs_sample_fwd
 *     (target, phi, I, dL_dphi, sample_err) MAY be only 4-byte aligned (a view such as tensor[1:]): the kernels
 *     move grid samples in 8-byte x-pairs only when all of them are 8-byte aligned and fall back to scalar
 *     accesses otherwise -- same results, never a misaligned-address fault.
 */
#ifndef GS_H_
#define GS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    GS_OK = 0,
    GS_ERR_INVALID_ARG = 1, /* null pointer, bad size, bad enum, non-positive spacing, ...            */
    GS_ERR_STATE = 2,       /* call order violated, or query differs from the one the accel was built for */
    GS_ERR_OOM = 3,         /* device allocation failed                                                 */
    GS_ERR_OVERFLOW = 4,    /* pair count T does not fit 32 bits, or a traversal stack overflowed       */
    GS_ERR_CUDA = 5         /* any other CUDA runtime error (message in gs_last_error)                  */
} gs_status;

typedef struct gs_ctx gs_ctx;

/* The model: N Gaussians with mean mu_i, scale S_i, rotation R_i, value v_i ("scalar")
 * and weight w_i ("opacity").  Values are ACTIVATED (DESIGN D2): scale is the linear standard deviation
 * per principal axis (> 0), opacity the weight in (0,1), scalar the value; the quaternion need not be
 * unit -- it is normalised inside gs_preprocess and gradients are w.r.t. the raw quaternion.
 * R is the standard rotation matrix of the unit quaternion and u = S^-1 R (p - mu) (Eq. 3 read
 * literally, DESIGN D1).  A Gaussian with a non-finite parameter, a non-positive scale or a
 * zero quaternion has empty support (contributes nowhere, receives zero gradient). */
typedef struct {
    uint32_t n;
    const float *mean;    /* [n,3] */
    const float *scale;   /* [n,3] */
    const float *quat;    /* [n,4] (w,x,y,z) */
    const float *opacity; /* [n]   */
    const float *scalar;  /* [n]   */
} gs_gaussians;

/* Axis-aligned box used to quantise Morton codes (unstructured path).  lo < hi on every axis. */
typedef struct {
    float lo[3], hi[3];
} gs_domain;

typedef enum { GS_QUERY_GRID = 0, GS_QUERY_POINTS = 1 } gs_query_kind;

/* Where to sample.
 * GS_QUERY_GRID (section 4.1): voxel centres of a regular grid, p_k = fmaf((float)i_k + 0.5f, spacing_k,
 *   origin_k) for global voxel index i (DESIGN D6).  A query is one BATCH: the brick-aligned sub-box
 *   of brick_cnt bricks starting at brick brick_lo, a brick being 8^3 voxels; voxels beyond dims are
 *   clipped.  Per-sample arrays are indexed x-fastest over the batch's clipped voxel box
 *   (bx = min(8*brick_cnt_x, dims_x - 8*brick_lo_x), ...), P = bx*by*bz.
 *   jitter != 0 ("a random position in each cell every iteration"): the sample of voxel i
 *   sits at p_k = fmaf(((float)i_k + 0.5f) + j_k, spacing_k, origin_k), j_k in [-0.5, 0.5) drawn by a
 *   counter-based generator from (jitter_seed, global voxel index), 21 bits per axis (DESIGN D26): the same seed
 *   gives the same samples in every batch and on every call; pass a new seed per training iteration.
 * GS_QUERY_POINTS (section 5.1): num_points arbitrary positions xyz[P,3]; per-sample arrays follow the
 *   caller's order.  presorted != 0 promises that xyz is already spatially coherent (skips the
 *   Morton sort of the queries; results are identical either way). */
typedef struct {
    int32_t kind; /* gs_query_kind */
    int32_t dims[3];
    float origin[3];
    float spacing[3];
    int32_t brick_lo[3];
    int32_t brick_cnt[3];
    uint64_t num_points;
    const float *xyz; /* [P,3] */
    int32_t presorted;
    int32_t jitter;       /* GS_QUERY_GRID: 0 = voxel centres */
    uint64_t jitter_seed; /* GS_QUERY_GRID with jitter */
} gs_query;

/* Gradient outputs, OVERWRITTEN (not accumulated): dL/dmean[N,3], dL/dscale[N,3], dL/dquat[N,4],
 * dL/dopacity[N], dL/dscalar[N] and the per-Gaussian sampling-error statistic err[N] (nullable;
 * DESIGN D10 -- E_i = sum over covered samples of |Phi_c - t_c| w_i G_ic / I_c).  E_i is a north_star
 * quantity: the PAPER DEFINES NO per-Gaussian error (it densifies from per-sample errors, which
 * gs_sample_fwd returns as sample_err), so its definition is this library's reading, not a result of the paper. */
typedef struct {
    float *dmean, *dscale, *dquat, *dopacity, *dscalar, *err;
} gs_grads;

/* Create a context bound to CUDA device `device`; cuda_stream is a cudaStream_t (NULL = default
 * stream).  *out receives the context.  Errors: INVALID_ARG, CUDA, OOM. */
gs_status gs_create(int device, void *cuda_stream, gs_ctx **out);
void gs_destroy(gs_ctx *ctx);
const char *gs_last_error(const gs_ctx *ctx);

/* S1 (section 4.1.1): per Gaussian, normalise the quaternion, build R, the whitening matrix
 * M = S^-1 R (M^T M is the paper's "conic" R^T S^-2 R), the cutoff ellipsoid {|M d|^2 <= -2 ln tau}
 * and its world AABB (inflated by 1 + 2^-8, a safe cull for the fp32 predicate).  Results are
 * stored in the context.  dom may be NULL for grid-only use.  tau in (0,1).
 * Errors: INVALID_ARG (null, n = 0 is allowed), OOM, CUDA. */
gs_status gs_preprocess(gs_ctx *ctx, const gs_gaussians *g, const gs_domain *dom, float tau);

/* S2 / S3: build the acceleration structure for one query.
 * Grid (section 4.1.2): the (brick, gaussian) pairs of the batch, sorted by
 *   (brick, gaussian), with per-brick ranges.  The sort is a radix sort taken most-significant
 *   digit first: a histogram over the bricks each AABB overlaps, its prefix sum (= the per-brick
 *   ranges), a fill that gives every pair a slot in its brick's run, and a sort of every run by
 *   Gaussian id, so each brick's list is in ascending Gaussian id whatever the fill order was.
 * Points (north_star (2); the paper uses a BVH over the samples instead):
 *   30-bit Morton codes of the Gaussian means in `dom`, radix sort of (code, id), Karras radix
 *   tree, bottom-up AABB refit; the query points are Morton-sorted for coherence unless presorted.
 *   Then every packet of 32 consecutive sorted points walks the tree once (short stack in shared
 *   memory) and its list of reachable Gaussians is stored for gs_sample_fwd AND gs_sample_bwd of this
 *   query; the pool of list chunks is context-owned, grow-only, and sized by count-and-repeat.
 *   The lists are conservative culls: membership is decided per pair by the canonical predicate (D4).
 *   The Gaussian side (codes, sort, tree, refit, records in leaf order) depends on the model alone: the FIRST point query
 *   after a gs_preprocess builds it, the following ones (the chunks of a decode, of gs_render) reuse it and only sort and
 *   cull their own points.  A training step calls gs_preprocess and therefore rebuilds the LBVH every step.
 * Errors: STATE (no preprocess; no domain for a point query), INVALID_ARG, OVERFLOW, OOM, CUDA. */
gs_status gs_build_accel(gs_ctx *ctx, const gs_query *q);

/* S4/S5/S6 (section 4.1.3; section 5.1.2): for every sample c
 *     I_c = sum_hits w_i G_i(p_c),  Phi_c = (sum_hits v_i w_i G_i(p_c)) / I_c  if I_c > tau, else 0
 * (strict compare, empty value 0, I_c always written: DESIGN D5).  If target != NULL the fused
 * epilogue also produces (each output nullable):
 *     *loss      += (1/P) sum_c (Phi_c - target_c)^2      (double, device; the CALLER zeroes it)
 *     dL_dphi[c]  = covered ? 2 (Phi_c - target_c) / P : 0
 *     sample_err[c] = |Phi_c - target_c|
 * q must be the query the accel was built for.  Errors: STATE, INVALID_ARG, OVERFLOW, CUDA. */
gs_status gs_sample_fwd(gs_ctx *ctx, const gs_query *q, const float *target, float *phi, float *I, double *loss,
                        float *dL_dphi, float *sample_err);

/* Context options.
 * GS_OPT_POINTS_ACCEL selects how the NEXT gs_build_accel of a point query (and the forward / backward on it) works:
 *   GS_POINTS_GATHER  (default; north_star (2)): LBVH over the Gaussians, per-packet traversal into cull lists, forward
 *                     with lane = point, backward with lane = Gaussian.
 *   GS_POINTS_SCATTER (the paper's own formulation, section 5.1, Fig. 7): a wide tree over the Morton-sorted
 *                     SAMPLE POSITIONS, one warp per Gaussian walking it with the Gaussian's cutoff box; the forward adds
 *                     (w G, v w G) to the samples with vector atomics and normalises in a second kernel; the backward
 *                     keeps the 12 per-Gaussian sums in registers and writes one row per Gaussian (no atomics).
 * Both modes decide membership with the same canonical predicate: ID sets are identical, values differ by summation
 * order only.  The LBVH debug items (nodes, parents, boxes) exist in gather mode only.
 * GS_OPT_ASYNC_BUILD (0 / 1, default 0) removes the host round trip from gs_build_accel of a GRID query in steady state.
 *   The first build for a model size is synchronous and leaves 50 % headroom in the pair list; the following builds fill
 *   the list speculatively and send the pair count T and the touched-Gaussian count M to pinned host memory WITHOUT
 *   waiting; forward, backward and finalize read M on the device.  The price is CUDA's own error model: if a later batch
 *   produces more than 1.5x the pairs of the sizing build, its kernels sample nothing (they check T against the capacity on
 *   the device) and a LATER call on the context returns GS_ERR_OVERFLOW (the following build is synchronous again and sizes
 *   the buffer).  What such a batch leaves behind: phi / I / dL_dphi / sample_err untouched; NaN added to *loss (loss_terms[0]
 *   of gs_sample_fwd_loss is NaN) -- the in-band sign that the batch did not happen; gs_sample_bwd writes ZERO gradients and
 *   err for every Gaussian (never the previous step's), so an optimiser step taken before the status arrives sees an empty
 *   batch.  The call that returns GS_ERR_OVERFLOW has itself done nothing (a gs_preprocess that reports it preprocessed
 *   nothing: call it again).  The counts are picked up without stalling the host, so the report can trail the batch by several builds:
 *   every batch built since the last call that WAITED for the counts (gs_status_query, gs_debug_get, a synchronous build) is
 *   suspect and should be repeated -- gs_decode_grid does exactly that.  Point queries always synchronise once.
 * GS_OPT_BWD_HIT_MASKS (0 / 1, default 1; point queries in gather mode): gs_sample_fwd / gs_sample_fwd_loss leave one bit per
 *   cull-list entry -- does the Gaussian hit any of the packet's 32 points -- and gs_sample_bwd on the same accel evaluates only
 *   the entries whose bit is set, compacted across list chunks so that every lane holds a Gaussian that reaches the packet
 *   (on configs[4] 44 % of the list entries hit nothing, on configs[2] 33 %).  Same per-entry arithmetic: the gradients differ
 *   from the unmasked backward's by the order of the atomic additions only.  0 = evaluate every entry (the A/B baseline);
 *   a gs_sample_bwd without a preceding forward on the accel falls back to that by itself.
 * Errors: INVALID_ARG (unknown key / value). */
typedef enum { GS_OPT_POINTS_ACCEL = 0, GS_OPT_ASYNC_BUILD = 1, GS_OPT_BWD_HIT_MASKS = 2 } gs_option;
typedef enum { GS_POINTS_GATHER = 0, GS_POINTS_SCATTER = 1 } gs_points_accel;
gs_status gs_set_option(gs_ctx *ctx, int32_t key, int64_t value);

/* Sample-sharded (multi-GPU) use: the number of samples the fused MSE mean of gs_sample_fwd runs over (loss,
 * dL_dphi = 2 res / total, and the error statistic of the fused backward).  0 (the default) = the query's own P.
 * A rank that holds 1/R of the samples sets the global count, so that the per-rank losses and gradients ADD UP
 * to the one-batch ones.  Errors: INVALID_ARG (null context). */
gs_status gs_set_sample_count(gs_ctx *ctx, uint64_t total_samples);

/* The same forward with the paper's training losses fused into the epilogue.
 * `defined` (device, uint8 [P], nullable = every sample) marks the samples that lie in the volume's
 * domain (set D); the others are the samples "undefined in the volume" (set U).
 *   reconstruction over D:  L_rec = (1/|D|) sum_D rho(Phi_d - target_d), rho = |.| for GS_LOSS_L1
 *     ("L1 reconstruction loss") or (.)^2 for GS_LOSS_MSE; an uncovered sample of D
 *     enters as rho(0 - target) and passes no gradient through Phi (DESIGN D5);
 *   false negatives, Eq. 4: D- = { d in D | I_d < (1 + eps_fn) tau },
 *     L_FN = lambda_fn sum_{D-} ((1 + eps_fn) tau - I_d) / |D-|;
 *   false positives, Eq. 5: U+ = { u in U | I_u >= tau },
 *     L_FP = lambda_fp sum_{U+} I_u / |U+|.
 * Membership of D- and U+ is decided on the fp32 I against (1.0f + eps_fn) * tau and tau.  The paper
 * gives no values for eps and the lambdas: they are the caller's.  num_defined = |D| (the caller
 * knows its mask; P when defined == NULL).
 * Outputs (device; nullable except phi, I):
 *   loss_terms[3] = (L_rec, L_FN, L_FP)   (double; OVERWRITTEN, not accumulated)
 *   dL_dphi[c] = covered and defined ? rho'(Phi_c - target_c) / |D| : 0        (|x|' = sign x, 0 at 0)
 *   dL_dI[c]   = -lambda_fn / |D-| on D-,  +lambda_fp / |U+| on U+,  0 elsewhere
 *   sample_err[c] = defined ? |Phi_c - target_c| : 0
 * |D-| and |U+| are only known once every sample has been seen: the epilogue writes dL_dI
 * un-normalised and a second, elementwise kernel divides by the counts and writes loss_terms.
 * Pass the outputs to gs_sample_bwd(phi, I, dL_dphi, dL_dI, target); on a GRID query the epilogue also keeps the
 * per-sample backward coefficients (alpha, beta, eps), so gs_sample_bwd(dL_dphi = NULL) differentiates this loss
 * without re-reading the five per-sample arrays.
 * Errors: STATE, INVALID_ARG (negative lambda / eps, unknown kind, num_defined = 0 with P > 0), CUDA. */
typedef enum { GS_LOSS_MSE = 0, GS_LOSS_L1 = 1 } gs_loss_kind;
typedef struct gs_loss {
    int32_t kind;            /* gs_loss_kind */
    float lambda_fn, eps_fn; /* Eq. 4; lambda_fn = 0 switches the term off */
    float lambda_fp;         /* Eq. 5; lambda_fp = 0 switches the term off */
    const uint8_t *defined;  /* device [P] or NULL */
    uint64_t num_defined;    /* |D| */
} gs_loss;
gs_status gs_sample_fwd_loss(gs_ctx *ctx, const gs_query *q, const gs_loss *loss, const float *target, float *phi, float *I,
                             double *loss_terms, float *dL_dphi, float *dL_dI, float *sample_err);

/* S7/S8 (section 4.1.4; section 5.1.2): gradients of L w.r.t. the Gaussian parameters
 * from dL_dphi[P] and dL_dI[P] (nullable = 0), re-computing the kernel weights from phi/I of the
 * forward pass (nothing else is kept from it).  dL_dphi of an uncovered sample (I_c <= tau) is
 * ignored.  target (nullable) is only used for the error statistic out->err.
 * Fused-loss form: dL_dphi == NULL means "the loss of the preceding forward on this accel" -- the MSE of
 * gs_sample_fwd(target != NULL), or (grid queries) the losses of gs_sample_fwd_loss: that forward keeps its
 * per-sample backward coefficients (alpha, beta, eps) in context scratch, so the backward reads them instead
 * of phi / I / dL_dphi / target (all ignored, may be NULL); dL_dI must be NULL.
 * STATE if no such forward preceded (or the scratch was overwritten by a non-fused gs_sample_bwd).
 * Errors: STATE, INVALID_ARG, OVERFLOW, CUDA. */
gs_status gs_sample_bwd(gs_ctx *ctx, const gs_query *q, const float *phi, const float *I, const float *dL_dphi,
                        const float *dL_dI, const float *target, const gs_grads *out);

/* One whole training-step pass of the hot path from HOST buffers (all pointers are host memory,
 * q->xyz included): copies the model, the query points and the target to the device, runs
 * preprocess -> build_accel -> forward (fused MSE) -> backward, copies phi, I, the loss and the
 * gradients back, and synchronises.  Output pointers may be NULL to skip their copy (loss excepted).
 * Errors: any of the above. */
gs_status gs_step_host(gs_ctx *ctx, const gs_gaussians *g_host, const gs_domain *dom, float tau, const gs_query *q_host,
                       const float *target_host, float *phi_host, float *I_host, double *loss_host,
                       const gs_grads *grads_host);

/* ---- parity / introspection: read-only views of context-owned device buffers ---------------- */
typedef enum {
    GS_DBG_RECORDS = 0,      /* float4 [4][N]: (mu.xyz,w) (M row0,v) (M row1,0) (M row2,0); count = N      */
    GS_DBG_AABB = 1,         /* float [N][6] lo.xyz hi.xyz                                                 */
    GS_DBG_BRICK_COUNT = 2,  /* uint32 [N] bricks of the current batch each Gaussian overlaps              */
    GS_DBG_PAIR_BRICK = 3,   /* uint32 [T] sorted brick ids (batch-local)                                  */
    GS_DBG_PAIR_GAUSS = 4,   /* uint32 [T] Gaussian ids, ascending inside a brick                          */
    GS_DBG_BRICK_START = 5,  /* uint32 [nbricks+1]                                                         */
    GS_DBG_LEAF_MORTON = 6,  /* uint32 [N] sorted Morton codes of the Gaussians                            */
    GS_DBG_LEAF_ORDER = 7,   /* uint32 [N] Gaussian id of each leaf in sorted order                        */
    GS_DBG_NODE_LEFT = 8,    /* int32 [N-1] child: >= 0 internal node, < 0 is ~leaf                        */
    GS_DBG_NODE_RIGHT = 9,   /* int32 [N-1]                                                                */
    GS_DBG_NODE_PARENT = 10, /* int32 [N-1], root = -1                                                     */
    GS_DBG_LEAF_PARENT = 11, /* int32 [N]                                                                  */
    GS_DBG_NODE_AABB = 12,   /* float [N-1][6]                                                             */
    GS_DBG_POINT_ORDER = 13, /* uint32 [P] caller index of the k-th point in traversal order               */
    GS_DBG_POINT_MORTON = 14 /* uint32 [P] sorted Morton codes of the query points                         */
} gs_debug_item;

/* *dev_ptr / *count describe the buffer as of the work enqueued so far (synchronise before reading).
 * Errors: STATE if the item has not been built, INVALID_ARG. */
gs_status gs_debug_get(gs_ctx *ctx, int32_t what, const void **dev_ptr, size_t *count);

/* Convenience: synchronise and copy the first `bytes` bytes of a debug buffer to HOST memory.
 * Errors: as gs_debug_get; INVALID_ARG if bytes exceeds the buffer. */
gs_status gs_debug_read(gs_ctx *ctx, int32_t what, void *dst_host, size_t bytes);

/* Per-sample intersection SETS for bit-exact comparison: number of Gaussians whose support contains
 * the sample, and the sum and xor over them of mix64(id) (splitmix64 finaliser of id + golden
 * gamma), through the same traversal as gs_sample_fwd.  Device outputs [P]; synchronises. */
gs_status gs_debug_point_sets(gs_ctx *ctx, const gs_query *q, uint32_t *count, uint64_t *hash_sum, uint64_t *hash_xor);

/* Counters of the last forward pass (device-side work statistics, for the roofline report):
 * pairs tested (predicate evaluated) and pairs hit.  Only collected by gs_debug_point_sets. */
gs_status gs_debug_counters(gs_ctx *ctx, uint64_t *tested_host, uint64_t *hits_host);

/* ---- training-step completion ---------------------------------------------
 * Raw parameters: scale = exp(raw_scale), opacity = sigmoid(raw_opacity),
 * scalar = sigmoid(raw_scalar); mean and quat are their own raw parameters (the quaternion is
 * normalised inside gs_preprocess).  All pointers are DEVICE memory owned by the caller. */
typedef struct gs_raw_params {
    uint32_t n;
    float *mean;        /* [n,3] */
    float *raw_scale;   /* [n,3] log of the scale */
    float *quat;        /* [n,4] (w,x,y,z), any non-zero norm */
    float *raw_opacity; /* [n]   logit of w */
    float *raw_scalar;  /* [n]   logit of v */
} gs_raw_params;
/* scale[n,3], opacity[n], scalar[n] = the activated values gs_preprocess takes.  Errors: INVALID_ARG, CUDA. */
gs_status gs_params_activate(gs_ctx *ctx, const gs_raw_params *p, float *scale, float *opacity, float *scalar);

/* One Adam step (Kingma & Ba, the paper's optimiser) on the raw parameters, in place:
 *     m = beta1 m + (1 - beta1) g;  v = beta2 v + (1 - beta2) g^2;
 *     p -= lr (m / (1 - beta1^step)) / (sqrt(v / (1 - beta2^step)) + eps)
 * `g` holds the gradients w.r.t. the ACTIVATED values exactly as gs_sample_bwd wrote them (err unused);
 * the chain rule of the activations is applied here: d/d raw_scale = dscale * scale,
 * d/d raw_opacity = dopacity * w (1 - w), d/d raw_scalar = dscalar * v (1 - v).
 * lr = (mean, scale, quat, opacity, scalar); the paper's values are
 * (0.00016, 0.001, 0.0001, 0.025, 0.0025) with Adam's defaults beta1 0.9, beta2 0.999, eps 1e-8.
 * m, v: device [12 n] moment blocks laid out mean 3n | scale 3n | quat 4n | opacity n | scalar n,
 * zeroed by the caller before step 1.  step >= 1.  scale_out / opacity_out / scalar_out (nullable)
 * receive the activations of the UPDATED parameters, i.e. the next gs_preprocess's inputs.
 * The paper's soft cap on the scales has no printed formula and is not applied.
 * Errors: INVALID_ARG (null pointers, step < 1, betas outside [0,1), negative lr / eps), CUDA. */
typedef struct gs_adam_cfg {
    float lr[5];
    float beta1, beta2, eps;
    int32_t step;
} gs_adam_cfg;
gs_status gs_adam_step(gs_ctx *ctx, const gs_raw_params *p, const gs_grads *g, float *m, float *v, const gs_adam_cfg *cfg,
                       float *scale_out, float *opacity_out, float *scalar_out);

/* Pruning (Gaussians below the weight threshold, 0.005 in the paper, are removed).  Keeps, in their
 * order, the Gaussians with opacity[i] >= tau2 (`opacity` = the ACTIVATED weights, device [n], e.g. the
 * opacity_out of gs_adam_step); parameters and both Adam moment blocks are compacted in place (the blocks are
 * re-laid-out for the new count).  *n_new_host = the new count; the caller updates p->n.  Synchronises.
 * Errors: INVALID_ARG, OOM, CUDA. */
gs_status gs_prune(gs_ctx *ctx, const gs_raw_params *p, float *m, float *v, const float *opacity, float tau2, uint32_t *n_new_host);

/* Sample-error densification: one new Gaussian at each of the k highest-error samples of the
 * query the accel was built for, false negatives (defined samples with I <= tau) first, equal errors by lower sample
 * index; only samples marked in `defined` (device uint8 [P], NULL = all; num_defined = their count) are candidates.
 * sample_err, I, target: device [P] (the outputs / input of the last forward).  At most capacity - p->n Gaussians
 * are added (`capacity` = Gaussians the caller's parameter arrays and [12 capacity] moment arrays can hold).
 * A new Gaussian is initialised as in PAPER.md:140 / :154: mean = the sample position, raw_scale = raw_scale_init on
 * all axes (the paper's density-dependent initial scale has no printed formula: the caller's), identity rotation,
 * raw_opacity = raw_opacity_init (logit of 0.01 in the paper), raw_scalar = logit(clip(target, 1e-4, 1 - 1e-4)),
 * zero Adam moments.  *n_new_host = the new count; the caller updates p->n.  Synchronises.
 * Errors: STATE (no accel), INVALID_ARG, OOM, CUDA. */
gs_status gs_densify(gs_ctx *ctx, const gs_raw_params *p, float *m, float *v, uint32_t capacity, const gs_query *q,
                     const float *sample_err, const float *I, const uint8_t *defined, uint64_t num_defined, const float *target,
                     uint32_t k, float raw_scale_init, float raw_opacity_init, uint32_t *n_new_host);

/* Status of the context's current model / accel.  Gaussians with a non-finite parameter, a non-positive scale
 * or a zero quaternion are not an error: they have empty support (see gs_gaussians) and are COUNTED by
 * gs_preprocess; this call surfaces the count.  HOST output; synchronises the stream.
 * Errors: INVALID_ARG, CUDA. */
typedef struct gs_status_info {
    uint64_t num_gaussians;       /* N of the last gs_preprocess (0 before it)                           */
    uint64_t invalid_gaussians;   /* of those, how many have empty support because a parameter is invalid */
    uint64_t grid_pairs;          /* grid accel: T = (brick, gaussian) pairs of the current batch          */
    uint64_t grid_touched;        /* grid accel: Gaussians that overlap a brick of the current batch       */
    uint64_t cull_chunk_capacity; /* point accel: 32-entry list chunks the pool holds                      */
    uint64_t decode_repeats;      /* batches gs_decode_grid repeated so far (asynchronous build overflow)  */
} gs_status_info;
gs_status gs_status_query(gs_ctx *ctx, gs_status_info *out_host);

/* ---- forward-only decode of a region of a structured grid in brick-aligned batches (BASELINE.json configs[3]: "decoded in
 * 128^3 brick-aligned batches, forward-only full decode"; the use the paper's models are made for) ----------
 * `region` is a GS_QUERY_GRID descriptor (no jitter) whose brick_lo / brick_cnt give the sub-box to decode (inside the grid:
 * brick_lo + brick_cnt <= ceil(dims / 8) per axis, checked before anything is enqueued); it is cut into
 * batches of batch_bricks[0..2] bricks (the last batch per axis may be smaller), enumerated x fastest.  Every batch is one
 * gs_build_accel + gs_sample_fwd; the batches are dealt round-robin to num_streams (1..8, 0 = 4) worker contexts that the
 * library keeps on CUDA streams of its own, each with its own gs_preprocess of the model, so that the build of one batch
 * runs beside the forward of another (a 128^3 batch is a chain of small kernels: launch- and tail-bound on one stream).
 * Output layout: BATCH-MAJOR.  phi / I (device, region's sample count) hold batch 0's samples first (in that batch's own
 * x-fastest order, exactly what gs_sample_fwd writes for it), then batch 1's, ...  The values are those of gs_sample_fwd.
 * g: device arrays, read on ctx's stream order (the workers wait for everything enqueued on it so far).  The call returns
 * when the decode is COMPLETE (it synchronises the worker streams -- on failure too: no work of this call is in flight once
 * it has returned, but phi / I may then hold the batches that did finish).  The context's own preprocess / accel state is not
 * touched.  Errors: INVALID_ARG, OOM, OVERFLOW, CUDA. */
gs_status gs_decode_grid(gs_ctx *ctx, const gs_gaussians *g, float tau, const gs_query *region, const int32_t *batch_bricks,
                         int32_t num_streams, float *phi, float *I);

/* ---- volume rendering over the sampler (Fig. 1, Fig. 9) ---------------
 * Emission-absorption ray marching of the current model (the one given to the last gs_preprocess, which must have had a
 * domain): every ray r takes spp samples at t_k = t_near + (k + 1/2) dt, dt = (t_far - t_near) / spp, p = o + t_k d
 * (float32: dt = (t1 - t0) / spp; t_k = fmaf((float)k + 0.5f, dt, t0); p = fmaf(t_k, d, o), DESIGN D27), evaluates the model
 * there with the point-query forward of this library, and composites front to back
 *     alpha_k = I_k > tau ? 1 - exp(-sigma(Phi_k) dt) : 0;   C += T alpha_k rgb(Phi_k);   T *= 1 - alpha_k
 * A sample the model does not cover (I <= tau) is empty space: the model's own domain test, no
 * surface mesh.  (rgb, sigma)(x) = linear interpolation of table[table_size][4] over x = clamp(Phi, 0, 1).
 * All pointers are DEVICE memory: origins[n,3], dirs[n,3], t_range[n,2] (a ray with t_far <= t_near sees nothing),
 * table (16-byte aligned), rgba[n,4] (16-byte aligned; OVERWRITTEN with (C, 1 - T)).  Rays are processed in chunks of
 * <= 2^24 samples; each chunk rebuilds the point acceleration structure in the mode of GS_OPT_POINTS_ACCEL, so a
 * caller's own accel is invalid afterwards (gs_build_accel again).  No window, swapchain or graphics API is involved:
 * the image is the rgba buffer.  Errors: STATE (no preprocess / no domain), INVALID_ARG, OOM, OVERFLOW, CUDA. */
gs_status gs_render(gs_ctx *ctx, uint32_t num_rays, const float *origins, const float *dirs, const float *t_range, uint32_t spp,
                    const float *table, uint32_t table_size, float *rgba);

/* ---- measurement: CUDA-event timing of the stages, on the context's stream --------------------
 * While enabled, every stage of the calls above is bracketed by a pair of CUDA events recorded on
 * the context's stream.  gs_profile_read synchronises the stream, adds up the elapsed time of all
 * pairs recorded since the last read and resets them.  ms_host[GS_PROF_STAGES] receives milliseconds,
 * calls_host[GS_PROF_STAGES] the number of times the stage ran, *launches_host the number of kernels
 * this library launched since the last read (memsets and copies not counted).  All outputs nullable.
 * Errors: INVALID_ARG, CUDA. */
typedef enum {
    GS_PROF_PREPROCESS = 0, /* S1 kernel                                                   */
    GS_PROF_BUILD = 1,      /* S2 or S3: every kernel of gs_build_accel                    */
    GS_PROF_FWD = 2,        /* S4/S5 + S6: the forward sampling kernel                     */
    GS_PROF_BWD_PACK = 3,   /* per-sample coefficients (structured backward only)          */
    GS_PROF_BWD = 4,        /* S7: the backward sampling kernel                            */
    GS_PROF_FINALIZE = 5,   /* S8                                                          */
    GS_PROF_CULL = 6,       /* unstructured: per-packet LBVH traversal + cull lists (inside gs_build_accel;
                               its time is ALSO part of GS_PROF_BUILD)                      */
    GS_PROF_STAGES = 7
} gs_prof_stage;
gs_status gs_profile_enable(gs_ctx *ctx, int32_t on);
gs_status gs_profile_read(gs_ctx *ctx, float *ms_host, uint32_t *calls_host, uint64_t *launches_host);

/* Measured denominators of the plain-ALU roofline the sampling kernels are held against (the path is
 * bound by FP32 issue, not by a dense contraction; north_star: "FP32/SFU issue utilisation against the
 * chip's peak"): FP32 FMA lane-instructions per second and MUFU.EX2 per second of this device at its
 * current clocks, from register-only loops timed with CUDA events on the context's stream; ffma2 (nullable) =
 * FMA lane-OPERATIONS per second through the packed fma.rn.f32x2 form (two per lane-instruction).
 * HOST outputs; synchronises.  Errors: INVALID_ARG, OOM, CUDA. */
gs_status gs_measure_alu_peaks2(gs_ctx *ctx, double *ffma_per_s_host, double *ex2_per_s_host, double *ffma2_per_s_host);
/* The same measurement under the name and prototype this header had before the packed-FMA figure was added (three
 * arguments, all required).  Kept so that a caller compiled against that header keeps working: an exported C symbol
 * carries no prototype, so its argument list must never change -- a new argument means a new name. */
gs_status gs_measure_alu_peaks(gs_ctx *ctx, double *ffma_per_s_host, double *ex2_per_s_host);

/* ---- sampling without device allocation ----------------------------------------------------------------------------
 * Forward sampling (Eq. 2 / Eq. 3; cutoff PAPER.md:116; coverage rule PAPER.md:126) of a SMALL model at a
 * list of points, for callers that cannot allocate device memory: a host application that handed the whole GPU to its own
 * memory pool at start-up (cudaMalloc then fails or eats the pool's head-room), a real-time loop that cannot take the
 * device-wide stall of cudaMalloc / cudaFree, a plug-in that may only touch buffers its host gives it.  Everything else in
 * this header works through a gs_ctx whose scratch arenas are cudaMalloc'd (gs_create already allocates); this call takes
 * no context and calls no cudaMalloc, cudaFree or other allocating routine, on any call.
 *
 * Its scratch (the per-Gaussian records of S1: means, weights, whitening matrices, cutoff boxes) is a fixed array inside
 * the library's device image, sized for GS_PROBE_MAX_GAUSSIANS Gaussians: about 1.9 MiB that EVERY GPU which loads this
 * library holds until the process exits, whether or not this call is ever made.  A model with more Gaussians is refused
 * (GS_ERR_INVALID_ARG, nothing launched); so are more than GS_PROBE_MAX_POINTS points per call -- split the list.
 *
 * device / cuda_stream: the GPU and the cudaStream_t (NULL = default stream) the work is enqueued on; the call returns
 * after enqueueing and leaves the thread's current device as it found it.  g, xyz[num_points,3], phi[num_points],
 * I[num_points]: DEVICE memory on that GPU, owned by the caller, layouts and value conventions as for gs_preprocess /
 * gs_sample_fwd (activated parameters, quaternion normalised inside, invalid Gaussians have empty support, a NaN point
 * gets I = 0, Phi = 0).  Outputs, valid once the stream is synchronised:
 *     I_c = sum_hits w_i G_i(p_c),   Phi_c = I_c > tau ? (sum_hits v_i w_i G_i(p_c)) / I_c : 0
 * with the same per-pair membership decision as gs_sample_fwd (the sets of contributing Gaussians are identical; values
 * differ from gs_sample_fwd's by fp32 summation order only).  Every Gaussian is tested against every point: the cost is
 * n * num_points pair tests, which is why the model size is capped.
 *
 * First call on a device: it looks up the device address of the scratch array (cudaGetSymbolAddress, once per device,
 * under a host mutex).  That lookup may make the CUDA runtime load the library's device code onto the GPU, so make the
 * first call on each device during start-up -- before any stream capture begins and before the time-critical part.
 * A call with num_points = 0 does the set-up and launches nothing.
 *
 * Sharing: all calls on a device use the ONE array, and it keeps the previous call's contents.  Each call overwrites the
 * rows of its own n Gaussians and clears its one counter before use, and never reads rows beyond n, so calls that run one
 * after the other (same stream, or ordered by events) are independent of each other.  Calls that may OVERLAP on the GPU
 * -- different streams without ordering, or several host threads on their own streams -- race on the array and produce
 * garbage: serialise them.  gs_ctx-based calls never touch the array and may overlap with it freely.
 *
 * err_host (nullable): a caller-owned HOST buffer of err_cap bytes that receives a NUL-terminated message for a non-OK
 * status (there is no context for gs_last_error to consult).
 * Errors: INVALID_ARG (null pointer, n > GS_PROBE_MAX_GAUSSIANS, num_points > GS_PROBE_MAX_POINTS, tau outside (0,1)),
 * CUDA (no such device, set-up or launch failure). */
#define GS_PROBE_MAX_GAUSSIANS 16384u
#define GS_PROBE_MAX_POINTS (1ull << 31)
gs_status gs_probe_points_static(int device, void *cuda_stream, const gs_gaussians *g, float tau, const float *xyz,
                                 uint64_t num_points, float *phi, float *I, char *err_host, size_t err_cap);

#ifdef __cplusplus
}
#endif
#endif /* GS_H_ */
