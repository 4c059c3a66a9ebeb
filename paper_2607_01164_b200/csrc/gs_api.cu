// gs_api.cu -- the C ABI of include/gs.h: argument validation, context-owned scratch, launch order.
// Every step of the path runs in the kernels of this directory; this file only orchestrates.
#include <math.h>
#include <stdio.h>
#include <string.h>
#include <new>
#include <thread>

#include "gs_internal.cuh"

using namespace gs;

namespace gs {
thread_local unsigned long long *tl_launches = nullptr;
}

namespace {

// binds the calling thread's launch counter to the context for the duration of one C-ABI call (nests)
struct LaunchScope {
    unsigned long long *prev;
    explicit LaunchScope(gs_ctx *c) : prev(gs::tl_launches) { if (c) gs::tl_launches = &c->launches; }
    ~LaunchScope() { gs::tl_launches = prev; }
};

// RAII bracket: two CUDA events around a stage on the context's stream while profiling is enabled
struct Stage {
    gs_ctx *ctx;
    gs_ctx::ProfPair pp{};
    bool on = false;
    Stage(gs_ctx *c, int stage) : ctx(c) {
        if (!c->prof) return;
        if (!c->prof_free.empty()) { pp = c->prof_free.back(); c->prof_free.pop_back(); }
        else if (cudaEventCreate(&pp.a) != cudaSuccess || cudaEventCreate(&pp.b) != cudaSuccess) { cudaGetLastError(); return; }
        pp.stage = stage;
        on = cudaEventRecord(pp.a, c->stream) == cudaSuccess;
    }
    ~Stage() {
        if (!on) return;
        cudaEventRecord(pp.b, ctx->stream);
        ctx->prof_pending.push_back(pp);
    }
};

gs_status fail(gs_ctx *ctx, gs_status st, const char *what) {
    if (ctx) ctx->err = what;
    return st;
}
gs_status fail_cuda(gs_ctx *ctx, cudaError_t e, const char *where) {
    if (ctx) {
        ctx->err = std::string(where) + ": " + cudaGetErrorString(e);
    }
    cudaGetLastError();  // clear sticky-less error state
    return e == cudaErrorMemoryAllocation ? GS_ERR_OOM : GS_ERR_CUDA;
}

#define CK(expr, where)                                        \
    do {                                                       \
        cudaError_t e__ = (expr);                              \
        if (e__ != cudaSuccess) return fail_cuda(ctx, e__, where); \
    } while (0)

bool same_query(const gs_query &a, const gs_query &b) {
    if (a.kind != b.kind) return false;
    if (a.kind == GS_QUERY_GRID) {
        for (int k = 0; k < 3; k++)
            if (a.dims[k] != b.dims[k] || a.origin[k] != b.origin[k] || a.spacing[k] != b.spacing[k] ||
                a.brick_lo[k] != b.brick_lo[k] || a.brick_cnt[k] != b.brick_cnt[k])
                return false;
        return (a.jitter != 0) == (b.jitter != 0) && (!a.jitter || a.jitter_seed == b.jitter_seed);
    }
    return a.num_points == b.num_points && a.xyz == b.xyz && a.presorted == b.presorted;
}

gs_status validate_query(gs_ctx *ctx, const gs_query *q, GridDesc *gd, uint64_t *P) {
    if (!q) return fail(ctx, GS_ERR_INVALID_ARG, "query is NULL");
    if (q->kind == GS_QUERY_GRID) {
        uint64_t p = 1, nb = 1;
        for (int k = 0; k < 3; k++) {
            if (q->dims[k] <= 0 || !(q->spacing[k] > 0.f) || !isfinite(q->spacing[k]) || !isfinite(q->origin[k]))
                return fail(ctx, GS_ERR_INVALID_ARG, "grid: dims and spacing must be positive and finite");
            const int nbk = (q->dims[k] + BRICK - 1) / BRICK;
            if (q->brick_lo[k] < 0 || q->brick_cnt[k] <= 0 || q->brick_lo[k] + q->brick_cnt[k] > nbk)
                return fail(ctx, GS_ERR_INVALID_ARG, "grid: brick_lo/brick_cnt outside the grid");
            gd->dims[k] = q->dims[k];
            gd->origin[k] = q->origin[k];
            gd->spacing[k] = q->spacing[k];
            gd->brick_lo[k] = q->brick_lo[k];
            gd->brick_cnt[k] = q->brick_cnt[k];
            const int ext = BRICK * q->brick_cnt[k], rest = q->dims[k] - BRICK * q->brick_lo[k];
            gd->bdim[k] = ext < rest ? ext : rest;
            gd->inv_brick[k] = 1.0f / (8.0f * q->spacing[k]);
            gd->nb_total[k] = nbk;
            p *= (uint64_t)gd->bdim[k];
            nb *= (uint64_t)q->brick_cnt[k];
        }
        if (nb >= (1ull << 31)) return fail(ctx, GS_ERR_INVALID_ARG, "grid: too many bricks in one batch");
        for (int k = 0; k < 3; k++)  // the kernels index samples with 32 bits and cells with 10 bits per axis
            if (gd->bdim[k] > 2048) return fail(ctx, GS_ERR_INVALID_ARG, "grid: a batch may span at most 2048 voxels per axis");
        if (p >= (1ull << 32)) return fail(ctx, GS_ERR_INVALID_ARG, "grid: a batch may hold at most 2^32-1 samples");
        gd->jitter = q->jitter != 0;
        gd->jitter_seed = q->jitter ? q->jitter_seed : 0ull;
        *P = p;
        return GS_OK;
    }
    if (q->kind == GS_QUERY_POINTS) {
        if (q->num_points > 0 && !q->xyz) return fail(ctx, GS_ERR_INVALID_ARG, "points: xyz is NULL");
        if (q->num_points >= (1ull << 32)) return fail(ctx, GS_ERR_INVALID_ARG, "points: more than 2^32-1 points in one query");
        *P = q->num_points;
        return GS_OK;
    }
    return fail(ctx, GS_ERR_INVALID_ARG, "query kind");
}

CullLists cull_lists(gs_ctx *ctx) {
    return CullLists{ctx->cull_ids.as<uint32_t>(), ctx->cull_link.as<uint32_t>(), ctx->cull_head.as<uint2>(),
                     ctx->counters.as<uint32_t>() + 2, ctx->cull_cap, nullptr};
}

// GS_OPT_ASYNC_BUILD: pick up the pair count T and the touched count M of the last grid build once they have arrived in
// pinned host memory.  If T outgrew the speculative buffer the kernels of that batch did nothing: grow, and report it.
gs_status resolve_grid_counts(gs_ctx *ctx, bool wait = true) {
    if (!ctx->grid_pending) return GS_OK;
    if (!wait) {   // between the batches of a stream of builds: take the counts if they have arrived, never stall the host
        const cudaError_t q = cudaEventQuery(ctx->grid_event);
        if (q == cudaErrorNotReady) return GS_OK;
        if (q != cudaSuccess) return fail_cuda(ctx, q, "query the pair count");
    } else {
        cudaError_t e = cudaEventSynchronize(ctx->grid_event);
        if (e != cudaSuccess) return fail_cuda(ctx, e, "wait for the pair count");
    }
    ctx->grid_pending = false;
    const unsigned long long T = ctx->grid_host[0], M = ctx->grid_host[1], sticky = ctx->grid_host[3];
    if (sticky) {   // some batch since the last look outgrew the speculative pair buffer: its kernels did nothing
        cudaMemsetAsync(ctx->counters.as<unsigned long long>() + 7, 0, 8, ctx->stream);
        ctx->accel_kind = -1;
        ctx->grid_warm_N = 0xffffffffu;   // the next build is synchronous and sizes the buffer
        return fail(ctx, GS_ERR_OVERFLOW, "asynchronous build: the pair list of an earlier batch outgrew its speculative capacity; "
                                          "that batch's outputs are invalid -- repeat it (the next gs_build_accel is synchronous)");
    }
    if (T >= (1ull << 32)) return fail(ctx, GS_ERR_OVERFLOW, "pair count T does not fit 32 bits");
    ctx->T = (uint32_t)T;
    ctx->M = ctx->M_hint = (uint32_t)M;
    return GS_OK;
}

DevCount dev_count(gs_ctx *ctx) {
    if (ctx->accel_kind == GS_QUERY_GRID && ctx->grid_pending)
        return DevCount{ctx->counters.as<unsigned long long>() + 4, (uint32_t)(ctx->pair_gauss.cap / 4 < 0xffffffffull ? ctx->pair_gauss.cap / 4 : 0xffffffffull)};
    return DevCount{nullptr, 0};
}

// number of order-list entries the backward / finalize launches are sized for: M, or (M still on the device) a bound from
// the last known M -- the kernels stride over the real one
uint32_t grid_M_launch(gs_ctx *ctx) {
    if (!ctx->grid_pending) return ctx->M;
    const uint64_t b = (uint64_t)ctx->M_hint + ctx->M_hint / 4 + 4096;
    return (uint32_t)(b < ctx->N ? b : ctx->N);
}

bool same_geometry(const GridDesc &a, const GridDesc &b) {
    for (int k = 0; k < 3; k++)
        if (a.dims[k] != b.dims[k] || a.origin[k] != b.origin[k] || a.spacing[k] != b.spacing[k]) return false;
    return true;
}

// Candidate Gaussians of a grid batch.  A batch that covers a small part of a large grid (configs[3]: a 128^3 batch touches
// 0.3 % of the model) should not look at every Gaussian: from the second such batch after a gs_preprocess on, a coarse index
// (cells of COARSE_B^3 bricks) built once over the whole model hands every batch the Gaussians of the <= 8 cells it overlaps.
gs_status batch_candidates(gs_ctx *ctx, const GridDesc &gd, uint32_t nbricks, CandSegs *cs) {
    memset(cs, 0, sizeof *cs);
    const uint32_t N = ctx->N;
    int nc[3], clo[3], chi[3];
    uint64_t total_bricks = 1, ncell = 1, nbatch = 1;
    for (int k = 0; k < 3; k++) {
        nc[k] = (gd.nb_total[k] + COARSE_B - 1) / COARSE_B;
        clo[k] = gd.brick_lo[k] / COARSE_B;
        chi[k] = (gd.brick_lo[k] + gd.brick_cnt[k] - 1) / COARSE_B;
        total_bricks *= (uint64_t)gd.nb_total[k];
        ncell *= (uint64_t)nc[k];
        nbatch *= (uint64_t)(chi[k] - clo[k] + 1);
    }
    const bool small = N >= 65536 && (uint64_t)nbricks * 8 <= total_bricks && nbatch <= 8 && ncell <= (1u << 24);
    if (!small || ctx->builds_since_pre < 1) return GS_OK;   // the first batch after a preprocess pays the full pass (a training step has only one)
    cudaStream_t s = ctx->stream;
    if (!ctx->cidx_valid || !same_geometry(ctx->cidx_geom, gd)) {
        ctx->prev_cand.ids = nullptr;   // the id list is about to be rebuilt (and may move): the counts are cleared wholesale
        ctx->bcount_exact = false;
        GridDesc full = gd;
        for (int k = 0; k < 3; k++) { full.brick_lo[k] = 0; full.brick_cnt[k] = gd.nb_total[k]; full.bdim[k] = gd.dims[k]; }
        CK(ctx->cidx_hist.reserve(ncell * 4), "alloc coarse index");
        CK(ctx->cidx_start.reserve((ncell + 1) * 4), "alloc coarse index");
        CK(launch_coarse_count(ctx->aabb.as<float>(), N, full, nc, ctx->cidx_hist.as<uint32_t>(), s), "coarse count");
        CK(exclusive_scan_u32(ctx->cidx_hist.as<uint32_t>(), ctx->cidx_start.as<uint32_t>(), ncell, ctx->scan_tmp, s), "coarse scan");
        ctx->cidx_start_host.resize(ncell + 1);
        CK(cudaMemcpyAsync(ctx->cidx_start_host.data(), ctx->cidx_start.p, (ncell + 1) * 4, cudaMemcpyDeviceToHost, s), "read coarse index");
        CK(cudaStreamSynchronize(s), "sync (coarse index)");   // once per index, i.e. once per decode
        CK(ctx->cidx_ids.reserve(((size_t)ctx->cidx_start_host[ncell] + 1) * 4), "alloc coarse index");
        CK(launch_coarse_fill(ctx->aabb.as<float>(), N, full, nc, ctx->cidx_hist.as<uint32_t>(), ctx->cidx_start.as<uint32_t>(),
                              ctx->cidx_ids.as<uint32_t>(), s), "coarse fill");
        ctx->cidx_valid = true;
        ctx->cidx_geom = gd;
        for (int k = 0; k < 3; k++) ctx->cidx_nc[k] = nc[k];
    }
    cs->ids = ctx->cidx_ids.as<uint32_t>();
    uint32_t n = 0, run = 0;
    for (int z = clo[2]; z <= chi[2]; z++)
        for (int y = clo[1]; y <= chi[1]; y++)
            for (int x = clo[0]; x <= chi[0]; x++) {
                const size_t c = ((size_t)z * nc[1] + y) * nc[0] + x;
                cs->start[n] = ctx->cidx_start_host[c];
                cs->prefix[n] = run;
                run += ctx->cidx_start_host[c + 1] - ctx->cidx_start_host[c];
                cs->cell[n][0] = x; cs->cell[n][1] = y; cs->cell[n][2] = z;
                n++;
            }
    for (uint32_t k = n; k <= 8; k++) cs->prefix[k] = run;
    cs->n = n;
    cs->total = run;
    for (int k = 0; k < 3; k++) cs->clo[k] = clo[k];
    return GS_OK;
}

int bits_for(uint64_t n) {  // bits needed to represent values in [0, n)
    int b = 0;
    while (b < 32 && (1ull << b) < n) b++;
    return b < 1 ? 1 : b;
}

}  // namespace

extern "C" {

gs_status gs_create(int device, void *cuda_stream, gs_ctx **out) {
    if (!out) return GS_ERR_INVALID_ARG;
    *out = nullptr;
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count) { cudaGetLastError(); return GS_ERR_CUDA; }
    if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return GS_ERR_CUDA; }
    gs_ctx *ctx = new (std::nothrow) gs_ctx();
    if (!ctx) return GS_ERR_OOM;
    ctx->device = device;
    ctx->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    if (ctx->counters.reserve(128) != cudaSuccess || cudaMemset(ctx->counters.p, 0, 128) != cudaSuccess) { delete ctx; cudaGetLastError(); return GS_ERR_OOM; }
    *out = ctx;
    return GS_OK;
}

void gs_destroy(gs_ctx *ctx) {
    if (!ctx) return;
    cudaSetDevice(ctx->device);
    for (gs_ctx *w : ctx->decode_workers) gs_destroy(w);
    for (cudaStream_t ws : ctx->decode_streams) cudaStreamDestroy(ws);
    if (ctx->decode_event) cudaEventDestroy(ctx->decode_event);
    cudaStreamSynchronize(ctx->stream);
    DevBuf *all[] = {&ctx->rec, &ctx->aabb, &ctx->params, &ctx->bcount, &ctx->bhist, &ctx->pair_gauss, &ctx->pair_brick,
                     &ctx->grid_order, &ctx->brick_start, &ctx->jit, &ctx->bwd_setup, &ctx->leaf_key[0], &ctx->leaf_key[1],
                     &ctx->leaf_val[0], &ctx->leaf_val[1], &ctx->node_left, &ctx->node_right, &ctx->node_parent,
                     &ctx->leaf_parent, &ctx->node_aabb, &ctx->node_flag, &ctx->bvh_nodes, &ctx->sorted_rec, &ctx->cull_ids, &ctx->cull_link, &ctx->cull_head, &ctx->cull_mask, &ctx->pt_key[0], &ctx->pt_key[1],
                     &ctx->pt_val[0], &ctx->pt_val[1], &ctx->scan_tmp, &ctx->sort_hist, &ctx->gacc, &ctx->misc, &ctx->counters, &ctx->dbg, &ctx->dens_work, &ctx->dens_scratch, &ctx->sel_key[0], &ctx->sel_key[1],
                     &ctx->sel_val[0], &ctx->sel_val[1], &ctx->sc_spt, &ctx->sc_box, &ctx->sc_acc, &ctx->sc_coef, &ctx->rn_xyz, &ctx->rn_phi, &ctx->rn_I, &ctx->cidx_hist, &ctx->cidx_start, &ctx->cidx_ids};
    for (DevBuf *b : all) b->release();
    for (DevBuf &b : ctx->h2d) b.release();
    for (auto *v : {&ctx->prof_pending, &ctx->prof_free})
        for (auto &pp : *v) { cudaEventDestroy(pp.a); cudaEventDestroy(pp.b); }
    if (ctx->aux_stream) { cudaStreamDestroy(ctx->aux_stream); cudaEventDestroy(ctx->aux_event); cudaEventDestroy(ctx->aux_event2); }
    if (ctx->grid_host) { cudaFreeHost(ctx->grid_host); cudaEventDestroy(ctx->grid_event); }
    delete ctx;
}

const char *gs_last_error(const gs_ctx *ctx) { return ctx ? ctx->err.c_str() : "null context"; }

gs_status gs_preprocess(gs_ctx *ctx, const gs_gaussians *g, const gs_domain *dom, float tau) {
    LaunchScope launch_scope(ctx);
    if (!ctx) return GS_ERR_INVALID_ARG;
    if (!g) return fail(ctx, GS_ERR_INVALID_ARG, "gaussians is NULL");
    if (g->n > 0 && (!g->mean || !g->scale || !g->quat || !g->opacity || !g->scalar))
        return fail(ctx, GS_ERR_INVALID_ARG, "gaussians: NULL parameter array");
    if (g->n >= (1u << 31)) return fail(ctx, GS_ERR_INVALID_ARG, "gaussians: n must be < 2^31");
    if (!(tau > 0.f && tau < 1.f)) return fail(ctx, GS_ERR_INVALID_ARG, "tau must lie in (0,1)");
    if (dom)
        for (int k = 0; k < 3; k++)
            if (!(dom->hi[k] > dom->lo[k]) || !isfinite(dom->hi[k]) || !isfinite(dom->lo[k]))
                return fail(ctx, GS_ERR_INVALID_ARG, "domain: need finite lo < hi");
    CK(cudaSetDevice(ctx->device), "cudaSetDevice");
    { gs_status rs__ = resolve_grid_counts(ctx); if (rs__ != GS_OK) return rs__; }
    ctx->have_pre = false;
    ctx->lbvh_state = 0;
    ctx->accel_kind = -1;
    ctx->have_hit_masks = false;
    ctx->fused_pack = 0;
    ctx->cidx_valid = false;
    ctx->builds_since_pre = 0;
    ctx->prev_cand.ids = nullptr;
    ctx->bcount_exact = false;
    const size_t n = g->n ? g->n : 1;
    CK(ctx->rec.reserve(n * 64), "alloc records");
    CK(ctx->aabb.reserve(n * 24), "alloc aabb");
    CK(ctx->params.reserve(n * 32), "alloc params");
    ctx->N = g->n;
    ctx->tau = tau;
    // support G >= tau  <=>  |u|^2 <= r2 = -2 ln tau (D3); both rounded to fp32 once, here
    ctx->r2 = (float)(-2.0 * log((double)tau));
    ctx->r = (float)sqrt((double)ctx->r2);
    ctx->have_dom = dom != nullptr;
    if (dom) ctx->dom = *dom;
    {
        Stage stage(ctx, GS_PROF_PREPROCESS);
        CK(launch_preprocess(*g, ctx->r, ctx->rec.as<float4>(), ctx->aabb.as<float>(), ctx->params.as<float>(),
                             ctx->counters.as<unsigned long long>() + 6, ctx->stream), "preprocess");
    }
    ctx->have_pre = true;
    return GS_OK;
}

gs_status gs_build_accel(gs_ctx *ctx, const gs_query *q) {
    LaunchScope launch_scope(ctx);
    if (!ctx) return GS_ERR_INVALID_ARG;
    if (!ctx->have_pre) return fail(ctx, GS_ERR_STATE, "gs_build_accel before gs_preprocess");
    GridDesc gd{};
    uint64_t P = 0;
    gs_status st = validate_query(ctx, q, &gd, &P);
    if (st != GS_OK) return st;
    CK(cudaSetDevice(ctx->device), "cudaSetDevice");
    if ((st = resolve_grid_counts(ctx, /*wait=*/false)) != GS_OK) return st;
    ctx->accel_kind = -1;
    ctx->fused_pack = 0;
    ctx->have_hit_masks = false;
    cudaStream_t s = ctx->stream;
    const uint32_t N = ctx->N;
    Stage stage(ctx, GS_PROF_BUILD);
    if (q->kind == GS_QUERY_GRID) {
        const uint32_t nbricks = (uint32_t)gd.brick_cnt[0] * gd.brick_cnt[1] * gd.brick_cnt[2];
        CK(ctx->bcount.reserve(((size_t)N + 1) * 4), "alloc brick counts");
        // the backward's processing order (Gaussians bucketed by the Morton code of their central brick, at most
        // 6 bits per axis) is built by the same two passes
        int axis_bits = 1;
        for (int k = 0; k < 3; k++) axis_bits = bits_for((uint64_t)gd.brick_cnt[k]) > axis_bits ? bits_for((uint64_t)gd.brick_cnt[k]) : axis_bits;
        const int order_shift = axis_bits > 6 ? axis_bits - 6 : 0;
        const uint32_t norder = 1u << (3 * (axis_bits - order_shift));
        const size_t nh = (size_t)nbricks + norder;
        CK(ctx->bhist.reserve(nh * 4), "alloc brick histogram");
        CK(ctx->brick_start.reserve((nh + 1) * 4), "alloc brick_start");
        const size_t n1 = N ? N : 1;
        CK(ctx->grid_order.reserve(n1 * 4), "alloc order");
        CK(ctx->bwd_setup.reserve(n1 * 32), "alloc backward setup");
        CK(ctx->pair_gauss.reserve(4), "alloc pair list");
        unsigned long long *total = ctx->counters.as<unsigned long long>() + 4;
        CandSegs cs;
        if ((st = batch_candidates(ctx, gd, nbricks, &cs)) != GS_OK) return st;
        ctx->builds_since_pre++;
        {   // reset of the counters in front of the passes: one launch (plus a whole-array memset the first time the index is used)
            CandSegs prev = ctx->prev_cand;
            if (cs.ids && !ctx->bcount_exact) {
                CK(cudaMemsetAsync(ctx->bcount.p, 0, (size_t)N * 4, s), "memset counts");
                prev.ids = nullptr;
            }
            if (!cs.ids) prev.ids = nullptr;   // a full pass writes every count itself
            CK(launch_build_reset(total, ctx->bhist.as<uint32_t>(), (uint32_t)nh, ctx->bcount.as<uint32_t>(), prev, s), "build reset");
            ctx->prev_cand = cs;
            ctx->bcount_exact = cs.ids != nullptr;
        }
        CK(launch_brick_count(ctx->aabb.as<float>(), ctx->rec.as<float4>(), N, gd, ctx->r, ctx->bcount.as<uint32_t>(), total,
                              ctx->bhist.as<uint32_t>(), nbricks, norder, order_shift, ctx->bwd_setup.as<float4>(), cs, s), "brick count");
        CK(exclusive_scan_u32(ctx->bhist.as<uint32_t>(), ctx->brick_start.as<uint32_t>(), nh, ctx->scan_tmp, s), "scan");
        // The pair list is filled speculatively into the buffer the previous step left; T is read back once, at the
        // end, and the fill is repeated only when the buffer had to grow (it writes nothing when T exceeds `cap`).
        unsigned long long T64[2] = {0, 0};
        // GS_OPT_ASYNC_BUILD, steady state (same model size as the last synchronous build, which left 50 % headroom): fill the
        // pair list speculatively and send T / M to pinned host memory WITHOUT waiting for them -- no host round trip in the step
        const bool async = ctx->opt_async_build && ctx->grid_warm_N == N && ctx->pair_gauss.cap >= 4;
        if (async) {
            const size_t cap = ctx->pair_gauss.cap / 4;
            CK(launch_pair_fill(ctx->aabb.as<float>(), ctx->bcount.as<uint32_t>(), N, gd, total, (uint32_t)(cap < 0xffffffffull ? cap : 0xffffffffull),
                                ctx->bhist.as<uint32_t>(), ctx->brick_start.as<uint32_t>(), nbricks, order_shift,
                                ctx->pair_gauss.as<uint32_t>(), ctx->grid_order.as<uint32_t>(), cs, s), "pair fill");
            CK(cudaMemcpyAsync(ctx->grid_host, total, 32, cudaMemcpyDeviceToHost, s), "read T (async)");   // T, M, (invalid count), sticky overflow
            CK(cudaEventRecord(ctx->grid_event, s), "event");
            ctx->grid_pending = true;
            T64[0] = ctx->T;        // last known values until the real ones arrive (debug views resolve first)
            T64[1] = ctx->M_hint;
        }
        for (int attempt = 0; attempt < 2 && !async; attempt++) {
            const size_t cap = ctx->pair_gauss.cap / 4;
            CK(launch_pair_fill(ctx->aabb.as<float>(), ctx->bcount.as<uint32_t>(), N, gd, total, (uint32_t)(cap < 0xffffffffull ? cap : 0xffffffffull),
                                ctx->bhist.as<uint32_t>(), ctx->brick_start.as<uint32_t>(), nbricks, order_shift,
                                ctx->pair_gauss.as<uint32_t>(), ctx->grid_order.as<uint32_t>(), cs, s), "pair fill");
            if (attempt == 0) {
                CK(cudaMemcpyAsync(T64, total, sizeof T64, cudaMemcpyDeviceToHost, s), "read T");
                CK(cudaStreamSynchronize(s), "sync (T)");
                if (T64[0] >= (1ull << 32)) return fail(ctx, GS_ERR_OVERFLOW, "pair count T does not fit 32 bits");
            }
            // with GS_OPT_ASYNC_BUILD the buffer keeps 50 % headroom for the speculative fills of the following steps
            const size_t need = ctx->opt_async_build ? (size_t)T64[0] + (size_t)T64[0] / 2 + 1024 : (size_t)T64[0];
            if (need <= cap) break;
            if ((size_t)T64[0] <= cap) {
                // the list fitted and IS written (the fill consumed the histogram, so it cannot be repeated): only the headroom
                // of the asynchronous builds to come is missing -- grow the buffer around its contents
                CK(ctx->pair_gauss.reserve_keep(need * 4, (size_t)T64[0] * 4, s), "grow pair list");
                break;
            }
            CK(ctx->pair_gauss.reserve(need * 4), "alloc pair list");
        }
        const uint32_t T = (uint32_t)T64[0];
        ctx->M = (uint32_t)T64[1];
        if (!async) {
            // the synchronous path handles an overflowing fill itself (grow + repeat): forget the device's sticky note of it
            if (ctx->opt_async_build) CK(cudaMemsetAsync(total + 3, 0, 8, s), "clear overflow note");
            ctx->M_hint = ctx->M;
            if (ctx->opt_async_build) {
                if (!ctx->grid_host) {
                    CK(cudaMallocHost(reinterpret_cast<void **>(&ctx->grid_host), 32), "alloc pinned counters");
                    CK(cudaEventCreateWithFlags(&ctx->grid_event, cudaEventDisableTiming), "event");
                }
                ctx->grid_warm_N = N;
            }
        }
        ctx->have_pair_brick = false;
        if (gd.jitter && P > 0) {
            CK(ctx->jit.reserve(P * sizeof(float4)), "alloc jitter table");
            CK(launch_jitter_table(gd, ctx->jit.as<float4>(), s), "jitter table");
        }
        ctx->T = T;
        ctx->nbricks = nbricks;
        ctx->grid = gd;
    } else {
        if (!ctx->have_dom) return fail(ctx, GS_ERR_STATE, "point query needs the domain given to gs_preprocess");
        const size_t n = N ? N : 1;
        for (int k = 0; k < 2; k++) {
            CK(ctx->leaf_key[k].reserve(n * 4), "alloc leaf keys");
            CK(ctx->leaf_val[k].reserve(n * 4), "alloc leaf vals");
        }
        CK(ctx->node_left.reserve(n * 4), "alloc nodes");
        CK(ctx->node_right.reserve(n * 4), "alloc nodes");
        CK(ctx->node_parent.reserve(n * 4), "alloc nodes");
        CK(ctx->leaf_parent.reserve(n * 4), "alloc nodes");
        CK(ctx->node_aabb.reserve(n * 24), "alloc nodes");
        CK(ctx->node_flag.reserve(n * 4), "alloc nodes");
        CK(ctx->bvh_nodes.reserve(n * 64), "alloc nodes");
        CK(ctx->sorted_rec.reserve(n * 64), "alloc sorted records");
        // The Gaussian side depends on the model alone: it is built by the first point query after a gs_preprocess and reused by
        // the following ones (the chunks of a decode or of gs_render; a training step calls gs_preprocess, so it rebuilds)
        const bool scatter = ctx->opt_points_accel == GS_POINTS_SCATTER;
        ctx->points_mode = ctx->opt_points_accel;
        uint32_t *keys[2] = {ctx->leaf_key[0].as<uint32_t>(), ctx->leaf_key[1].as<uint32_t>()};
        uint32_t *vals[2] = {ctx->leaf_val[0].as<uint32_t>(), ctx->leaf_val[1].as<uint32_t>()};
        if (ctx->lbvh_state < 1) {
            // Morton codes of the means (record plane 0: mu.xyz, w; NaN marks an invalid Gaussian)
            CK(launch_morton(ctx->rec.as<float>(), 4, ctx->rec.as<float>(), N, ctx->dom, ctx->leaf_key[0].as<uint32_t>(),
                             ctx->leaf_val[0].as<uint32_t>(), s), "morton (gaussians)");
            CK(radix_sort_pairs(keys, vals, N, 31, ctx->sort_hist, ctx->scan_tmp, s, &ctx->leaf_sel), "morton sort (gaussians)");
            ctx->lbvh_state = 1;
        }
        if (!scatter && ctx->lbvh_state < 2) {   // the scatter mode only needs the Morton ORDER of the Gaussians (processing order), no tree over them
            CK(launch_lbvh(keys[ctx->leaf_sel], vals[ctx->leaf_sel], ctx->aabb.as<float>(), ctx->rec.as<float4>(), N,
                           ctx->node_left.as<int32_t>(), ctx->node_right.as<int32_t>(), ctx->node_parent.as<int32_t>(),
                           ctx->leaf_parent.as<int32_t>(), ctx->node_aabb.as<float>(),
                           ctx->node_flag.as<uint32_t>(), ctx->bvh_nodes.as<float4>(), ctx->sorted_rec.as<float4>(), s), "lbvh");
            ctx->lbvh_state = 2;
        }
        // coherence sort of the queries
        ctx->have_pt_order = false;
        if (ctx->points_ready) {   // gs_step_host: the points' H2D copy ran on the aux stream beside preprocess and the LBVH build
            CK(cudaStreamWaitEvent(s, ctx->points_ready, 0), "wait for the points");
            ctx->points_ready = nullptr;
        }
        if (!q->presorted && P > 0) {
            for (int k = 0; k < 2; k++) {
                CK(ctx->pt_key[k].reserve(P * 4), "alloc point keys");
                CK(ctx->pt_val[k].reserve(P * 4), "alloc point order");
            }
            CK(launch_morton(q->xyz, 3, nullptr, P, ctx->dom, ctx->pt_key[0].as<uint32_t>(), ctx->pt_val[0].as<uint32_t>(), s),
               "morton (points)");
            uint32_t *pk[2] = {ctx->pt_key[0].as<uint32_t>(), ctx->pt_key[1].as<uint32_t>()};
            uint32_t *pv[2] = {ctx->pt_val[0].as<uint32_t>(), ctx->pt_val[1].as<uint32_t>()};
            CK(radix_sort_pairs(pk, pv, P, 30, ctx->sort_hist, ctx->scan_tmp, s, &ctx->pt_sel), "morton sort (points)");
            ctx->have_pt_order = true;
        }
        // per-packet cull lists (the LBVH traversal; shared by the forward and the backward of this step).  The pool of
        // list chunks grows on demand: the kernel counts the chunks it needs, the host reads that count back (the one
        // device->host crossing of the unstructured path, like T of the structured path) and repeats the pass if it
        // did not fit.
        // sorted copy of the query points: every point kernel reads positions from it (one coalesced 16-byte load per lane)
        CK(ctx->sc_spt.reserve(scatter_padded_points(P ? P : 1) * 16), "alloc sorted points");
        CK(launch_sorted_points(q->xyz, ctx->have_pt_order ? ctx->pt_val[ctx->pt_sel].as<uint32_t>() : nullptr, P, ctx->sc_spt.as<float4>(), s),
           "sorted points");
        if (scatter) {
            // the paper's structure: a wide tree over the SORTED SAMPLE POSITIONS, rebuilt per query
            const uint32_t nodes = scatter_tree_shape(P, &ctx->sc_tree);
            CK(ctx->sc_box.reserve((size_t)nodes * 24), "alloc point tree");
            ctx->sc_tree.box = ctx->sc_box.as<float>();
            CK(launch_scatter_build(P, ctx->sc_tree, ctx->sc_spt.as<float4>(), ctx->sc_box.as<float>(), s), "point tree");
        } else if (P > 0) {
            Stage cull_stage(ctx, GS_PROF_CULL);
            const uint64_t packets = (P + 31) / 32;
            CK(ctx->cull_head.reserve(packets * 8), "alloc cull heads");
            if (ctx->cull_cap == 0) {
                const uint64_t guess = packets * 8 + 1024;   // 256 Gaussians per point-packet; grown below when exceeded
                CK(ctx->cull_ids.reserve(guess * 128), "alloc cull pool");
                CK(ctx->cull_link.reserve(guess * 4), "alloc cull pool");
                ctx->cull_cap = (uint32_t)guess;
            }
            uint32_t *ovf = ctx->counters.as<uint32_t>();
            for (int attempt = 0;; attempt++) {
                CK(cudaMemsetAsync(ovf, 0, 4, s), "memset");
                CK(launch_points_cull(ctx->sorted_rec.as<float4>(), N, ctx->bvh_nodes.as<float4>(), ctx->sc_spt.as<float4>(),
                                      ctx->have_pt_order ? ctx->pt_val[ctx->pt_sel].as<uint32_t>() : nullptr, P, ctx->dom, ctx->r,
                                      cull_lists(ctx), ovf, ctx->cull_per_packet > 512.0 ? 2 : 4, s), "points cull");
                uint32_t host[3] = {0, 0, 0};   // [0] stack overflow flag, [2] chunks requested
                CK(cudaMemcpyAsync(host, ctx->counters.p, 12, cudaMemcpyDeviceToHost, s), "read cull counters");
                CK(cudaStreamSynchronize(s), "sync");
                if (host[0]) return fail(ctx, GS_ERR_OVERFLOW, "BVH traversal stack overflow");
                ctx->cull_per_packet = 32.0 * (double)host[2] / (double)packets;
                if (host[2] <= ctx->cull_cap) break;
                if (attempt >= 2) return fail(ctx, GS_ERR_OVERFLOW, "cull list pool did not converge");
                const uint64_t want = (uint64_t)host[2] + host[2] / 8 + 1024;
                if (want >= 0xffffffffull) return fail(ctx, GS_ERR_OVERFLOW, "cull lists exceed 2^32 chunks");
                CK(ctx->cull_ids.reserve(want * 128), "alloc cull pool");
                CK(ctx->cull_link.reserve(want * 4), "alloc cull pool");
                ctx->cull_cap = (uint32_t)want;
            }
        }
    }
    ctx->P = P;
    ctx->accel_q = *q;
    ctx->accel_kind = q->kind;
    return GS_OK;
}

static gs_status check_ready(gs_ctx *ctx, const gs_query *q, const char *who) {
    if (!ctx->have_pre || ctx->accel_kind < 0) return fail(ctx, GS_ERR_STATE, who);
    if (!q) return fail(ctx, GS_ERR_INVALID_ARG, "query is NULL");
    if (!same_query(*q, ctx->accel_q)) return fail(ctx, GS_ERR_STATE, "query differs from the one gs_build_accel was called with");
    return GS_OK;
}

static gs_status run_fwd(gs_ctx *ctx, const FwdOut &o) {
    cudaStream_t s = ctx->stream;
    if (ctx->accel_kind == GS_QUERY_GRID) {
        Stage stage(ctx, GS_PROF_FWD);
        CK(launch_grid_fwd(ctx->rec.as<float4>(), ctx->N, ctx->grid, ctx->pair_gauss.as<uint32_t>(),
                           ctx->brick_start.as<uint32_t>(), ctx->tau, ctx->r2, o, ctx->jit.as<float4>(), dev_count(ctx), s), "grid forward");
    } else if (ctx->points_mode == GS_POINTS_SCATTER) {
        Stage stage(ctx, GS_PROF_FWD);
        CK(ctx->sc_acc.reserve(scatter_padded_points(ctx->P ? ctx->P : 1) * 8), "alloc accumulators");
        CK(launch_scatter_fwd(ctx->rec.as<float4>(), ctx->aabb.as<float>(), ctx->leaf_val[ctx->leaf_sel].as<uint32_t>(), ctx->N, ctx->sc_tree,
                              ctx->sc_spt.as<float4>(), ctx->sc_acc.as<float2>(),
                              ctx->have_pt_order ? ctx->pt_val[ctx->pt_sel].as<uint32_t>() : nullptr, ctx->P, ctx->tau, ctx->r2, o, s),
           "points forward (scatter)");
    } else {
        // the forward leaves one hit bit per list entry for gs_sample_bwd (k_points_bwd_masked); the debug-set variant does not
        CullLists lists = cull_lists(ctx);
        const bool sets = o.set_count || o.set_sum || o.set_xor || o.counters;
        if (ctx->opt_bwd_hit_masks && !sets && ctx->P > 0) {
            CK(ctx->cull_mask.reserve(((size_t)ctx->cull_cap + 1) * 8), "alloc hit masks");
            lists.mask = ctx->cull_mask.as<uint2>();
        }
        Stage stage(ctx, GS_PROF_FWD);
        CK(launch_points_fwd(ctx->sorted_rec.as<float4>(), ctx->sc_spt.as<float4>(),
                             ctx->have_pt_order ? ctx->pt_val[ctx->pt_sel].as<uint32_t>() : nullptr, ctx->P, lists, ctx->tau,
                             ctx->r2, o, s), "points forward");
        if (lists.mask) ctx->have_hit_masks = true;
    }
    return GS_OK;
}

gs_status gs_sample_fwd(gs_ctx *ctx, const gs_query *q, const float *target, float *phi, float *I, double *loss, float *dL_dphi,
                        float *sample_err) {
    LaunchScope launch_scope(ctx);
    if (!ctx) return GS_ERR_INVALID_ARG;
    gs_status st = check_ready(ctx, q, "gs_sample_fwd before gs_preprocess/gs_build_accel");
    if (st != GS_OK) return st;
    if (ctx->P > 0 && (!phi || !I)) return fail(ctx, GS_ERR_INVALID_ARG, "phi and I must be given");
    if (ctx->P > 0 && !target && (loss || dL_dphi || sample_err)) return fail(ctx, GS_ERR_INVALID_ARG, "loss outputs need a target");
    CK(cudaSetDevice(ctx->device), "cudaSetDevice");
    FwdOut o{target, phi, I, loss, dL_dphi, sample_err, nullptr, nullptr, nullptr, nullptr, nullptr};
    o.inv_count = ctx->sample_count ? 1.0 / (double)ctx->sample_count : 0.0;
    // x-pairs of a grid batch are moved as float2 only when every per-sample array the caller passed is 8-byte aligned
    // (a 4-byte-aligned view such as tensor[1:] takes the scalar epilogue: same values)
    o.vec_ok = !(((uintptr_t)target | (uintptr_t)phi | (uintptr_t)I | (uintptr_t)dL_dphi | (uintptr_t)sample_err) & 7);
    ctx->fused_pack = 0;
    if (target && ctx->P > 0) {  // keep the backward coefficients of the fused MSE for gs_sample_bwd(dL_dphi = NULL)
        CK(ctx->misc.reserve(ctx->P * 16), "alloc sample pack");
        o.pack2 = ctx->misc.as<float2>();
    }
    st = run_fwd(ctx, o);
    if (st == GS_OK && o.pack2) ctx->fused_pack = 1;
    return st;
}

gs_status gs_sample_fwd_loss(gs_ctx *ctx, const gs_query *q, const gs_loss *loss, const float *target, float *phi, float *I,
                             double *loss_terms, float *dL_dphi, float *dL_dI, float *sample_err) {
    LaunchScope launch_scope(ctx);
    if (!ctx) return GS_ERR_INVALID_ARG;
    gs_status st = check_ready(ctx, q, "gs_sample_fwd_loss before gs_preprocess/gs_build_accel");
    if (st != GS_OK) return st;
    if (!loss) return fail(ctx, GS_ERR_INVALID_ARG, "loss is NULL");
    if (loss->kind != GS_LOSS_MSE && loss->kind != GS_LOSS_L1) return fail(ctx, GS_ERR_INVALID_ARG, "unknown loss kind");
    if (!(loss->lambda_fn >= 0.f) || !(loss->lambda_fp >= 0.f) || !(loss->eps_fn >= 0.f) || !isfinite(loss->lambda_fn) ||
        !isfinite(loss->lambda_fp) || !isfinite(loss->eps_fn))
        return fail(ctx, GS_ERR_INVALID_ARG, "lambda_fn, lambda_fp and eps_fn must be finite and >= 0");
    if (ctx->P > 0 && (!phi || !I || !target)) return fail(ctx, GS_ERR_INVALID_ARG, "phi, I and target must be given");
    if (ctx->P > 0 && (loss->num_defined == 0 || loss->num_defined > ctx->P || (!loss->defined && loss->num_defined != ctx->P)))
        return fail(ctx, GS_ERR_INVALID_ARG, "num_defined must be |D| (P when defined is NULL)");
    CK(cudaSetDevice(ctx->device), "cudaSetDevice");
    cudaStream_t s = ctx->stream;
    // accumulators of the epilogue: 3 sums (double) and 2 counts, in the context's counter block
    double *sums = reinterpret_cast<double *>(ctx->counters.as<char>() + 64);
    unsigned long long *counts = reinterpret_cast<unsigned long long *>(ctx->counters.as<char>() + 88);
    CK(cudaMemsetAsync(sums, 0, 40, s), "memset loss sums");
    FwdOut o{target, phi, I, nullptr, dL_dphi, sample_err, nullptr, nullptr, nullptr, nullptr, nullptr, {}};
    o.gen.on = 1;
    o.gen.kind = loss->kind;
    o.gen.defined = loss->defined;
    o.gen.dL_dI = dL_dI;
    o.gen.lam_fn = loss->lambda_fn;
    o.gen.thr_fn = (1.0f + loss->eps_fn) * ctx->tau;
    o.gen.lam_fp = loss->lambda_fp;
    o.gen.inv_nd = ctx->P ? (float)(1.0 / (double)loss->num_defined) : 0.f;
    o.gen.sums = sums;
    o.gen.counts = counts;
    ctx->fused_pack = 0;
    if (ctx->accel_kind == GS_QUERY_GRID && ctx->P > 0) {  // keep the backward coefficients for gs_sample_bwd(dL_dphi = NULL)
        CK(ctx->misc.reserve(ctx->P * 16), "alloc sample pack");
        o.gen.pack4 = ctx->misc.as<float4>();
    }
    if (ctx->P > 0) {
        st = run_fwd(ctx, o);
        if (st != GS_OK) return st;
    }
    Stage stage(ctx, GS_PROF_FWD);
    CK(launch_loss_finish(o.gen, ctx->P, (double)loss->num_defined, loss_terms, s), "loss finish");
    if (o.gen.pack4) ctx->fused_pack = 2;
    return GS_OK;
}

gs_status gs_sample_bwd(gs_ctx *ctx, const gs_query *q, const float *phi, const float *I, const float *dL_dphi, const float *dL_dI,
                        const float *target, const gs_grads *out) {
    LaunchScope launch_scope(ctx);
    if (!ctx) return GS_ERR_INVALID_ARG;
    gs_status st = check_ready(ctx, q, "gs_sample_bwd before gs_preprocess/gs_build_accel");
    if (st != GS_OK) return st;
    if (!out || (ctx->N > 0 && (!out->dmean || !out->dscale || !out->dquat || !out->dopacity || !out->dscalar)))
        return fail(ctx, GS_ERR_INVALID_ARG, "gradient outputs must be given");
    const bool fused = dL_dphi == nullptr;
    if (fused && ctx->P > 0 && (!ctx->fused_pack || dL_dI))
        return fail(ctx, GS_ERR_STATE, "dL_dphi = NULL needs a preceding gs_sample_fwd with a target (or, on a grid, gs_sample_fwd_loss) on the same accel, and dL_dI = NULL");
    if (!fused && ctx->P > 0 && (!phi || !I)) return fail(ctx, GS_ERR_INVALID_ARG, "phi and I must be given with dL_dphi");
    if (ctx->N > 0 && ((uintptr_t)out->dquat & 15)) return fail(ctx, GS_ERR_INVALID_ARG, "dquat must be 16-byte aligned");
    CK(cudaSetDevice(ctx->device), "cudaSetDevice");
    cudaStream_t s = ctx->stream;
    const uint32_t N = ctx->N;
    if (N == 0) return GS_OK;
    CK(ctx->gacc.reserve((size_t)N * GACC_GRID * 4), "alloc gradient accumulator");
    const bool fused2 = fused && ctx->fused_pack == 1;  // float2 coefficients of the fused MSE; otherwise float4 coefficients
    BwdIn in{phi, I, dL_dphi, dL_dI, target, fused2 ? ctx->misc.as<float2>() : nullptr,
             0.5f * (float)(ctx->sample_count ? ctx->sample_count : ctx->P)};
    if (ctx->accel_kind == GS_QUERY_GRID) {
        if (!fused) {
            ctx->fused_pack = 0;  // misc is overwritten with the caller's coefficients
            CK(ctx->misc.reserve((ctx->P ? ctx->P : 1) * 16), "alloc sample pack");
            Stage stage(ctx, GS_PROF_BWD_PACK);
            CK(launch_pack_samples(in, ctx->P, ctx->tau, ctx->misc.as<float4>(), s), "pack samples");
        }
        Stage stage(ctx, GS_PROF_BWD);
        CK(launch_grid_bwd(ctx->rec.as<float4>(), ctx->bwd_setup.as<float4>(), N, ctx->grid, ctx->misc.p, fused2, ctx->r2,
                           ctx->gacc.as<float>(), ctx->grid_order.as<uint32_t>(), grid_M_launch(ctx), ctx->jit.as<float4>(), dev_count(ctx), s), "grid backward");
    } else if (ctx->points_mode == GS_POINTS_SCATTER) {
        CK(ctx->sc_coef.reserve(scatter_padded_points(ctx->P ? ctx->P : 1) * 32), "alloc backward coefficients");
        Stage stage(ctx, GS_PROF_BWD);
        CK(launch_scatter_bwd(ctx->rec.as<float4>(), ctx->aabb.as<float>(), ctx->leaf_val[ctx->leaf_sel].as<uint32_t>(), N, ctx->sc_tree,
                              ctx->sc_spt.as<float4>(), ctx->sc_coef.as<float4>(),
                              ctx->have_pt_order ? ctx->pt_val[ctx->pt_sel].as<uint32_t>() : nullptr, ctx->P, ctx->tau, ctx->r2, in,
                              ctx->gacc.as<float>(), s), "points backward (scatter)");
    } else {
        CK(cudaMemsetAsync(ctx->gacc.p, 0, (size_t)N * GACC * 4, s), "memset gacc");
        Stage stage(ctx, GS_PROF_BWD);
        CullLists lists = cull_lists(ctx);
        const bool masked = ctx->have_hit_masks && ctx->opt_bwd_hit_masks;   // a forward on these lists left its hit bits
        if (masked) lists.mask = ctx->cull_mask.as<uint2>();
        CK(launch_points_bwd(ctx->sorted_rec.as<float4>(), ctx->sc_spt.as<float4>(),
                             ctx->have_pt_order ? ctx->pt_val[ctx->pt_sel].as<uint32_t>() : nullptr, ctx->P, lists, ctx->tau,
                             ctx->r2, in, ctx->gacc.as<float>(), masked, s), "points backward");
    }
    Stage stage(ctx, GS_PROF_FINALIZE);
    const bool grid = ctx->accel_kind == GS_QUERY_GRID;
    CK(launch_finalize(ctx->rec.as<float4>(), ctx->params.as<float>(), ctx->gacc.as<float>(), N, grid, (grid && fused2) ? in.eps_scale : 1.f,
                       *out, grid ? ctx->bcount.as<uint32_t>() : nullptr, grid ? dev_count(ctx) : DevCount{nullptr, 0},
                       grid ? grid_M_launch(ctx) : N, s), "finalize");
    return GS_OK;
}

gs_status gs_debug_get(gs_ctx *ctx, int32_t what, const void **dev_ptr, size_t *count) {
    LaunchScope launch_scope(ctx);
    if (ctx && ctx->grid_pending) { gs_status rs__ = resolve_grid_counts(ctx); if (rs__ != GS_OK) return rs__; }
    if (!ctx || !dev_ptr || !count) return GS_ERR_INVALID_ARG;
    if (!ctx->have_pre) return fail(ctx, GS_ERR_STATE, "nothing built yet");
    const size_t N = ctx->N;
    const bool grid = ctx->accel_kind == GS_QUERY_GRID, pts = ctx->accel_kind == GS_QUERY_POINTS;
    const bool tree = pts && ctx->points_mode == GS_POINTS_GATHER;   // the scatter mode builds no tree over the Gaussians
    const size_t ni = N >= 1 ? N - 1 : 0;
    switch (what) {
        case GS_DBG_RECORDS: *dev_ptr = ctx->rec.p; *count = N; return GS_OK;
        case GS_DBG_AABB: *dev_ptr = ctx->aabb.p; *count = N; return GS_OK;
        case GS_DBG_BRICK_COUNT: if (!grid) break; *dev_ptr = ctx->bcount.p; *count = N; return GS_OK;
        case GS_DBG_PAIR_BRICK:
            if (!grid) break;
            if (!ctx->have_pair_brick) {  // the sorted list stores no brick ids: they are the runs of brick_start
                CK(cudaSetDevice(ctx->device), "cudaSetDevice");
                CK(ctx->pair_brick.reserve(((size_t)ctx->T + 1) * 4), "alloc debug view");
                CK(launch_expand_bricks(ctx->brick_start.as<uint32_t>(), ctx->nbricks, ctx->pair_brick.as<uint32_t>(), ctx->stream),
                   "expand bricks");
                ctx->have_pair_brick = true;
            }
            *dev_ptr = ctx->pair_brick.p; *count = ctx->T; return GS_OK;
        case GS_DBG_PAIR_GAUSS: if (!grid) break; *dev_ptr = ctx->pair_gauss.p; *count = ctx->T; return GS_OK;
        case GS_DBG_BRICK_START: if (!grid) break; *dev_ptr = ctx->brick_start.p; *count = (size_t)ctx->nbricks + 1; return GS_OK;
        case GS_DBG_LEAF_MORTON: if (!pts) break; *dev_ptr = ctx->leaf_key[ctx->leaf_sel].p; *count = N; return GS_OK;
        case GS_DBG_LEAF_ORDER: if (!pts) break; *dev_ptr = ctx->leaf_val[ctx->leaf_sel].p; *count = N; return GS_OK;
        case GS_DBG_NODE_LEFT: if (!tree) break; *dev_ptr = ctx->node_left.p; *count = ni; return GS_OK;
        case GS_DBG_NODE_RIGHT: if (!tree) break; *dev_ptr = ctx->node_right.p; *count = ni; return GS_OK;
        case GS_DBG_NODE_PARENT: if (!tree) break; *dev_ptr = ctx->node_parent.p; *count = ni; return GS_OK;
        case GS_DBG_LEAF_PARENT: if (!tree) break; *dev_ptr = ctx->leaf_parent.p; *count = N; return GS_OK;
        case GS_DBG_NODE_AABB: if (!tree) break; *dev_ptr = ctx->node_aabb.p; *count = ni; return GS_OK;
        case GS_DBG_POINT_ORDER: if (!pts || !ctx->have_pt_order) break; *dev_ptr = ctx->pt_val[ctx->pt_sel].p; *count = ctx->P; return GS_OK;
        case GS_DBG_POINT_MORTON: if (!pts || !ctx->have_pt_order) break; *dev_ptr = ctx->pt_key[ctx->pt_sel].p; *count = ctx->P; return GS_OK;
        default: return fail(ctx, GS_ERR_INVALID_ARG, "unknown debug item");
    }
    return fail(ctx, GS_ERR_STATE, "debug item not built for the current accel");
}

gs_status gs_debug_read(gs_ctx *ctx, int32_t what, void *dst_host, size_t bytes) {
    if (!ctx || (!dst_host && bytes)) return GS_ERR_INVALID_ARG;
    const void *p = nullptr;
    size_t count = 0;
    gs_status st = gs_debug_get(ctx, what, &p, &count);
    if (st != GS_OK) return st;
    static const size_t elem[] = {64, 24, 4, 4, 4, 4, 4, 4, 4, 4, 4, 4, 24, 4, 4};
    if (bytes > count * elem[what]) return fail(ctx, GS_ERR_INVALID_ARG, "gs_debug_read: more bytes than the buffer holds");
    CK(cudaSetDevice(ctx->device), "cudaSetDevice");
    CK(cudaStreamSynchronize(ctx->stream), "sync");
    if (bytes) CK(cudaMemcpy(dst_host, p, bytes, cudaMemcpyDeviceToHost), "debug read");
    return GS_OK;
}

gs_status gs_debug_point_sets(gs_ctx *ctx, const gs_query *q, uint32_t *count, uint64_t *hash_sum, uint64_t *hash_xor) {
    LaunchScope launch_scope(ctx);
    if (!ctx) return GS_ERR_INVALID_ARG;
    gs_status st = check_ready(ctx, q, "gs_debug_point_sets before gs_preprocess/gs_build_accel");
    if (st != GS_OK) return st;
    CK(cudaSetDevice(ctx->device), "cudaSetDevice");
    CK(ctx->dbg.reserve((ctx->P ? ctx->P : 1) * 8), "alloc scratch");
    unsigned long long *ctr = ctx->counters.as<unsigned long long>() + 2;
    CK(cudaMemsetAsync(ctr, 0, 16, ctx->stream), "memset");
    float *phi = ctx->dbg.as<float>();
    float *I = phi + (ctx->P ? ctx->P : 1);
    FwdOut o{nullptr, phi, I, nullptr, nullptr, nullptr, count, reinterpret_cast<unsigned long long *>(hash_sum),
             reinterpret_cast<unsigned long long *>(hash_xor), ctr, nullptr};
    st = run_fwd(ctx, o);
    if (st != GS_OK) return st;
    CK(cudaStreamSynchronize(ctx->stream), "sync");
    return GS_OK;
}

gs_status gs_debug_counters(gs_ctx *ctx, uint64_t *tested_host, uint64_t *hits_host) {
    if (!ctx || !tested_host || !hits_host) return GS_ERR_INVALID_ARG;
    unsigned long long v[2] = {0, 0};
    CK(cudaSetDevice(ctx->device), "cudaSetDevice");
    CK(cudaStreamSynchronize(ctx->stream), "sync");
    CK(cudaMemcpy(v, ctx->counters.as<unsigned long long>() + 2, 16, cudaMemcpyDeviceToHost), "read counters");
    *tested_host = v[0];
    *hits_host = v[1];
    return GS_OK;
}

gs_status gs_params_activate(gs_ctx *ctx, const gs_raw_params *p, float *scale, float *opacity, float *scalar) {
    LaunchScope launch_scope(ctx);
    if (!ctx || !p) return GS_ERR_INVALID_ARG;
    if (p->n > 0 && (!p->raw_scale || !p->raw_opacity || !p->raw_scalar || !scale || !opacity || !scalar))
        return fail(ctx, GS_ERR_INVALID_ARG, "gs_params_activate: null pointer");
    CK(cudaSetDevice(ctx->device), "cudaSetDevice");
    CK(launch_activate(*p, scale, opacity, scalar, ctx->stream), "activate");
    return GS_OK;
}

gs_status gs_adam_step(gs_ctx *ctx, const gs_raw_params *p, const gs_grads *g, float *m, float *v, const gs_adam_cfg *cfg,
                       float *scale_out, float *opacity_out, float *scalar_out) {
    LaunchScope launch_scope(ctx);
    if (!ctx || !p || !g || !cfg) return GS_ERR_INVALID_ARG;
    if (p->n > 0 && (!p->mean || !p->raw_scale || !p->quat || !p->raw_opacity || !p->raw_scalar || !g->dmean || !g->dscale ||
                     !g->dquat || !g->dopacity || !g->dscalar || !m || !v))
        return fail(ctx, GS_ERR_INVALID_ARG, "gs_adam_step: null pointer");
    if (cfg->step < 1 || !(cfg->beta1 >= 0.f && cfg->beta1 < 1.f) || !(cfg->beta2 >= 0.f && cfg->beta2 < 1.f) || !(cfg->eps >= 0.f))
        return fail(ctx, GS_ERR_INVALID_ARG, "gs_adam_step: step >= 1, betas in [0,1), eps >= 0");
    for (int k = 0; k < 5; k++)
        if (!(cfg->lr[k] >= 0.f) || !isfinite(cfg->lr[k])) return fail(ctx, GS_ERR_INVALID_ARG, "gs_adam_step: lr must be finite and >= 0");
    CK(cudaSetDevice(ctx->device), "cudaSetDevice");
    CK(launch_adam_step(*p, *g, m, v, *cfg, scale_out, opacity_out, scalar_out, ctx->stream), "adam step");
    return GS_OK;
}

gs_status gs_prune(gs_ctx *ctx, const gs_raw_params *p, float *m, float *v, const float *opacity, float tau2, uint32_t *n_new_host) {
    LaunchScope launch_scope(ctx);
    if (!ctx || !p || !n_new_host) return GS_ERR_INVALID_ARG;
    const uint32_t n = p->n;
    if (n > 0 && (!p->mean || !p->raw_scale || !p->quat || !p->raw_opacity || !p->raw_scalar || !m || !v || !opacity))
        return fail(ctx, GS_ERR_INVALID_ARG, "gs_prune: null pointer");
    CK(cudaSetDevice(ctx->device), "cudaSetDevice");
    cudaStream_t s = ctx->stream;
    CK(ctx->dens_work.reserve((3 * (size_t)n + 2) * 4), "alloc prune index");
    uint32_t *work = ctx->dens_work.as<uint32_t>();
    CK(launch_prune_index(opacity, n, tau2, work, ctx->scan_tmp, s), "prune index");
    uint32_t kept = 0;
    CK(cudaMemcpyAsync(&kept, work + 2 * (size_t)n, 4, cudaMemcpyDeviceToHost, s), "read kept count");
    CK(cudaStreamSynchronize(s), "sync");
    if (kept < n) {
        CK(ctx->dens_scratch.reserve(37 * (size_t)(kept ? kept : 1) * 4), "alloc prune scratch");
        CK(launch_regather(*p, m, v, kept, work + 2 * (size_t)n + 1, kept, ctx->dens_scratch.as<float>(), true, s), "prune gather");
        CK(cudaStreamSynchronize(s), "sync");
    }
    *n_new_host = kept;
    return GS_OK;
}

gs_status gs_densify(gs_ctx *ctx, const gs_raw_params *p, float *m, float *v, uint32_t capacity, const gs_query *q,
                     const float *sample_err, const float *I, const uint8_t *defined, uint64_t num_defined, const float *target,
                     uint32_t k, float raw_scale_init, float raw_opacity_init, uint32_t *n_new_host) {
    LaunchScope launch_scope(ctx);
    if (ctx && ctx->grid_pending) { gs_status rs__ = resolve_grid_counts(ctx); if (rs__ != GS_OK) return rs__; }
    if (!ctx || !p || !n_new_host) return GS_ERR_INVALID_ARG;
    gs_status st = check_ready(ctx, q, "gs_densify before gs_preprocess/gs_build_accel");
    if (st != GS_OK) return st;
    const uint32_t n = p->n;
    const uint64_t P = ctx->P;
    if (capacity < n) return fail(ctx, GS_ERR_INVALID_ARG, "gs_densify: capacity < n");
    if (!p->mean || !p->raw_scale || !p->quat || !p->raw_opacity || !p->raw_scalar || !m || !v)
        return fail(ctx, GS_ERR_INVALID_ARG, "gs_densify: null pointer");
    if (P > 0 && (!sample_err || !I || !target)) return fail(ctx, GS_ERR_INVALID_ARG, "gs_densify: sample_err, I and target must be given");
    if (num_defined > P || (!defined && num_defined != P)) return fail(ctx, GS_ERR_INVALID_ARG, "gs_densify: num_defined must be |D| (P when defined is NULL)");
    if (!isfinite(raw_scale_init) || !isfinite(raw_opacity_init)) return fail(ctx, GS_ERR_INVALID_ARG, "gs_densify: init values must be finite");
    uint64_t add64 = k;
    if (add64 > capacity - n) add64 = capacity - n;
    if (add64 > num_defined) add64 = num_defined;
    const uint32_t add = (uint32_t)add64, n_new = n + add;
    *n_new_host = n_new;
    if (add == 0) return GS_OK;
    CK(cudaSetDevice(ctx->device), "cudaSetDevice");
    cudaStream_t s = ctx->stream;
    for (int b = 0; b < 2; b++) {
        CK(ctx->sel_key[b].reserve(P * 4), "alloc selection keys");
        CK(ctx->sel_val[b].reserve(P * 4), "alloc selection values");
    }
    uint32_t *keys[2] = {ctx->sel_key[0].as<uint32_t>(), ctx->sel_key[1].as<uint32_t>()};
    uint32_t *vals[2] = {ctx->sel_val[0].as<uint32_t>(), ctx->sel_val[1].as<uint32_t>()};
    CK(launch_select_keys(sample_err, I, defined, P, ctx->tau, keys[0], vals[0], s), "selection keys");
    int sel = 0;
    CK(radix_sort_pairs(keys, vals, P, 32, ctx->sort_hist, ctx->scan_tmp, s, &sel), "selection sort");
    CK(ctx->dens_scratch.reserve(37 * (size_t)n_new * 4), "alloc densify scratch");
    float *scratch = ctx->dens_scratch.as<float>();
    CK(launch_regather(*p, m, v, n_new, nullptr, n, scratch, false, s), "densify gather");
    const float *xyz = ctx->accel_kind == GS_QUERY_POINTS ? ctx->accel_q.xyz : nullptr;
    CK(launch_new_gaussians(*p, m, v, n_new, vals[sel], ctx->grid, ctx->jit.as<float4>(), xyz, target, raw_scale_init, raw_opacity_init, 1e-4f, scratch, s),
       "new gaussians");
    CK(cudaStreamSynchronize(s), "sync");
    return GS_OK;
}

gs_status gs_measure_alu_peaks(gs_ctx *ctx, double *ffma_per_s_host, double *ex2_per_s_host) {
    return gs_measure_alu_peaks2(ctx, ffma_per_s_host, ex2_per_s_host, nullptr);
}

gs_status gs_measure_alu_peaks2(gs_ctx *ctx, double *ffma_per_s_host, double *ex2_per_s_host, double *ffma2_per_s_host) {
    LaunchScope launch_scope(ctx);
    if (!ctx || !ffma_per_s_host || !ex2_per_s_host) return GS_ERR_INVALID_ARG;
    CK(cudaSetDevice(ctx->device), "cudaSetDevice");
    CK(ctx->dbg.reserve(64), "alloc scratch");
    CK(measure_alu_peaks(ctx->dbg.as<float>(), ctx->stream, ffma_per_s_host, ex2_per_s_host, ffma2_per_s_host), "alu peaks");
    return GS_OK;
}

gs_status gs_render(gs_ctx *ctx, uint32_t num_rays, const float *origins, const float *dirs, const float *t_range, uint32_t spp,
                    const float *table, uint32_t table_size, float *rgba) {
    LaunchScope launch_scope(ctx);
    if (!ctx) return GS_ERR_INVALID_ARG;
    if (!ctx->have_pre) return fail(ctx, GS_ERR_STATE, "gs_render before gs_preprocess");
    if (!ctx->have_dom) return fail(ctx, GS_ERR_STATE, "gs_render needs the domain given to gs_preprocess");
    if (num_rays > 0 && (!origins || !dirs || !t_range || !rgba)) return fail(ctx, GS_ERR_INVALID_ARG, "gs_render: null pointer");
    if (spp == 0 || spp > 65535u || !table || table_size < 2) return fail(ctx, GS_ERR_INVALID_ARG, "gs_render: spp in [1, 65535], table of >= 2 entries");
    if (((uintptr_t)table | (uintptr_t)rgba) & 15) return fail(ctx, GS_ERR_INVALID_ARG, "gs_render: table and rgba must be 16-byte aligned");
    CK(cudaSetDevice(ctx->device), "cudaSetDevice");
    cudaStream_t s = ctx->stream;
    // chunks of rays whose samples fit one point query of <= 2^24 points
    const uint32_t chunk_rays = (1u << 24) / spp ? (1u << 24) / spp : 1u;
    for (uint32_t r0 = 0; r0 < num_rays; r0 += chunk_rays) {
        const uint32_t nr = num_rays - r0 < chunk_rays ? num_rays - r0 : chunk_rays;
        const size_t ns = (size_t)nr * spp;
        CK(ctx->rn_xyz.reserve(ns * 12), "alloc ray samples");
        CK(ctx->rn_phi.reserve(ns * 4), "alloc ray samples");
        CK(ctx->rn_I.reserve(ns * 4), "alloc ray samples");
        CK(launch_ray_samples(origins + 3 * (size_t)r0, dirs + 3 * (size_t)r0, t_range + 2 * (size_t)r0, nr, spp, ctx->rn_xyz.as<float>(), s),
           "ray samples");
        gs_query q{};
        q.kind = GS_QUERY_POINTS;
        q.num_points = ns;
        q.xyz = ctx->rn_xyz.as<float>();
        gs_status st = gs_build_accel(ctx, &q);
        if (st != GS_OK) return st;
        st = gs_sample_fwd(ctx, &q, nullptr, ctx->rn_phi.as<float>(), ctx->rn_I.as<float>(), nullptr, nullptr, nullptr);
        if (st != GS_OK) return st;
        CK(launch_composite(ctx->rn_phi.as<float>(), ctx->rn_I.as<float>(), t_range + 2 * (size_t)r0, nr, spp, ctx->tau,
                            reinterpret_cast<const float4 *>(table), table_size, reinterpret_cast<float4 *>(rgba) + r0, s), "composite");
    }
    ctx->accel_kind = -1;   // the accel now belongs to the last chunk of ray samples, not to a query of the caller
    return GS_OK;
}

gs_status gs_decode_grid(gs_ctx *ctx, const gs_gaussians *g, float tau, const gs_query *region, const int32_t *batch_bricks,
                         int32_t num_streams, float *phi, float *I) {
    LaunchScope launch_scope(ctx);
    if (!ctx) return GS_ERR_INVALID_ARG;
    if (!g || !region || !batch_bricks) return fail(ctx, GS_ERR_INVALID_ARG, "gs_decode_grid: NULL argument");
    if (region->kind != GS_QUERY_GRID || region->jitter) return fail(ctx, GS_ERR_INVALID_ARG, "gs_decode_grid: region must be a grid query without jitter");
    if (num_streams == 0) num_streams = 4;
    if (num_streams < 1 || num_streams > 8) return fail(ctx, GS_ERR_INVALID_ARG, "gs_decode_grid: num_streams must lie in [1, 8] (0 = 4)");
    uint64_t nbatch[3], total_batches = 1;
    for (int k = 0; k < 3; k++) {
        if (batch_bricks[k] < 1 || batch_bricks[k] > 256) return fail(ctx, GS_ERR_INVALID_ARG, "gs_decode_grid: batch_bricks must lie in [1, 256]");
        if (region->dims[k] < 1 || region->brick_lo[k] < 0 || region->brick_cnt[k] < 1 || BRICK * (int64_t)region->brick_lo[k] >= region->dims[k])
            return fail(ctx, GS_ERR_INVALID_ARG, "gs_decode_grid: empty or misplaced region");
        // the same rules as gs_build_accel applies to every batch, checked ONCE here: a bad region fails before anything is enqueued
        // instead of inside a worker thread after other batches have already written into phi / I
        if (!(region->spacing[k] > 0.f) || !isfinite(region->spacing[k]) || !isfinite(region->origin[k]))
            return fail(ctx, GS_ERR_INVALID_ARG, "gs_decode_grid: spacing must be positive and finite, origin finite");
        if ((int64_t)region->brick_lo[k] + region->brick_cnt[k] > ((int64_t)region->dims[k] + BRICK - 1) / BRICK)
            return fail(ctx, GS_ERR_INVALID_ARG, "gs_decode_grid: brick_lo + brick_cnt reaches beyond the grid");
        nbatch[k] = ((uint64_t)region->brick_cnt[k] + batch_bricks[k] - 1) / batch_bricks[k];
        total_batches *= nbatch[k];
    }
    uint64_t Ptot = 1;
    for (int k = 0; k < 3; k++) {
        const int64_t ext = BRICK * (int64_t)region->brick_cnt[k], rest = (int64_t)region->dims[k] - BRICK * (int64_t)region->brick_lo[k];
        Ptot *= (uint64_t)(ext < rest ? ext : rest);
    }
    if (Ptot > 0 && (!phi || !I)) return fail(ctx, GS_ERR_INVALID_ARG, "gs_decode_grid: phi and I must be given");
    CK(cudaSetDevice(ctx->device), "cudaSetDevice");
    // ---- workers: one context per stream, each with its own preprocess of the model (records, index, build buffers)
    while ((int)ctx->decode_workers.size() < num_streams) {
        cudaStream_t ws = nullptr;
        CK(cudaStreamCreateWithFlags(&ws, cudaStreamNonBlocking), "decode stream");
        gs_ctx *w = nullptr;
        if (gs_create(ctx->device, ws, &w) != GS_OK) { cudaStreamDestroy(ws); return fail(ctx, GS_ERR_OOM, "gs_decode_grid: worker context"); }
        gs_set_option(w, GS_OPT_ASYNC_BUILD, 1);
        ctx->decode_streams.push_back(ws);
        ctx->decode_workers.push_back(w);
    }
    if (!ctx->decode_event) CK(cudaEventCreateWithFlags(&ctx->decode_event, cudaEventDisableTiming), "event");
    CK(cudaEventRecord(ctx->decode_event, ctx->stream), "event");   // the model arrays may be produced on the caller's stream
    // every way out of this call, failures included, first waits for all worker streams: nothing of this call may still be reading
    // the caller's model or writing the caller's phi / I once it has returned
    auto worker_fail = [&](gs_ctx *w, gs_status st) {
        const std::string msg = gs_last_error(w);
        for (int k = 0; k < num_streams; k++) cudaStreamSynchronize(ctx->decode_streams[(size_t)k]);
        cudaGetLastError();
        return fail(ctx, st, msg.c_str());
    };
    for (int k = 0; k < num_streams; k++) {
        gs_ctx *w = ctx->decode_workers[k];
        const cudaError_t we = cudaStreamWaitEvent(ctx->decode_streams[k], ctx->decode_event, 0);
        if (we != cudaSuccess) { w->err = std::string("wait: ") + cudaGetErrorString(we); return worker_fail(w, GS_ERR_CUDA); }
        const gs_status st = gs_preprocess(w, g, nullptr, tau);
        if (st != GS_OK) return worker_fail(w, st);
    }
    // ---- batches, round-robin over the workers; every worker is driven by a host thread of its own (a 128^3 batch is ~7 CUDA
    //      calls of a few microseconds each: one thread issuing for all streams would be the bottleneck).  Builds are asynchronous
    //      (gs.h GS_OPT_ASYNC_BUILD): a batch whose pair list outgrows the worker's speculative buffer does nothing and is reported
    //      by the worker's next call; it is then repeated.
    struct Job { gs_query q; uint64_t off; };
    std::vector<std::vector<Job>> jobs((size_t)num_streams);
    {
        uint64_t off = 0, b = 0;
        for (uint64_t bz = 0; bz < nbatch[2]; bz++)
            for (uint64_t by = 0; by < nbatch[1]; by++)
                for (uint64_t bx = 0; bx < nbatch[0]; bx++, b++) {
                    Job j{*region, off};
                    const uint64_t bi[3] = {bx, by, bz};
                    uint64_t Pb = 1;
                    for (int k = 0; k < 3; k++) {
                        const int lo = region->brick_lo[k] + (int)bi[k] * batch_bricks[k];
                        const int left = region->brick_lo[k] + region->brick_cnt[k] - lo;
                        j.q.brick_lo[k] = lo;
                        j.q.brick_cnt[k] = left < batch_bricks[k] ? left : batch_bricks[k];
                        const int64_t ext = BRICK * (int64_t)j.q.brick_cnt[k], rest = (int64_t)region->dims[k] - BRICK * (int64_t)lo;
                        Pb *= (uint64_t)(rest <= 0 ? 0 : (ext < rest ? ext : rest));
                    }
                    if (Pb == 0) continue;   // the region's upper end lies beyond the grid
                    jobs[(size_t)(b % (uint64_t)num_streams)].push_back(j);
                    off += Pb;
                }
    }
    std::vector<gs_status> wst((size_t)num_streams, GS_OK);
    std::vector<uint64_t> wrep((size_t)num_streams, 0);
    auto drive = [&](int k) {
        gs_ctx *w = ctx->decode_workers[(size_t)k];
        if (cudaSetDevice(ctx->device) != cudaSuccess) { wst[(size_t)k] = GS_ERR_CUDA; return; }
        auto run = [&](const Job &j) -> gs_status {
            const gs_status bs = gs_build_accel(w, &j.q);
            if (bs != GS_OK) return bs;
            return gs_sample_fwd(w, &j.q, nullptr, phi + j.off, I + j.off, nullptr, nullptr, nullptr);
        };
        const std::vector<Job> &mine = jobs[(size_t)k];
        // An overflow is reported by a LATER call (the counts are picked up without stalling the host, so the report can trail the
        // batch by several builds): every batch since the last checkpoint -- a call that waited for the counts and found them
        // fine -- is then suspect and is done again with SYNCHRONOUS builds (each sizes the grow-only pair list for itself, so the
        // batch that overflowed fits afterwards and the loop terminates).
        constexpr size_t CHECK_EVERY = 32;
        gs_status st = GS_OK;
        size_t ckpt = 0, n = 0;
        while (n < mine.size() && st == GS_OK) {
            st = run(mine[n]);
            if (st == GS_OK) {
                n++;
                if (n - ckpt < CHECK_EVERY && n < mine.size()) continue;
                gs_status_info info;
                st = gs_status_query(w, &info);   // waits for the counts of the builds so far
                if (st == GS_OK) { ckpt = n; continue; }
            }
            if (st != GS_ERR_OVERFLOW) break;
            wrep[(size_t)k] += n - ckpt;
            st = gs_set_option(w, GS_OPT_ASYNC_BUILD, 0);
            for (size_t m = ckpt; m < n && st == GS_OK; m++) st = run(mine[m]);
            if (st == GS_OK) st = gs_set_option(w, GS_OPT_ASYNC_BUILD, 1);
            ckpt = n;
        }
        const cudaError_t se = cudaStreamSynchronize(ctx->decode_streams[(size_t)k]);   // whatever the status: see worker_fail
        if (st == GS_OK && se != cudaSuccess) { st = GS_ERR_CUDA; w->err = std::string("gs_decode_grid: ") + cudaGetErrorString(se); }
        wst[(size_t)k] = st;
    };
    {
        std::vector<std::thread> threads;
        for (int k = 1; k < num_streams; k++) threads.emplace_back(drive, k);
        drive(0);
        for (std::thread &t : threads) t.join();
    }
    for (int k = 0; k < num_streams; k++) {
        gs_ctx *w = ctx->decode_workers[(size_t)k];
        ctx->launches += w->launches;
        w->launches = 0;
        ctx->decode_repeats += wrep[(size_t)k];
        if (wst[(size_t)k] != GS_OK) return worker_fail(w, wst[(size_t)k]);
    }
    return GS_OK;
}

gs_status gs_set_option(gs_ctx *ctx, int32_t key, int64_t value) {
    if (!ctx) return GS_ERR_INVALID_ARG;
    switch (key) {
        case GS_OPT_POINTS_ACCEL:
            if (value != GS_POINTS_GATHER && value != GS_POINTS_SCATTER) return fail(ctx, GS_ERR_INVALID_ARG, "GS_OPT_POINTS_ACCEL: unknown mode");
            ctx->opt_points_accel = (int)value;
            return GS_OK;
        case GS_OPT_ASYNC_BUILD:
            if (value != 0 && value != 1) return fail(ctx, GS_ERR_INVALID_ARG, "GS_OPT_ASYNC_BUILD: 0 or 1");
            if (!value) { gs_status rs__ = resolve_grid_counts(ctx); if (rs__ != GS_OK) return rs__; }
            ctx->opt_async_build = (int)value;
            ctx->grid_warm_N = 0xffffffffu;
            return GS_OK;
        case GS_OPT_BWD_HIT_MASKS:
            if (value != 0 && value != 1) return fail(ctx, GS_ERR_INVALID_ARG, "GS_OPT_BWD_HIT_MASKS: 0 or 1");
            ctx->opt_bwd_hit_masks = (int)value;
            ctx->have_hit_masks = false;
            return GS_OK;
        default: return fail(ctx, GS_ERR_INVALID_ARG, "unknown option");
    }
}

gs_status gs_set_sample_count(gs_ctx *ctx, uint64_t total_samples) {
    if (!ctx) return GS_ERR_INVALID_ARG;
    ctx->sample_count = total_samples;
    ctx->fused_pack = 0;
    return GS_OK;
}

gs_status gs_status_query(gs_ctx *ctx, gs_status_info *out_host) {
    if (ctx && ctx->grid_pending) { gs_status rs__ = resolve_grid_counts(ctx); if (rs__ != GS_OK) return rs__; }
    if (!ctx || !out_host) return GS_ERR_INVALID_ARG;
    CK(cudaSetDevice(ctx->device), "cudaSetDevice");
    CK(cudaStreamSynchronize(ctx->stream), "sync");
    unsigned long long inv = 0;
    CK(cudaMemcpy(&inv, ctx->counters.as<unsigned long long>() + 6, 8, cudaMemcpyDeviceToHost), "read counters");
    memset(out_host, 0, sizeof *out_host);
    out_host->num_gaussians = ctx->have_pre ? ctx->N : 0;
    out_host->invalid_gaussians = ctx->have_pre ? inv : 0;
    if (ctx->accel_kind == GS_QUERY_GRID) { out_host->grid_pairs = ctx->T; out_host->grid_touched = ctx->M; }
    if (ctx->accel_kind == GS_QUERY_POINTS) out_host->cull_chunk_capacity = ctx->cull_cap;
    out_host->decode_repeats = ctx->decode_repeats;
    return GS_OK;
}

gs_status gs_profile_enable(gs_ctx *ctx, int32_t on) {
    if (!ctx) return GS_ERR_INVALID_ARG;
    ctx->prof = on != 0;
    return GS_OK;
}

gs_status gs_profile_read(gs_ctx *ctx, float *ms_host, uint32_t *calls_host, uint64_t *launches_host) {
    if (!ctx) return GS_ERR_INVALID_ARG;
    CK(cudaSetDevice(ctx->device), "cudaSetDevice");
    CK(cudaStreamSynchronize(ctx->stream), "sync");
    float ms[GS_PROF_STAGES] = {0};
    uint32_t calls[GS_PROF_STAGES] = {0};
    for (auto &pp : ctx->prof_pending) {
        float t = 0.f;
        CK(cudaEventElapsedTime(&t, pp.a, pp.b), "event elapsed");
        ms[pp.stage] += t;
        calls[pp.stage]++;
        ctx->prof_free.push_back(pp);
    }
    ctx->prof_pending.clear();
    for (int k = 0; k < GS_PROF_STAGES; k++) {
        if (ms_host) ms_host[k] = ms[k];
        if (calls_host) calls_host[k] = calls[k];
    }
    if (launches_host) *launches_host = ctx->launches;
    ctx->launches = 0;
    return GS_OK;
}

gs_status gs_step_host(gs_ctx *ctx, const gs_gaussians *gh, const gs_domain *dom, float tau, const gs_query *qh,
                       const float *target_host, float *phi_host, float *I_host, double *loss_host, const gs_grads *grads_host) {
    LaunchScope launch_scope(ctx);
    if (!ctx) return GS_ERR_INVALID_ARG;
    if (!gh || !qh || !target_host || !loss_host) return fail(ctx, GS_ERR_INVALID_ARG, "gs_step_host: NULL argument");
    GridDesc gd{};
    uint64_t P = 0;
    gs_status st = validate_query(ctx, qh, &gd, &P);
    if (st != GS_OK) return st;
    CK(cudaSetDevice(ctx->device), "cudaSetDevice");
    cudaStream_t s = ctx->stream;
    const size_t N = gh->n, n1 = N ? N : 1, p1 = P ? P : 1;
    // staging layout: 0 mean 1 scale 2 quat 3 opacity 4 scalar 5 xyz 6 target 7 phi 8 I 9 dL_dphi 10 loss 11.. grads
    const size_t sizes[16] = {n1 * 12, n1 * 12, n1 * 16, n1 * 4, n1 * 4, qh->kind == GS_QUERY_POINTS ? p1 * 12 : 4, p1 * 4, p1 * 4, p1 * 4, 4, 8,
                              n1 * 12, n1 * 12, n1 * 16, n1 * 4, n1 * 8};
    for (int k = 0; k < 16; k++) CK(ctx->h2d[k].reserve(sizes[k]), "alloc staging");
    const void *src[5] = {gh->mean, gh->scale, gh->quat, gh->opacity, gh->scalar};
    for (int k = 0; k < 5; k++)
        if (N) CK(cudaMemcpyAsync(ctx->h2d[k].p, src[k], N * (sizes[k] / n1), cudaMemcpyHostToDevice, s), "H2D model");
    gs_query q = *qh;
    // The model is needed first (preprocess, LBVH over the Gaussians): its copy leads on the context's stream.  The query
    // points are first needed by the coherence sort inside gs_build_accel and the target by the forward's epilogue: their
    // copies run on a second stream beside preprocess and the Gaussian side of the build.
    if (!ctx->aux_stream) {
        CK(cudaStreamCreateWithFlags(&ctx->aux_stream, cudaStreamNonBlocking), "aux stream");
        CK(cudaEventCreateWithFlags(&ctx->aux_event, cudaEventDisableTiming), "aux event");
        CK(cudaEventCreateWithFlags(&ctx->aux_event2, cudaEventDisableTiming), "aux event");
    }
    if (P) {
        CK(cudaEventRecord(ctx->aux_event, s), "event");                       // after everything enqueued so far
        CK(cudaStreamWaitEvent(ctx->aux_stream, ctx->aux_event, 0), "wait");
        if (q.kind == GS_QUERY_POINTS) {
            CK(cudaMemcpyAsync(ctx->h2d[5].p, qh->xyz, P * 12, cudaMemcpyHostToDevice, ctx->aux_stream), "H2D points");
            CK(cudaEventRecord(ctx->aux_event2, ctx->aux_stream), "event");
            ctx->points_ready = ctx->aux_event2;
        }
        CK(cudaMemcpyAsync(ctx->h2d[6].p, target_host, P * 4, cudaMemcpyHostToDevice, ctx->aux_stream), "H2D target");
        CK(cudaEventRecord(ctx->aux_event, ctx->aux_stream), "event");
    }
    if (q.kind == GS_QUERY_POINTS) q.xyz = ctx->h2d[5].as<float>();
    CK(cudaMemsetAsync(ctx->h2d[10].p, 0, 8, s), "zero loss");
    gs_gaussians gdv{gh->n, ctx->h2d[0].as<float>(), ctx->h2d[1].as<float>(), ctx->h2d[2].as<float>(), ctx->h2d[3].as<float>(),
                     ctx->h2d[4].as<float>()};
    if ((st = gs_preprocess(ctx, &gdv, dom, tau)) != GS_OK) return st;
    if ((st = gs_build_accel(ctx, &q)) != GS_OK) return st;
    float *phi = ctx->h2d[7].as<float>(), *I = ctx->h2d[8].as<float>();
    if (P) CK(cudaStreamWaitEvent(s, ctx->aux_event, 0), "wait for the target");
    if ((st = gs_sample_fwd(ctx, &q, ctx->h2d[6].as<float>(), phi, I, ctx->h2d[10].as<double>(), nullptr, nullptr)) != GS_OK) return st;
    gs_grads gdev{ctx->h2d[11].as<float>(), ctx->h2d[12].as<float>(), ctx->h2d[13].as<float>(), ctx->h2d[14].as<float>(),
                  ctx->h2d[15].as<float>(), ctx->h2d[15].as<float>() + n1};
    if ((st = gs_sample_bwd(ctx, &q, nullptr, nullptr, nullptr, nullptr, nullptr, &gdev)) != GS_OK) return st;  // fused MSE backward
    if (phi_host && P) CK(cudaMemcpyAsync(phi_host, phi, P * 4, cudaMemcpyDeviceToHost, s), "D2H phi");
    if (I_host && P) CK(cudaMemcpyAsync(I_host, I, P * 4, cudaMemcpyDeviceToHost, s), "D2H I");
    CK(cudaMemcpyAsync(loss_host, ctx->h2d[10].p, 8, cudaMemcpyDeviceToHost, s), "D2H loss");
    if (grads_host && N) {
        float *dst[6] = {grads_host->dmean, grads_host->dscale, grads_host->dquat, grads_host->dopacity, grads_host->dscalar, grads_host->err};
        const float *srcd[6] = {gdev.dmean, gdev.dscale, gdev.dquat, gdev.dopacity, gdev.dscalar, gdev.err};
        const size_t bytes[6] = {N * 12, N * 12, N * 16, N * 4, N * 4, N * 4};
        for (int k = 0; k < 6; k++)
            if (dst[k]) CK(cudaMemcpyAsync(dst[k], srcd[k], bytes[k], cudaMemcpyDeviceToHost, s), "D2H grads");
    }
    CK(cudaStreamSynchronize(s), "sync");
    return GS_OK;
}

}  // extern "C"
