/*
 * wveg_oracle.c -- CPU ORACLE for the W-VEG sampling path.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, double-precision restatement of what arxiv/paper_2607_01164 ("Efficient
 * Compression of Structured and Unstructured Volumes via Learned 3D Gaussian
 * Representation") computes when it samples a collection of world-space volume-encoding
 * Gaussians (W-VEG) at 3D positions, and of the analytic gradients of that computation.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, load or call this file.  It shares no code with the CUDA path.
 *
 * Citations are PAPER.md:<line> (+ equation / section).  "DESIGN Dn" refers to the numbered
 * readings in DESIGN.md, taken where the paper is silent.
 *
 *   value arithmetic : double everywhere (inputs are the fp32 arrays promoted to double)
 *   decisions        : where floating point decides an integer (is Gaussian i in point c's
 *                      set; which bricks does an AABB touch; which Morton cell) the decision
 *                      is taken in fp32 with a fixed operation order -- the kernel's
 *                      precision -- restated here in plain C float arithmetic (compiled with
 *                      -ffp-contract=off so that only the fmaf() written below fuses).
 *
 * Parity pins (tests/test_oracle_*.py): closed form of one Gaussian, G(mu)=1, G=tau at
 * Mahalanobis radius sqrt(-2 ln tau), textbook normal pdf (scipy), rotation about z by hand,
 * constant-scalar collections, convexity, weight splitting, central finite
 * differences of every gradient, sum rules, brute force vs culled, Morton/Karras brute force.
 * The per-Gaussian error statistic E_i (DESIGN D10) is NOT defined by the paper (it is north_star's): its
 * DEFINITION is "parity unpinned"; its arithmetic is pinned by the sum rule and by two closed forms
 * (disjoint supports, coincident Gaussians: tests/test_oracle_atsize.py).
 * The cell-grid cull (mode 1) is pinned against all pairs (mode 0) on tiny inputs AND against the full
 * configs[1] / configs[2] models on point subsets (tests/test_oracle_atsize.py).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int64_t n;
    const float *mean;    /* [n,3] */
    const float *scale;   /* [n,3] linear sigma per principal axis, > 0 (PAPER.md:140 exp activation already applied) */
    const float *quat;    /* [n,4] (w,x,y,z), normalised here ("normalization activation") */
    const float *opacity; /* [n]   the paper's weight w_i */
    const float *scalar;  /* [n]   the paper's value v_i */
} wo_gaussians;

typedef struct {
    int32_t dims[3];      /* voxels of the whole grid */
    float origin[3];
    float spacing[3];
    int32_t brick_lo[3];  /* batch = brick-aligned sub-box, bricks of 8^3 voxels */
    int32_t brick_cnt[3];
} wo_grid;

int wo_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------------------- */
/* Constants of the cutoff (tau_1 = 0.01 "influence is the cutoff").        */
/* DESIGN D3: support of Gaussian i = { p : G_i(p) >= tau }  <=>  |u|^2 <= r2 = -2 ln tau. */
/* ------------------------------------------------------------------------------------- */
float wo_r2_f32(float tau) { return (float)(-2.0 * log((double)tau)); }
float wo_r_f32(float tau) { return (float)sqrt((double)wo_r2_f32(tau)); }

/* ------------------------------------------------------------------------------------- */
/* Rotation matrix of a unit quaternion (w,x,y,z): the standard v' = R v matrix.          */
/* Eq. 3 uses R_i inside R^T S^-2 R; DESIGN D1: rows of R are the principal  */
/* axes, u = S^-1 R (p - mu).                                                             */
/* ------------------------------------------------------------------------------------- */
static void rotation_f64(const double q[4], double R[9]) {
    double w = q[0], x = q[1], y = q[2], z = q[3];
    R[0] = 1.0 - 2.0 * (y * y + z * z); R[1] = 2.0 * (x * y - w * z);       R[2] = 2.0 * (x * z + w * y);
    R[3] = 2.0 * (x * y + w * z);       R[4] = 1.0 - 2.0 * (x * x + z * z); R[5] = 2.0 * (y * z - w * x);
    R[6] = 2.0 * (x * z - w * y);       R[7] = 2.0 * (y * z + w * x);       R[8] = 1.0 - 2.0 * (x * x + y * y);
}

static int gaussian_valid(const wo_gaussians *g, int64_t i) {
    /* DESIGN (boundary): non-finite parameters, non-positive scale or a zero quaternion => empty support */
    for (int k = 0; k < 3; k++) {
        if (!isfinite(g->mean[3 * i + k])) return 0;
        if (!(g->scale[3 * i + k] > 0.0f) || !isfinite(g->scale[3 * i + k])) return 0;
    }
    float n2 = 0.0f;
    for (int k = 0; k < 4; k++) {
        if (!isfinite(g->quat[4 * i + k])) return 0;
        n2 += g->quat[4 * i + k] * g->quat[4 * i + k];
    }
    if (!(n2 > 0.0f) || !isfinite(n2)) return 0;
    if (!isfinite(g->opacity[i]) || !isfinite(g->scalar[i])) return 0;
    return 1;
}

/* Whitening matrix M = S^-1 R in double (value arithmetic). M^T M = R^T S^-2 R (Eq. 3). */
static void whiten_f64(const wo_gaussians *g, int64_t i, double M[9], double R[9], double qhat[4], double *qnorm) {
    double q[4], n = 0.0;
    for (int k = 0; k < 4; k++) { q[k] = (double)g->quat[4 * i + k]; n += q[k] * q[k]; }
    n = sqrt(n);
    for (int k = 0; k < 4; k++) qhat[k] = q[k] / n;
    *qnorm = n;
    rotation_f64(qhat, R);
    for (int j = 0; j < 3; j++)
        for (int k = 0; k < 3; k++) M[3 * j + k] = R[3 * j + k] / (double)g->scale[3 * i + j];
}

/* ------------------------------------------------------------------------------------- */
/* S1 in the kernel's precision (DESIGN D4/D7): the fp32 sequence whose results feed       */
/* integer decisions.  Plain float ops, each rounded to nearest; fmaf only where written.  */
/* ------------------------------------------------------------------------------------- */
void wo_preprocess_f32(const wo_gaussians *g, float tau, float *M_out /*[n,9]*/, float *aabb_out /*[n,6] lo,hi*/,
                       uint8_t *valid_out /*[n]*/) {
    const float rf = wo_r_f32(tau);
    for (int64_t i = 0; i < g->n; i++) {
        float *M = M_out + 9 * i, *bb = aabb_out + 6 * i;
        if (!gaussian_valid(g, i)) {
            valid_out[i] = 0;
            for (int k = 0; k < 9; k++) M[k] = 0.0f;
            for (int k = 0; k < 3; k++) { bb[k] = INFINITY; bb[3 + k] = -INFINITY; } /* empty box */
            continue;
        }
        valid_out[i] = 1;
        const float qw = g->quat[4 * i], qx = g->quat[4 * i + 1], qy = g->quat[4 * i + 2], qz = g->quat[4 * i + 3];
        const float n2 = fmaf(qz, qz, fmaf(qy, qy, fmaf(qx, qx, qw * qw)));
        const float nrm = sqrtf(n2);
        const float w = qw / nrm, x = qx / nrm, y = qy / nrm, z = qz / nrm;
        const float xx = x * x, yy = y * y, zz = z * z;
        const float xy = x * y, xz = x * z, yz = y * z;
        const float wx = w * x, wy = w * y, wz = w * z;
        float R[9];
        R[0] = 1.0f - 2.0f * (yy + zz); R[1] = 2.0f * (xy - wz);        R[2] = 2.0f * (xz + wy);
        R[3] = 2.0f * (xy + wz);        R[4] = 1.0f - 2.0f * (xx + zz); R[5] = 2.0f * (yz - wx);
        R[6] = 2.0f * (xz - wy);        R[7] = 2.0f * (yz + wx);        R[8] = 1.0f - 2.0f * (xx + yy);
        const float *s = g->scale + 3 * i;
        for (int j = 0; j < 3; j++)
            for (int k = 0; k < 3; k++) M[3 * j + k] = R[3 * j + k] / s[j];
        /* cutoff ellipsoid { d : |S^-1 R d| <= r } -> half extent along world axis k is
           r * sqrt(sum_j (s_j R_jk)^2)  ("convert this ellipsoid to an AABB"),
           inflated by (1 + 2^-8) so that the box is a safe cull for the fp32 predicate. */
        for (int k = 0; k < 3; k++) {
            const float a0 = s[0] * R[k], a1 = s[1] * R[3 + k], a2 = s[2] * R[6 + k];
            const float e = rf * sqrtf(fmaf(a2, a2, fmaf(a1, a1, a0 * a0)));
            const float ei = e * 1.00390625f;
            bb[k] = g->mean[3 * i + k] - ei;
            bb[3 + k] = g->mean[3 * i + k] + ei;
        }
    }
}

/* The inclusion predicate in the kernel's precision (DESIGN D4): is p inside G_i's support? */
static inline int hit_f32(const float *M, const float *mu, const float *p, float r2f) {
    const float dx = p[0] - mu[0], dy = p[1] - mu[1], dz = p[2] - mu[2];
    const float u0 = fmaf(M[2], dz, fmaf(M[1], dy, M[0] * dx));
    const float u1 = fmaf(M[5], dz, fmaf(M[4], dy, M[3] * dx));
    const float u2 = fmaf(M[8], dz, fmaf(M[7], dy, M[6] * dx));
    const float qd = fmaf(u2, u2, fmaf(u1, u1, u0 * u0));
    return qd <= r2f;
}

int wo_hit_f32(const float *M, const float *mu, const float *p, float tau) { return hit_f32(M, mu, p, wo_r2_f32(tau)); }

/* Sample positions of a grid batch (DESIGN D6): voxel centre, p = fmaf((float)i + 0.5f, spacing, origin);
   x fastest.  The fp32 result IS the sample position. */
static void grid_batch_dims(const wo_grid *gr, int32_t bd[3]) {
    for (int k = 0; k < 3; k++) {
        int32_t e = 8 * gr->brick_cnt[k], rest = gr->dims[k] - 8 * gr->brick_lo[k];
        bd[k] = e < rest ? e : rest;
    }
}
int64_t wo_grid_num_points(const wo_grid *gr) {
    int32_t bd[3]; grid_batch_dims(gr, bd);
    return (int64_t)bd[0] * bd[1] * bd[2];
}
static inline float grid_coord(const wo_grid *gr, int axis, int32_t i_global) {
    return fmaf((float)i_global + 0.5f, gr->spacing[axis], gr->origin[axis]);
}
void wo_grid_points(const wo_grid *gr, float *xyz /*[P,3]*/) {
    int32_t bd[3]; grid_batch_dims(gr, bd);
    int64_t c = 0;
    for (int32_t z = 0; z < bd[2]; z++)
        for (int32_t y = 0; y < bd[1]; y++)
            for (int32_t x = 0; x < bd[0]; x++, c++) {
                xyz[3 * c + 0] = grid_coord(gr, 0, x + 8 * gr->brick_lo[0]);
                xyz[3 * c + 1] = grid_coord(gr, 1, y + 8 * gr->brick_lo[1]);
                xyz[3 * c + 2] = grid_coord(gr, 2, z + 8 * gr->brick_lo[2]);
            }
}

/* In-cell jitter of the grid samples ("we select a random position in each cell every iteration of     */
/* training").  The random numbers come from a counter-based generator so that both sides can draw the same ones      */
/* (DESIGN D26): the voxel with global index L = (gz * dims_y + gy) * dims_x + gx draws ONE 64-bit number              */
/*   h = splitmix64-finaliser(seed + L + golden gamma)                                                                 */
/* and axis a takes 21 of its bits:  j_a = ((h >> 21 a) & (2^21 - 1)) * 2^-21 - 0.5  in [-0.5, 0.5).                   */
/* The sample position is p_a = fmaf(((float)i_a + 0.5f) + j_a, spacing_a, origin_a) (every step exact or one fp32     */
/* rounding; that fp32 value IS the position, as for voxel centres, D6).                                               */
static inline uint64_t mix64_u64(uint64_t z) {
    z += 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}
float wo_jitter(uint64_t seed, uint64_t voxel_linear, int axis) {
    const uint64_t h = mix64_u64(seed + voxel_linear);
    return (float)((h >> (21 * axis)) & 0x1FFFFFull) * 4.76837158203125e-7f - 0.5f;
}
void wo_grid_points_jitter(const wo_grid *gr, uint64_t seed, float *xyz /*[P,3]*/) {
    int32_t bd[3]; grid_batch_dims(gr, bd);
    int64_t c = 0;
    for (int32_t z = 0; z < bd[2]; z++)
        for (int32_t y = 0; y < bd[1]; y++)
            for (int32_t x = 0; x < bd[0]; x++, c++) {
                const int32_t g[3] = {x + 8 * gr->brick_lo[0], y + 8 * gr->brick_lo[1], z + 8 * gr->brick_lo[2]};
                const uint64_t L = ((uint64_t)g[2] * (uint64_t)gr->dims[1] + (uint64_t)g[1]) * (uint64_t)gr->dims[0] + (uint64_t)g[0];
                for (int a = 0; a < 3; a++) {
                    const float t = ((float)g[a] + 0.5f) + wo_jitter(seed, L, a);
                    xyz[3 * c + a] = fmaf(t, gr->spacing[a], gr->origin[a]);
                }
            }
}

/* id hash used to compare per-point intersection SETS (order-free): count, sum and xor of mix(id). */
static inline uint64_t mix_id(uint32_t id) {
    uint64_t z = (uint64_t)id + 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

/* ------------------------------------------------------------------------------------- */
/* Candidate cull for large inputs: a uniform cell grid over the points' bounding box.     */
/* Gaussian i is a candidate for every point whose cell overlaps i's (inflated, fp32)      */
/* cutoff AABB.  The predicate is re-applied per pair, so the cull only removes pairs that */
/* the plain all-pairs definition would reject too (tested: culled == all-pairs).          */
/* ------------------------------------------------------------------------------------- */
typedef struct {
    double lo[3], hi[3], inv_h[3];   /* lo/hi: bounding box of the points */
    int32_t n[3];
    int64_t *cell_start;   /* [ncell+1] CSR over points */
    int64_t *cell_points;  /* [P] */
    int64_t *gcell_start;  /* [ncell+1] CSR over candidate Gaussians */
    int32_t *gcell_ids;    /* [sum] ascending Gaussian id inside each cell */
} cellgrid;

static inline int32_t cell_coord(const cellgrid *cg, int k, double x) {
    double f = floor((x - cg->lo[k]) * cg->inv_h[k]);
    if (f < 0.0) f = 0.0;
    if (f > (double)(cg->n[k] - 1)) f = (double)(cg->n[k] - 1);
    return (int32_t)f;
}

static void cellgrid_free(cellgrid *cg) {
    free(cg->cell_start); free(cg->cell_points); free(cg->gcell_start); free(cg->gcell_ids);
    memset(cg, 0, sizeof *cg);
}

/* need_points: build cell -> points; need_gauss: build cell -> candidate Gaussians */
static int cellgrid_build(cellgrid *cg, const float *xyz, int64_t P, const float *aabb, const uint8_t *valid, int64_t N,
                          int need_points, int need_gauss) {
    memset(cg, 0, sizeof *cg);
    double lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
    for (int64_t c = 0; c < P; c++)
        for (int k = 0; k < 3; k++) {
            double x = (double)xyz[3 * c + k];
            if (x < lo[k]) lo[k] = x;
            if (x > hi[k]) hi[k] = x;
        }
    /* resolution: about 4 points per cell, but cells no finer than half the mean Gaussian box
       (keeps the candidate lists small); any resolution gives the same result. */
    double target = cbrt((double)(P > 0 ? P : 1) / 4.0);
    double wsum = 0.0, ext_max = 0.0;
    int64_t nv = 0;
    for (int k = 0; k < 3; k++)
        if (hi[k] - lo[k] > ext_max) ext_max = hi[k] - lo[k];
    for (int64_t i = 0; i < N; i++) {
        if (!valid[i]) continue;
        double w = 0.0;
        for (int k = 0; k < 3; k++) {
            double e = (double)aabb[6 * i + 3 + k] - (double)aabb[6 * i + k];
            if (e > w) w = e;
        }
        wsum += w; nv++;
    }
    if (nv > 0 && wsum > 0.0 && ext_max > 0.0) {
        double cap = 2.0 * ext_max / (wsum / (double)nv);
        if (cap < target) target = cap;
    }
    int32_t res = (int32_t)target;
    if (res < 1) res = 1;
    if (res > 160) res = 160;
    for (int k = 0; k < 3; k++) {
        double ext = hi[k] - lo[k];
        cg->lo[k] = lo[k];
        cg->hi[k] = hi[k];
        cg->n[k] = (P > 0 && ext > 0.0) ? res : 1;
        cg->inv_h[k] = (cg->n[k] > 1) ? (double)cg->n[k] / ext : 0.0;
    }
    const int64_t ncell = (int64_t)cg->n[0] * cg->n[1] * cg->n[2];
    if (need_points) {
        cg->cell_start = (int64_t *)calloc((size_t)ncell + 1, sizeof(int64_t));
        cg->cell_points = (int64_t *)malloc(sizeof(int64_t) * (size_t)(P > 0 ? P : 1));
        if (!cg->cell_start || !cg->cell_points) return -1;
        for (int64_t c = 0; c < P; c++) {
            int64_t id = ((int64_t)cell_coord(cg, 2, xyz[3 * c + 2]) * cg->n[1] + cell_coord(cg, 1, xyz[3 * c + 1])) * cg->n[0] +
                         cell_coord(cg, 0, xyz[3 * c + 0]);
            cg->cell_start[id + 1]++;
        }
        for (int64_t k = 0; k < ncell; k++) cg->cell_start[k + 1] += cg->cell_start[k];
        int64_t *cur = (int64_t *)malloc(sizeof(int64_t) * (size_t)ncell);
        if (!cur) return -1;
        memcpy(cur, cg->cell_start, sizeof(int64_t) * (size_t)ncell);
        for (int64_t c = 0; c < P; c++) {
            int64_t id = ((int64_t)cell_coord(cg, 2, xyz[3 * c + 2]) * cg->n[1] + cell_coord(cg, 1, xyz[3 * c + 1])) * cg->n[0] +
                         cell_coord(cg, 0, xyz[3 * c + 0]);
            cg->cell_points[cur[id]++] = c;
        }
        free(cur);
    }
    if (need_gauss) {
        cg->gcell_start = (int64_t *)calloc((size_t)ncell + 1, sizeof(int64_t));
        if (!cg->gcell_start) return -1;
        for (int pass = 0; pass < 2; pass++) {
            int64_t *cur = NULL;
            if (pass == 1) {
                for (int64_t k = 0; k < ncell; k++) cg->gcell_start[k + 1] += cg->gcell_start[k];
                cg->gcell_ids = (int32_t *)malloc(sizeof(int32_t) * (size_t)(cg->gcell_start[ncell] > 0 ? cg->gcell_start[ncell] : 1));
                cur = (int64_t *)malloc(sizeof(int64_t) * (size_t)ncell);
                if (!cg->gcell_ids || !cur) return -1;
                memcpy(cur, cg->gcell_start, sizeof(int64_t) * (size_t)ncell);
            }
            for (int64_t i = 0; i < N; i++) {
                if (!valid[i]) continue;
                int32_t a[3], b[3], empty = 0;
                for (int k = 0; k < 3; k++) {
                    double blo = (double)aabb[6 * i + k], bhi = (double)aabb[6 * i + 3 + k];
                    if (bhi < lo[k] || blo > hi[k]) empty = 1;
                    a[k] = cell_coord(cg, k, blo);
                    b[k] = cell_coord(cg, k, bhi);
                }
                if (empty) continue;
                for (int32_t z = a[2]; z <= b[2]; z++)
                    for (int32_t y = a[1]; y <= b[1]; y++)
                        for (int32_t x = a[0]; x <= b[0]; x++) {
                            int64_t id = ((int64_t)z * cg->n[1] + y) * cg->n[0] + x;
                            if (pass == 0) cg->gcell_start[id + 1]++;
                            else cg->gcell_ids[cur[id]++] = (int32_t)i;
                        }
            }
            free(cur);
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------------------- */
/* Per-Gaussian tables shared by forward and backward: fp32 decision data + double values  */
/* ------------------------------------------------------------------------------------- */
typedef struct {
    float *Mf;       /* [n,9] fp32 whitening matrix (decisions) */
    float *aabb;     /* [n,6] */
    uint8_t *valid;  /* [n] */
    double *Md;      /* [n,9] double whitening matrix (values) */
    double *Rd;      /* [n,9] rotation of the normalised quaternion */
    double *qhat;    /* [n,4] */
    double *qnorm;   /* [n] */
} gtables;

static void gtables_free(gtables *t) {
    free(t->Mf); free(t->aabb); free(t->valid); free(t->Md); free(t->Rd); free(t->qhat); free(t->qnorm);
    memset(t, 0, sizeof *t);
}

static int gtables_build(gtables *t, const wo_gaussians *g, float tau) {
    size_t n = (size_t)(g->n > 0 ? g->n : 1);
    memset(t, 0, sizeof *t);
    t->Mf = (float *)malloc(n * 9 * sizeof(float));
    t->aabb = (float *)malloc(n * 6 * sizeof(float));
    t->valid = (uint8_t *)malloc(n);
    t->Md = (double *)malloc(n * 9 * sizeof(double));
    t->Rd = (double *)malloc(n * 9 * sizeof(double));
    t->qhat = (double *)malloc(n * 4 * sizeof(double));
    t->qnorm = (double *)malloc(n * sizeof(double));
    if (!t->Mf || !t->aabb || !t->valid || !t->Md || !t->Rd || !t->qhat || !t->qnorm) { gtables_free(t); return -1; }
    wo_preprocess_f32(g, tau, t->Mf, t->aabb, t->valid);
    for (int64_t i = 0; i < g->n; i++)
        if (t->valid[i]) whiten_f64(g, i, t->Md + 9 * i, t->Rd + 9 * i, t->qhat + 4 * i, t->qnorm + i);
    return 0;
}

/* One (point, Gaussian) pair, values in double.  Eq. 3: G = exp(-1/2 d^T R^T S^-2 R d)
   = exp(-|u|^2/2) with u = S^-1 R d. */
static inline double pair_G(const double *M, const float *mu, const float *p, double u[3]) {
    const double d0 = (double)p[0] - (double)mu[0], d1 = (double)p[1] - (double)mu[1], d2 = (double)p[2] - (double)mu[2];
    u[0] = M[0] * d0 + M[1] * d1 + M[2] * d2;
    u[1] = M[3] * d0 + M[4] * d1 + M[5] * d2;
    u[2] = M[6] * d0 + M[7] * d1 + M[8] * d2;
    return exp(-0.5 * (u[0] * u[0] + u[1] * u[1] + u[2] * u[2]));
}

/* ------------------------------------------------------------------------------------- */
/* FORWARD (S4/S5 + the normalisation of S6).                                              */
/*   I_c   = sum_{i in hits(c)} w_i G_i(p_c)           ("I_c += w_i G_i(p)")   */
/*   Nacc  = sum_{i in hits(c)} v_i w_i G_i(p_c)       ("V_c += v_i w_i G_i")  */
/*   Phi_c = Nacc / I_c  if I_c > tau  else 0          (Eq. 2; rule PAPER.md:126;*/
/*                                                      empty value DESIGN D5)              */
/* mode 0: all pairs; mode 1: cell-grid cull.  hit_mask_in (all-pairs only, [P,n] bytes)    */
/* freezes the membership, covered_in ([P] bytes) freezes the coverage decision: both are   */
/* for finite-difference checks, where the sets must not change under a perturbation.       */
/* Outputs count/hsum/hxor describe the per-point ID SET (order free).  All nullable except */
/* phi and I.  Returns 0, or -1 on allocation failure / bad arguments.                      */
/* ------------------------------------------------------------------------------------- */
int wo_forward(const wo_gaussians *g, const float *xyz, int64_t P, float tau, int mode, const uint8_t *hit_mask_in,
               const uint8_t *covered_in, double *phi, double *I, uint32_t *count, uint64_t *hsum, uint64_t *hxor,
               uint8_t *hit_mask_out) {
    if ((hit_mask_in || hit_mask_out) && mode != 0) return -1;
    gtables t;
    if (gtables_build(&t, g, tau)) return -1;
    const float r2f = wo_r2_f32(tau);
    const double taud = (double)tau;
    cellgrid cg;
    memset(&cg, 0, sizeof cg);
    if (mode == 1 && cellgrid_build(&cg, xyz, P, t.aabb, t.valid, g->n, 0, 1)) { gtables_free(&t); return -1; }
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t c = 0; c < P; c++) {
        const float *p = xyz + 3 * c;
        double Ic = 0.0, Nacc = 0.0;
        uint32_t cnt = 0;
        uint64_t hs = 0, hx = 0;
        const int32_t *cand = NULL;
        int64_t ncand = g->n;
        if (mode == 1) {
            int64_t id = ((int64_t)cell_coord(&cg, 2, p[2]) * cg.n[1] + cell_coord(&cg, 1, p[1])) * cg.n[0] + cell_coord(&cg, 0, p[0]);
            cand = cg.gcell_ids + cg.gcell_start[id];
            ncand = cg.gcell_start[id + 1] - cg.gcell_start[id];
        }
        for (int64_t k = 0; k < ncand; k++) {
            const int64_t i = cand ? cand[k] : k;
            int hit;
            if (hit_mask_in) hit = hit_mask_in[c * g->n + i];
            else hit = t.valid[i] && hit_f32(t.Mf + 9 * i, g->mean + 3 * i, p, r2f);
            if (hit_mask_out) hit_mask_out[c * g->n + i] = (uint8_t)hit;
            if (!hit) continue;
            double u[3];
            const double G = pair_G(t.Md + 9 * i, g->mean + 3 * i, p, u);
            const double wG = (double)g->opacity[i] * G;
            Ic += wG;
            Nacc += (double)g->scalar[i] * wG;
            cnt++;
            const uint64_t m = mix_id((uint32_t)i);
            hs += m; hx ^= m;
        }
        /* coverage decision in the kernel's precision (DESIGN D5): strict fp32 compare of the
           fp32-rounded accumulated influence against tau */
        int covered = covered_in ? covered_in[c] : ((float)Ic > tau);
        (void)taud;
        phi[c] = covered ? Nacc / Ic : 0.0;
        I[c] = Ic;
        if (count) count[c] = cnt;
        if (hsum) hsum[c] = hs;
        if (hxor) hxor[c] = hx;
    }
    if (mode == 1) cellgrid_free(&cg);
    gtables_free(&t);
    return 0;
}

/* ------------------------------------------------------------------------------------- */
/* S6: loss epilogue.  north_star fixes MSE (the paper trains with L1):       */
/*   L = (1/P) sum_c (Phi_c - t_c)^2 over ALL samples (uncovered ones enter as (0 - t)^2),  */
/*   dL/dPhi_c = 2 (Phi_c - t_c) / P where covered, 0 elsewhere (DESIGN D5),                */
/*   sample_err_c = |Phi_c - t_c|  (the per-sample error densification ranks).*/
/* ------------------------------------------------------------------------------------- */
void wo_mse(const double *phi, const double *I, const float *target, int64_t P, float tau, double *loss, double *dL_dphi,
            double *sample_err) {
    double acc = 0.0;
    for (int64_t c = 0; c < P; c++) {
        const double res = phi[c] - (double)target[c];
        const int covered = (float)I[c] > tau;
        acc += res * res;
        if (dL_dphi) dL_dphi[c] = covered ? 2.0 * res / (double)P : 0.0;
        if (sample_err) sample_err[c] = fabs(res);
    }
    if (loss) *loss = P > 0 ? acc / (double)P : 0.0;
}

/* ------------------------------------------------------------------------------------- */
/* S6, the paper's training losses.  `defined` (nullable = all) marks the */
/* samples that lie in the volume's domain (set D); the others form the set U of samples     */
/* "undefined in the volume".  With nD = |D|:                                 */
/*   reconstruction over D: L_rec = (1/nD) sum_D rho(Phi_d - t_d), rho = |.| ("L1            */
/*     reconstruction loss"; kind 1) or (.)^2 (north_star's MSE; kind 0);      */
/*     an uncovered sample of D enters as rho(0 - t) and passes no gradient through Phi      */
/*     (DESIGN D5); d|x|/dx = sign(x), 0 at x = 0.                                           */
/*   false negatives, Eq. 4: D- = { d in D | I_d < (1 + eps) tau },       */
/*     L_FN = lambda_FN sum_{D-} ((1 + eps) tau - I_d) / |D-|   (0 when D- is empty)         */
/*     => dL/dI_d = -lambda_FN / |D-| on D-.                                                 */
/*   false positives, Eq. 5: U+ = { u in U | I_u >= tau },                    */
/*     L_FP = lambda_FP sum_{U+} I_u / |U+|   => dL/dI_u = +lambda_FP / |U+| on U+.          */
/* Membership of D- and U+ is decided on the fp32 value of I against fp32 thresholds         */
/* ((1.0f + eps) * tau and tau), like the coverage rule.  The paper gives no eps / lambda.   */
/* loss3 = (L_rec, L_FN, L_FP); counts3 = (nD, |D-|, |U+|); sample_err = |Phi - t| on D, 0 on U. */
/* ------------------------------------------------------------------------------------- */
void wo_loss(const double *phi, const double *I, const float *target, const uint8_t *defined, int64_t P, float tau, int kind,
             float lambda_fn, float eps_fn, float lambda_fp, double *loss3, double *dL_dphi, double *dL_dI, double *sample_err,
             int64_t *counts3) {
    const float thr_fn = (1.0f + eps_fn) * tau;
    int64_t nD = 0, nFN = 0, nFP = 0;
    for (int64_t c = 0; c < P; c++) {
        const int def = defined ? defined[c] != 0 : 1;
        const float If = (float)I[c];
        if (def) {
            nD++;
            if (If < thr_fn) nFN++;
        } else if (If >= tau) {
            nFP++;
        }
    }
    double rec = 0.0, fn = 0.0, fp = 0.0;
    for (int64_t c = 0; c < P; c++) {
        const int def = defined ? defined[c] != 0 : 1;
        const float If = (float)I[c];
        const int covered = If > tau;
        double a = 0.0, b = 0.0, e = 0.0;
        if (def) {
            const double res = phi[c] - (double)target[c];
            e = fabs(res);
            if (kind == 1) {
                rec += fabs(res);
                if (covered) a = (res > 0.0 ? 1.0 : res < 0.0 ? -1.0 : 0.0) / (double)nD;
            } else {
                rec += res * res;
                if (covered) a = 2.0 * res / (double)nD;
            }
            if (If < thr_fn) {
                fn += (double)thr_fn - I[c];
                b = -(double)lambda_fn / (double)nFN;
            }
        } else if (If >= tau) {
            fp += I[c];
            b = (double)lambda_fp / (double)nFP;
        }
        if (dL_dphi) dL_dphi[c] = a;
        if (dL_dI) dL_dI[c] = b;
        if (sample_err) sample_err[c] = e;
    }
    if (loss3) {
        loss3[0] = nD ? rec / (double)nD : 0.0;
        loss3[1] = nFN ? (double)lambda_fn * fn / (double)nFN : 0.0;
        loss3[2] = nFP ? (double)lambda_fp * fp / (double)nFP : 0.0;
    }
    if (counts3) { counts3[0] = nD; counts3[1] = nFN; counts3[2] = nFP; }
}

/* ------------------------------------------------------------------------------------- */
/* Training-step completion.  Raw parameters and their activations        */
/* (PAPER.md:140): "sigmoid activation functions for v_i and w_i", "an exponential            */
/* activation for S_i" (the normalisation of R_i is part of the preprocess, DESIGN D2):       */
/*   scale = exp(raw_scale), opacity = sigmoid(raw_opacity), scalar = sigmoid(raw_scalar).    */
/* ------------------------------------------------------------------------------------- */
static double wo_sigmoid(double x) { return 1.0 / (1.0 + exp(-x)); }

void wo_activate(int64_t n, const float *raw_scale, const float *raw_opacity, const float *raw_scalar, double *scale,
                 double *opacity, double *scalar) {
    for (int64_t i = 0; i < n; i++) {
        for (int k = 0; k < 3; k++) scale[3 * i + k] = exp((double)raw_scale[3 * i + k]);
        opacity[i] = wo_sigmoid((double)raw_opacity[i]);
        scalar[i] = wo_sigmoid((double)raw_scalar[i]);
    }
}

/* Adam (Kingma & Ba, the paper's [20]), one step t >= 1 on one tensor of `count` elements: */
/*   m = b1 m + (1 - b1) g;  v = b2 v + (1 - b2) g^2;  p -= lr (m / (1 - b1^t)) / (sqrt(v / (1 - b2^t)) + eps) */
static void adam_tensor(int64_t count, double *p, const double *g, double *m, double *v, double lr, double b1, double b2,
                        double eps, int t) {
    const double c1 = 1.0 - pow(b1, (double)t), c2 = 1.0 - pow(b2, (double)t);
    for (int64_t k = 0; k < count; k++) {
        m[k] = b1 * m[k] + (1.0 - b1) * g[k];
        v[k] = b2 * v[k] + (1.0 - b2) * g[k] * g[k];
        p[k] -= lr * (m[k] / c1) / (sqrt(v[k] / c2) + eps);
    }
}

/* One optimiser step on the RAW parameters given the gradients w.r.t. the ACTIVATED values (what the */
/* backward returns).  Chain rule of the activations: d/d raw_scale = dscale * scale (exp' = exp),    */
/* d/d raw_opacity = dopacity * w (1 - w), d/d raw_scalar = dscalar * v (1 - v) (sigmoid' = s (1 - s)); */
/* mean and quaternion are their own raw parameters.  lr = (mean, scale, quat, opacity, scalar); the    */
/* paper's values are 0.00016, 0.001, 0.0001, 0.025 (weights), 0.0025 (values).         */
/* p* are updated in place; m*, v* are the Adam moments (same shapes).                                */
void wo_adam_step(int64_t n, double *mean, double *raw_scale, double *quat, double *raw_opacity, double *raw_scalar,
                  const double *dmean, const double *dscale, const double *dquat, const double *dopacity, const double *dscalar,
                  double *m, double *v, const double *lr, double b1, double b2, double eps, int t) {
    /* moments are laid out as one block of 12 n doubles: mean 3n | scale 3n | quat 4n | opacity n | scalar n */
    double *graw_s = (double *)malloc(sizeof(double) * 3 * (size_t)(n ? n : 1));
    double *graw_w = (double *)malloc(sizeof(double) * (size_t)(n ? n : 1));
    double *graw_v = (double *)malloc(sizeof(double) * (size_t)(n ? n : 1));
    for (int64_t i = 0; i < n; i++) {
        for (int k = 0; k < 3; k++) graw_s[3 * i + k] = dscale[3 * i + k] * exp(raw_scale[3 * i + k]);
        const double w = wo_sigmoid(raw_opacity[i]), s = wo_sigmoid(raw_scalar[i]);
        graw_w[i] = dopacity[i] * w * (1.0 - w);
        graw_v[i] = dscalar[i] * s * (1.0 - s);
    }
    adam_tensor(3 * n, mean, dmean, m, v, lr[0], b1, b2, eps, t);
    adam_tensor(3 * n, raw_scale, graw_s, m + 3 * n, v + 3 * n, lr[1], b1, b2, eps, t);
    adam_tensor(4 * n, quat, dquat, m + 6 * n, v + 6 * n, lr[2], b1, b2, eps, t);
    adam_tensor(n, raw_opacity, graw_w, m + 10 * n, v + 10 * n, lr[3], b1, b2, eps, t);
    adam_tensor(n, raw_scalar, graw_v, m + 11 * n, v + 11 * n, lr[4], b1, b2, eps, t);
    free(graw_s); free(graw_w); free(graw_v);
}

/* ------------------------------------------------------------------------------------- */
/* BACKWARD (S7 + S8): analytic gradients of any loss L(Phi, I) w.r.t. the inputs of the    */
/* forward, given a_c = dL/dPhi_c and b_c = dL/dI_c ("(I_c, V_c, dL/dI_c,      */
/* dL/dV_c)"; "backpropagating gradients to (mu_i, S_i, R_i, v_i, w_i)").      */
/* The paper does not print the derivatives; they follow from Eq. 2/3 by the chain rule:    */
/*   Phi = Nacc/I:   dL/dNacc = a/I =: alpha,  dL/dI(total) = b - alpha Phi =: beta         */
/*   each hit adds w G to I and v w G to Nacc:  dL/d(wG) = alpha v + beta =: gamma          */
/*   dL/dv_i = sum_c alpha w G          dL/dw_i = sum_c gamma G                             */
/*   G = exp(-|u|^2/2), u = S^-1 R (p - mu):  dL/du = -t u,  t = gamma w G                  */
/*   dL/dmu = M^T U,  U = sum_c t u        (d = p - mu, dd/dmu = -1)                        */
/*   dL/ds_j = W_jj / s_j,  W = sum_c t u u^T   (du_j/ds_j = -u_j/s_j)                      */
/*   dL/dR_jk = -(1/s_j) sum_l W_jl s_l R_lk    (du_j/dR_jk = d_k/s_j, d = R^T S u)         */
/*   dL/dqhat by differentiating the rotation formula, then through qhat = q/|q|:           */
/*   dL/dq = (dL/dqhat - qhat (qhat . dL/dqhat)) / |q|                                      */
/* a_c of an uncovered sample is ignored (Phi is the constant 0 there, DESIGN D5).          */
/* Error statistic (DESIGN D10, not from the paper): E_i = sum_{c covered} |Phi_c - t_c| w_i G_ic / I_c. */
/* hit_mask_in as in wo_forward (mode 0 only).  phi, I are the forward's outputs.           */
/* ------------------------------------------------------------------------------------- */
int wo_backward(const wo_gaussians *g, const float *xyz, int64_t P, float tau, int mode, const uint8_t *hit_mask_in,
                const uint8_t *covered_in, const double *phi, const double *I, const double *a, const double *b,
                const float *target, double *dmean, double *dscale, double *dquat, double *dopacity, double *dscalar,
                double *err) {
    if (hit_mask_in && mode != 0) return -1;
    gtables t;
    if (gtables_build(&t, g, tau)) return -1;
    const float r2f = wo_r2_f32(tau);
    cellgrid cg;
    memset(&cg, 0, sizeof cg);
    if (mode == 1 && cellgrid_build(&cg, xyz, P, t.aabb, t.valid, g->n, 1, 0)) { gtables_free(&t); return -1; }
    /* per-sample coefficients */
    double *alpha = (double *)malloc(sizeof(double) * (size_t)(P > 0 ? P : 1));
    double *beta = (double *)malloc(sizeof(double) * (size_t)(P > 0 ? P : 1));
    double *eps = (double *)malloc(sizeof(double) * (size_t)(P > 0 ? P : 1));
    if (!alpha || !beta || !eps) { free(alpha); free(beta); free(eps); gtables_free(&t); cellgrid_free(&cg); return -1; }
    for (int64_t c = 0; c < P; c++) {
        const int covered = covered_in ? covered_in[c] : ((float)I[c] > tau);
        const double al = covered ? a[c] / I[c] : 0.0;
        alpha[c] = al;
        beta[c] = (b ? b[c] : 0.0) - al * phi[c];
        eps[c] = (covered && target) ? fabs(phi[c] - (double)target[c]) / I[c] : 0.0;
    }
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < g->n; i++) {
        double dv = 0.0, dw = 0.0, U[3] = {0, 0, 0}, W[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0}, E = 0.0;
        const double w = (double)g->opacity[i], v = (double)g->scalar[i];
        if (t.valid[i]) {
            int32_t ca[3] = {0, 0, 0}, cb[3] = {0, 0, 0};
            int skip = 0;
            if (mode == 1) {
                for (int k = 0; k < 3; k++) {
                    /* an AABB that misses the points' bounding box holds no point: same skip as the forward's
                       candidate lists (cellgrid_build), so that a small batch of a large model costs O(touched) */
                    if ((double)t.aabb[6 * i + 3 + k] < cg.lo[k] || (double)t.aabb[6 * i + k] > cg.hi[k]) skip = 1;
                    ca[k] = cell_coord(&cg, k, (double)t.aabb[6 * i + k]);
                    cb[k] = cell_coord(&cg, k, (double)t.aabb[6 * i + 3 + k]);
                }
            }
            for (int32_t cz = ca[2]; cz <= cb[2] && !skip; cz++)
                for (int32_t cy = ca[1]; cy <= cb[1]; cy++)
                    for (int32_t cx = ca[0]; cx <= cb[0]; cx++) {
                        int64_t k0 = 0, k1 = P;
                        if (mode == 1) {
                            int64_t id = ((int64_t)cz * cg.n[1] + cy) * cg.n[0] + cx;
                            k0 = cg.cell_start[id]; k1 = cg.cell_start[id + 1];
                        }
                        for (int64_t k = k0; k < k1; k++) {
                            const int64_t c = mode == 1 ? cg.cell_points[k] : k;
                            const float *p = xyz + 3 * c;
                            const int hit = hit_mask_in ? hit_mask_in[c * g->n + i] : hit_f32(t.Mf + 9 * i, g->mean + 3 * i, p, r2f);
                            if (!hit) continue;
                            double u[3];
                            const double G = pair_G(t.Md + 9 * i, g->mean + 3 * i, p, u);
                            const double gamma = alpha[c] * v + beta[c];
                            const double tt = gamma * w * G;
                            dv += alpha[c] * w * G;
                            dw += gamma * G;
                            E += eps[c] * w * G;
                            for (int j = 0; j < 3; j++) {
                                U[j] += tt * u[j];
                                for (int l = 0; l < 3; l++) W[3 * j + l] += tt * u[j] * u[l];
                            }
                        }
                    }
        }
        /* S8: from (U, W) to the parameters */
        double dmu[3] = {0, 0, 0}, ds[3] = {0, 0, 0}, dq[4] = {0, 0, 0, 0};
        if (t.valid[i]) {
            const double *M = t.Md + 9 * i, *R = t.Rd + 9 * i, *qh = t.qhat + 4 * i;
            const float *s = g->scale + 3 * i;
            for (int k = 0; k < 3; k++) dmu[k] = M[k] * U[0] + M[3 + k] * U[1] + M[6 + k] * U[2];
            for (int j = 0; j < 3; j++) ds[j] = W[3 * j + j] / (double)s[j];
            double D[9];
            for (int j = 0; j < 3; j++)
                for (int k = 0; k < 3; k++) {
                    double acc = 0.0;
                    for (int l = 0; l < 3; l++) acc += W[3 * j + l] * (double)s[l] * R[3 * l + k];
                    D[3 * j + k] = -acc / (double)s[j];
                }
            const double qw = qh[0], qx = qh[1], qy = qh[2], qz = qh[3];
            double dh[4];
            dh[0] = 2.0 * (-qz * D[1] + qy * D[2] + qz * D[3] - qx * D[5] - qy * D[6] + qx * D[7]);
            dh[1] = 2.0 * (qy * D[1] + qz * D[2] + qy * D[3] - 2.0 * qx * D[4] - qw * D[5] + qz * D[6] + qw * D[7] - 2.0 * qx * D[8]);
            dh[2] = 2.0 * (-2.0 * qy * D[0] + qx * D[1] + qw * D[2] + qx * D[3] + qz * D[5] - qw * D[6] + qz * D[7] - 2.0 * qy * D[8]);
            dh[3] = 2.0 * (-2.0 * qz * D[0] - qw * D[1] + qx * D[2] + qw * D[3] - 2.0 * qz * D[4] + qy * D[5] + qx * D[6] + qy * D[7]);
            const double dot = qh[0] * dh[0] + qh[1] * dh[1] + qh[2] * dh[2] + qh[3] * dh[3];
            for (int k = 0; k < 4; k++) dq[k] = (dh[k] - qh[k] * dot) / t.qnorm[i];
        }
        for (int k = 0; k < 3; k++) { dmean[3 * i + k] = dmu[k]; dscale[3 * i + k] = ds[k]; }
        for (int k = 0; k < 4; k++) dquat[4 * i + k] = dq[k];
        dopacity[i] = dw;
        dscalar[i] = dv;
        if (err) err[i] = E;
    }
    free(alpha); free(beta); free(eps);
    if (mode == 1) cellgrid_free(&cg);
    gtables_free(&t);
    return 0;
}

/* ------------------------------------------------------------------------------------- */
/* S2 (integer): which 8^3 bricks of the batch does each Gaussian's AABB touch            */
/* ("AABB in blocks of the structured grid ... number of blocks intersected", */
/* PAPER.md:120-122 pairs sorted by block ID, per-block index ranges).  DESIGN D7:         */
/*   inv_brick_k = 1.0f / (8.0f * spacing_k)                                               */
/*   b = floorf((aabb - origin_k) * inv_brick_k), clamped in float to [-1, nb_k], -> int   */
/*   range = [max(b_lo, first_k), min(b_hi, last_k)], empty if lo > hi                     */
/* brick id is batch-local: ((bz-lo_z)*cnt_y + (by-lo_y))*cnt_x + (bx-lo_x).               */
/* ------------------------------------------------------------------------------------- */
void wo_brick_ranges(const float *aabb, const uint8_t *valid, int64_t n, const wo_grid *gr, int32_t *blo /*[n,3]*/,
                     int32_t *bhi /*[n,3]*/, uint32_t *count /*[n]*/) {
    for (int64_t i = 0; i < n; i++) {
        int64_t cnt = valid[i] ? 1 : 0;
        for (int k = 0; k < 3; k++) {
            const float inv_brick = 1.0f / (8.0f * gr->spacing[k]);
            const float nb = (float)((gr->dims[k] + 7) / 8);
            float fl = floorf((aabb[6 * i + k] - gr->origin[k]) * inv_brick);
            float fh = floorf((aabb[6 * i + 3 + k] - gr->origin[k]) * inv_brick);
            int32_t lo, hi;
            if (!valid[i]) { lo = 0; hi = -1; }
            else {
                fl = fminf(fmaxf(fl, -1.0f), nb);
                fh = fminf(fmaxf(fh, -1.0f), nb);
                lo = (int32_t)fl; hi = (int32_t)fh;
                const int32_t first = gr->brick_lo[k], last = gr->brick_lo[k] + gr->brick_cnt[k] - 1;
                if (lo < first) lo = first;
                if (hi > last) hi = last;
            }
            blo[3 * i + k] = lo; bhi[3 * i + k] = hi;
            cnt *= (hi >= lo) ? (int64_t)(hi - lo + 1) : 0;
        }
        count[i] = (uint32_t)cnt;
    }
}

static int cmp_u64(const void *a, const void *b) {
    const uint64_t x = *(const uint64_t *)a, y = *(const uint64_t *)b;
    return x < y ? -1 : (x > y ? 1 : 0);
}

/* keys[T] = (brick_id << 32 | gaussian_id) sorted ascending; brick_start[nbricks+1].
   T = sum(count) must be the caller's allocation size.  Returns T. */
int64_t wo_brick_keys(const int32_t *blo, const int32_t *bhi, const uint32_t *count, int64_t n, const wo_grid *gr,
                      uint64_t *keys, int64_t *brick_start) {
    int64_t T = 0;
    for (int64_t i = 0; i < n; i++) {
        if (!count[i]) continue;
        for (int32_t z = blo[3 * i + 2]; z <= bhi[3 * i + 2]; z++)
            for (int32_t y = blo[3 * i + 1]; y <= bhi[3 * i + 1]; y++)
                for (int32_t x = blo[3 * i]; x <= bhi[3 * i]; x++) {
                    const uint64_t brick = ((uint64_t)(z - gr->brick_lo[2]) * (uint64_t)gr->brick_cnt[1] + (uint64_t)(y - gr->brick_lo[1])) *
                                               (uint64_t)gr->brick_cnt[0] + (uint64_t)(x - gr->brick_lo[0]);
                    keys[T++] = (brick << 32) | (uint64_t)(uint32_t)i;
                }
    }
    qsort(keys, (size_t)T, sizeof(uint64_t), cmp_u64);
    const int64_t nbricks = (int64_t)gr->brick_cnt[0] * gr->brick_cnt[1] * gr->brick_cnt[2];
    int64_t k = 0;
    for (int64_t b = 0; b <= nbricks; b++) {
        while (k < T && (int64_t)(keys[k] >> 32) < b) k++;
        brick_start[b] = k;
    }
    return T;
}

/* ------------------------------------------------------------------------------------- */
/* S3 (integer): 30-bit Morton codes, LBVH topology and boxes (north_star (2); the paper    */
/* itself uses a cuBQL BVH over the sample positions).  DESIGN D8:            */
/*   scale_k = 1024.0f / (hi_k - lo_k)   (fp32, computed once)                              */
/*   q_k = (int) fminf(fmaxf((x_k - lo_k) * scale_k, 0.0f), 1023.0f)   (truncation)         */
/*   code = interleave, x in the lowest bit of each triple; invalid Gaussian -> 1<<30       */
/*   sort key = (code << 32 | id): unique, so the radix tree has no ties.                   */
/* ------------------------------------------------------------------------------------- */
static inline uint32_t expand10(uint32_t v) {
    uint32_t r = 0;
    for (int b = 0; b < 10; b++) r |= ((v >> b) & 1u) << (3 * b);
    return r;
}
void wo_morton_codes(const float *xyz, const uint8_t *valid /*nullable*/, int64_t n, const float lo[3], const float hi[3],
                     uint32_t *codes) {
    float scale[3];
    for (int k = 0; k < 3; k++) scale[k] = 1024.0f / (hi[k] - lo[k]);
    for (int64_t i = 0; i < n; i++) {
        if (valid && !valid[i]) { codes[i] = 1u << 30; continue; }
        uint32_t q[3];
        for (int k = 0; k < 3; k++) {
            const float t = (xyz[3 * i + k] - lo[k]) * scale[k];
            q[k] = (uint32_t)(int32_t)fminf(fmaxf(t, 0.0f), 1023.0f);
        }
        codes[i] = expand10(q[0]) | (expand10(q[1]) << 1) | (expand10(q[2]) << 2);
    }
}

/* order[n] = ids sorted by (code, id); sorted_keys[n] (nullable) = the 64-bit keys in that order */
void wo_morton_order(const uint32_t *codes, int64_t n, uint32_t *order, uint64_t *sorted_keys) {
    uint64_t *k = (uint64_t *)malloc(sizeof(uint64_t) * (size_t)(n > 0 ? n : 1));
    for (int64_t i = 0; i < n; i++) k[i] = ((uint64_t)codes[i] << 32) | (uint64_t)(uint32_t)i;
    qsort(k, (size_t)n, sizeof(uint64_t), cmp_u64);
    for (int64_t i = 0; i < n; i++) { order[i] = (uint32_t)(k[i] & 0xffffffffu); if (sorted_keys) sorted_keys[i] = k[i]; }
    free(k);
}

/* The binary radix tree over n sorted unique keys, written as its plain top-down definition:
   a node covering [l, r] (l < r) splits after the last key that shares with key_l a longer
   common prefix than key_l shares with key_r.  Numbering (Karras 2012's layout): the root is
   internal node 0; the left child [l, s] is internal node s (or leaf s if l == s), the right
   child [s+1, r] is internal node s+1 (or leaf s+1 if s+1 == r).  Children are encoded as
   index >= 0 for an internal node and ~leaf (< 0) for a leaf (leaf = position in sorted order).
   Boxes: the exact min/max union of the leaves' fp32 AABBs (leaf_aabb is in SORTED order).
   Outputs: left/right/parent [n-1], leaf_parent [n], node_aabb [n-1,6], range_lo/hi [n-1]. */
static inline int clz64(uint64_t x) { return x ? __builtin_clzll(x) : 64; }
int wo_lbvh_build(const uint64_t *keys, int64_t n, const float *leaf_aabb, int32_t *left, int32_t *right, int32_t *parent,
                  int32_t *leaf_parent, float *node_aabb, int32_t *range_lo, int32_t *range_hi) {
    if (n < 2) { if (n == 1 && leaf_parent) leaf_parent[0] = -1; return 0; }
    typedef struct { int64_t l, r; int32_t idx, par; } item;
    item *stack = (item *)malloc(sizeof(item) * (size_t)(n + 8));
    int32_t *order = (int32_t *)malloc(sizeof(int32_t) * (size_t)n); /* internal nodes in visit (pre-)order */
    if (!stack || !order) { free(stack); free(order); return -1; }
    int64_t sp = 0, nvisit = 0;
    stack[sp++] = (item){0, n - 1, 0, -1};
    while (sp > 0) {
        item it = stack[--sp];
        const int common = clz64(keys[it.l] ^ keys[it.r]);
        int64_t s = it.l;
        for (int64_t k = it.l; k < it.r; k++)
            if (clz64(keys[it.l] ^ keys[k]) > common) s = k; /* k = l gives clz = 64 > common */
        parent[it.idx] = it.par;
        range_lo[it.idx] = (int32_t)it.l; range_hi[it.idx] = (int32_t)it.r;
        order[nvisit++] = it.idx;
        if (s == it.l) { left[it.idx] = ~(int32_t)s; leaf_parent[s] = it.idx; }
        else { left[it.idx] = (int32_t)s; stack[sp++] = (item){it.l, s, (int32_t)s, it.idx}; }
        if (s + 1 == it.r) { right[it.idx] = ~(int32_t)(s + 1); leaf_parent[s + 1] = it.idx; }
        else { right[it.idx] = (int32_t)(s + 1); stack[sp++] = (item){s + 1, it.r, (int32_t)(s + 1), it.idx}; }
    }
    for (int64_t v = 0; v < nvisit; v++) {
        const int32_t i = order[v];
        float *bb = node_aabb + 6 * i;
        for (int k = 0; k < 3; k++) { bb[k] = INFINITY; bb[3 + k] = -INFINITY; }
        for (int64_t k = range_lo[i]; k <= range_hi[i]; k++)
            for (int d = 0; d < 3; d++) {
                bb[d] = fminf(bb[d], leaf_aabb[6 * k + d]);
                bb[3 + d] = fmaxf(bb[3 + d], leaf_aabb[6 * k + 3 + d]);
            }
    }
    free(stack); free(order);
    return 0;
}
