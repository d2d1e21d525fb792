/*
 * tofmlem_oracle.c -- plain, slow, fp64 CPU oracle for list-mode TOF-weighted MLEM.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no code,
 * header, table or helper with the CUDA path under paper_1706_07075_b200/ and neither imports the
 * other.
 *
 * What it computes, and the passages it follows (PAPER.md = /root/reference/PAPER.md; "R<n>" are the
 * readings listed in DESIGN.md / SURVEY.md section 8(c) where the paper is silent):
 *
 *   - list-mode MLEM with a TOF probability density in the system model (the
 *     update equation is never printed -> R1: x_j <- (x_j / s_j) * sum_e a_ej / sum_k a_ek x_k);
 *   - the TOF kernel is a Gaussian of the coincidence time resolution (300 ps FWHM), centred on the
 *     measured time difference of the two photons, truncated at ~3 sigma
 *     (PAPER.md:105, :206 -> R5: exactly trunc_sigmas * sigma, default 3);
 *   - events are filled directly into the voxels under the kernel ("direct technique for voxel
 *     filling").  The paper's own kernel is K sampled points;
 *     BASELINE.json's north_star fixes the graded projector instead as *Siddon exact voxel chord
 *     lengths times a normalised Gaussian evaluated at each chord midpoint, truncated at +-3 sigma*
 *     (R2, R4, R6, R7: the window is CLIPPED, end chords are weighted with their clipped length and
 *     clipped midpoint; no renormalisation after truncation);
 *   - sigma_x = c * FWHM / (2 * 2 sqrt(2 ln 2))  (pinned by PAPER.md:111, "sigma = 19.11 mm" at 300 ps);
 *   - TOF-assisted division of the events into axial body regions by the TOF-estimated annihilation
 *     position (R12, R13: single assignment by z of the kernel centre, first region
 *     double width as in "200 + 8 x 100" slices);
 *   - locality bin keys (BASELINE.json north_star bullet 1; arithmetic specification F1 in DESIGN.md),
 *     evaluated in float32 with a fixed operation order so that integer results are bit-exact.
 *
 * The algorithm is written step by step as a definition (collect plane crossings, sort, take
 * consecutive pairs); there is no incremental traversal, blocking or fusion.  All floating point is
 * fp64 except where a float32 decision must match the CUDA path bit for bit (mask, keys, regions).
 *
 * Pins (tests/test_oracle_pins.py): P1 sigma; P2 uniform-box line integral = analytic chord;
 * P3 axis-aligned / diagonal chords; P4 TOF weights sum to erf(3/sqrt 2); P5 closed-form weights;
 * P6 sigma->inf reduces to non-TOF; P7 sum(x*sens)=n_valid; P8 one-voxel MLEM; P9 brute-force
 * quadrature on 8^3; P10 adjointness; P11 region partition 200+8x100; P12 hand-built keys;
 * P17 the float32 mask rule (orc_mask_f32) on a hand-written array with the expected bytes typed in.
 * Unpinned: the image after N iterations on realistic data has no independent pin beyond
 * P7/P8/P10 ("parity unpinned" for image values on realistic data is NOT claimed pinned);
 * split-vs-unsplit agreement is parity unpinned (PAPER.md:212 is visual only).
 *
 *
 * Widened rows (added after the hot path):
 *   - NEXT-1, the paper's own K-sample TOF kernel (Fig. 3): K equally spaced samples inside
 *     the truncated Gaussian, Gaussian weights normalised to sum to one, each sample filled into the voxel
 *     that contains it ("direct technique for voxel filling") -- orc_sample_lut, orc_*_k.
 *     Pins P13: weights sum to 1 / symmetric / printed K = 15, 32; uniform image -> fwd = 1; K -> inf
 *     converges to the Siddon-TOF forward value / erf(T/sqrt 2).
 *   - NEXT-2, the median filter applied to the image estimate after each iteration (size
 *     unstated -> R23: 3x3x3, edges replicated) -- orc_median3.  Pin P14: scipy.ndimage.median_filter.
 *   - NEXT-3, attenuation correction as a per-event weight (PAPER.md:93 -> R19: w_e = 1 / P(both photons
 *     survive) = exp(+ line integral of mu along the LOR), multiplying the backprojected ratio)
 *     -- orc_attenuation_weights, the `evw` argument of orc_em_correction_w.  Pins P15.
 *   - NEXT-4, TOF-based scatter rejection: an event is kept iff the 95 % confidence
 *     interval of its TOF-estimated annihilation point (+-1.96 sigma along the LOR) meets the body outline,
 *     here a union of ellipsoids; float32 specification F2 -- orc_scatter_keep.  Pins P16.
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -fPIC -shared (no -ffast-math).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int32_t nx, ny, nz;
    double vx, vy, vz; /* voxel size, mm */
    double ox, oy, oz; /* mm coordinate of the low corner of voxel (0,0,0) */
} orc_grid;

typedef struct {
    const float *x1, *y1, *z1, *x2, *y2, *z2, *dt; /* SoA; dt (ps) may be NULL for non-TOF */
} orc_events;

typedef struct {
    uint64_t n_valid, n_skipped, visits;
    double sum_image_sens;
} orc_stats;

#define ORC_C_MM_PER_PS 0.299792458

/* FWHM (ps) of the coincidence time difference -> sigma (mm) along the LOR.
 * The factor 1/2: a time difference dt moves the annihilation point by c*dt/2. */
double orc_sigma_mm(double fwhm_ps, double c_mm_per_ps) {
    return c_mm_per_ps * fwhm_ps / (2.0 * 2.0 * sqrt(2.0 * log(2.0)));
}

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

static int cmp_double(const void *a, const void *b) {
    double x = *(const double *)a, y = *(const double *)b;
    return (x > y) - (x < y);
}

/* Capacity needed for the per-LOR scratch arrays. */
int orc_lor_capacity(const orc_grid *g) { return g->nx + g->ny + g->nz + 16; }

/*
 * System-matrix row of one LOR (steps 1-4 of DESIGN.md "Oracle algorithm").
 *   sigma_mm > 0 : TOF weights  a_j = l_j * exp(-(s_m - s_c)^2 / (2 sigma^2)) / (sigma sqrt(2 pi))
 *   sigma_mm <= 0: non-TOF      a_j = l_j  over the whole chord inside the grid
 * p1,p2 in mm, dt_ps = t1 - t2 (positive => annihilation nearer endpoint 2, R22).
 * scratch: cap doubles.  idx/w: cap entries.  Returns the number of (voxel, weight) pairs,
 * 0 if the LOR is skipped or misses, -1 if cap is too small.
 */
int orc_lor_weights(const orc_grid *g, double sigma_mm, double trunc_sigmas, const double p1[3],
                    const double p2[3], double dt_ps, int64_t *idx, double *w, double *scratch, int cap) {
    const int n[3] = {g->nx, g->ny, g->nz};
    const double v[3] = {g->vx, g->vy, g->vz};
    const double o[3] = {g->ox, g->oy, g->oz};
    double d[3], u[3];
    int a;
    for (a = 0; a < 3; ++a) {
        if (!isfinite(p1[a]) || !isfinite(p2[a])) return 0;
        d[a] = p2[a] - p1[a];
    }
    if (sigma_mm > 0.0 && !isfinite(dt_ps)) return 0;
    const double L = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    if (!(L > 0.0)) return 0;
    for (a = 0; a < 3; ++a) u[a] = d[a] / L;

    /* step 3: slab method against the grid box -> [s_in, s_out] */
    double s_in = -INFINITY, s_out = INFINITY;
    for (a = 0; a < 3; ++a) {
        const double lo = o[a], hi = o[a] + n[a] * v[a];
        if (u[a] == 0.0) {
            if (p1[a] < lo || p1[a] >= hi) return 0; /* parallel and outside */
        } else {
            double t0 = (lo - p1[a]) / u[a], t1 = (hi - p1[a]) / u[a];
            if (t0 > t1) { double t = t0; t0 = t1; t1 = t; }
            if (t0 > s_in) s_in = t0;
            if (t1 < s_out) s_out = t1;
        }
    }
    double s_lo = s_in > 0.0 ? s_in : 0.0;
    double s_hi = s_out < L ? s_out : L;
    double s_c = 0.0;
    if (sigma_mm > 0.0) {
        /* step 2: kernel centre on the measured time difference */
        s_c = 0.5 * L + 0.5 * ORC_C_MM_PER_PS * dt_ps;
        const double hw = trunc_sigmas * sigma_mm;
        if (s_c - hw > s_lo) s_lo = s_c - hw;
        if (s_c + hw < s_hi) s_hi = s_c + hw;
    }
    if (!(s_hi > s_lo)) return 0;

    /* step 4: every plane crossing strictly inside the window, plus the window ends */
    int m = 0;
    scratch[m++] = s_lo;
    scratch[m++] = s_hi;
    for (a = 0; a < 3; ++a) {
        if (u[a] == 0.0) continue;
        /* conservative plane index range touched by the window, then the exact filter */
        const double qa = (p1[a] + u[a] * s_lo - o[a]) / v[a];
        const double qb = (p1[a] + u[a] * s_hi - o[a]) / v[a];
        long k0 = (long)floor(qa < qb ? qa : qb) - 1;
        long k1 = (long)ceil(qa < qb ? qb : qa) + 1;
        if (k0 < 0) k0 = 0;
        if (k1 > n[a]) k1 = n[a];
        for (long k = k0; k <= k1; ++k) {
            const double s = (o[a] + (double)k * v[a] - p1[a]) / u[a];
            if (s > s_lo && s < s_hi) {
                if (m >= cap) return -1;
                scratch[m++] = s;
            }
        }
    }
    qsort(scratch, (size_t)m, sizeof(double), cmp_double);

    const double inv_norm = sigma_mm > 0.0 ? 1.0 / (sigma_mm * sqrt(2.0 * M_PI)) : 1.0;
    int cnt = 0;
    for (int i = 0; i + 1 < m; ++i) {
        const double sa = scratch[i], sb = scratch[i + 1];
        const double len = sb - sa;
        if (!(len > 0.0)) continue;
        const double sm = 0.5 * (sa + sb);
        int64_t ijk[3];
        int inside = 1;
        for (a = 0; a < 3; ++a) {
            ijk[a] = (int64_t)floor((p1[a] + u[a] * sm - o[a]) / v[a]);
            if (ijk[a] < 0 || ijk[a] >= n[a]) inside = 0;
        }
        if (!inside) continue;
        double wt = len;
        if (sigma_mm > 0.0) {
            const double r = (sm - s_c) / sigma_mm;
            wt = len * exp(-0.5 * r * r) * inv_norm;
        }
        if (cnt >= cap) return -1;
        idx[cnt] = (ijk[2] * g->ny + ijk[1]) * (int64_t)g->nx + ijk[0];
        w[cnt] = wt;
        ++cnt;
    }
    return cnt;
}

/* ------------------------------------------------------------------------------------------
 * NEXT-1: the paper's K-sample TOF kernel (Fig. 3 :83; SURVEY.md 8(c) "variant V").
 * offset_k = -T sigma + k * 2 T sigma / (K - 1), k = 0..K-1  ("equally spaced inside the ... Gaussian");
 * weight_k = exp(-offset_k^2 / 2 sigma^2) / sum_m exp(-offset_m^2 / 2 sigma^2)  ("the sum of the weights
 * equaled one").  K = 1 degenerates to one sample at the centre with weight 1.
 * ------------------------------------------------------------------------------------------ */
void orc_sample_lut(int K, double sigma_mm, double trunc_sigmas, double *offset, double *weight) {
    double sum = 0.0;
    for (int k = 0; k < K; ++k) {
        offset[k] = K > 1 ? -trunc_sigmas * sigma_mm + (double)k * (2.0 * trunc_sigmas * sigma_mm) / (double)(K - 1) : 0.0;
        const double r = offset[k] / sigma_mm;
        weight[k] = exp(-0.5 * r * r);
        sum += weight[k];
    }
    for (int k = 0; k < K; ++k) weight[k] /= sum;
}

/* Row of one event under the K-sample kernel: sample k sits at s_k = s_c + offset_k on the LOR
 * ("centered in the coincidence time difference") and is filled into the voxel that contains
 * it; samples beyond the LOR's end points or outside the grid are dropped (R8).  Returns the number of
 * (voxel, weight) pairs kept (<= K); the same voxel may appear more than once. */
int orc_lor_samples(const orc_grid *g, int K, const double *offset, const double *weight, const double p1[3],
                    const double p2[3], double dt_ps, int64_t *idx, double *w) {
    const int n[3] = {g->nx, g->ny, g->nz};
    const double v[3] = {g->vx, g->vy, g->vz};
    const double o[3] = {g->ox, g->oy, g->oz};
    double d[3], u[3];
    int a;
    for (a = 0; a < 3; ++a) {
        if (!isfinite(p1[a]) || !isfinite(p2[a])) return 0;
        d[a] = p2[a] - p1[a];
    }
    if (!isfinite(dt_ps)) return 0;
    const double L = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    if (!(L > 0.0)) return 0;
    for (a = 0; a < 3; ++a) u[a] = d[a] / L;
    const double s_c = 0.5 * L + 0.5 * ORC_C_MM_PER_PS * dt_ps;
    int cnt = 0;
    for (int k = 0; k < K; ++k) {
        const double s = s_c + offset[k];
        if (s < 0.0 || s > L) continue;
        int64_t ijk[3];
        int inside = 1;
        for (a = 0; a < 3; ++a) {
            ijk[a] = (int64_t)floor((p1[a] + u[a] * s - o[a]) / v[a]);
            if (ijk[a] < 0 || ijk[a] >= n[a]) inside = 0;
        }
        if (!inside) continue;
        idx[cnt] = (ijk[2] * g->ny + ijk[1]) * (int64_t)g->nx + ijk[0];
        w[cnt] = weight[k];
        ++cnt;
    }
    return cnt;
}

typedef struct {
    int64_t *idx;
    double *w, *scratch;
    int cap;
} lor_buf;

static void lor_buf_init(lor_buf *b, const orc_grid *g) {
    b->cap = orc_lor_capacity(g);
    b->idx = (int64_t *)malloc(sizeof(int64_t) * (size_t)b->cap);
    b->w = (double *)malloc(sizeof(double) * (size_t)b->cap);
    b->scratch = (double *)malloc(sizeof(double) * (size_t)b->cap);
}
static void lor_buf_free(lor_buf *b) {
    free(b->idx);
    free(b->w);
    free(b->scratch);
}

/* Which system-matrix row an entry point uses: K = 0 -> Siddon chords x Gaussian at the chord midpoints (the graded
 * projector, R2); K >= 1 -> the paper's K-sample kernel (NEXT-1). */
typedef struct {
    int K;
    double *offset, *weight;
} row_model;

static void row_model_init(row_model *rm, int K, double sigma_mm, double trunc) {
    rm->K = K;
    rm->offset = rm->weight = NULL;
    if (K > 0) {
        rm->offset = (double *)malloc(sizeof(double) * (size_t)K);
        rm->weight = (double *)malloc(sizeof(double) * (size_t)K);
        orc_sample_lut(K, sigma_mm, trunc, rm->offset, rm->weight);
    }
}
static void row_model_free(row_model *rm) {
    free(rm->offset);
    free(rm->weight);
}

static void lor_buf_init_k(lor_buf *b, const orc_grid *g, int K) {
    lor_buf_init(b, g);
    if (K > b->cap) {
        lor_buf_free(b);
        b->cap = K;
        b->idx = (int64_t *)malloc(sizeof(int64_t) * (size_t)K);
        b->w = (double *)malloc(sizeof(double) * (size_t)K);
        b->scratch = (double *)malloc(sizeof(double) * (size_t)K);
    }
}

static int event_row(const orc_grid *g, double sigma_mm, double trunc, const row_model *rm, const orc_events *ev,
                     uint64_t e, lor_buf *b) {
    const double p1[3] = {ev->x1[e], ev->y1[e], ev->z1[e]};
    const double p2[3] = {ev->x2[e], ev->y2[e], ev->z2[e]};
    const double dt = (sigma_mm > 0.0 && ev->dt) ? (double)ev->dt[e] : 0.0;
    if (rm->K > 0) return orc_lor_samples(g, rm->K, rm->offset, rm->weight, p1, p2, dt, b->idx, b->w);
    return orc_lor_weights(g, sigma_mm, trunc, p1, p2, dt, b->idx, b->w, b->scratch, b->cap);
}

/* step 5: fwd_e = sum_j a_ej x_j */
void orc_forward_k(const orc_grid *g, double sigma_mm, double trunc, int K, const orc_events *ev, uint64_t n,
                   const double *image, double *fwd) {
    row_model rm;
    row_model_init(&rm, K, sigma_mm, trunc);
#pragma omp parallel
    {
        lor_buf b;
        lor_buf_init_k(&b, g, K);
#pragma omp for schedule(dynamic, 1024)
        for (int64_t e = 0; e < (int64_t)n; ++e) {
            const int cnt = event_row(g, sigma_mm, trunc, &rm, ev, (uint64_t)e, &b);
            double acc = 0.0;
            for (int k = 0; k < cnt; ++k) acc += b.w[k] * image[b.idx[k]];
            fwd[e] = acc;
        }
        lor_buf_free(&b);
    }
    row_model_free(&rm);
}
void orc_forward(const orc_grid *g, double sigma_mm, double trunc, const orc_events *ev, uint64_t n,
                 const double *image, double *fwd) {
    orc_forward_k(g, sigma_mm, trunc, 0, ev, n, image, fwd);
}

/* step 5: out_j += a_ej * val_e   (values == NULL => 1) */
void orc_backproject_k(const orc_grid *g, double sigma_mm, double trunc, int K, const orc_events *ev, uint64_t n,
                       const double *values, double *out) {
    const int64_t nvox = (int64_t)g->nx * g->ny * g->nz;
    row_model rm;
    row_model_init(&rm, K, sigma_mm, trunc);
#pragma omp parallel
    {
        lor_buf b;
        lor_buf_init_k(&b, g, K);
        double *priv = (double *)calloc((size_t)nvox, sizeof(double));
#pragma omp for schedule(dynamic, 1024)
        for (int64_t e = 0; e < (int64_t)n; ++e) {
            const int cnt = event_row(g, sigma_mm, trunc, &rm, ev, (uint64_t)e, &b);
            const double val = values ? values[e] : 1.0;
            for (int k = 0; k < cnt; ++k) priv[b.idx[k]] += b.w[k] * val;
        }
#pragma omp critical
        for (int64_t j = 0; j < nvox; ++j) out[j] += priv[j];
        free(priv);
        lor_buf_free(&b);
    }
    row_model_free(&rm);
}
void orc_backproject(const orc_grid *g, double sigma_mm, double trunc, const orc_events *ev, uint64_t n,
                     const double *values, double *out) {
    orc_backproject_k(g, sigma_mm, trunc, 0, ev, n, values, out);
}

/* step 7: sens_j = (1/m) sum_i l_ij over the m given LORs (non-TOF chords), R10 */
void orc_sensitivity(const orc_grid *g, const orc_events *lors, uint64_t m, double *sens) {
    const int64_t nvox = (int64_t)g->nx * g->ny * g->nz;
    memset(sens, 0, sizeof(double) * (size_t)nvox);
    orc_backproject(g, 0.0, 0.0, lors, m, NULL, sens);
    for (int64_t j = 0; j < nvox; ++j) sens[j] /= (double)m;
}

/* R11: mask_j = sens_j >= floor_rel * max_k sens_k, decided in float32 (the CUDA path's precision,
 * so the integer decision is taken identically on both sides). */
void orc_mask_f32(const float *sens, int64_t nvox, float floor_rel, uint8_t *mask) {
    float mx = 0.0f;
    for (int64_t j = 0; j < nvox; ++j)
        if (sens[j] > mx) mx = sens[j];
    const float thr = floor_rel * mx;
    for (int64_t j = 0; j < nvox; ++j) mask[j] = (sens[j] >= thr && sens[j] > 0.0f) ? 1 : 0;
}

/* EM correction image of one pass (step 6, first half): corr_j = sum_{e: fwd_e>0} evw_e * a_ej / fwd_e.
 * evw (optional, NULL => 1) is the per-event weight of NEXT-3 (R19).  corr is overwritten.
 * Returns n_valid; *visits (optional) counts voxel visits; *sum_w (optional) = sum of evw over the valid events. */
uint64_t orc_em_correction_w(const orc_grid *g, double sigma_mm, double trunc, int K, const orc_events *ev, uint64_t n,
                             const double *evw, const double *image, double *corr, uint64_t *visits, double *sum_w) {
    const int64_t nvox = (int64_t)g->nx * g->ny * g->nz;
    uint64_t n_valid = 0, vis = 0;
    double sw = 0.0;
    row_model rm;
    row_model_init(&rm, K, sigma_mm, trunc);
    memset(corr, 0, sizeof(double) * (size_t)nvox);
#pragma omp parallel reduction(+ : n_valid, vis, sw)
    {
        lor_buf b;
        lor_buf_init_k(&b, g, K);
        double *priv = (double *)calloc((size_t)nvox, sizeof(double));
#pragma omp for schedule(dynamic, 1024)
        for (int64_t e = 0; e < (int64_t)n; ++e) {
            const int cnt = event_row(g, sigma_mm, trunc, &rm, ev, (uint64_t)e, &b);
            double fwd = 0.0;
            for (int k = 0; k < cnt; ++k) fwd += b.w[k] * image[b.idx[k]];
            vis += (uint64_t)(cnt > 0 ? cnt : 0);
            if (fwd > 0.0) { /* R9 */
                const double we = evw ? evw[e] : 1.0;
                const double r = we / fwd;
                for (int k = 0; k < cnt; ++k) priv[b.idx[k]] += b.w[k] * r;
                ++n_valid;
                sw += we;
            }
        }
#pragma omp critical
        for (int64_t j = 0; j < nvox; ++j) corr[j] += priv[j];
        free(priv);
        lor_buf_free(&b);
    }
    row_model_free(&rm);
    if (visits) *visits = vis;
    if (sum_w) *sum_w = sw;
    return n_valid;
}
uint64_t orc_em_correction(const orc_grid *g, double sigma_mm, double trunc, const orc_events *ev, uint64_t n,
                           const double *image, double *corr, uint64_t *visits) {
    return orc_em_correction_w(g, sigma_mm, trunc, 0, ev, n, NULL, image, corr, visits, NULL);
}

/* step 6, second half: x_j <- mask_j ? x_j * corr_j / sens_j : 0 */
void orc_update(int64_t nvox, double *image, const double *corr, const float *sens, const uint8_t *mask) {
    for (int64_t j = 0; j < nvox; ++j) image[j] = mask[j] ? image[j] * corr[j] / (double)sens[j] : 0.0;
}

/* NEXT-2: 3x3x3 median filter ("we introduced a median filter between MLEM iterations"; the size is
 * not stated -> R23: the 27-voxel cube, edges replicated, i.e. neighbour indices are clamped to the volume).
 * out_j = the 14th smallest of the 27 values.  in and out must not alias. */
void orc_median3(int32_t nx, int32_t ny, int32_t nz, const double *in, double *out) {
#pragma omp parallel for schedule(static)
    for (int64_t z = 0; z < nz; ++z)
        for (int64_t y = 0; y < ny; ++y)
            for (int64_t x = 0; x < nx; ++x) {
                double v[27];
                int m = 0;
                for (int dz = -1; dz <= 1; ++dz)
                    for (int dy = -1; dy <= 1; ++dy)
                        for (int dx = -1; dx <= 1; ++dx) {
                            int64_t xx = x + dx, yy = y + dy, zz = z + dz;
                            xx = xx < 0 ? 0 : (xx >= nx ? nx - 1 : xx);
                            yy = yy < 0 ? 0 : (yy >= ny ? ny - 1 : yy);
                            zz = zz < 0 ? 0 : (zz >= nz ? nz - 1 : zz);
                            v[m++] = in[(zz * ny + yy) * nx + xx];
                        }
                qsort(v, 27, sizeof(double), cmp_double);
                out[(z * ny + y) * nx + x] = v[13];
            }
}

/* `iters` MLEM iterations in fp64 (R1). image: in x0, out x_iters.  sens is the float32 buffer
 * that is also given to the CUDA path (R11).  K: row model; evw: optional per-event weights (NEXT-3);
 * median != 0: the 3x3x3 median filter is applied to the image estimate after every iteration
 * ("applied to the image estimate after each iteration", R23). */
void orc_mlem_x(const orc_grid *g, double sigma_mm, double trunc, int K, const orc_events *ev, uint64_t n,
                const double *evw, double *image, const float *sens, int iters, float sens_floor_rel, int median,
                orc_stats *stats) {
    const int64_t nvox = (int64_t)g->nx * g->ny * g->nz;
    uint8_t *mask = (uint8_t *)malloc((size_t)nvox);
    double *corr = (double *)malloc(sizeof(double) * (size_t)nvox);
    double *tmp = median ? (double *)malloc(sizeof(double) * (size_t)nvox) : NULL;
    orc_mask_f32(sens, nvox, sens_floor_rel, mask);
    uint64_t n_valid = 0, visits = 0;
    for (int it = 0; it < iters; ++it) {
        n_valid = orc_em_correction_w(g, sigma_mm, trunc, K, ev, n, evw, image, corr, &visits, NULL);
        orc_update(nvox, image, corr, sens, mask);
        if (median) {
            orc_median3(g->nx, g->ny, g->nz, image, tmp);
            memcpy(image, tmp, sizeof(double) * (size_t)nvox);
        }
    }
    if (stats) {
        double s = 0.0;
        for (int64_t j = 0; j < nvox; ++j) s += image[j] * (double)sens[j];
        stats->n_valid = n_valid;
        stats->n_skipped = n - n_valid;
        stats->visits = visits;
        stats->sum_image_sens = s;
    }
    free(mask);
    free(corr);
    free(tmp);
}
void orc_mlem(const orc_grid *g, double sigma_mm, double trunc, const orc_events *ev, uint64_t n, double *image,
              const float *sens, int iters, float sens_floor_rel, orc_stats *stats) {
    orc_mlem_x(g, sigma_mm, trunc, 0, ev, n, NULL, image, sens, iters, sens_floor_rel, 0, stats);
}

/* NEXT-3 (R19): per-event attenuation weight w_e = 1 / P(both photons reach the detectors)
 * = exp(+ sum_j l_ej mu_j), the non-TOF Siddon line integral of the attenuation map mu (1/mm, on the
 * reconstruction grid) over the LOR's whole chord inside the grid.  Skipped LORs get weight 1. */
void orc_attenuation_weights(const orc_grid *g, const orc_events *ev, uint64_t n, const double *mu, double *w) {
    orc_events lor = *ev;
    lor.dt = NULL;
    orc_forward_k(g, 0.0, 0.0, 0, &lor, n, mu, w);
    for (uint64_t e = 0; e < n; ++e) w[e] = exp(w[e]);
}

/* ------------------------------------------------------------------------------------------
 * Integer-valued parts, float32 arithmetic specification F1: every operation below is
 * a single IEEE binary32 operation, round-to-nearest-even, in exactly this order, no FMA
 * contraction (compile with -ffp-contract=off).
 * ------------------------------------------------------------------------------------------ */
#define ORC_HALF_C_F32 0.149896229f /* c/2 in mm/ps */

typedef struct {
    int32_t nx, ny, nz;
    float vx, vy, vz, ox, oy, oz;
} orc_grid_f32;

/* TOF-estimated annihilation point (kernel centre), float32.  Returns 0 for an invalid event. */
static int tof_centre_f32(const orc_events *ev, uint64_t e, float c[3], float d[3]) {
    const float x1 = ev->x1[e], y1 = ev->y1[e], z1 = ev->z1[e];
    const float x2 = ev->x2[e], y2 = ev->y2[e], z2 = ev->z2[e];
    const float dt = ev->dt ? ev->dt[e] : 0.0f;
    if (!isfinite(x1) || !isfinite(y1) || !isfinite(z1) || !isfinite(x2) || !isfinite(y2) || !isfinite(z2) ||
        !isfinite(dt))
        return 0;
    const float dx = x2 - x1, dy = y2 - y1, dz = z2 - z1;
    const float xx = dx * dx, yy = dy * dy, zz = dz * dz;
    const float sxy = xx + yy;
    const float L2 = sxy + zz;
    if (!(L2 > 0.0f) || !isfinite(L2)) return 0;
    const float L = sqrtf(L2);
    const float h = ORC_HALF_C_F32 * dt;
    const float q = h / L;
    const float mx = 0.5f * (x1 + x2), my = 0.5f * (y1 + y2), mz = 0.5f * (z1 + z2);
    const float qx = q * dx, qy = q * dy, qz = q * dz;
    c[0] = mx + qx;
    c[1] = my + qy;
    c[2] = mz + qz;
    d[0] = dx;
    d[1] = dy;
    d[2] = dz;
    return 1;
}

static int32_t centre_voxel_f32(float c, float o, float v, int32_t n) {
    const float t = c - o;
    const float q = t / v;
    const float f = floorf(q);
    if (!(f >= 0.0f)) return 0; /* also catches NaN */
    if (f >= (float)n) return n - 1;
    return (int32_t)f;
}

uint32_t orc_num_bins(const orc_grid_f32 *g, int tile_log2) {
    const int32_t t = 1 << tile_log2;
    const uint32_t Tx = (uint32_t)((g->nx + t - 1) >> tile_log2), Ty = (uint32_t)((g->ny + t - 1) >> tile_log2),
                   Tz = (uint32_t)((g->nz + t - 1) >> tile_log2);
    return 12u * Tx * Ty * Tz;
}

/* key = dirclass * (Tx*Ty*Tz) + tile; invalid events get 0xFFFFFFFF. */
void orc_bin_keys(const orc_grid_f32 *g, const orc_events *ev, uint64_t n, int tile_log2, uint32_t *key) {
    const int32_t t = 1 << tile_log2;
    const uint32_t Tx = (uint32_t)((g->nx + t - 1) >> tile_log2), Ty = (uint32_t)((g->ny + t - 1) >> tile_log2),
                   Tz = (uint32_t)((g->nz + t - 1) >> tile_log2);
    for (uint64_t e = 0; e < n; ++e) {
        float c[3], d[3];
        if (!tof_centre_f32(ev, e, c, d)) {
            key[e] = 0xFFFFFFFFu;
            continue;
        }
        const int32_t ix = centre_voxel_f32(c[0], g->ox, g->vx, g->nx);
        const int32_t iy = centre_voxel_f32(c[1], g->oy, g->vy, g->ny);
        const int32_t iz = centre_voxel_f32(c[2], g->oz, g->vz, g->nz);
        const uint32_t tile =
            (((uint32_t)(iz >> tile_log2)) * Ty + (uint32_t)(iy >> tile_log2)) * Tx + (uint32_t)(ix >> tile_log2);
        int a = 0;
        float best = fabsf(d[0]);
        if (fabsf(d[1]) > best) { a = 1; best = fabsf(d[1]); }
        if (fabsf(d[2]) > best) { a = 2; }
        const float sgn = d[a] < 0.0f ? -1.0f : 1.0f;
        const float db = sgn * d[(a + 1) % 3], dc = sgn * d[(a + 2) % 3];
        const uint32_t dirclass = 4u * (uint32_t)a + 2u * (db < 0.0f ? 1u : 0u) + (dc < 0.0f ? 1u : 0u);
        key[e] = dirclass * (Tx * Ty * Tz) + tile;
    }
}

/* Default region boundaries in slices: first region double width, R regions in all
 * (200 + 8 x 100 of 1000 slices). k[j] = nz * {0,2,3,...,R+1} / (R+1), integer division. */
void orc_default_region_slices(int32_t nz, int n_regions, int32_t *k /* n_regions+1 */) {
    k[0] = 0;
    for (int j = 1; j <= n_regions; ++j) k[j] = (int32_t)(((int64_t)nz * (j + 1)) / (n_regions + 1));
}

/* zb[j] = (float)k_j * vz + oz (multiply, then add), float32. */
void orc_region_zbounds(const orc_grid_f32 *g, int n_regions, float *zb /* n_regions+1 */) {
    int32_t *k = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n_regions + 1));
    orc_default_region_slices(g->nz, n_regions, k);
    for (int j = 0; j <= n_regions; ++j) {
        const float kv = (float)k[j] * g->vz;
        zb[j] = kv + g->oz;
    }
    free(k);
}

/* region_e = #{ j in 1..R-1 : zb[j] <= cz_e } (R13: single assignment by the kernel centre's z);
 * invalid events get -1.  counts[R] receives the per-region totals. */
void orc_region_ids(const orc_events *ev, uint64_t n, int n_regions, const float *zb, int32_t *region,
                    uint64_t *counts) {
    for (int r = 0; r < n_regions; ++r) counts[r] = 0;
    for (uint64_t e = 0; e < n; ++e) {
        float c[3], d[3];
        if (!tof_centre_f32(ev, e, c, d)) {
            region[e] = -1;
            continue;
        }
        int32_t r = 0;
        for (int j = 1; j < n_regions; ++j)
            if (zb[j] <= c[2]) ++r;
        region[e] = r;
        ++counts[r];
    }
}

/* Reading R27 (an event "always contributed to 1 or 2 image regions", e.g. "a 40% probability ... within
 * image 5, and a 60% probability ... image region number 6"): the event belongs to EVERY region whose core the axial
 * extent of its +-T sigma window meets.  Integer result -> float32 specification F3 (conventions of F1):
 *   c, (dx,dy,dz), L as in F1;  q = hw / L;  hz = q * |dz|;  zlo = cz - hz;  zhi = cz + hz;
 *   lo = #{ j in 1..R-1 : zb[j] <= zlo },  hi = #{ j in 1..R-1 : zb[j] <= zhi };  regions lo..hi.
 * hw = (float)(trunc * sigma).  Invalid events: lo = hi = -1.  counts[r] = events whose span contains r. */
void orc_region_spans(const orc_events *ev, uint64_t n, int n_regions, const float *zb, float hw, int32_t *lo,
                      int32_t *hi, uint64_t *counts) {
    for (int r = 0; r < n_regions; ++r) counts[r] = 0;
    for (uint64_t e = 0; e < n; ++e) {
        float c[3], d[3];
        if (!tof_centre_f32(ev, e, c, d)) {
            lo[e] = hi[e] = -1;
            continue;
        }
        const float xx = d[0] * d[0], yy = d[1] * d[1], zz = d[2] * d[2];
        const float sxy = xx + yy;
        const float L2 = sxy + zz;
        const float L = sqrtf(L2);
        const float q = hw / L;
        const float hz = q * fabsf(d[2]);
        const float zlo = c[2] - hz, zhi = c[2] + hz;
        int32_t a = 0, b = 0;
        for (int j = 1; j < n_regions; ++j) {
            if (zb[j] <= zlo) ++a;
            if (zb[j] <= zhi) ++b;
        }
        lo[e] = a;
        hi[e] = b;
        for (int r = a; r <= b; ++r) ++counts[r];
    }
}

/* R12: margin in slices on each open side of a region core: ceil((trunc*sigma + shell_mm)/vz). */
int32_t orc_region_margin_slices(double sigma_mm, double trunc, double shell_mm, double vz) {
    return (int32_t)ceil((trunc * sigma_mm + shell_mm) / vz);
}

/* ------------------------------------------------------------------------------------------
 * NEXT-4: TOF-based scatter rejection (PAPER.md:63 Fig. 2, :69-71).  "The annihilation point determined
 * along the scatter LOR had a certain probability of being inside the human body, according to the TOF
 * resolution.  The limits of rejection were estimated at a 95% confidence level.  The body outline was
 * determined from knowledge of the NCAT outline" -> reading R24: the event is KEPT iff the segment
 * { c + u t : |t| <= h }, h = 1.959964 sigma (two-sided 95 % of the TOF Gaussian), c = TOF-estimated
 * annihilation point, u = LOR direction, meets the body outline; the outline is a union of ellipsoids
 * (the NCAT outline is not available; a measured one would be a CT mask).  Integer result -> float32
 * specification F2, same conventions as F1 (single RN operations in this order, no contraction):
 *   c, (dx,dy,dz), L as in F1;  ux = dx / L, uy = dy / L, uz = dz / L;
 *   per ellipsoid (centre e, reciprocal semi-axes i, both float32 from the caller):
 *     rx = (cx - ex) * ix ...;  wx = ux * ix ...;
 *     A = (wx*wx + wy*wy) + wz*wz;  B = (rx*wx + ry*wy) + rz*wz;
 *     t = -(B / A);  t = fminf(fmaxf(t, -h), h);          (point of the segment closest to the centre in the
 *     px = rx + wx * t ...;                                  ellipsoid's unit-sphere coordinates)
 *     Q = (px*px + py*py) + pz*pz;  hit iff Q <= 1.
 *   keep = hit for any ellipsoid; invalid events (F1) are not kept.
 * ------------------------------------------------------------------------------------------ */
void orc_scatter_keep(const orc_events *ev, uint64_t n, const float *ell /* n_ell x {cx,cy,cz,1/ax,1/ay,1/az} */,
                      int n_ell, float h, uint8_t *keep, uint64_t *n_kept) {
    uint64_t kept = 0;
    const float mh = -h;
    for (uint64_t e = 0; e < n; ++e) {
        float c[3], d[3];
        keep[e] = 0;
        if (!tof_centre_f32(ev, e, c, d)) continue;
        const float xx = d[0] * d[0], yy = d[1] * d[1], zz = d[2] * d[2];
        const float sxy = xx + yy;
        const float L = sqrtf(sxy + zz);
        const float ux = d[0] / L, uy = d[1] / L, uz = d[2] / L;
        uint8_t hit = 0;
        for (int k = 0; k < n_ell && !hit; ++k) {
            const float *q = ell + 6 * k;
            const float tx = c[0] - q[0], ty = c[1] - q[1], tz = c[2] - q[2];
            const float rx = tx * q[3], ry = ty * q[4], rz = tz * q[5];
            const float wx = ux * q[3], wy = uy * q[4], wz = uz * q[5];
            const float a0 = wx * wx, a1 = wy * wy, a2 = wz * wz;
            const float a01 = a0 + a1;
            const float A = a01 + a2;
            const float b0 = rx * wx, b1 = ry * wy, b2 = rz * wz;
            const float b01 = b0 + b1;
            const float B = b01 + b2;
            const float t0 = B / A;
            float t = -t0;
            t = fminf(fmaxf(t, mh), h);
            const float mx = wx * t, my = wy * t, mz = wz * t;
            const float px = rx + mx, py = ry + my, pz = rz + mz;
            const float q0 = px * px, q1 = py * py, q2 = pz * pz;
            const float q01 = q0 + q1;
            const float Q = q01 + q2;
            if (Q <= 1.0f) hit = 1;
        }
        keep[e] = hit;
        kept += hit;
    }
    if (n_kept) *n_kept = kept;
}
