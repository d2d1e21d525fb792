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
 * quadrature on 8^3; P10 adjointness; P11 region partition 200+8x100; P12 hand-built keys.
 * Unpinned: the image after N iterations on realistic data has no independent pin beyond
 * P7/P8/P10 ("parity unpinned" for image values on realistic data is NOT claimed pinned);
 * split-vs-unsplit agreement is parity unpinned (PAPER.md:212 is visual only).
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

static int event_row(const orc_grid *g, double sigma_mm, double trunc, const orc_events *ev, uint64_t e, lor_buf *b) {
    const double p1[3] = {ev->x1[e], ev->y1[e], ev->z1[e]};
    const double p2[3] = {ev->x2[e], ev->y2[e], ev->z2[e]};
    const double dt = (sigma_mm > 0.0 && ev->dt) ? (double)ev->dt[e] : 0.0;
    return orc_lor_weights(g, sigma_mm, trunc, p1, p2, dt, b->idx, b->w, b->scratch, b->cap);
}

/* step 5: fwd_e = sum_j a_ej x_j */
void orc_forward(const orc_grid *g, double sigma_mm, double trunc, const orc_events *ev, uint64_t n,
                 const double *image, double *fwd) {
#pragma omp parallel
    {
        lor_buf b;
        lor_buf_init(&b, g);
#pragma omp for schedule(dynamic, 1024)
        for (int64_t e = 0; e < (int64_t)n; ++e) {
            const int cnt = event_row(g, sigma_mm, trunc, ev, (uint64_t)e, &b);
            double acc = 0.0;
            for (int k = 0; k < cnt; ++k) acc += b.w[k] * image[b.idx[k]];
            fwd[e] = acc;
        }
        lor_buf_free(&b);
    }
}

/* step 5: out_j += a_ej * val_e   (values == NULL => 1) */
void orc_backproject(const orc_grid *g, double sigma_mm, double trunc, const orc_events *ev, uint64_t n,
                     const double *values, double *out) {
    const int64_t nvox = (int64_t)g->nx * g->ny * g->nz;
#pragma omp parallel
    {
        lor_buf b;
        lor_buf_init(&b, g);
        double *priv = (double *)calloc((size_t)nvox, sizeof(double));
#pragma omp for schedule(dynamic, 1024)
        for (int64_t e = 0; e < (int64_t)n; ++e) {
            const int cnt = event_row(g, sigma_mm, trunc, ev, (uint64_t)e, &b);
            const double val = values ? values[e] : 1.0;
            for (int k = 0; k < cnt; ++k) priv[b.idx[k]] += b.w[k] * val;
        }
#pragma omp critical
        for (int64_t j = 0; j < nvox; ++j) out[j] += priv[j];
        free(priv);
        lor_buf_free(&b);
    }
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

/* EM correction image of one pass (step 6, first half): corr_j = sum_{e: fwd_e>0} a_ej / fwd_e.
 * corr is overwritten.  Returns n_valid; *visits (optional) counts voxel visits. */
uint64_t orc_em_correction(const orc_grid *g, double sigma_mm, double trunc, const orc_events *ev, uint64_t n,
                           const double *image, double *corr, uint64_t *visits) {
    const int64_t nvox = (int64_t)g->nx * g->ny * g->nz;
    uint64_t n_valid = 0, vis = 0;
    memset(corr, 0, sizeof(double) * (size_t)nvox);
#pragma omp parallel reduction(+ : n_valid, vis)
    {
        lor_buf b;
        lor_buf_init(&b, g);
        double *priv = (double *)calloc((size_t)nvox, sizeof(double));
#pragma omp for schedule(dynamic, 1024)
        for (int64_t e = 0; e < (int64_t)n; ++e) {
            const int cnt = event_row(g, sigma_mm, trunc, ev, (uint64_t)e, &b);
            double fwd = 0.0;
            for (int k = 0; k < cnt; ++k) fwd += b.w[k] * image[b.idx[k]];
            vis += (uint64_t)(cnt > 0 ? cnt : 0);
            if (fwd > 0.0) { /* R9 */
                const double r = 1.0 / fwd;
                for (int k = 0; k < cnt; ++k) priv[b.idx[k]] += b.w[k] * r;
                ++n_valid;
            }
        }
#pragma omp critical
        for (int64_t j = 0; j < nvox; ++j) corr[j] += priv[j];
        free(priv);
        lor_buf_free(&b);
    }
    if (visits) *visits = vis;
    return n_valid;
}

/* step 6, second half: x_j <- mask_j ? x_j * corr_j / sens_j : 0 */
void orc_update(int64_t nvox, double *image, const double *corr, const float *sens, const uint8_t *mask) {
    for (int64_t j = 0; j < nvox; ++j) image[j] = mask[j] ? image[j] * corr[j] / (double)sens[j] : 0.0;
}

/* `iters` MLEM iterations in fp64 (R1). image: in x0, out x_iters.  sens is the float32 buffer
 * that is also given to the CUDA path (R11). */
void orc_mlem(const orc_grid *g, double sigma_mm, double trunc, const orc_events *ev, uint64_t n, double *image,
              const float *sens, int iters, float sens_floor_rel, orc_stats *stats) {
    const int64_t nvox = (int64_t)g->nx * g->ny * g->nz;
    uint8_t *mask = (uint8_t *)malloc((size_t)nvox);
    double *corr = (double *)malloc(sizeof(double) * (size_t)nvox);
    orc_mask_f32(sens, nvox, sens_floor_rel, mask);
    uint64_t n_valid = 0, visits = 0;
    for (int it = 0; it < iters; ++it) {
        n_valid = orc_em_correction(g, sigma_mm, trunc, ev, n, image, corr, &visits);
        orc_update(nvox, image, corr, sens, mask);
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

/* R12: margin in slices on each open side of a region core: ceil((trunc*sigma + shell_mm)/vz). */
int32_t orc_region_margin_slices(double sigma_mm, double trunc, double shell_mm, double vz) {
    return (int32_t)ceil((trunc * sigma_mm + shell_mm) / vz);
}
