/*
 * tofmlem.h -- C ABI of libtofmlem: list-mode TOF-weighted MLEM hot path on one NVIDIA B200 (sm_100a).
 *
 * Source of every operation: arxiv 1706.07075 ("PAPER.md" = /root/reference/PAPER.md) as read in
 * DESIGN.md (readings R1..R26).  The paper states the problem in prose only (events with a TOF time
 * difference -> image by TOF-weighted list-mode MLEM; nine-region TOF-assisted
 * data division); the call list follows BASELINE.json's north_star.
 *
 * Conventions
 *   - Units: millimetres and picoseconds.  Scanner = cylinder of radius R and axial length A around the
 *     z axis, centred at the origin.  Image layout: flat index = (iz*ny + iy)*nx + ix (x fastest), float32.
 *   - An event is two detection points p1, p2 (mm) and dt = t1 - t2 (ps); dt > 0 puts the annihilation
 *     nearer p2 (the TOF kernel centre is at arc length L/2 + c*dt/2 from p1).
 *     Events are struct-of-arrays float32.
 *   - Pointers named d_* and the members of tofmlem_events are DEVICE pointers, pointers named h_* are
 *     HOST pointers.  All buffers are owned by the caller; the library never frees or reallocates them.
 *     The only library-owned objects are the opaque context and its internal scratch.
 *   - Every call enqueues work on the CUDA stream given at tofmlem_create and returns without
 *     synchronising, unless stated otherwise.  A context must not be used from two host threads at once.
 *   - Return value: TOFMLEM_OK (0) or a negative tofmlem_status.  No exceptions, no exit().
 *     After TOFMLEM_ECUDA the text of the CUDA error is available from tofmlem_last_error().
 *   - System matrix (north_star; R2,R4-R8): a_ej = l_ej * g_sigma(s_mid,ej - s_c,e) with l_ej the
 *     exact (Siddon) chord of LOR e in voxel j clipped to the window [s_c - T sigma, s_c + T sigma] n grid
 *     n [0, L], g the unit-area Gaussian evaluated at the clipped chord's midpoint, T = trunc_sigmas = 3,
 *     sigma = c * FWHM / (2 * 2 sqrt(2 ln 2)).  Non-TOF contexts use a_ej = l_ej.
 *   - Arithmetic: per-event ray set-up in fp64, per-voxel stepping/weights/accumulation in fp32,
 *     accumulation into images with float32 atomics (order not deterministic).  Bin keys and region
 *     ids follow the float32 specification F1 of DESIGN.md and are bit-exact.
 */
#ifndef TOFMLEM_H
#define TOFMLEM_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    TOFMLEM_OK = 0,
    TOFMLEM_EINVAL = -1,       /* NULL / out-of-range argument */
    TOFMLEM_ENOMEM = -2,       /* device or host allocation failed */
    TOFMLEM_ECUDA = -3,        /* a CUDA call failed; see tofmlem_last_error */
    TOFMLEM_ESTATE = -4,       /* call not valid in the context's current state */
    TOFMLEM_EUNSUPPORTED = -5  /* option or mode not available */
} tofmlem_status;

typedef struct tofmlem_ctx tofmlem_ctx; /* opaque, owned by the library */

typedef struct { float radius_mm, axial_length_mm; } tofmlem_scanner;

typedef struct {
    int32_t nx, ny, nz;
    float vx, vy, vz;  /* voxel size, mm */
    float ox, oy, oz;  /* mm coordinate of the low corner of voxel (0,0,0) */
} tofmlem_grid;

/* Struct-of-arrays events (float32, n entries each).  dt may be NULL for LOR-only use
 * (sensitivity LORs, non-TOF contexts); then dt = 0 is assumed. */
typedef struct { const float *x1, *y1, *z1, *x2, *y2, *z2, *dt; } tofmlem_events;
typedef struct { float *x1, *y1, *z1, *x2, *y2, *z2, *dt; } tofmlem_events_mut;

typedef struct {
    uint64_t n_valid;      /* events with forward projection > 0 in the last EM pass (R9) */
    uint64_t n_skipped;    /* n - n_valid of that pass */
    uint64_t visits;       /* voxel visits of the forward walk of that pass */
    double sum_image_sens; /* sum_j image_j * sens_j after the last tofmlem_iterate (= n_valid, P7) */
    uint64_t reductions;   /* reduction instructions (scalar or 16-byte) the scatter walk of that pass sent to the L2
                              atomic units: the unit of the l2_atomic roofline */
    uint64_t tile_events;  /* of n_valid: events accumulated through a shared-memory tile (tofmlem_plan_events) */
    uint64_t tile_oob;     /* TOFMLEM_OPT_TILE_CHECK: tile accesses found out of range; must be 0 */
    uint64_t tile_visits;  /* of visits: voxel visits of the forward walk on shared-memory tiles */
} tofmlem_stats;

/* What tofmlem_plan_events decided (tofmlem_plan_info). */
typedef struct {
    int32_t active;           /* 1: the context holds ray records for the planned list */
    int32_t sorted;           /* 1: the list was found sorted by locality key (0 also when tiles do not fit: not looked at) */
    uint32_t n_tile_items;    /* pieces of locality bins that are accumulated in shared-memory tiles (0: none) */
    uint32_t n_direct_chunks; /* 32-event pieces of the list that hold events of the direct pass on records */
    uint64_t n_tile_events;   /* events that run on a tile */
    uint64_t n_direct_events; /* n - n_tile_events */
    uint64_t n_stragglers;    /* of n_direct_events: valid events of tile items whose window leaves the item's tile */
} tofmlem_plan;

/* Option keys for tofmlem_set_option. */
enum {
    TOFMLEM_OPT_TRUNC_SIGMAS = 1,   /* half-width of the TOF window in sigmas, default 3.0 (R5) */
    TOFMLEM_OPT_SENS_FLOOR_REL = 2, /* mask_j = sens_j >= value * max(sens), default 1e-2 (R11) */
    TOFMLEM_OPT_TILE_LOG2 = 3,      /* locality bins are cubes of 2^value voxels, default 3 */
    TOFMLEM_OPT_PROJECTOR = 4,      /* 0 = Siddon x Gaussian (default); 1 = paper's K-sample LUT */
    TOFMLEM_OPT_SAMPLES_K = 5,      /* K of the sampled projector, default 32 */
    TOFMLEM_OPT_SHELL_MM = 6,       /* extra shell added to the region margin, default 6 mm */
    TOFMLEM_OPT_EM_VARIANT = 8,     /* fused EM pass scheduling (performance only): 0 = persistent kernel with one work
                                       queue per SM (default), 1 = one CTA per 256-event chunk in grid order, 2 = one
                                       1024-thread CTA per SM whose warps reduce partly through a shared-memory
                                       write-back cache (see TOFMLEM_OPT_CACHE_SHARE) */
    TOFMLEM_OPT_CTA_INTERLEAVE = 7, /* scatter kernels: number of list segments advanced in parallel (default 64;
                                       1 = natural order).  Performance only, results are the same up to the
                                       order of the float32 reductions. */
    TOFMLEM_OPT_CORR_BRICKS = 12,   /* 1 (default): correction images of the fused pass are kept in the context's internal
                                       order (2x2x1-voxel bricks per 16 bytes: 11 % fewer reductions at L2).  This
                                       concerns d_corr of tofmlem_em_correction[_weighted] and tofmlem_update: between
                                       those calls it may be zeroed, copied, or summed element-wise with the d_corr of
                                       an equally configured context (multi-GPU), but not read as an image.  0: d_corr
                                       is a plain image (x fastest).  Applies when nx and ny are even, the Siddon
                                       projector is selected and d_corr is 16-byte aligned;
                                       otherwise d_corr is a plain image anyway.  Do not change options between a pass
                                       and its update. */
    TOFMLEM_OPT_CACHE_SHARE = 11,   /* EM variant 2 (performance only): how many warps of every 8 reduce through the
                                       shared-memory write-back cache (0..8); the others reduce at L2 directly */
    TOFMLEM_OPT_MEDIAN = 10,        /* 1: tofmlem_iterate applies the 3x3x3 median filter to the image estimate after
                                       every update (R23); default 0 */
    TOFMLEM_OPT_TILE_MIN_EVENTS = 14, /* tofmlem_plan_events: a locality bin with at least this many events is
                                       accumulated in a shared-memory tile (default 1024; performance only) */
    TOFMLEM_OPT_TILE_MAX_EVENTS = 16, /* ... in pieces of at most this many events per CTA (default 8192) */
    TOFMLEM_OPT_CONCURRENT = 22,    /* planned fused pass: k > 0 runs the direct pass on records on a second stream BESIDE the tile
                                       pass, the tile pass limited to k CTAs per SM (0, the default: one after the
                                       other).  Performance only. */
    TOFMLEM_OPT_WARP_WALK = 23,     /* 1 (default): whole-chord walks -- tofmlem_sensitivity, tofmlem_attenuation_weights and every
                                       projection / fused pass of a non-TOF context -- run with a WARP per LOR: the 32 lanes
                                       take 32 consecutive slabs along the chord's dominant axis, on images stored with that
                                       axis fastest (2 x nvox floats of scratch kept by the context); 0: a thread per LOR as
                                       for TOF windows.  Same result up to float32 rounding (both within the parity
                                       tolerances against the fp64 oracle).  With 1 the correction image of a non-TOF
                                       context is in grid order, not in bricks (see TOFMLEM_OPT_CORR_BRICKS). */
    TOFMLEM_OPT_SENS_SORT = 21,     /* 1: tofmlem_sensitivity orders the LORs by locality key and chord length first (32 B per
                                       LOR of scratch during the call; from 2^18 LORs on); 0 (default): as they come.
                                       Performance only (the image is the same up to the order of the float32 sums);
                                       measured: 94.6 against 95.8 ms per 100 M LORs -- the pass is bound by the L2
                                       reduction requests, not by the lanes idling in uneven warps. */
    TOFMLEM_OPT_TILE_MIN_ITEMS = 20, /* tofmlem_plan_events: with fewer tile items than this the list is planned without tiles
                                       (default -1: twice the number of tile CTAs the GPU holds at once -- fewer would
                                       run on a fraction of the SMs before the direct pass starts; performance only) */
    TOFMLEM_OPT_TILE_CHECK = 15,    /* 1: bounds-test every access to the shared-memory tiles and count violations in
                                       tofmlem_stats.tile_oob (a debugging aid; default 0).  The plan has already
                                       dry-run every tile event against its tile, so the count must stay 0 */
    TOFMLEM_OPT_L2_PERSIST = 19,    /* 1 (default): the fused passes put a persisting L2 access-policy window on their correction
                                       image (north_star: "the image kept L2-resident where it fits"); 0: no window.
                                       Performance only. */
    TOFMLEM_OPT_REGION_OVERLAP = 18, /* tofmlem_reconstruct_regions / tofmlem_region_grid: 0 (default) = reading R13, every event in
                                       the ONE region that holds its TOF centre (bit-exact split), extended images summed;
                                       1 = reading R27, an event in every region its window reaches (1 or 2),
                                       wider margins, cores only */
    TOFMLEM_OPT_REGION_PLAN = 17,   /* tofmlem_reconstruct_regions plans every region's binned list (ray records + tiles;
                                       48 B per event more scratch), the phases of the nine plans interleaved so that
                                       the host waits twice in all: 0 never, 1 always (when iters > 1), 2 (default) from
                                       6 iterations on.  Measured at cfg-4: an iteration of the nine concurrent regions
                                       takes 21.4 ms with plans against 25.1 ms without, the plans 14 ms: 5 iterations
                                       141.5 against 142.3 ms, 9 iterations 226.9 against 242.6 ms. */
    TOFMLEM_OPT_DETERMINISTIC = 13, /* run-to-run bit-identical accumulation (the paper's LUT kernel "always
                                       generated an identically reconstructed image").  1: the iterations of
                                       tofmlem_iterate[_weighted] on a PLANNED list (tofmlem_plan_events; else
                                       TOFMLEM_EUNSUPPORTED) round every contribution a_ej w_e / fwd_e to an integer number
                                       of quanta -- a power of two fixed per iteration by max(image) alone, ~2^26 per
                                       typical contribution, clamped at 2^48 -- and add it to a 64-bit integer correction
                                       image: integer sums do not depend on the order of the events, so the image is the
                                       same bit for bit in every run and for every ordering of the list.  About 2.5 x
                                       the time of the default pass (scalar 64-bit reductions, no tiles).  0 (default):
                                       float32 sums, order not fixed (run-to-run differences ~1e-7 relative).  TOF Siddon
                                       projector only.  tofmlem_em_correction / tofmlem_iterate_host are not affected. */
    TOFMLEM_OPT_SUBBINS = 9         /* tofmlem_bin_events: order the events INSIDE each locality bin by predicted
                                       voxel-visit count, in `value` sub-bins (1..64, default 16; 1 = off), so that
                                       the events of a warp walk windows of nearly equal length.  Keys, bin offsets
                                       and bin membership do not change (the order inside a bin is unspecified). */
};

/* Create a context.  tof_fwhm_ps <= 0 makes a non-TOF context (full-chord traversal).
 * cuda_stream is a cudaStream_t (NULL = default stream) on the current device; every later call with
 * this context enqueues there.  Errors: EINVAL (NULL, non-positive sizes), ENOMEM, ECUDA. */
int tofmlem_create(const tofmlem_scanner *scanner, const tofmlem_grid *grid, float tof_fwhm_ps,
                   void *cuda_stream, tofmlem_ctx **out);
/* Synchronises the stream, frees internal scratch and the context.  NULL is allowed. */
int tofmlem_destroy(tofmlem_ctx *ctx);
int tofmlem_set_option(tofmlem_ctx *ctx, int key, double value);
/* sigma along the LOR in mm for this context (0 for non-TOF). */
double tofmlem_sigma_mm(const tofmlem_ctx *ctx);
/* Scratch memory.  The context allocates device scratch at first use and keeps it until tofmlem_destroy: the
 * correction image of tofmlem_iterate (4 B per voxel), the histogram of tofmlem_bin_events (8 B per locality bin and
 * sub-bin, 1 B per event), the records of tofmlem_permute_events (32 B per event), the event copies of
 * tofmlem_reconstruct_regions (64 B per event), the staging buffers of tofmlem_iterate_host, the axis-fastest image copies of
 * the whole-chord walks (TOFMLEM_OPT_WARP_WALK: 8 B per voxel, also allocated by tofmlem_reserve).  cudaMalloc inside a
 * call synchronises the device, so a caller who times calls or runs several contexts concurrently reserves first:
 * tofmlem_reserve allocates what iterate / bin_events / permute_events need for up to n_events events under the
 * context's CURRENT options (call it after tofmlem_set_option).  tofmlem_trim SYNCHRONISES and releases every
 * per-event scratch buffer (they are allocated again on demand); ENOMEM / ECUDA as usual. */
int tofmlem_reserve(tofmlem_ctx *ctx, uint64_t n_events);
int tofmlem_trim(tofmlem_ctx *ctx);

/* Sensitivity image (north_star; R10): d_sens[j] = (1/m) sum_i l_ij over m detector-pair LORs
 * (non-TOF chords over the whole grid).  d_sens (nvox floats) is overwritten.  lors->dt is ignored. */
int tofmlem_sensitivity(tofmlem_ctx *ctx, const tofmlem_events *lors, uint64_t m, float *d_sens);

/* TOF-weighted forward projection: d_fwd[e] = sum_j a_ej d_image[j], n floats.
 * Skipped events (non-finite fields, L = 0, empty window) give 0. */
int tofmlem_forward(tofmlem_ctx *ctx, const tofmlem_events *ev, uint64_t n, const float *d_image, float *d_fwd);

/* TOF-weighted backprojection ("direct voxel filling"; the paper's "starting
 * backprojection", :247, is d_values = NULL): d_out[j] += a_ej * d_values[e] (NULL => 1).
 * d_out (nvox floats) is accumulated into; the caller zeroes it. */
int tofmlem_backproject(tofmlem_ctx *ctx, const tofmlem_events *ev, uint64_t n, const float *d_values, float *d_out);

/* One fused forward+back EM pass (R1, R9): d_corr[j] += sum_{e: fwd_e > 0} a_ej / fwd_e with
 * fwd_e = sum_k a_ek d_image[k].  d_corr is accumulated into (caller zeroes it), so that a data set can be
 * passed in several calls or its partial corrections summed across GPUs before tofmlem_update.
 * Updates the context's n_valid / visits counters (reset them with tofmlem_reset_stats). */
int tofmlem_em_correction(tofmlem_ctx *ctx, const tofmlem_events *ev, uint64_t n, const float *d_image, float *d_corr);
int tofmlem_reset_stats(tofmlem_ctx *ctx);

/* Planned event list: ray records + shared-memory tiles for the fused pass (north_star bullets 3 and 4: a fused pass that
 * "recomputes or caches the weights", "shared-memory tile accumulation rather than naive global atomics"; the paper's
 * "direct technique for voxel filling").  For a TOF context with the Siddon projector the call
 * computes, once, a 48-byte ray record per event (the fp64 ray set-up, quantised so that the float32 voxel walk adds
 * exactly) and keeps it in the context; tofmlem_em_correction[_weighted], tofmlem_iterate[_weighted] and
 * tofmlem_forward calls with THIS list (same x1 pointer and n; the records are a snapshot: changing the arrays in place
 * needs a new plan) then run on the records.  If ev is sorted by locality key (the output of tofmlem_bin_events +
 * tofmlem_permute_events) and the +-T sigma neighbourhood of a locality bin fits in shared memory, bins with at least
 * TOFMLEM_OPT_TILE_MIN_EVENTS events are walked with the image and the correction image of that neighbourhood held in
 * shared memory ("tile items"); every event of such a bin is dry-run against the tile at plan time and the few whose
 * window leaves it join the other events in the direct pass.  Results equal the unplanned pass up to float32 rounding
 * (forward values within 1e-4 of the oracle like the unplanned ones).  Changing sigma-related options, the tile size,
 * the projector or the layout of the correction image makes later calls ignore the plan (they take the unplanned path);
 * tofmlem_trim drops it.  A non-TOF context or the K-sample projector leave the plan inactive (no error).  Replaces any
 * earlier plan.  SYNCHRONISES; keeps 48 B per event of device memory. */
int tofmlem_plan_events(tofmlem_ctx *ctx, const tofmlem_events *ev, uint64_t n);
int tofmlem_plan_info(const tofmlem_ctx *ctx, tofmlem_plan *h_out);

/* Multiplicative update (R1, R11): d_image[j] = mask_j ? d_image[j] * d_corr[j] / d_sens[j] : 0 with
 * mask_j = d_sens[j] >= sens_floor_rel * max_k d_sens[k] (and d_sens[j] > 0), decided in float32.
 * d_corr is zeroed afterwards (ready for the next pass). */
int tofmlem_update(tofmlem_ctx *ctx, float *d_image, float *d_corr, const float *d_sens);

/* `iters` MLEM iterations: for each, zero the internal correction image, one fused EM pass
 * over all n events, multiplicative update.  d_image: in x0, out x_iters.  d_image and d_sens must not alias.
 * n <= 2^32 - 1. */
int tofmlem_iterate(tofmlem_ctx *ctx, const tofmlem_events *ev, uint64_t n, float *d_image, const float *d_sens,
                    int iters);

/* Same as tofmlem_iterate with HOST buffers (pinned memory recommended): uploads the events in chunks
 * overlapped with the first pass, the image and the sensitivity, runs `iters` iterations and downloads
 * the image.  SYNCHRONISES before returning.  h_events members are host pointers here. */
int tofmlem_iterate_host(tofmlem_ctx *ctx, const tofmlem_events *h_events, uint64_t n, float *h_image,
                         const float *h_sens, int iters);

/* Locality binning (north_star bullet 1; specification F1 in DESIGN.md): key = dirclass * T + tile of the
 * TOF kernel centre (12 direction classes x cubes of 2^tile_log2 voxels); invalid events get 0xFFFFFFFF.
 * d_key[n] receives the keys (input order); d_perm[n] a permutation that sorts events by key (order inside
 * a bin unspecified; invalid events last); d_bin_offsets (bins+1 entries, may be NULL) the start of each
 * bin in d_perm, with d_bin_offsets[bins] = number of valid events. */
int tofmlem_bin_events(tofmlem_ctx *ctx, const tofmlem_events *ev, uint64_t n, uint32_t *d_key, uint32_t *d_perm,
                       uint32_t *d_bin_offsets);
uint32_t tofmlem_num_bins(const tofmlem_ctx *ctx);
/* out[i] = in[d_perm[i]], i < n, for every member (dt skipped if either dt pointer is NULL).  in/out must not alias.
 * tofmlem_gather_events accepts any index list (e.g. the kept events of tofmlem_scatter_reject, whose indices exceed
 * n); tofmlem_permute_events REQUIRES d_perm to be a permutation of 0..n-1 (what tofmlem_bin_events and
 * tofmlem_split_regions produce) and is 4x faster: it interleaves the members into 32-byte records first, in scratch
 * of 32 B per event that the context keeps until tofmlem_destroy. */
int tofmlem_gather_events(tofmlem_ctx *ctx, const tofmlem_events *in, const uint32_t *d_perm, uint64_t n,
                          const tofmlem_events_mut *out);
int tofmlem_permute_events(tofmlem_ctx *ctx, const tofmlem_events *in, const uint32_t *d_perm, uint64_t n,
                           const tofmlem_events_mut *out);

/* TOF-assisted data division (R12, R13): d_region[e] = #{ j in 1..R-1 : zb[j] <= cz_e } with
 * cz_e the z of the TOF kernel centre (float32, F1); invalid events get -1.  h_zbounds: n_regions+1 ascending
 * HOST floats, or NULL for the paper's partition (first region double width: "200 + 8 x 100").
 * d_perm groups event indices by region (invalid last; order inside a region unspecified); h_counts
 * (HOST, n_regions entries) is valid on return (this call SYNCHRONISES). n_regions <= 64. */
int tofmlem_split_regions(tofmlem_ctx *ctx, const tofmlem_events *ev, uint64_t n, int n_regions,
                          const float *h_zbounds, int32_t *d_region, uint32_t *d_perm, uint64_t *h_counts);
/* The other reading of PAPER.md:101 ("a 40% probability ... within image 5, and a 60% probability ... image region
 * number 6 ... always contributed to 1 or 2 image regions"; reading R27): an event belongs to EVERY region whose core
 * the axial extent of its +-trunc_sigmas*sigma window meets.  float32 specification F3: c, d, L as in F1;
 * hz = (hw / L) * |dz| with hw = (float)(trunc_sigmas * sigma); lo = #{j : zb[j] <= cz - hz}, hi = #{j : zb[j] <= cz + hz}
 * (j in 1..R-1); d_span[e] = lo | hi << 16, -1 for an invalid event.  d_perm (may be NULL; perm_capacity entries, 2 n
 * always suffice while the cores are longer than the window) lists the event indices region by region, an event once
 * in every region of its span; h_counts[r] = length of region r's list.  TOF contexts only.  SYNCHRONISES. */
int tofmlem_split_regions_overlap(tofmlem_ctx *ctx, const tofmlem_events *ev, uint64_t n, int n_regions,
                                  const float *h_zbounds, int32_t *d_span, uint32_t *d_perm, uint64_t perm_capacity,
                                  uint64_t *h_counts);
/* Default boundaries zb[j] = (float)k_j * vz + oz, k_j = nz * {0,2,3,..,R+1} / (R+1) (integer division). */
int tofmlem_region_zbounds(const tofmlem_ctx *ctx, int n_regions, float *h_zbounds);
/* Sub-grid of region r: its core slices plus ceil((trunc_sigmas*sigma + shell_mm)/vz) slices on each side,
 * clamped to the volume (R12); with TOFMLEM_OPT_REGION_OVERLAP the margin is ceil((2*trunc_sigmas*sigma + shell_mm)/vz):
 * the whole window of an event centred up to one half-width outside the core.  *z0,*z1 = slice range [z0, z1) in the
 * parent volume. */
int tofmlem_region_grid(const tofmlem_ctx *ctx, int n_regions, const float *h_zbounds, int r, tofmlem_grid *sub,
                        int32_t *z0, int32_t *z1);
/* Whole cfg-4 pipeline: split, gather each region's events, reconstruct every region independently on its
 * own sub-grid and CUDA stream (`iters` iterations from x0 = mask), and SUM the extended region images into
 * d_image_out (nvox floats, overwritten) as the paper does.  With TOFMLEM_OPT_REGION_OVERLAP = 1 the
 * split is tofmlem_split_regions_overlap (an event reconstructed in every region its window reaches), the margins are
 * the wider ones of tofmlem_region_grid and d_image_out is made of the region CORES only (margins discarded).  The
 * sub-contexts, streams and region images are kept by the context between calls (tofmlem_trim releases them).
 * SYNCHRONISES. */
int tofmlem_reconstruct_regions(tofmlem_ctx *ctx, const tofmlem_events *ev, uint64_t n, int n_regions,
                                const float *h_zbounds, float *d_image_out, const float *d_sens, int iters);

/* ---- Widened rows: the steps the paper runs around the hot path -------------------------
 *
 * NEXT-1, the paper's own TOF kernel (Fig. 3): tofmlem_set_option(TOFMLEM_OPT_PROJECTOR, 1) switches
 * forward / backproject / em_correction / iterate of a TOF context to K equally spaced samples inside the truncated
 * Gaussian (offset_k = -T sigma + k 2 T sigma/(K-1), Gaussian weights normalised to sum to one, K =
 * TOFMLEM_OPT_SAMPLES_K, default 32), centred on the measured time difference; each sample is filled into the voxel
 * that contains it; samples beyond the LOR's end points or outside the grid are dropped.  The voxel of a sample is
 * decided in fp64.  `visits` then counts the samples kept. */

/* NEXT-2 ("we introduced a median filter between MLEM iterations"; size unstated -> R23): 3x3x3 median
 * filter, edges replicated: d_out[j] = the 14th smallest of the 27 values around voxel j.  d_in, d_out: nvox floats,
 * must not alias.  Bit-exact (the result is one of the inputs).  TOFMLEM_OPT_MEDIAN = 1 makes tofmlem_iterate
 * apply it after every update. */
int tofmlem_median3(tofmlem_ctx *ctx, const float *d_in, float *d_out);

/* NEXT-3 ("Attenuation correction was implemented in the forward projection by a weight inversely
 * proportional to the probability of the event being attenuated" -> R19): d_weight[e] = exp(+ sum_j l_ej d_mu[j]),
 * the reciprocal of the probability that both photons of LOR e survive; l_ej = non-TOF Siddon chords over the whole
 * grid, d_mu = attenuation map (1/mm, nvox floats on the context's grid).  LORs that miss the grid get 1. */
int tofmlem_attenuation_weights(tofmlem_ctx *ctx, const tofmlem_events *lors, uint64_t n, const float *d_mu,
                                float *d_weight);
/* EM pass / iterations with a per-event weight: d_corr[j] += d_weight[e] * a_ej / fwd_e (d_weight = NULL => 1, i.e.
 * tofmlem_em_correction / tofmlem_iterate).  d_weight: n floats in the SAME order as the events (after
 * tofmlem_bin_events, permute it with tofmlem_gather_f32). */
int tofmlem_em_correction_weighted(tofmlem_ctx *ctx, const tofmlem_events *ev, uint64_t n, const float *d_weight,
                                   const float *d_image, float *d_corr);
int tofmlem_iterate_weighted(tofmlem_ctx *ctx, const tofmlem_events *ev, uint64_t n, const float *d_weight,
                             float *d_image, const float *d_sens, int iters);
/* d_out[i] = d_in[d_perm[i]], n floats; d_in and d_out must not alias. */
int tofmlem_gather_f32(tofmlem_ctx *ctx, const float *d_in, const uint32_t *d_perm, uint64_t n, float *d_out);

/* NEXT-4, TOF-based scatter rejection (PAPER.md:63 Fig. 2, :69-71 -> R24): d_keep[e] = 1 iff the segment
 * {c + u t : |t| <= half_width_mm} meets the body outline, else 0; c = TOF-estimated annihilation point, u = LOR
 * direction, half_width_mm <= 0 selects 1.959964 sigma ("limits of rejection ... at a 95% confidence level").
 * The outline is a union of n_ellipsoids <= 64 ellipsoids, h_ellipsoids = HOST array of 6 floats each
 * (centre x, y, z, then the RECIPROCAL semi-axes 1/ax, 1/ay, 1/az).  float32 specification F2: the flags
 * are bit-exact.  Invalid events are not kept.  d_perm (may be NULL) receives the indices of the kept events in its
 * first *h_n_kept entries (order unspecified), ready for tofmlem_gather_events.  SYNCHRONISES (h_n_kept is HOST). */
int tofmlem_scatter_reject(tofmlem_ctx *ctx, const tofmlem_events *ev, uint64_t n, const float *h_ellipsoids,
                           int n_ellipsoids, float half_width_mm, uint8_t *d_keep, uint32_t *d_perm,
                           uint64_t *h_n_kept);

/* Roofline probe (measurement aid; north_star asks for the MEASURED atomic / L2 roofline): issues n_ops float32
 * operations against d_buf[0..n_elems) and returns the elapsed milliseconds in *h_ms (second of two passes, so
 * the array is L2-resident when it fits).  kind 0: RED.ADD.F32 to unrelated random elements per lane; 1: RED to
 * 32 consecutive elements of a random row per warp; 2 / 3: the same two patterns with 4-byte loads; 4 / 5: random
 * 8-byte / 16-byte vector reductions (one n_ops unit = one instruction per lane); 6 / 7: random 32-bit integer adds /
 * 4-byte loads on a 72 KB SHARED-MEMORY tile, three CTAs per SM (the tile pass's own access pattern; d_buf untouched).
 * d_buf is modified by kinds 0, 1, 4, 5.  SYNCHRONISES. */
int tofmlem_probe(tofmlem_ctx *ctx, int kind, float *d_buf, uint64_t n_elems, uint64_t n_ops, float *h_ms);

/* Copies the counters of the last pass to *h_out.  SYNCHRONISES the context's stream. */
int tofmlem_get_stats(tofmlem_ctx *ctx, tofmlem_stats *h_out);
/* Device time of the kernels of the LAST planned fused pass (tofmlem_plan_events), in milliseconds, measured with CUDA
 * events on the context's stream: h_ms[0] = tile pass (tile.cu), h_ms[1] = direct pass on records, h_ms[2] = the
 * unplanned pass over the sliver windows (prepared.cuh, kRecTiny); 0 for a part that did not run (all 0 after an
 * unplanned pass).  SYNCHRONISES. */
int tofmlem_pass_timing(tofmlem_ctx *ctx, float h_ms[3]);
/* Text of the last error of this context ("" if none).  Valid until the next call on the context. */
const char *tofmlem_last_error(const tofmlem_ctx *ctx);
/* Number of kernel launches this context has enqueued since creation (bench.py's gpu_launches). */
uint64_t tofmlem_launch_count(const tofmlem_ctx *ctx);
const char *tofmlem_version(void);

/* The fused forward+back EM pass of tofmlem_em_correction (R1, R9) WITHOUT a context and without
 * any allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid it): d_corr[j] += sum_{e: fwd_e > 0} a_ej / fwd_e, fwd_e = sum_k a_ek d_image[k], over the n events in
 * the order given (binned or not), on the current device.  The call itself calls no cudaMalloc, cudaFree or allocating
 * library routine: the only scratch of the pass, the work-queue counters of its persistent kernel, is a file-scope
 * __device__ array of TOFMLEM_STATIC_MAX_QUEUES 32-bit words (4 KB) that every GPU which loads the library holds until
 * the process exits.
 *   grid, tof_fwhm_ps (0 = non-TOF: ev->dt may be NULL), trunc_sigmas (3.0 = the context default): as tofmlem_create /
 *     TOFMLEM_OPT_TRUNC_SIGMAS.  ev: device arrays, n <= 2^32 - 1 entries.
 *   d_image: nvox floats (device), read.  d_corr: nvox floats (device) in GRID order (never bricks), accumulated into:
 *     the caller zeroes it.  16-byte aligned d_corr with nvox % 4 == 0 takes the 16-byte reductions, else scalar ones.
 *   queues_per_sm: work queues (list segments) per SM, 1..8, or 0 = chosen from the window length like the context
 *     path (1, 3 or 4).  Performance only.
 *   cuda_stream: a cudaStream_t on the current device (NULL = default stream); the call enqueues one memset of the
 *     counters and one kernel there and returns without synchronising.
 * Limit: (SM count of the device) x queues_per_sm <= TOFMLEM_STATIC_MAX_QUEUES, else TOFMLEM_EINVAL (a B200 has 148 SMs).
 * ALL calls in the process share the array on a device: it is cleared on the caller's stream before every launch, and
 * two calls that OVERLAP on the GPU (different streams with no dependency between them, or two host threads) race on
 * the counters and give wrong sums -- the caller serialises them.  No statistics counters are kept.
 * Returns TOFMLEM_OK or a negative status; the text of the error is in tofmlem_static_error() (per host thread).
 * Same arithmetic as the unplanned pass of a context with TOFMLEM_OPT_CORR_BRICKS = 0 (tests/test_zz_no_alloc.py). */
#define TOFMLEM_STATIC_MAX_QUEUES 1024
int tofmlem_em_correction_static(const tofmlem_grid *grid, double tof_fwhm_ps, double trunc_sigmas,
                                 const tofmlem_events *ev, uint64_t n, const float *d_image, float *d_corr,
                                 int queues_per_sm, void *cuda_stream);
const char *tofmlem_static_error(void);

#ifdef __cplusplus
}
#endif
#endif /* TOFMLEM_H */
