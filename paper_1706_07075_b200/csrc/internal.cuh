// internal.cuh -- declarations shared by the translation units of libtofmlem (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>

#include "prepared.cuh"
#include "tofmlem.h"

namespace tofmlem {

constexpr double kCmmPerPs = 0.299792458;  // speed of light, mm/ps

// Geometry + TOF constants of one context, passed by value to the projector kernels.
// Per-event ray set-up is done in fp64 from these; the voxel walk is fp32 in a window-local frame.
struct ProjParams {
    int n[3];              // nx, ny, nz
    double v[3], iv[3];    // voxel size and its reciprocal
    double o[3], h[3];     // low corner, high corner o + n*v
    double half_window;    // trunc_sigmas * sigma (mm); unused for non-TOF
    float gauss_a;         // -log2(e) / (2 sigma^2): weight = l * 2^(gauss_a * t^2)
    float gauss_norm;      // 1 / (sigma sqrt(2 pi))
    unsigned stride;       // CTA interleave of the scatter kernels (<= 1: natural order)
    int variant;           // fused EM pass: 0 = persistent per-SM queues (default), 1 = grid order, 2 = smem cache
    int cache_share;       // variant 2: warps (of every 8) that reduce through the shared-memory cache
    int brick;             // fused EM pass: the correction image is in the 2x2x1 brick layout (needs even nx, ny)
    int n_sm;              // SM count of the context's device (persistent kernels: one work queue per SM)
};

struct EventPtrs {
    const float *x1, *y1, *z1, *x2, *y2, *z2, *dt;
};

struct DeviceStats {
    unsigned long long n_valid;
    unsigned long long visits;
    unsigned long long reds;  // reduction instructions (requests to the L2 atomic units) of the scatter walk
    unsigned long long tile_events;  // valid events whose window was accumulated in a shared-memory tile (tile.cu)
    unsigned long long tile_oob;     // TOFMLEM_OPT_TILE_CHECK: tile accesses found out of range (must stay 0)
    unsigned long long tile_visits;  // voxel visits of the forward walk on tiles
    double sum_image_sens;
};
constexpr int kStatsCounters = 6;  // leading unsigned long long members, reset before every pass

// float32 grid for the bit-exact key / region arithmetic (specification F1)
struct GridF32 {
    int nx, ny, nz;
    float vx, vy, vz, ox, oy, oz;
};

// ---- projector.cu
void launch_forward(const ProjParams &p, bool tof, const EventPtrs &ev, uint64_t n, const float *image, float *fwd,
                    cudaStream_t s);
// vec_ok: `out`/`corr` is 16-byte aligned and its allocation covers whole groups of 4 voxels
void launch_backproject(const ProjParams &p, bool tof, const EventPtrs &ev, uint64_t n, const float *values,
                        float *out, bool vec_ok, cudaStream_t s);
// queues: kMaxQueues work counters owned by the context (persistent variant), may be NULL
constexpr int kMaxQueues = 2048;
// the counters of kernels that space them kQueueStride words apart (one 128-byte line each: 148 counters side by side sit in
// five lines, i.e. on a few L2 slices, which then carry every warp's polling and atomics); the array holds
// kMaxQueues * kQueueStride words
constexpr int kQueueStride = 32;
// evw: optional per-event weights (NEXT-3), NULL => 1
void launch_em_correction(const ProjParams &p, bool tof, const EventPtrs &ev, uint64_t n, const float *evw,
                          const float *image, float *corr, bool vec_ok, DeviceStats *stats, unsigned *queues,
                          cudaStream_t s);

// chunks (optional): the pass runs over a list of (first event, count <= 32) pieces instead of 0..n-1 (the events the
// tile-mode pass leaves over); then n_chunks pieces are processed and `n` only bounds the event indices.
void launch_em_correction_chunks(const ProjParams &p, bool tof, const EventPtrs &ev, uint64_t n, const uint2 *chunks,
                                 uint32_t n_chunks, const float *evw, const float *image, float *corr, bool vec_ok,
                                 DeviceStats *stats, unsigned *queues, cudaStream_t s,
                                 bool gather /* the pieces are single events: a warp takes 32 of them, a lane each */);

// ---- warpwalk.cu: a warp per LOR for whole chords (non-TOF); scratch = 2 (forward: 1) x nvox floats
bool warp_walk_ok(const ProjParams &p);
void launch_warp_backproject(const ProjParams &p, const EventPtrs &ev, uint64_t n, const float *values, float *out,
                             float *scratch, cudaStream_t s);
void launch_warp_forward(const ProjParams &p, const EventPtrs &ev, uint64_t n, const float *image, float *fwd,
                         float *scratch, cudaStream_t s);
void launch_warp_em(const ProjParams &p, const EventPtrs &ev, uint64_t n, const float *evw, const float *image,
                    float *corr, float *scratch, DeviceStats *stats, cudaStream_t s);

// ---- tile.cu: fused EM pass with the image and the correction image of one locality bin held in shared memory
constexpr int kTileMaxPlanes = 96;
// Footprint of a locality bin (cube of T voxels, direction class with dominant axis a): the union of the +-T sigma
// windows of all events whose TOF centre lies in the cube and whose direction is in the class is a double cone.  It is
// stored plane by plane along a: plane p (p = i_a - cube origin + RA) holds a W[0] x W[1] rectangle of the two lateral
// axes (fast axis f = the lower-numbered one, slow axis s) whose low corner, in cell coordinates mirrored so that the
// class's rays run towards +f and +s, is (lo[0][p], lo[1][p]).
// Two variants: [0] the item is one cube, [1] the item is a PAIR of cubes that are neighbours along a (the tile is T
// planes longer, the lateral rectangles are the same): fewer, larger items -- the per-item cost (tile load, flush,
// barriers) is shared by twice the events, and bins too sparse on their own become tile work.
struct TileGeom {
    int T;                 // cube edge in voxels
    int ok;                // tile mode is available for this context (all three dominant axes fit)
    int pairs;             // variant [1] may be used (it fits without lowering the number of CTAs per SM)
    int RA[3];             // planes below the first cube, per dominant axis
    int PA[2][3];          // planes in all
    int W[2][3][2];        // rectangle width along f and s
    int PS[2][3];          // words per plane (odd, >= W[0] * W[1])
    int words;             // words of the largest tile in use: max PA * PS
    signed char lo[2][3][2][kTileMaxPlanes];
};
struct TileItem {
    uint32_t start, count;    // events [start, start + count) of the sorted list: the item's (first) cube, key `key`
    uint32_t start2, count2;  // pair items: the events of the second cube (key + one step along a), else count2 = 0
    uint32_t key, variant, pad0, pad1;
};
// A contiguous run of events of the sorted list that belongs to a tile item (the plan's event -> item look-up).
struct TileRange {
    uint32_t start, count, item, pad;
};
// false (g.ok = 0) when a tile pair does not fit in `smem_budget` bytes of shared memory
void build_tile_geom(const ProjParams &p, int tile_log2, size_t smem_budget, size_t smem_per_sm, TileGeom &g);
int tile_ctas_per_sm(size_t tile_bytes, size_t smem_per_sm);
size_t tile_smem_bytes(const TileGeom &g);
// d_geom: the same structure in device memory; rec: the ray records of the planned list (prepared.cuh)
void launch_em_tile(const ProjParams &p, const TileGeom &g, const TileGeom *d_geom, int tile_log2, const RecPtrs &rec,
                    const float *evw, const float *image, float *corr, DeviceStats *stats, const TileItem *items,
                    uint32_t n_items, unsigned *counter /* one word, zeroed by the call */, int n_sm,
                    size_t smem_per_sm, bool check, double sigma, uint32_t max_item_events /* no item holds more */,
                    float *ev_scale /* one float per event of the list: scratch between the two phases */,
                    int cap_ctas /* > 0: at most this many CTAs per SM */, cudaStream_t s);

// ---- prepared.cu: ray records of a planned list and the passes that run on them
// Writes one record per event (p.brick says which group count the direct records carry), one flag per 32-event piece of
// the list (1: the piece holds events for the direct pass on records), the kRecTiny events as one-event pieces, and
// fills the counters (plan_counter_bytes() bytes of device memory; read_plan_counters: valid events, tile events,
// events of tile items that do not fit their tile, visits, kRecTiny events).
size_t plan_counter_bytes();
void launch_prepare_rays(const ProjParams &p, double sigma, const TileGeom *d_geom /* NULL: no tiles */, int tile_log2,
                         const EventPtrs &ev, uint64_t n, const TileItem *items, const TileRange *ranges,
                         uint32_t n_ranges, const RecPtrs &rec, uint32_t *chunk_flags /* ceil(n / 32) */,
                         uint2 *tiny_list /* (event, 1) pieces of the kRecTiny events */, uint32_t tiny_cap,
                         void *d_counters, cudaStream_t s);
void read_plan_counters(const void *h_counters, uint64_t out[5]);  // ... and the kRecTiny events
// ev: the raw events of the planned list (the kRecTiny records are walked from them)
void launch_planned_forward(const ProjParams &p, double sigma, const EventPtrs &ev, const RecPtrs &rec, uint64_t n,
                            const float *image, float *fwd, cudaStream_t s);
// pieces: n_pieces indices of the 32-event pieces of the list that hold work for this pass, ascending
// sparse: the pieces are what a tile pass leaves over (the sparse bins), not a whole list
void launch_em_planned(const ProjParams &p, const RecPtrs &rec, uint64_t n, const uint32_t *pieces, uint32_t n_pieces,
                       const float *evw, const float *image, float *corr, bool vec_ok, DeviceStats *stats,
                       unsigned *queues, int n_sm, bool sparse, cudaStream_t s);

// reproducible accumulation (TOFMLEM_OPT_DETERMINISTIC): every event of the planned list, 64-bit integer correction image
void launch_em_det(const ProjParams &p, const RecPtrs &rec, uint64_t n, const float *evw, const float *image,
                   unsigned long long *corr_q, const float *gscale /* [0] quanta per unit */, DeviceStats *stats,
                   unsigned *queues, int n_sm, cudaStream_t s);

// ---- image_ops.cu
void launch_det_scale(const float *d_img_max, float *gscale /* [2]: G, 1 / G */, cudaStream_t s);
void launch_update_det(float *image, unsigned long long *corr_q, const float *sens, const float *d_max, float floor_rel,
                       const float *gscale, uint64_t n, cudaStream_t s);
void launch_max_nonneg(const float *x, uint64_t n, float *d_max /* zeroed by the call */, cudaStream_t s);
void launch_update(float *image, float *corr, const float *sens, const float *d_max, float floor_rel, uint64_t n,
                   cudaStream_t s);
// corr in the brick layout: index = ((z * ny/2 + y/2) * nx/2 + x/2) * 4 + (y & 1) * 2 + (x & 1); nx, ny even
void launch_update_brick(float *image, float *corr, const float *sens, const float *d_max, float floor_rel, int nx,
                         int ny, int nz, cudaStream_t s);
void launch_mask_init(float *image, const float *sens, const float *d_max, float floor_rel, uint64_t n,
                      cudaStream_t s);
void launch_dot_f64(const float *a, const float *b, uint64_t n, double *d_out /* zeroed by the call */,
                    cudaStream_t s);
void launch_scale(float *x, float a, uint64_t n, cudaStream_t s);
void launch_add(float *dst, const float *src, uint64_t n, cudaStream_t s);
void launch_median3(const float *in, float *out, int nx, int ny, int nz, cudaStream_t s);
void launch_exp(float *w, uint64_t n, cudaStream_t s);

// ---- binning.cu
// Sub-bins: the events of one locality bin are ordered by predicted visit count (S sub-bins of `quantum` visits;
// sub-bin 0 = the window misses the grid).  S = 1 switches the ordering off.
struct SubBin {
    uint32_t S, quantum;
    float half_window;  // trunc_sigmas * sigma (mm); 0 for non-TOF
};
void launch_plan_hist(const GridF32 &g, int tile_log2, const EventPtrs &ev, uint64_t n, uint32_t *hist /* zeroed */,
                      uint32_t nbins, unsigned *unsorted /* zeroed; set to 1 when a key is below its predecessor's */,
                      cudaStream_t s);
void launch_bin_keys(const GridF32 &g, int tile_log2, const SubBin &sb, const EventPtrs &ev, uint64_t n, uint32_t *key,
                     uint8_t *sub /* n, or NULL */, uint32_t *hist /* nbins*S+1, zeroed by caller */, uint32_t nbins,
                     cudaStream_t s);
uint32_t scan_tmp_elems(uint32_t n);
// returns the number of kernels launched; tmp: scan_tmp_elems(n) words (NULL: single-block scan)
int launch_exclusive_scan_u32(const uint32_t *in, uint32_t *out, uint32_t *tmp, uint32_t n, cudaStream_t s);
// list[pos[i]] = i for flags[i] != 0 (pos: exclusive scan of flags): the flagged indices in ascending order
void launch_compact_flags(const uint32_t *flags, const uint32_t *pos, uint32_t n, uint32_t *list, cudaStream_t s);
void launch_scatter_perm(const uint32_t *key, const uint8_t *sub, uint32_t S, uint64_t n, uint32_t nbins,
                         uint32_t *cursor, uint32_t *perm, cudaStream_t s);
void launch_strided_copy(const uint32_t *fine, uint32_t S, uint32_t count, uint32_t *out, cudaStream_t s);
void launch_gather(const float *in, const uint32_t *perm, uint64_t n, float *out, cudaStream_t s);
// all members at once through 32-byte records; rec: 8 n floats of scratch (16-byte aligned); out[6] may be NULL
void launch_gather_packed(const EventPtrs &in, const uint32_t *perm, uint64_t n, float *rec, float *const out[7],
                          cudaStream_t s);
constexpr int kMaxRegions = 64;
struct RegionBounds {
    float zb[kMaxRegions + 1];
    int n_regions;
};
void launch_region_ids(const EventPtrs &ev, uint64_t n, const RegionBounds &rb, int32_t *region,
                       unsigned long long *counts /* n_regions+1, zeroed by caller; last = invalid */,
                       cudaStream_t s);
void launch_region_scatter(const int32_t *region, uint64_t n, int n_regions,
                           unsigned long long *cursor /* n_regions+1 start offsets, advanced */, uint32_t *perm,
                           cudaStream_t s);

// reading R27 / F3: span[e] = lo | hi << 16 (-1 invalid); counts as launch_region_ids, with multiplicity
void launch_region_spans(const EventPtrs &ev, uint64_t n, const RegionBounds &rb, float hw, int32_t *span,
                         unsigned long long *counts /* n_regions+1, zeroed by caller */, cudaStream_t s);
void launch_region_span_scatter(const int32_t *span, uint64_t n, int n_regions,
                                unsigned long long *cursor /* start offsets, advanced */, uint32_t *perm,
                                cudaStream_t s);

constexpr int kMaxEllipsoids = 64;
struct EllipsoidSet {
    float v[6 * kMaxEllipsoids];  // per ellipsoid: centre x, y, z, reciprocal semi-axes 1/ax, 1/ay, 1/az
    int n;
};
void launch_scatter_keep(const EventPtrs &ev, uint64_t n, const EllipsoidSet &es, float h, uint8_t *keep,
                         uint32_t *perm /* may be NULL */, unsigned long long *counter /* zeroed by caller */,
                         cudaStream_t s);

// ---- sampled.cu (the paper's K-sample TOF kernel, NEXT-1)
struct SampleLutEntry {
    double offset;  // mm along the LOR from the kernel centre
    float weight;   // Gaussian weight, the K weights sum to one
    float offset_f; // offset rounded to float32 (fast path of the voxel decision)
};
void launch_sampled_forward(const ProjParams &p, const SampleLutEntry *lut, int K, const EventPtrs &ev, uint64_t n,
                            const float *image, float *fwd, cudaStream_t s);
void launch_sampled_backproject(const ProjParams &p, const SampleLutEntry *lut, int K, const EventPtrs &ev, uint64_t n,
                                const float *values, float *out, cudaStream_t s);
void launch_sampled_em(const ProjParams &p, const SampleLutEntry *lut, int K, const EventPtrs &ev, uint64_t n,
                       const float *evw, const float *image, float *corr, DeviceStats *stats,
                       unsigned *queues /* kMaxQueues work counters */, cudaStream_t s);

// ---- probe.cu
int run_probe(int kind, float *d_buf, uint64_t n_elems, uint64_t n_ops, float *ms, cudaStream_t s);

}  // namespace tofmlem
