// api.cu -- the C ABI of libtofmlem (include/tofmlem.h): context, argument checks, stream orchestration.
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <new>
#include <vector>

#include "internal.cuh"

using namespace tofmlem;

struct tofmlem_ctx {
    tofmlem_ctx() { memset(&h_geom_sent, 0xff, sizeof h_geom_sent); }
    tofmlem_scanner scanner;
    tofmlem_grid grid;
    bool tof;
    double sigma;  // mm
    double trunc_sigmas = 3.0, sens_floor_rel = 1e-2, shell_mm = 6.0;
    int tile_log2 = 3, projector = 0, samples_k = 32;
    cudaStream_t stream = nullptr;
    uint64_t nvox = 0;
    // scratch owned by the context
    float *d_corr = nullptr;  // padded to whole groups of 4 voxels
    unsigned cta_interleave = 64;
    int em_variant = 0;
    int cache_share = 4;
    int corr_bricks = 1;  // correction images of the fused pass in the 2x2x1 brick layout (TOFMLEM_OPT_CORR_BRICKS)
    float *d_max = nullptr;          // max(sens) of the current iterate call
    const float *d_max_ext = nullptr;  // region sub-contexts use the parent's global max
    DeviceStats *d_stats = nullptr;
    unsigned *d_queues = nullptr;  // work counters of the persistent EM kernel
    uint32_t *d_hist = nullptr, *d_cursor = nullptr, *d_scan_tmp = nullptr;
    size_t hist_cap = 0;
    // scratch of tofmlem_reconstruct_regions, kept between calls (64 B per event): region ids / keys, permutation,
    // region-sorted and region-binned event copies
    int32_t *d_rg_region = nullptr;
    uint32_t *d_rg_perm = nullptr;
    float *d_rg_sorted = nullptr, *d_rg_binned = nullptr;
    size_t rg_cap = 0;
    float *d_pack = nullptr;   // 32-byte event records of tofmlem_gather_events
    size_t pack_cap = 0;
    uint8_t *d_sub = nullptr;  // sub-bin of every event of the last tofmlem_bin_events
    size_t sub_cap = 0;
    int subbins = 16;
    int median = 0;                    // 3x3x3 median filter after every update of tofmlem_iterate (NEXT-2)
    float *d_tmp_image = nullptr;      // median filter output
    SampleLutEntry *d_lut = nullptr;   // K-sample TOF kernel (NEXT-1)
    int lut_k = 0;
    double lut_sigma = 0.0, lut_trunc = 0.0;
    std::vector<SampleLutEntry> h_lut;
    unsigned long long *d_rcounts = nullptr;  // 2*(kMaxRegions+1)
    // host-buffer path
    float *d_hev = nullptr;
    size_t hev_cap = 0;
    float *d_himg = nullptr, *d_hsens = nullptr;
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t chunk_done[2] = {nullptr, nullptr};
    uint64_t last_n = 0;
    uint64_t launches = 0;
    // tile-mode plan of the fused pass (tofmlem_plan_events; tile.cu)
    int tile_min_events = 1024, tile_max_events = 8192, tile_check = 0;
    int deterministic = 0;        // TOFMLEM_OPT_DETERMINISTIC: integer accumulation (prepared.cu, em_det_kernel)
    unsigned long long *d_corr_q = nullptr;  // its 64-bit correction image
    float *d_gscale = nullptr;               // [0] quanta per unit, [1] its reciprocal, [2] max(image) of the pass
    int l2_persist = 1;           // TOFMLEM_OPT_L2_PERSIST
    const float *l2_ptr = nullptr;  // correction image the stream's access-policy window currently covers
    cudaStream_t l2_stream = nullptr;
    int region_overlap = 0;  // reading R27: an event goes to every region its window meets (TOFMLEM_OPT_REGION_OVERLAP)
    int warp_walk = 1;            // TOFMLEM_OPT_WARP_WALK: whole-chord (non-TOF) walks with a warp per LOR (warpwalk.cu)
    float *d_axis = nullptr;      // its scratch: image / target stored y-fastest or z-fastest (2 nvox floats)
    int sens_sort = 0;            // TOFMLEM_OPT_SENS_SORT: tofmlem_sensitivity orders the LORs by locality and chord length
    bool bin_whole_chords = false;  // tofmlem_bin_events: sub-bins by the visits of the WHOLE chord (non-TOF walks)
    int tile_min_items = -1;  // TOFMLEM_OPT_TILE_MIN_ITEMS (-1: twice the number of tile CTAs the GPU holds)
    int region_plan = 2;  // tofmlem_reconstruct_regions plans every region's list: 0 never, 1 always, 2 from 6 iterations on
    int n_sm = 0;
    size_t smem_optin = 0;  // largest dynamic shared memory a CTA may opt in to on this device
    TileGeom *d_geom = nullptr;
    TileGeom h_geom_sent;   // what d_geom currently holds (valid when d_geom != nullptr)
    TileItem *d_items = nullptr;
    size_t items_cap = 0;
    TileRange *d_ranges = nullptr;
    size_t ranges_cap = 0;
    uint32_t *d_chunk_flags = nullptr;  // one per 32-event piece of the planned list: 1 = work for the direct pass
    uint32_t *d_chunk_pos = nullptr, *d_chunk_list = nullptr, *d_chunk_tmp = nullptr;  // scan of the flags, flagged pieces
    uint32_t *h_hist_pinned = nullptr;  // staging of the bin counts for the plan's host part
    size_t h_hist_cap = 0;
    unsigned *d_plan_flags = nullptr;  // [0] tile work counter, [1] "keys not sorted" flag
    RecPtrs d_rec{nullptr, nullptr, nullptr};  // ray records of the planned list (prepared.cuh), 48 B per event
    size_t rec_cap = 0;
    uint2 *d_tiny = nullptr;           // one-event pieces of the kRecTiny events (kTinyCap entries)
    float *d_ev_scale = nullptr;       // w_e / fwd_e of the tile events between the two phases of tile.cu (rec_cap floats)
    size_t smem_per_sm = 0;
    void *d_plan_counters = nullptr;
    // tofmlem_reconstruct_regions: sub-contexts, streams, events and region images, kept between calls (creating and
    // destroying them per call put nine cudaMalloc / cudaFree device-wide syncs in the middle of nine running streams)
    struct RegionCache {
        std::vector<float> zb;       // region bounds the cache was built for (n_regions + 1)
        double sigma = 0.0, trunc = 0.0, shell = 0.0;
        std::vector<tofmlem_ctx *> subs;
        std::vector<cudaStream_t> streams;
        std::vector<cudaEvent_t> done;
        std::vector<float *> images;
        std::vector<int32_t> z0, z1;
        cudaEvent_t ready = nullptr;
    } rgc;
    cudaEvent_t t_ev[4] = {nullptr, nullptr, nullptr, nullptr};  // tofmlem_pass_timing: around the planned kernels
    int concurrent = 0;            // TOFMLEM_OPT_CONCURRENT: tile CTAs per SM while the direct pass runs beside them
    cudaStream_t side_stream = nullptr;
    cudaEvent_t fork_ev = nullptr, join_ev = nullptr;
    int t_have = 0;                                              // bit k: part k of the last planned pass ran
    struct {
        bool valid = false;
        const float *x1 = nullptr;  // the plan describes THIS event list (first member array) ...
        uint64_t n = 0;             // ... of this length, binned with
        int tile_log2 = 0;          // ... this cube size, for a context with
        double sigma = 0.0, trunc = 0.0;  // ... this TOF kernel
        int brick = 0;              // ... and this layout of the correction image
        uint32_t n_items = 0, n_strag = 0, n_tiny = 0, max_item_events = 0;
        uint64_t direct_valid = 0;  // valid events of the direct pass on records
        uint32_t n_pieces = 0;      // 32-event pieces of the list that hold some of them
        uint64_t tile_events = 0, direct_events = 0, valid_events = 0, visits = 0;
        int sorted = 0;
    } plan;
    // state of a plan between the phases of tofmlem_plan_events (plan_begin / plan_build / plan_finish)
    struct PlanJob {
        tofmlem_events ev{};
        uint64_t n = 0;
        ProjParams p{};
        TileGeom g{};
        std::vector<TileItem> items;
        std::vector<TileRange> ranges;
        std::vector<uint64_t> start;
        std::vector<uint8_t> state;
        unsigned flags[2] = {0, 0};
        uint32_t n_pieces = 0;
        std::vector<unsigned char> hc;
    } job;
    std::string err;
};

namespace {

constexpr uint32_t kTinyCap = 1u << 20;  // kRecTiny events a plan can hold (more: the list is not planned at all)

int fail(tofmlem_ctx *c, int code, const char *what) {
    if (c) c->err = what ? what : "";
    return code;
}

int cuda_fail(tofmlem_ctx *c, cudaError_t e, const char *where) {
    if (c) {
        char buf[512];
        snprintf(buf, sizeof buf, "%s: %s (%s)", where, cudaGetErrorString(e), cudaGetErrorName(e));
        c->err = buf;
    }
    return e == cudaErrorMemoryAllocation ? TOFMLEM_ENOMEM : TOFMLEM_ECUDA;
}

#define CU(call)                                                  \
    do {                                                          \
        cudaError_t e_ = (call);                                  \
        if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call);  \
    } while (0)

#define CHECK_LAUNCH(k)                                                       \
    do {                                                                      \
        cudaError_t e_ = cudaGetLastError();                                  \
        if (e_ != cudaSuccess) return cuda_fail(ctx, e_, "kernel launch");    \
        ctx->launches += (k);                                                 \
    } while (0)

double sigma_from_fwhm(double fwhm_ps) { return kCmmPerPs * fwhm_ps / (2.0 * 2.0 * sqrt(2.0 * log(2.0))); }

ProjParams make_params(const tofmlem_ctx *c, bool tof) {
    ProjParams p;
    const tofmlem_grid &g = c->grid;
    p.n[0] = g.nx; p.n[1] = g.ny; p.n[2] = g.nz;
    p.v[0] = g.vx; p.v[1] = g.vy; p.v[2] = g.vz;
    p.o[0] = g.ox; p.o[1] = g.oy; p.o[2] = g.oz;
    for (int a = 0; a < 3; ++a) {
        p.iv[a] = 1.0 / p.v[a];
        p.h[a] = p.o[a] + p.n[a] * p.v[a];
    }
    if (tof) {
        p.half_window = c->trunc_sigmas * c->sigma;
        p.gauss_a = (float)(-1.4426950408889634 / (2.0 * c->sigma * c->sigma));
        p.gauss_norm = (float)(1.0 / (c->sigma * sqrt(2.0 * M_PI)));
    } else {
        p.half_window = 0.0;
        p.gauss_a = 0.0f;
        p.gauss_norm = 1.0f;
    }
    p.stride = c->cta_interleave;
    p.variant = c->em_variant;
    p.cache_share = c->cache_share;
    p.brick = 0;
    p.n_sm = c->n_sm;
    return p;
}

// 16-byte vector reductions need an aligned array made of whole groups of 4 voxels
bool vec_ok(const tofmlem_ctx *c, const float *out) {
    return (c->nvox & 3) == 0 && (reinterpret_cast<uintptr_t>(out) & 15) == 0;
}

// Whole-chord walks (sensitivity, attenuation line integrals, every projection of a non-TOF context) run with a warp per
// LOR (warpwalk.cu) unless switched off or the grid does not fit its index packing.
bool warp_on(const tofmlem_ctx *c) { return c->warp_walk && c->projector == 0 && warp_walk_ok(make_params(c, false)); }
// ... and so does the fused pass of a non-TOF context (default scheduling variant only); its correction image is in
// grid order (the walk wants the ray's dominant axis fastest, not bricks).
bool warp_em_on(const tofmlem_ctx *c) { return !c->tof && c->em_variant == 0 && warp_on(c); }

int ensure_axis_scratch(tofmlem_ctx *c) {
    if (c->d_axis) return TOFMLEM_OK;
    if (cudaMalloc(&c->d_axis, 2 * c->nvox * sizeof(float)) != cudaSuccess) {
        cudaGetLastError();
        c->d_axis = nullptr;
        c->err = "out of device memory (axis-major scratch of the warp-per-LOR walk)";
        return TOFMLEM_ENOMEM;
    }
    return TOFMLEM_OK;
}

// Is the correction image `corr` of this context's fused pass / update in the brick layout?  Depends only on the
// context's options and the pointer, so tofmlem_em_correction and tofmlem_update agree without further state.
bool bricks_on(const tofmlem_ctx *c, const float *corr) {
    return c->corr_bricks && c->projector == 0 && (c->grid.nx & 1) == 0 && (c->grid.ny & 1) == 0 && vec_ok(c, corr) &&
           !warp_em_on(c);
}

// The brick-order update reads image and sens as float2: both must be 8-byte aligned there (checked by the callers
// through update_aligned; the layout decision itself depends on corr and the options only).
bool update_aligned(const tofmlem_ctx *c, const float *image, const float *corr, const float *sens) {
    return !bricks_on(c, corr) ||
           (((reinterpret_cast<uintptr_t>(image) | reinterpret_cast<uintptr_t>(sens)) & 7) == 0);
}

void update_any(const tofmlem_ctx *c, float *image, float *corr, const float *sens, const float *dmax, cudaStream_t s) {
    if (bricks_on(c, corr))
        launch_update_brick(image, corr, sens, dmax, (float)c->sens_floor_rel, c->grid.nx, c->grid.ny, c->grid.nz, s);
    else
        launch_update(image, corr, sens, dmax, (float)c->sens_floor_rel, c->nvox, s);
}

EventPtrs ev_ptrs(const tofmlem_events *e, uint64_t off = 0) {
    EventPtrs p{e->x1 + off, e->y1 + off, e->z1 + off, e->x2 + off, e->y2 + off, e->z2 + off,
                e->dt ? e->dt + off : nullptr};
    return p;
}

bool ev_ok(const tofmlem_events *e, bool need_dt) {
    return e && e->x1 && e->y1 && e->z1 && e->x2 && e->y2 && e->z2 && (!need_dt || e->dt);
}

GridF32 grid_f32(const tofmlem_ctx *c) {
    const tofmlem_grid &g = c->grid;
    return GridF32{g.nx, g.ny, g.nz, g.vx, g.vy, g.vz, g.ox, g.oy, g.oz};
}

uint32_t num_bins(const tofmlem_ctx *c) {
    const int t = 1 << c->tile_log2;
    const uint64_t T = (uint64_t)((c->grid.nx + t - 1) >> c->tile_log2) * ((c->grid.ny + t - 1) >> c->tile_log2) *
                       ((c->grid.nz + t - 1) >> c->tile_log2);
    return (uint32_t)(12u * T);
}

int ensure_corr(tofmlem_ctx *ctx) {
    if (!ctx->d_corr) {
        CU(cudaMalloc(&ctx->d_corr, (ctx->nvox + 4) * sizeof(float)));
        CU(cudaMemsetAsync(ctx->d_corr, 0, (ctx->nvox + 4) * sizeof(float), ctx->stream));
    }
    return TOFMLEM_OK;
}

// Scratch of tofmlem_bin_events: fine histogram, cursors and scan space for `nfine` counters, one sub-bin byte per
// event (n_sub = 0: none).  Grows only; cudaFree synchronises the device, so no launch can still be using the old one.
int ensure_bin_scratch(tofmlem_ctx *ctx, size_t nfine, uint64_t n_sub) {
    if (ctx->hist_cap < nfine) {
        cudaFree(ctx->d_hist);
        cudaFree(ctx->d_cursor);
        cudaFree(ctx->d_scan_tmp);
        ctx->d_hist = ctx->d_cursor = ctx->d_scan_tmp = nullptr;
        ctx->hist_cap = 0;
        CU(cudaMalloc(&ctx->d_hist, nfine * sizeof(uint32_t)));
        CU(cudaMalloc(&ctx->d_cursor, nfine * sizeof(uint32_t)));
        CU(cudaMalloc(&ctx->d_scan_tmp, (size_t)scan_tmp_elems((uint32_t)nfine) * sizeof(uint32_t)));
        ctx->hist_cap = nfine;
    }
    if (ctx->sub_cap < n_sub) {
        cudaFree(ctx->d_sub);
        ctx->d_sub = nullptr;
        ctx->sub_cap = 0;
        CU(cudaMalloc(&ctx->d_sub, n_sub));
        ctx->sub_cap = n_sub;
    }
    return TOFMLEM_OK;
}

void free_region_cache(tofmlem_ctx *ctx) {
    auto &c = ctx->rgc;
    for (size_t r = 0; r < c.subs.size(); ++r) {
        if (c.subs[r]) tofmlem_destroy(c.subs[r]);
        if (c.streams[r]) cudaStreamDestroy(c.streams[r]);
        if (c.done[r]) cudaEventDestroy(c.done[r]);
        cudaFree(c.images[r]);
    }
    if (c.ready) cudaEventDestroy(c.ready);
    c = tofmlem_ctx::RegionCache();
}

void free_records(tofmlem_ctx *ctx) {
    cudaFree(ctx->d_rec.a);
    cudaFree(ctx->d_rec.b);
    cudaFree(ctx->d_rec.c);
    cudaFree(ctx->d_chunk_flags);
    cudaFree(ctx->d_chunk_pos);
    cudaFree(ctx->d_chunk_list);
    cudaFree(ctx->d_chunk_tmp);
    ctx->d_chunk_flags = ctx->d_chunk_pos = ctx->d_chunk_list = ctx->d_chunk_tmp = nullptr;
    cudaFree(ctx->d_ev_scale);
    cudaFree(ctx->d_tiny);
    ctx->d_tiny = nullptr;
    ctx->d_rec = RecPtrs{nullptr, nullptr, nullptr};
    ctx->d_ev_scale = nullptr;
    ctx->rec_cap = 0;
    ctx->plan.valid = false;
}

// Scratch of tofmlem_plan_events for a list of n events (grows only): ray records (48 B per event), w_e / fwd_e of the
// tile pass (4 B), per-piece flags, the sliver list, pinned staging for the bin counts.
int ensure_plan_scratch(tofmlem_ctx *ctx, uint64_t n) {
    if (ctx->rec_cap < n) {
        free_records(ctx);
        CU(cudaMalloc(&ctx->d_rec.a, n * sizeof(float4)));
        CU(cudaMalloc(&ctx->d_rec.b, n * sizeof(float4)));
        CU(cudaMalloc(&ctx->d_rec.c, n * sizeof(uint4)));
        CU(cudaMalloc(&ctx->d_ev_scale, n * sizeof(float)));
        CU(cudaMalloc(&ctx->d_tiny, kTinyCap * sizeof(uint2)));
        {
            const size_t nc = (size_t)((n + 31) / 32) + 1;  // + the total
            CU(cudaMalloc(&ctx->d_chunk_flags, nc * sizeof(uint32_t)));
            CU(cudaMalloc(&ctx->d_chunk_pos, nc * sizeof(uint32_t)));
            CU(cudaMalloc(&ctx->d_chunk_list, nc * sizeof(uint32_t)));
            CU(cudaMalloc(&ctx->d_chunk_tmp, (size_t)scan_tmp_elems((uint32_t)nc) * sizeof(uint32_t)));
        }
        ctx->rec_cap = n;
    }
    const uint32_t nb = num_bins(ctx);
    if (ctx->h_hist_cap < nb) {  // pinned: the 18 MB of counts at cfg-3 come back at PCIe speed
        if (ctx->h_hist_pinned) cudaFreeHost(ctx->h_hist_pinned);
        ctx->h_hist_pinned = nullptr;
        ctx->h_hist_cap = 0;
        CU(cudaMallocHost(&ctx->h_hist_pinned, (size_t)nb * sizeof(uint32_t)));
        ctx->h_hist_cap = nb;
    }
    return ensure_bin_scratch(ctx, (size_t)nb + 1, 0);
}

// 32-byte event records of tofmlem_permute_events (grows only).  false: not enough memory (the caller falls back).
bool ensure_pack(tofmlem_ctx *ctx, uint64_t n) {
    if (ctx->pack_cap >= n) return true;
    cudaFree(ctx->d_pack);
    ctx->d_pack = nullptr;
    ctx->pack_cap = 0;
    if (cudaMalloc(&ctx->d_pack, n * 8 * sizeof(float)) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    ctx->pack_cap = n;
    return true;
}

// number of sub-bins tofmlem_bin_events uses for a sorting call (the fine histogram must fit 32-bit indices)
uint32_t effective_subbins(const tofmlem_ctx *c) {
    uint32_t S = (uint32_t)c->subbins;
    const uint32_t nb = num_bins(c);
    while (S > 1 && (uint64_t)nb * S + 1 > 0x7FFFFFFFull) S >>= 1;
    return S;
}

void default_region_slices(int nz, int R, std::vector<int32_t> &k) {
    k.resize(R + 1);
    k[0] = 0;
    for (int j = 1; j <= R; ++j) k[j] = (int32_t)(((int64_t)nz * (j + 1)) / (R + 1));
}

// zb[j] = (float)k_j * vz + oz : one float multiply, then one float add (F1); volatile blocks contraction.
void default_zbounds(const tofmlem_ctx *c, int R, float *zb) {
    std::vector<int32_t> k;
    default_region_slices(c->grid.nz, R, k);
    for (int j = 0; j <= R; ++j) {
        volatile float kv = (float)k[j] * c->grid.vz;
        volatile float z = kv + c->grid.oz;
        zb[j] = z;
    }
}

// Look-up table of the paper's K-sample TOF kernel (Fig. 3): offset_k = -T sigma + k 2 T sigma/(K-1),
// weight_k = exp(-offset_k^2 / 2 sigma^2) / sum_m exp(-offset_m^2 / 2 sigma^2); K = 1: one sample at the centre.
int ensure_lut(tofmlem_ctx *ctx) {
    const int K = ctx->samples_k;
    if (ctx->d_lut && ctx->lut_k == K && ctx->lut_sigma == ctx->sigma && ctx->lut_trunc == ctx->trunc_sigmas)
        return TOFMLEM_OK;
    CU(cudaStreamSynchronize(ctx->stream));  // a previous launch may still read the old table
    cudaFree(ctx->d_lut);
    ctx->d_lut = nullptr;
    std::vector<double> w(K);
    ctx->h_lut.assign(K, SampleLutEntry{});
    const double hw = ctx->trunc_sigmas * ctx->sigma;
    double sum = 0.0;
    for (int k = 0; k < K; ++k) {
        const double off = K > 1 ? -hw + (double)k * (2.0 * hw) / (double)(K - 1) : 0.0;
        const double r = off / ctx->sigma;
        w[k] = exp(-0.5 * r * r);
        sum += w[k];
        ctx->h_lut[k].offset = off;
        ctx->h_lut[k].offset_f = (float)off;
    }
    for (int k = 0; k < K; ++k) ctx->h_lut[k].weight = (float)(w[k] / sum);
    CU(cudaMalloc(&ctx->d_lut, K * sizeof(SampleLutEntry)));
    CU(cudaMemcpyAsync(ctx->d_lut, ctx->h_lut.data(), K * sizeof(SampleLutEntry), cudaMemcpyHostToDevice, ctx->stream));
    ctx->lut_k = K;
    ctx->lut_sigma = ctx->sigma;
    ctx->lut_trunc = ctx->trunc_sigmas;
    return TOFMLEM_OK;
}

// Does the context hold ray records for exactly this list and this TOF kernel?
bool plan_matches(const tofmlem_ctx *c, const float *x1, uint64_t n) {
    return c->plan.valid && c->plan.x1 == x1 && c->plan.n == n && c->plan.tile_log2 == c->tile_log2 && c->tof &&
           c->projector == 0 && c->plan.sigma == c->sigma && c->plan.trunc == c->trunc_sigmas;
}

// BASELINE.json north_star bullet 4: "the image kept L2-resident where it fits".  The correction image is the target of
// every reduction; a persisting access-policy window on it keeps its sectors from being evicted by the streaming event /
// record loads (ncu r04: the correction image was written back to DRAM ~20 times per pass).  Set once per (stream,
// pointer); TOFMLEM_OPT_L2_PERSIST = 0 switches it off.
void corr_l2_window(tofmlem_ctx *ctx, const float *d_corr, cudaStream_t s) {
    if (!ctx->l2_persist || (ctx->l2_ptr == d_corr && ctx->l2_stream == s)) return;
    ctx->l2_ptr = d_corr;
    ctx->l2_stream = s;
    int dev = 0, max_persist = 0, max_window = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&max_persist, cudaDevAttrMaxPersistingL2CacheSize, dev);
    cudaDeviceGetAttribute(&max_window, cudaDevAttrMaxAccessPolicyWindowSize, dev);
    size_t bytes = ctx->nvox * sizeof(float);
    if (max_persist <= 0 || max_window <= 0) return;
    size_t want = bytes < (size_t)max_persist ? bytes : (size_t)max_persist;
    cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, want);
    cudaStreamAttrValue attr;
    memset(&attr, 0, sizeof attr);
    attr.accessPolicyWindow.base_ptr = const_cast<float *>(d_corr);
    attr.accessPolicyWindow.num_bytes = bytes < (size_t)max_window ? bytes : (size_t)max_window;
    attr.accessPolicyWindow.hitRatio = (float)((double)want / (double)attr.accessPolicyWindow.num_bytes);
    if (attr.accessPolicyWindow.hitRatio > 1.0f) attr.accessPolicyWindow.hitRatio = 1.0f;
    attr.accessPolicyWindow.hitProp = cudaAccessPropertyPersisting;
    attr.accessPolicyWindow.missProp = cudaAccessPropertyStreaming;
    cudaStreamSetAttribute(s, cudaStreamAttributeAccessPolicyWindow, &attr);
    cudaGetLastError();  // not supported (e.g. MPS / MIG): the pass runs without the window
}

// One fused EM pass with the context's projector (0 = Siddon x Gaussian, 1 = K-sample kernel).
int em_pass(tofmlem_ctx *ctx, const ProjParams &p_in, const EventPtrs &ev, uint64_t n, const float *evw,
            const float *d_image, float *d_corr, bool vec, cudaStream_t s) {
    if (n == 0) return TOFMLEM_OK;
    ProjParams p = p_in;
    p.brick = bricks_on(ctx, d_corr) ? 1 : 0;
    corr_l2_window(ctx, d_corr, s);
    if (ctx->projector == 1) {
        int rc = ensure_lut(ctx);
        if (rc) return rc;
        launch_sampled_em(p, ctx->d_lut, ctx->samples_k, ev, n, evw, d_image, d_corr, ctx->d_stats, ctx->d_queues, s);
    } else if (warp_em_on(ctx)) {
        int rc = ensure_axis_scratch(ctx);
        if (rc) return rc;
        launch_warp_em(p, ev, n, evw, d_image, d_corr, ctx->d_axis, ctx->d_stats, s);
    } else if (plan_matches(ctx, ev.x1, n) && ctx->plan.brick == p.brick && ctx->em_variant == 0) {
        // Planned list (tofmlem_plan_events): the pass runs on the ray records -- the items on shared-memory tiles
        // (tile.cu), the other events and the stragglers of the items through the direct pass on records (prepared.cu).
        const int n_sm = ctx->n_sm > 0 ? ctx->n_sm : 1;
        if (!ctx->t_ev[0])
            for (auto &te : ctx->t_ev) CU(cudaEventCreate(&te));
        ctx->t_have = (ctx->plan.n_items ? 1 : 0) | (ctx->plan.direct_valid ? 2 : 0) | (ctx->plan.n_tiny ? 4 : 0);
        // TOFMLEM_OPT_CONCURRENT = k > 0: the direct pass (bound by L2 reduction requests, issue slots half idle) on a
        // second stream beside the tile pass (issue-bound, L2 idle), the tile pass limited to k CTAs per SM so that CTAs
        // of both fit an SM.  Both only add to the correction image and to the counters.
        cudaStream_t ds = s;
        const bool conc = ctx->concurrent > 0 && ctx->plan.n_items && ctx->plan.direct_valid;
        if (conc) {
            if (!ctx->side_stream) {
                CU(cudaStreamCreateWithFlags(&ctx->side_stream, cudaStreamNonBlocking));
                CU(cudaEventCreateWithFlags(&ctx->fork_ev, cudaEventDisableTiming));
                CU(cudaEventCreateWithFlags(&ctx->join_ev, cudaEventDisableTiming));
            }
            ds = ctx->side_stream;
            CU(cudaEventRecord(ctx->fork_ev, s));
            CU(cudaStreamWaitEvent(ds, ctx->fork_ev, 0));
        }
        CU(cudaEventRecord(ctx->t_ev[0], s));
        if (ctx->plan.n_items) {
            TileGeom g;
            build_tile_geom(p, ctx->tile_log2, ctx->smem_optin, ctx->smem_per_sm, g);  // as at plan time (sigma, trunc match)
            launch_em_tile(p, g, ctx->d_geom, ctx->tile_log2, ctx->d_rec, evw, d_image, d_corr, ctx->d_stats,
                           ctx->d_items, ctx->plan.n_items, ctx->d_plan_flags, n_sm, ctx->smem_per_sm,
                           ctx->tile_check != 0, ctx->sigma, ctx->plan.max_item_events, ctx->d_ev_scale,
                           conc ? ctx->concurrent : 0, s);
            CHECK_LAUNCH(1);
        }
        CU(cudaEventRecord(ctx->t_ev[1], s));
        if (ctx->plan.direct_valid) {
            launch_em_planned(p, ctx->d_rec, n, ctx->d_chunk_list, ctx->plan.n_pieces, evw, d_image, d_corr, vec,
                              ctx->d_stats, ctx->d_queues, n_sm, ctx->plan.n_items > 0, ds);
            CHECK_LAUNCH(1);
        }
        if (!conc) CU(cudaEventRecord(ctx->t_ev[2], s));
        if (ctx->plan.n_tiny) {  // kRecTiny: the unplanned walk (fp64 set-up), one event per piece
            launch_em_correction_chunks(p, true, ev, n, ctx->d_tiny, ctx->plan.n_tiny, evw, d_image, d_corr, vec,
                                        ctx->d_stats, ctx->d_queues, ds, true);
            CHECK_LAUNCH(1);
        }
        if (conc) {
            CU(cudaEventRecord(ctx->join_ev, ds));
            CU(cudaStreamWaitEvent(s, ctx->join_ev, 0));
            CU(cudaEventRecord(ctx->t_ev[2], s));  // [1] -> [2]: what the direct pass added after the tile pass ended
        }
        CU(cudaEventRecord(ctx->t_ev[3], s));
        return TOFMLEM_OK;
    } else {
        launch_em_correction(p, ctx->tof, ev, n, evw, d_image, d_corr, vec, ctx->d_stats, ctx->d_queues, s);
    }
    ctx->t_have = 0;
    CHECK_LAUNCH(1);
    return TOFMLEM_OK;
}

int median_in_place(tofmlem_ctx *ctx, float *d_image, cudaStream_t s) {
    if (!ctx->d_tmp_image) CU(cudaMalloc(&ctx->d_tmp_image, ctx->nvox * sizeof(float)));
    launch_median3(d_image, ctx->d_tmp_image, ctx->grid.nx, ctx->grid.ny, ctx->grid.nz, s);
    CHECK_LAUNCH(1);
    CU(cudaMemcpyAsync(d_image, ctx->d_tmp_image, ctx->nvox * sizeof(float), cudaMemcpyDeviceToDevice, s));
    return TOFMLEM_OK;
}

int iterate_device(tofmlem_ctx *ctx, const EventPtrs &ev, uint64_t n, const float *evw, float *d_image,
                   const float *d_sens, int iters, bool compute_max) {
    int rc = ensure_corr(ctx);
    if (rc) return rc;
    const ProjParams p = make_params(ctx, ctx->tof);
    const float *dmax = ctx->d_max_ext ? ctx->d_max_ext : ctx->d_max;
    if (compute_max && !ctx->d_max_ext) {
        launch_max_nonneg(d_sens, ctx->nvox, ctx->d_max, ctx->stream);
        CHECK_LAUNCH(1);
    }
    const bool det = ctx->deterministic && n > 0 && iters > 0;
    if (det) {
        if (!plan_matches(ctx, ev.x1, n))
            return fail(ctx, TOFMLEM_EUNSUPPORTED, "deterministic iterations need a planned list (tofmlem_plan_events)");
        if (!ctx->d_corr_q) {
            CU(cudaMalloc(&ctx->d_corr_q, ctx->nvox * sizeof(unsigned long long)));
            CU(cudaMalloc(&ctx->d_gscale, 4 * sizeof(float)));
        }
        CU(cudaMemsetAsync(ctx->d_corr_q, 0, ctx->nvox * sizeof(unsigned long long), ctx->stream));
    }
    CU(cudaMemsetAsync(ctx->d_corr, 0, ctx->nvox * sizeof(float), ctx->stream));
    for (int it = 0; it < iters; ++it) {
        CU(cudaMemsetAsync(ctx->d_stats, 0, kStatsCounters * sizeof(unsigned long long), ctx->stream));
        if (det) {
            // quanta per unit from max(image) alone (order-independent), integer pass, integer update
            launch_max_nonneg(d_image, ctx->nvox, ctx->d_gscale + 2, ctx->stream);
            launch_det_scale(ctx->d_gscale + 2, ctx->d_gscale, ctx->stream);
            launch_em_det(p, ctx->d_rec, n, evw, d_image, ctx->d_corr_q, ctx->d_gscale, ctx->d_stats, ctx->d_queues,
                          ctx->n_sm, ctx->stream);
            launch_update_det(d_image, ctx->d_corr_q, d_sens, dmax, (float)ctx->sens_floor_rel, ctx->d_gscale, ctx->nvox,
                              ctx->stream);
            CHECK_LAUNCH(4);
            ctx->t_have = 0;
        } else {
            rc = em_pass(ctx, p, ev, n, evw, d_image, ctx->d_corr, true, ctx->stream);
            if (rc) return rc;
            update_any(ctx, d_image, ctx->d_corr, d_sens, dmax, ctx->stream);
            CHECK_LAUNCH(1);
        }
        if (ctx->median) {  // the filter is applied to the image estimate after each iteration (R23)
            rc = median_in_place(ctx, d_image, ctx->stream);
            if (rc) return rc;
        }
    }
    launch_dot_f64(d_image, d_sens, ctx->nvox, &ctx->d_stats->sum_image_sens, ctx->stream);
    CHECK_LAUNCH(1);
    ctx->last_n = n;
    return TOFMLEM_OK;
}

}  // namespace

extern "C" {

const char *tofmlem_version(void) { return "tofmlem 0.1 (sm_100a)"; }

int tofmlem_create(const tofmlem_scanner *scanner, const tofmlem_grid *grid, float tof_fwhm_ps, void *cuda_stream,
                   tofmlem_ctx **out) {
    if (!scanner || !grid || !out) return TOFMLEM_EINVAL;
    *out = nullptr;
    if (grid->nx <= 0 || grid->ny <= 0 || grid->nz <= 0 || !(grid->vx > 0) || !(grid->vy > 0) || !(grid->vz > 0) ||
        !isfinite(grid->ox) || !isfinite(grid->oy) || !isfinite(grid->oz) || !(scanner->radius_mm > 0) ||
        !(scanner->axial_length_mm > 0) || isnan(tof_fwhm_ps))
        return TOFMLEM_EINVAL;
    const uint64_t nvox = (uint64_t)grid->nx * grid->ny * grid->nz;
    if (nvox >= (1ull << 31)) return TOFMLEM_EINVAL;
    tofmlem_ctx *ctx = new (std::nothrow) tofmlem_ctx;
    if (!ctx) return TOFMLEM_ENOMEM;
    ctx->scanner = *scanner;
    ctx->grid = *grid;
    ctx->tof = tof_fwhm_ps > 0.0f;
    ctx->sigma = ctx->tof ? sigma_from_fwhm(tof_fwhm_ps) : 0.0;
    ctx->stream = (cudaStream_t)cuda_stream;
    ctx->nvox = nvox;
    {
        int dev = 0, v = 0;
        if (cudaGetDevice(&dev) == cudaSuccess) {
            if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess) ctx->n_sm = v;
            if (cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) == cudaSuccess) ctx->smem_optin = (size_t)v;
            if (cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev) == cudaSuccess) ctx->smem_per_sm = (size_t)v;
        }
        cudaGetLastError();
    }
    cudaError_t e = cudaMalloc(&ctx->d_max, sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc(&ctx->d_stats, sizeof(DeviceStats));
    if (e == cudaSuccess) e = cudaMalloc(&ctx->d_queues, (size_t)kMaxQueues * kQueueStride * sizeof(unsigned));
    if (e == cudaSuccess) e = cudaMalloc(&ctx->d_rcounts, 2 * (kMaxRegions + 1) * sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMalloc(&ctx->d_plan_flags, 2 * sizeof(unsigned));
    if (e == cudaSuccess) e = cudaMalloc(&ctx->d_plan_counters, plan_counter_bytes());
    if (e == cudaSuccess) e = cudaMemsetAsync(ctx->d_stats, 0, sizeof(DeviceStats), ctx->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(ctx->d_max, 0, sizeof(float), ctx->stream);
    if (e != cudaSuccess) {
        int rc = e == cudaErrorMemoryAllocation ? TOFMLEM_ENOMEM : TOFMLEM_ECUDA;
        cudaFree(ctx->d_max);
        cudaFree(ctx->d_stats);
        cudaFree(ctx->d_queues);
        cudaFree(ctx->d_rcounts);
        cudaFree(ctx->d_plan_flags);
        cudaFree(ctx->d_plan_counters);
        delete ctx;
        return rc;
    }
    *out = ctx;
    return TOFMLEM_OK;
}

int tofmlem_destroy(tofmlem_ctx *ctx) {
    if (!ctx) return TOFMLEM_OK;
    cudaStreamSynchronize(ctx->stream);
    if (ctx->copy_stream) {
        cudaStreamSynchronize(ctx->copy_stream);
        cudaStreamDestroy(ctx->copy_stream);
    }
    for (auto &ev : ctx->chunk_done)
        if (ev) cudaEventDestroy(ev);
    cudaFree(ctx->d_corr);
    cudaFree(ctx->d_max);
    cudaFree(ctx->d_stats);
    cudaFree(ctx->d_queues);
    cudaFree(ctx->d_hist);
    cudaFree(ctx->d_cursor);
    cudaFree(ctx->d_scan_tmp);
    cudaFree(ctx->d_sub);
    cudaFree(ctx->d_pack);
    cudaFree(ctx->d_rg_region);
    cudaFree(ctx->d_rg_perm);
    cudaFree(ctx->d_rg_sorted);
    cudaFree(ctx->d_rg_binned);
    cudaFree(ctx->d_tmp_image);
    cudaFree(ctx->d_axis);
    cudaFree(ctx->d_lut);
    cudaFree(ctx->d_rcounts);
    cudaFree(ctx->d_hev);
    cudaFree(ctx->d_himg);
    cudaFree(ctx->d_hsens);
    cudaFree(ctx->d_plan_flags);
    cudaFree(ctx->d_geom);
    cudaFree(ctx->d_items);
    cudaFree(ctx->d_ranges);
    if (ctx->h_hist_pinned) cudaFreeHost(ctx->h_hist_pinned);
    cudaFree(ctx->d_plan_counters);
    cudaFree(ctx->d_corr_q);
    cudaFree(ctx->d_gscale);
    if (ctx->side_stream) {
        cudaStreamSynchronize(ctx->side_stream);
        cudaStreamDestroy(ctx->side_stream);
        cudaEventDestroy(ctx->fork_ev);
        cudaEventDestroy(ctx->join_ev);
    }
    for (auto &te : ctx->t_ev)
        if (te) cudaEventDestroy(te);
    free_records(ctx);
    free_region_cache(ctx);
    delete ctx;
    return TOFMLEM_OK;
}

int tofmlem_set_option(tofmlem_ctx *ctx, int key, double value) {
    if (!ctx) return TOFMLEM_EINVAL;
    switch (key) {
        case TOFMLEM_OPT_TRUNC_SIGMAS:
            if (!(value > 0.0) || !isfinite(value)) return fail(ctx, TOFMLEM_EINVAL, "trunc_sigmas must be > 0");
            ctx->trunc_sigmas = value;
            return TOFMLEM_OK;
        case TOFMLEM_OPT_SENS_FLOOR_REL:
            if (!(value >= 0.0) || !(value <= 1.0)) return fail(ctx, TOFMLEM_EINVAL, "sens_floor_rel in [0,1]");
            ctx->sens_floor_rel = value;
            return TOFMLEM_OK;
        case TOFMLEM_OPT_TILE_LOG2:
            if (value < 0 || value > 8 || value != floor(value)) return fail(ctx, TOFMLEM_EINVAL, "tile_log2 in 0..8");
            ctx->tile_log2 = (int)value;
            return TOFMLEM_OK;
        case TOFMLEM_OPT_PROJECTOR:
            if (value != 0.0 && value != 1.0) return fail(ctx, TOFMLEM_EINVAL, "projector is 0 (Siddon) or 1 (K samples)");
            if (value == 1.0 && !ctx->tof) return fail(ctx, TOFMLEM_EUNSUPPORTED, "the K-sample kernel needs a TOF context");
            ctx->projector = (int)value;
            return TOFMLEM_OK;
        case TOFMLEM_OPT_SAMPLES_K:
            if (value < 1 || value > 1024 || value != floor(value)) return fail(ctx, TOFMLEM_EINVAL, "K in 1..1024");
            ctx->samples_k = (int)value;
            return TOFMLEM_OK;
        case TOFMLEM_OPT_SHELL_MM:
            if (!(value >= 0.0) || !isfinite(value)) return fail(ctx, TOFMLEM_EINVAL, "shell_mm must be >= 0");
            ctx->shell_mm = value;
            return TOFMLEM_OK;
        case TOFMLEM_OPT_CTA_INTERLEAVE:
            if (value < 1 || value > 65536 || value != floor(value)) return fail(ctx, TOFMLEM_EINVAL, "cta_interleave in 1..65536");
            ctx->cta_interleave = (unsigned)value;
            return TOFMLEM_OK;
        case TOFMLEM_OPT_EM_VARIANT:
            if (value < 0 || value > 2 || value != floor(value)) return fail(ctx, TOFMLEM_EINVAL, "em_variant in 0..2");
            ctx->em_variant = (int)value;
            return TOFMLEM_OK;
        case TOFMLEM_OPT_CORR_BRICKS:
            if (value != 0.0 && value != 1.0) return fail(ctx, TOFMLEM_EINVAL, "corr_bricks is 0 or 1");
            ctx->corr_bricks = (int)value;
            return TOFMLEM_OK;
        case TOFMLEM_OPT_CACHE_SHARE:
            if (value < 0 || value > 8 || value != floor(value)) return fail(ctx, TOFMLEM_EINVAL, "cache_share in 0..8");
            ctx->cache_share = (int)value;
            return TOFMLEM_OK;
        case TOFMLEM_OPT_MEDIAN:
            if (value != 0.0 && value != 1.0) return fail(ctx, TOFMLEM_EINVAL, "median is 0 or 1");
            ctx->median = (int)value;
            return TOFMLEM_OK;
        case TOFMLEM_OPT_SUBBINS:
            if (value < 1 || value > 64 || value != floor(value)) return fail(ctx, TOFMLEM_EINVAL, "subbins in 1..64");
            ctx->subbins = (int)value;
            return TOFMLEM_OK;
        case TOFMLEM_OPT_TILE_MIN_EVENTS:
            if (value < 1 || value > 1e9 || value != floor(value)) return fail(ctx, TOFMLEM_EINVAL, "tile_min_events in 1..1e9");
            ctx->tile_min_events = (int)value;
            return TOFMLEM_OK;
        case TOFMLEM_OPT_TILE_MAX_EVENTS:
            if (value < 32 || value > 1e9 || value != floor(value)) return fail(ctx, TOFMLEM_EINVAL, "tile_max_events in 32..1e9");
            ctx->tile_max_events = (int)value;
            return TOFMLEM_OK;
        case TOFMLEM_OPT_CONCURRENT:
            if (value < 0 || value > 4 || value != floor(value)) return fail(ctx, TOFMLEM_EINVAL, "concurrent in 0..4");
            ctx->concurrent = (int)value;
            return TOFMLEM_OK;
        case TOFMLEM_OPT_WARP_WALK:
            if (value != 0.0 && value != 1.0) return fail(ctx, TOFMLEM_EINVAL, "warp_walk is 0 or 1");
            ctx->warp_walk = (int)value;
            return TOFMLEM_OK;
        case TOFMLEM_OPT_SENS_SORT:
            if (value != 0.0 && value != 1.0) return fail(ctx, TOFMLEM_EINVAL, "sens_sort is 0 or 1");
            ctx->sens_sort = (int)value;
            return TOFMLEM_OK;
        case TOFMLEM_OPT_TILE_MIN_ITEMS:
            if (value < -1 || value > 1e9 || value != floor(value)) return fail(ctx, TOFMLEM_EINVAL, "tile_min_items in -1..1e9");
            ctx->tile_min_items = (int)value;
            return TOFMLEM_OK;
        case TOFMLEM_OPT_TILE_CHECK:
            if (value != 0.0 && value != 1.0) return fail(ctx, TOFMLEM_EINVAL, "tile_check is 0 or 1");
            ctx->tile_check = (int)value;
            return TOFMLEM_OK;
        case TOFMLEM_OPT_L2_PERSIST:
            if (value != 0.0 && value != 1.0) return fail(ctx, TOFMLEM_EINVAL, "l2_persist is 0 or 1");
            ctx->l2_persist = (int)value;
            ctx->l2_ptr = nullptr;
            if (!ctx->l2_persist) {
                cudaStreamAttrValue attr;
                memset(&attr, 0, sizeof attr);
                cudaStreamSetAttribute(ctx->stream, cudaStreamAttributeAccessPolicyWindow, &attr);
                cudaCtxResetPersistingL2Cache();
                cudaGetLastError();
            }
            return TOFMLEM_OK;
        case TOFMLEM_OPT_REGION_OVERLAP:
            if (value != 0.0 && value != 1.0) return fail(ctx, TOFMLEM_EINVAL, "region_overlap is 0 or 1");
            ctx->region_overlap = (int)value;
            return TOFMLEM_OK;
        case TOFMLEM_OPT_REGION_PLAN:
            if (value != 0.0 && value != 1.0 && value != 2.0) return fail(ctx, TOFMLEM_EINVAL, "region_plan is 0, 1 or 2");
            ctx->region_plan = (int)value;
            return TOFMLEM_OK;
        case TOFMLEM_OPT_DETERMINISTIC:
            // the paper's LUT kernel "always generated an identically reconstructed image".  1: the
            // iterations of tofmlem_iterate[_weighted] on a PLANNED list accumulate in 64-bit integers (prepared.cu,
            // em_det_kernel): run-to-run bit-identical images.  The float32 paths stay unordered.
            if (value != 0.0 && value != 1.0) return fail(ctx, TOFMLEM_EINVAL, "deterministic is 0 or 1");
            if (value == 1.0 && (!ctx->tof || ctx->projector != 0))
                return fail(ctx, TOFMLEM_EUNSUPPORTED, "deterministic accumulation exists for the TOF Siddon projector only");
            ctx->deterministic = (int)value;
            return TOFMLEM_OK;
        default:
            return fail(ctx, TOFMLEM_EINVAL, "unknown option key");
    }
}

double tofmlem_sigma_mm(const tofmlem_ctx *ctx) { return ctx ? ctx->sigma : 0.0; }

int tofmlem_reserve(tofmlem_ctx *ctx, uint64_t n_events) {
    if (!ctx || n_events > 0xFFFFFFFFull) return TOFMLEM_EINVAL;
    int rc = ensure_corr(ctx);
    if (rc) return rc;
    if (warp_on(ctx)) {  // axis-fastest scratch of the whole-chord walks (sensitivity, attenuation weights, non-TOF passes)
        rc = ensure_axis_scratch(ctx);
        if (rc) return rc;
    }
    if (n_events) {
        const uint32_t S = effective_subbins(ctx);
        rc = ensure_bin_scratch(ctx, (size_t)num_bins(ctx) * S + 1, S > 1 ? n_events : 0);
        if (rc) return rc;
        if (!ensure_pack(ctx, n_events)) return fail(ctx, TOFMLEM_ENOMEM, "reserve: no memory for the 32-byte event records");
        if (ctx->tof && ctx->projector == 0) {  // tofmlem_plan_events: ray records and their side arrays, pinned bin counts
            rc = ensure_plan_scratch(ctx, n_events);
            if (rc) return rc;
        }
    }
    return TOFMLEM_OK;
}

int tofmlem_trim(tofmlem_ctx *ctx) {
    if (!ctx) return TOFMLEM_EINVAL;
    CU(cudaStreamSynchronize(ctx->stream));
    if (ctx->copy_stream) CU(cudaStreamSynchronize(ctx->copy_stream));
    cudaFree(ctx->d_pack);
    cudaFree(ctx->d_sub);
    cudaFree(ctx->d_rg_region);
    cudaFree(ctx->d_rg_perm);
    cudaFree(ctx->d_rg_sorted);
    cudaFree(ctx->d_rg_binned);
    cudaFree(ctx->d_tmp_image);
    cudaFree(ctx->d_axis);
    ctx->d_axis = nullptr;
    cudaFree(ctx->d_hev);
    cudaFree(ctx->d_himg);
    cudaFree(ctx->d_hsens);
    free_records(ctx);  // the plan goes with its records
    free_region_cache(ctx);
    ctx->d_pack = nullptr;
    ctx->d_sub = nullptr;
    ctx->d_rg_region = nullptr;
    ctx->d_rg_perm = nullptr;
    ctx->d_rg_sorted = ctx->d_rg_binned = nullptr;
    ctx->d_tmp_image = nullptr;
    ctx->d_hev = ctx->d_himg = ctx->d_hsens = nullptr;
    ctx->pack_cap = ctx->sub_cap = ctx->rg_cap = ctx->hev_cap = 0;
    return TOFMLEM_OK;
}

int tofmlem_sensitivity(tofmlem_ctx *ctx, const tofmlem_events *lors, uint64_t m, float *d_sens) {
    if (!ctx) return TOFMLEM_EINVAL;
    if (!ev_ok(lors, false) || !d_sens || m == 0 || m > 0xFFFFFFFFull) return fail(ctx, TOFMLEM_EINVAL, "sensitivity: bad argument");
    const ProjParams p = make_params(ctx, false);
    CU(cudaMemsetAsync(d_sens, 0, ctx->nvox * sizeof(float), ctx->stream));
    EventPtrs ev = ev_ptrs(lors);
    ev.dt = nullptr;
    // Random detector pairs give chords of 0 .. 900 voxels side by side in a warp (ncu r05: 11 of 32 lanes active, the
    // sensitivity image written back to DRAM 700 times).  Order the LORs first: locality key of the chord's midpoint,
    // sub-bins by the chord's visit count (the binning of a1 with dt = 0 and whole-chord sub-bins), 32 B per LOR of scratch
    // for the duration of the call.  The result is the same up to the order of the float32 sums.
    uint32_t *d_key = nullptr, *d_perm = nullptr;
    float *d_sorted = nullptr;
    if (ctx->sens_sort && m >= (1u << 18)) {
        const uint64_t stride = (m + 3) & ~3ull;
        if (cudaMalloc(&d_key, m * sizeof(uint32_t)) == cudaSuccess && cudaMalloc(&d_perm, m * sizeof(uint32_t)) == cudaSuccess &&
            cudaMalloc(&d_sorted, 6 * stride * sizeof(float)) == cudaSuccess) {
            tofmlem_events in = *lors;
            in.dt = nullptr;
            tofmlem_events_mut out{d_sorted, d_sorted + stride, d_sorted + 2 * stride, d_sorted + 3 * stride,
                                   d_sorted + 4 * stride, d_sorted + 5 * stride, nullptr};
            ctx->bin_whole_chords = true;
            int rc = tofmlem_bin_events(ctx, &in, m, d_key, d_perm, nullptr);
            ctx->bin_whole_chords = false;
            if (rc == TOFMLEM_OK) rc = tofmlem_permute_events(ctx, &in, d_perm, m, &out);
            if (rc == TOFMLEM_OK) {
                ev = EventPtrs{out.x1, out.y1, out.z1, out.x2, out.y2, out.z2, nullptr};
            } else {
                cudaGetLastError();
            }
        } else {
            cudaGetLastError();  // not enough memory for the scratch: the LORs as they come
        }
    }
    if (warp_on(ctx)) {
        int rc = ensure_axis_scratch(ctx);
        if (rc) return rc;
        launch_warp_backproject(p, ev, m, nullptr, d_sens, ctx->d_axis, ctx->stream);
    } else {
        launch_backproject(p, false, ev, m, nullptr, d_sens, vec_ok(ctx, d_sens), ctx->stream);
    }
    if (d_key || d_perm || d_sorted) {
        cudaStreamSynchronize(ctx->stream);
        cudaFree(d_key);
        cudaFree(d_perm);
        cudaFree(d_sorted);
    }
    CHECK_LAUNCH(1);
    launch_scale(d_sens, (float)(1.0 / (double)m), ctx->nvox, ctx->stream);
    CHECK_LAUNCH(1);
    return TOFMLEM_OK;
}

int tofmlem_forward(tofmlem_ctx *ctx, const tofmlem_events *ev, uint64_t n, const float *d_image, float *d_fwd) {
    if (!ctx) return TOFMLEM_EINVAL;
    if (n == 0) return TOFMLEM_OK;
    if (!ev_ok(ev, ctx->tof) || !d_image || !d_fwd || n > 0xFFFFFFFFull) return fail(ctx, TOFMLEM_EINVAL, "forward: bad argument");
    if (ctx->projector == 1) {
        int rc = ensure_lut(ctx);
        if (rc) return rc;
        launch_sampled_forward(make_params(ctx, true), ctx->d_lut, ctx->samples_k, ev_ptrs(ev), n, d_image, d_fwd,
                               ctx->stream);
    } else if (plan_matches(ctx, ev->x1, n)) {  // planned list: the walk of the fused pass, on the ray records
        launch_planned_forward(make_params(ctx, true), ctx->sigma, ev_ptrs(ev), ctx->d_rec, n, d_image, d_fwd, ctx->stream);
    } else if (!ctx->tof && warp_on(ctx)) {
        int rc = ensure_axis_scratch(ctx);
        if (rc) return rc;
        launch_warp_forward(make_params(ctx, false), ev_ptrs(ev), n, d_image, d_fwd, ctx->d_axis, ctx->stream);
    } else {
        launch_forward(make_params(ctx, ctx->tof), ctx->tof, ev_ptrs(ev), n, d_image, d_fwd, ctx->stream);
    }
    CHECK_LAUNCH(1);
    return TOFMLEM_OK;
}

int tofmlem_backproject(tofmlem_ctx *ctx, const tofmlem_events *ev, uint64_t n, const float *d_values, float *d_out) {
    if (!ctx) return TOFMLEM_EINVAL;
    if (n == 0) return TOFMLEM_OK;
    if (!ev_ok(ev, ctx->tof) || !d_out || n > 0xFFFFFFFFull) return fail(ctx, TOFMLEM_EINVAL, "backproject: bad argument");
    if (ctx->projector == 1) {
        int rc = ensure_lut(ctx);
        if (rc) return rc;
        launch_sampled_backproject(make_params(ctx, true), ctx->d_lut, ctx->samples_k, ev_ptrs(ev), n, d_values, d_out,
                                   ctx->stream);
    } else if (!ctx->tof && warp_on(ctx)) {
        int rc = ensure_axis_scratch(ctx);
        if (rc) return rc;
        launch_warp_backproject(make_params(ctx, false), ev_ptrs(ev), n, d_values, d_out, ctx->d_axis, ctx->stream);
    } else {
        launch_backproject(make_params(ctx, ctx->tof), ctx->tof, ev_ptrs(ev), n, d_values, d_out, vec_ok(ctx, d_out),
                           ctx->stream);
    }
    CHECK_LAUNCH(1);
    return TOFMLEM_OK;
}

int tofmlem_reset_stats(tofmlem_ctx *ctx) {
    if (!ctx) return TOFMLEM_EINVAL;
    CU(cudaMemsetAsync(ctx->d_stats, 0, sizeof(DeviceStats), ctx->stream));
    ctx->last_n = 0;
    return TOFMLEM_OK;
}

int tofmlem_em_correction_weighted(tofmlem_ctx *ctx, const tofmlem_events *ev, uint64_t n, const float *d_weight,
                                   const float *d_image, float *d_corr) {
    if (!ctx) return TOFMLEM_EINVAL;
    if (n == 0) return TOFMLEM_OK;
    if (!ev_ok(ev, ctx->tof) || !d_image || !d_corr || n > 0xFFFFFFFFull) return fail(ctx, TOFMLEM_EINVAL, "em_correction: bad argument");
    int rc = em_pass(ctx, make_params(ctx, ctx->tof), ev_ptrs(ev), n, d_weight, d_image, d_corr, vec_ok(ctx, d_corr),
                     ctx->stream);
    if (rc) return rc;
    ctx->last_n += n;
    return TOFMLEM_OK;
}

int tofmlem_em_correction(tofmlem_ctx *ctx, const tofmlem_events *ev, uint64_t n, const float *d_image, float *d_corr) {
    return tofmlem_em_correction_weighted(ctx, ev, n, nullptr, d_image, d_corr);
}

int tofmlem_update(tofmlem_ctx *ctx, float *d_image, float *d_corr, const float *d_sens) {
    if (!ctx) return TOFMLEM_EINVAL;
    if (!d_image || !d_corr || !d_sens) return fail(ctx, TOFMLEM_EINVAL, "update: NULL argument");
    if (!update_aligned(ctx, d_image, d_corr, d_sens))
        return fail(ctx, TOFMLEM_EINVAL, "update: d_image and d_sens must be 8-byte aligned with the brick layout of d_corr");
    launch_max_nonneg(d_sens, ctx->nvox, ctx->d_max, ctx->stream);
    CHECK_LAUNCH(1);
    update_any(ctx, d_image, d_corr, d_sens, ctx->d_max, ctx->stream);
    CHECK_LAUNCH(1);
    return TOFMLEM_OK;
}

int tofmlem_iterate_weighted(tofmlem_ctx *ctx, const tofmlem_events *ev, uint64_t n, const float *d_weight,
                             float *d_image, const float *d_sens, int iters) {
    if (!ctx) return TOFMLEM_EINVAL;
    if ((n && !ev_ok(ev, ctx->tof)) || !d_image || !d_sens || iters < 0 || n > 0xFFFFFFFFull || d_image == d_sens)
        return fail(ctx, TOFMLEM_EINVAL, "iterate: bad argument");
    if (((reinterpret_cast<uintptr_t>(d_image) | reinterpret_cast<uintptr_t>(d_sens)) & 7) != 0)
        return fail(ctx, TOFMLEM_EINVAL, "iterate: d_image and d_sens must be 8-byte aligned");
    EventPtrs p = n ? ev_ptrs(ev) : EventPtrs{};
    return iterate_device(ctx, p, n, d_weight, d_image, d_sens, iters, true);
}

int tofmlem_iterate(tofmlem_ctx *ctx, const tofmlem_events *ev, uint64_t n, float *d_image, const float *d_sens,
                    int iters) {
    return tofmlem_iterate_weighted(ctx, ev, n, nullptr, d_image, d_sens, iters);
}

int tofmlem_median3(tofmlem_ctx *ctx, const float *d_in, float *d_out) {
    if (!ctx) return TOFMLEM_EINVAL;
    if (!d_in || !d_out || d_in == d_out) return fail(ctx, TOFMLEM_EINVAL, "median3: NULL or aliased argument");
    launch_median3(d_in, d_out, ctx->grid.nx, ctx->grid.ny, ctx->grid.nz, ctx->stream);
    CHECK_LAUNCH(1);
    return TOFMLEM_OK;
}

int tofmlem_attenuation_weights(tofmlem_ctx *ctx, const tofmlem_events *lors, uint64_t n, const float *d_mu,
                                float *d_weight) {
    if (!ctx) return TOFMLEM_EINVAL;
    if (n == 0) return TOFMLEM_OK;
    if (!ev_ok(lors, false) || !d_mu || !d_weight || n > 0xFFFFFFFFull)
        return fail(ctx, TOFMLEM_EINVAL, "attenuation_weights: bad argument");
    EventPtrs ev = ev_ptrs(lors);
    ev.dt = nullptr;
    if (warp_on(ctx)) {  // line integral of mu
        int rc = ensure_axis_scratch(ctx);
        if (rc) return rc;
        launch_warp_forward(make_params(ctx, false), ev, n, d_mu, d_weight, ctx->d_axis, ctx->stream);
    } else {
        launch_forward(make_params(ctx, false), false, ev, n, d_mu, d_weight, ctx->stream);
    }
    CHECK_LAUNCH(1);
    launch_exp(d_weight, n, ctx->stream);
    CHECK_LAUNCH(1);
    return TOFMLEM_OK;
}

int tofmlem_gather_f32(tofmlem_ctx *ctx, const float *d_in, const uint32_t *d_perm, uint64_t n, float *d_out) {
    if (!ctx) return TOFMLEM_EINVAL;
    if (n == 0) return TOFMLEM_OK;
    if (!d_in || !d_perm || !d_out || d_in == d_out) return fail(ctx, TOFMLEM_EINVAL, "gather_f32: bad argument");
    launch_gather(d_in, d_perm, n, d_out, ctx->stream);
    CHECK_LAUNCH(1);
    return TOFMLEM_OK;
}

int tofmlem_scatter_reject(tofmlem_ctx *ctx, const tofmlem_events *ev, uint64_t n, const float *h_ellipsoids,
                           int n_ellipsoids, float half_width_mm, uint8_t *d_keep, uint32_t *d_perm,
                           uint64_t *h_n_kept) {
    if (!ctx) return TOFMLEM_EINVAL;
    if ((n && !ev_ok(ev, true)) || !h_ellipsoids || n_ellipsoids < 1 || n_ellipsoids > kMaxEllipsoids ||
        (n && !d_keep) || !h_n_kept || n > 0xFFFFFFFFull || isnan(half_width_mm))
        return fail(ctx, TOFMLEM_EINVAL, "scatter_reject: bad argument");
    EllipsoidSet es;
    es.n = n_ellipsoids;
    for (int i = 0; i < 6 * n_ellipsoids; ++i) es.v[i] = h_ellipsoids[i];
    // default half width: the two-sided 95 % point of the TOF Gaussian ("95% confidence level")
    const float h = half_width_mm > 0.0f ? half_width_mm : (float)(1.959964 * ctx->sigma);
    unsigned long long *counter = ctx->d_rcounts;
    CU(cudaMemsetAsync(counter, 0, sizeof(unsigned long long), ctx->stream));
    if (n) {
        launch_scatter_keep(ev_ptrs(ev), n, es, h, d_keep, d_perm, counter, ctx->stream);
        CHECK_LAUNCH(1);
    }
    unsigned long long kept = 0;
    CU(cudaMemcpyAsync(&kept, counter, sizeof kept, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    *h_n_kept = kept;
    return TOFMLEM_OK;
}

int tofmlem_iterate_host(tofmlem_ctx *ctx, const tofmlem_events *h_ev, uint64_t n, float *h_image,
                         const float *h_sens, int iters) {
    if (!ctx) return TOFMLEM_EINVAL;
    if ((n && !ev_ok(h_ev, ctx->tof)) || !h_image || !h_sens || iters < 0 || n > 0xFFFFFFFFull)
        return fail(ctx, TOFMLEM_EINVAL, "iterate_host: bad argument");
    const size_t vbytes = ctx->nvox * sizeof(float);
    if (!ctx->copy_stream) {
        CU(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
        for (auto &e : ctx->chunk_done) CU(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    }
    if (!ctx->d_himg) {
        CU(cudaMalloc(&ctx->d_himg, vbytes));
        CU(cudaMalloc(&ctx->d_hsens, vbytes));
    }
    const uint64_t stride = (n + 3) & ~3ull;  // keep every member array 16-byte aligned
    if (ctx->hev_cap < 7 * stride) {
        cudaFree(ctx->d_hev);
        ctx->d_hev = nullptr;
        ctx->hev_cap = 0;
        CU(cudaMalloc(&ctx->d_hev, 7 * stride * sizeof(float) + 16));
        ctx->hev_cap = 7 * stride;
    }
    int rc = ensure_corr(ctx);
    if (rc) return rc;
    cudaStream_t s = ctx->stream, cs = ctx->copy_stream;
    CU(cudaMemcpyAsync(ctx->d_himg, h_image, vbytes, cudaMemcpyHostToDevice, s));
    CU(cudaMemcpyAsync(ctx->d_hsens, h_sens, vbytes, cudaMemcpyHostToDevice, s));
    launch_max_nonneg(ctx->d_hsens, ctx->nvox, ctx->d_max, s);
    CHECK_LAUNCH(1);
    CU(cudaMemsetAsync(ctx->d_corr, 0, vbytes, s));
    CU(cudaMemsetAsync(ctx->d_stats, 0, sizeof(DeviceStats), s));
    float *d = ctx->d_hev;
    tofmlem_events dev{d, d + stride, d + 2 * stride, d + 3 * stride, d + 4 * stride, d + 5 * stride,
                       h_ev && h_ev->dt ? d + 6 * stride : nullptr};
    const float *hsrc[7] = {n ? h_ev->x1 : nullptr, n ? h_ev->y1 : nullptr, n ? h_ev->z1 : nullptr,
                            n ? h_ev->x2 : nullptr, n ? h_ev->y2 : nullptr, n ? h_ev->z2 : nullptr,
                            n ? h_ev->dt : nullptr};
    const ProjParams p = make_params(ctx, ctx->tof);
    if (iters > 0 && n > 0) {
        // first pass: upload chunk k+1 on the copy stream while chunk k is projected on the compute stream
        const uint64_t chunk = 8ull << 20;
        int slot = 0;
        for (uint64_t off = 0; off < n; off += chunk, slot ^= 1) {
            const uint64_t m = n - off < chunk ? n - off : chunk;
            for (int f = 0; f < 7; ++f)
                if (hsrc[f])
                    CU(cudaMemcpyAsync(d + f * stride + off, hsrc[f] + off, m * sizeof(float), cudaMemcpyHostToDevice, cs));
            CU(cudaEventRecord(ctx->chunk_done[slot], cs));
            CU(cudaStreamWaitEvent(s, ctx->chunk_done[slot], 0));
            rc = em_pass(ctx, p, ev_ptrs(&dev, off), m, nullptr, ctx->d_himg, ctx->d_corr, true, s);
            if (rc) return rc;
        }
        update_any(ctx, ctx->d_himg, ctx->d_corr, ctx->d_hsens, ctx->d_max, s);
        CHECK_LAUNCH(1);
        if (ctx->median && (rc = median_in_place(ctx, ctx->d_himg, s))) return rc;
        for (int it = 1; it < iters; ++it) {
            CU(cudaMemsetAsync(ctx->d_stats, 0, kStatsCounters * sizeof(unsigned long long), s));
            rc = em_pass(ctx, p, ev_ptrs(&dev), n, nullptr, ctx->d_himg, ctx->d_corr, true, s);
            if (rc) return rc;
            update_any(ctx, ctx->d_himg, ctx->d_corr, ctx->d_hsens, ctx->d_max, s);
            CHECK_LAUNCH(1);
            if (ctx->median && (rc = median_in_place(ctx, ctx->d_himg, s))) return rc;
        }
    } else if (iters > 0) {
        for (int it = 0; it < iters; ++it) {
            update_any(ctx, ctx->d_himg, ctx->d_corr, ctx->d_hsens, ctx->d_max, s);
            CHECK_LAUNCH(1);
        }
    }
    launch_dot_f64(ctx->d_himg, ctx->d_hsens, ctx->nvox, &ctx->d_stats->sum_image_sens, s);
    CHECK_LAUNCH(1);
    CU(cudaMemcpyAsync(h_image, ctx->d_himg, vbytes, cudaMemcpyDeviceToHost, s));
    CU(cudaStreamSynchronize(s));
    ctx->last_n = n;
    return TOFMLEM_OK;
}

// tofmlem_plan_events in three phases, so that a caller with several contexts on several streams
// (tofmlem_reconstruct_regions) can enqueue phase 1 everywhere, then phase 2 everywhere, then phase 3: each phase ends with
// asynchronous copies to the host, and the NEXT phase starts after a synchronisation of the context's stream -- two rounds
// of waiting in all instead of two per context with the other streams idle meanwhile.
//   plan_begin  : validation, scratch, key histogram of the list -> host (asynchronous).  1 = nothing to plan, 0 = started.
//   plan_build  : (stream synchronised) tile items from the bin counts; ray records, dry run, piece list -> counters to host
//   plan_finish : (stream synchronised) the plan becomes valid
namespace {

int plan_begin(tofmlem_ctx *ctx, const tofmlem_events *ev, uint64_t n) {
    ctx->plan.valid = false;
    ctx->plan.n_items = ctx->plan.n_strag = 0;
    ctx->plan.direct_valid = 0;
    ctx->plan.tile_events = ctx->plan.direct_events = ctx->plan.valid_events = ctx->plan.visits = 0;
    ctx->plan.sorted = 0;
    if (n == 0) return 1;
    if (!ev_ok(ev, ctx->tof) || n > 0xFFFFFFFFull) return fail(ctx, TOFMLEM_EINVAL, "plan_events: bad argument");
    if (!ctx->tof || ctx->projector != 0) return 1;  // records exist for the TOF Siddon pass only
    auto &J = ctx->job;
    J.ev = *ev;
    J.n = n;
    J.p = make_params(ctx, true);
    // the layout the context's own correction image will have (ensure_corr aligns it): decides which group count the
    // direct records carry; a pass into another layout ignores the plan
    J.p.brick = ctx->corr_bricks && (ctx->grid.nx & 1) == 0 && (ctx->grid.ny & 1) == 0 && (ctx->nvox & 3) == 0 ? 1 : 0;
    build_tile_geom(J.p, ctx->tile_log2, ctx->smem_optin, ctx->smem_per_sm, J.g);
    cudaStream_t s = ctx->stream;
    {
        int rc0 = ensure_plan_scratch(ctx, n);
        if (rc0) return rc0;
    }
    J.items.clear();
    J.ranges.clear();
    J.flags[0] = J.flags[1] = 0;
    // ---- which bins become tile items?  Needs a list sorted by key (tofmlem_permute_events) and tiles that fit.
    if (J.g.ok) {
        const uint32_t nb = num_bins(ctx);
        int rc = ensure_bin_scratch(ctx, (size_t)nb + 1, 0);
        if (rc) return rc;
        CU(cudaMemsetAsync(ctx->d_hist, 0, ((size_t)nb + 1) * sizeof(uint32_t), s));
        CU(cudaMemsetAsync(ctx->d_plan_flags, 0, 2 * sizeof(unsigned), s));
        launch_plan_hist(grid_f32(ctx), ctx->tile_log2, ev_ptrs(ev), n, ctx->d_hist, nb, ctx->d_plan_flags + 1, s);
        CHECK_LAUNCH(1);
        CU(cudaMemcpyAsync(ctx->h_hist_pinned, ctx->d_hist, (size_t)nb * sizeof(uint32_t), cudaMemcpyDeviceToHost, s));
        CU(cudaMemcpyAsync(J.flags, ctx->d_plan_flags, sizeof J.flags, cudaMemcpyDeviceToHost, s));
    }
    return 0;
}

int plan_build(tofmlem_ctx *ctx) {
    auto &J = ctx->job;
    const TileGeom &g = J.g;
    const ProjParams &p = J.p;
    const tofmlem_events *ev = &J.ev;
    const uint64_t n = J.n;
    cudaStream_t s = ctx->stream;
    std::vector<TileItem> &items = J.items;
    std::vector<TileRange> &ranges = J.ranges;
    bool sorted = false;
    if (g.ok) {
        const uint32_t nb = num_bins(ctx);
        const uint32_t *cnt = ctx->h_hist_pinned;
        sorted = J.flags[1] == 0;
        if (sorted) {
            // Tile items: a bin with at least tile_min_events events (pieces of at most tile_max_events, whole warps), or
            // a PAIR of bins that are neighbours along the class's dominant axis and hold tile_min_events .. tile_max_events
            // events together (one tile, T planes longer: the per-item cost is shared by more events and bins too sparse
            // on their own become tile work).  Maximal runs of the other bins are cut into 32-event pieces for the
            // direct pass.
            const uint32_t thr = (uint32_t)ctx->tile_min_events, mx = (uint32_t)ctx->tile_max_events;
            const int t = 1 << ctx->tile_log2;
            const uint32_t Tx = (uint32_t)((ctx->grid.nx + t - 1) >> ctx->tile_log2),
                           Ty = (uint32_t)((ctx->grid.ny + t - 1) >> ctx->tile_log2),
                           Tz = (uint32_t)((ctx->grid.nz + t - 1) >> ctx->tile_log2), T3 = Tx * Ty * Tz;
            const auto add_pieces = [&](uint64_t first, uint32_t c, uint32_t b) {
                const uint32_t pieces = (c + mx - 1) / mx;
                uint32_t per = (c + pieces - 1) / pieces;
                per = (per + 31u) & ~31u;
                for (uint32_t k = 0; k < c; k += per)
                    items.push_back(TileItem{(uint32_t)(first + k), c - k < per ? c - k : per, 0u, 0u, b, 0u, 0u, 0u});
            };
            if (!g.pairs) {
                // no pair items (they do not fit at this window length): one pass over the bin counts with a running offset
                // (the general form below costs 4 ms of host time at 384 k bins: an array of bin starts, and four integer
                // divisions per bin to find its neighbour along the dominant axis)
                uint64_t off = 0;
                for (uint32_t b = 0; b < nb; ++b) {
                    const uint32_t c = cnt[b];
                    if (c >= thr) add_pieces(off, c, b);
                    off += c;
                }
            } else {
                std::vector<uint64_t> &start = J.start;  // kept by the job: no fresh pages per plan
                start.resize((size_t)nb + 1);
                uint64_t off = 0;
                for (uint32_t b = 0; b < nb; ++b) {
                    start[b] = off;
                    off += cnt[b];
                }
                start[nb] = off;
                std::vector<uint8_t> &state = J.state;  // 0: direct, 1: item (first cube or single), 2: second cube of a pair
                state.assign(nb, 0);
                for (uint32_t b = 0; b < nb; ++b) {
                    const uint32_t c = cnt[b];
                    if (c == 0 || state[b]) continue;
                    const uint32_t D = b / T3, tl = b - D * T3, a = D >> 2;
                    const uint32_t step = a == 0 ? 1u : (a == 1 ? Tx : Tx * Ty);
                    const uint32_t ca = a == 0 ? tl % Tx : (a == 1 ? (tl / Tx) % Ty : tl / (Tx * Ty));
                    const uint32_t na = a == 0 ? Tx : (a == 1 ? Ty : Tz);
                    const uint32_t b2 = b + step;
                    const uint32_t c2 = (ca + 1 < na && !state[b2]) ? cnt[b2] : 0u;
                    if (c2 > 0 && c + c2 >= thr && c + c2 <= mx) {
                        state[b] = 1;
                        state[b2] = 2;
                        items.push_back(TileItem{(uint32_t)start[b], c, (uint32_t)start[b2], c2, b, 1u, 0u, 0u});
                    } else if (c >= thr) {
                        state[b] = 1;
                        add_pieces(start[b], c, b);
                    }
                }
            }
            // the items' event ranges in list order: the record set-up finds the item of an event by bisection
            for (size_t i = 0; i < items.size(); ++i) {
                ranges.push_back(TileRange{items[i].start, items[i].count, (uint32_t)i, 0u});
                if (items[i].count2) ranges.push_back(TileRange{items[i].start2, items[i].count2, (uint32_t)i, 0u});
            }
            // single-cube items come out in list order already; only the second cubes of pair items break it
            if (!std::is_sorted(ranges.begin(), ranges.end(), [](const TileRange &x, const TileRange &y) { return x.start < y.start; }))
                std::sort(ranges.begin(), ranges.end(), [](const TileRange &x, const TileRange &y) { return x.start < y.start; });
        }
    }
    // too few items to fill the GPU twice over: the tile pass would run on a fraction of the SMs before the direct pass
    // starts (measured at 10 M events on the cfg-3 grid: 2.33 ms with 243 items against 2.02 ms all direct)
    {
        const size_t auto_min = 2u * (size_t)(ctx->n_sm > 0 ? ctx->n_sm : 1) *
                                (size_t)tile_ctas_per_sm(tile_smem_bytes(g), ctx->smem_per_sm);
        const size_t min_items = ctx->tile_min_items >= 0 ? (size_t)ctx->tile_min_items : auto_min;
        if (items.size() < min_items) items.clear();
    }
    ctx->plan.sorted = sorted ? 1 : 0;
    if (items.empty()) ranges.clear();  // no tiles (window too wide, unsorted list, sparse bins): the whole list in order
    // ---- scratch (grows only)
    if (ctx->items_cap < items.size()) {
        cudaFree(ctx->d_items);
        ctx->d_items = nullptr;
        ctx->items_cap = 0;
        CU(cudaMalloc(&ctx->d_items, items.size() * sizeof(TileItem)));
        ctx->items_cap = items.size();
    }
    if (ctx->ranges_cap < ranges.size()) {
        cudaFree(ctx->d_ranges);
        ctx->d_ranges = nullptr;
        ctx->ranges_cap = 0;
        CU(cudaMalloc(&ctx->d_ranges, ranges.size() * sizeof(TileRange)));
        ctx->ranges_cap = ranges.size();
    }
    if (!items.empty()) {
        if (!ctx->d_geom) CU(cudaMalloc(&ctx->d_geom, sizeof(TileGeom)));
        if (memcmp(&g, &ctx->h_geom_sent, sizeof g) != 0) {
            ctx->h_geom_sent = g;
            CU(cudaMemcpyAsync(ctx->d_geom, &ctx->h_geom_sent, sizeof g, cudaMemcpyHostToDevice, s));
        }
        CU(cudaMemcpyAsync(ctx->d_items, items.data(), items.size() * sizeof(TileItem), cudaMemcpyHostToDevice, s));
        CU(cudaMemcpyAsync(ctx->d_ranges, ranges.data(), ranges.size() * sizeof(TileRange), cudaMemcpyHostToDevice, s));
    }
    // ---- the records: fp64 set-up, quantisation, dry run against the tile (prepared.cu)
    launch_prepare_rays(p, ctx->sigma, items.empty() ? nullptr : ctx->d_geom, ctx->tile_log2, ev_ptrs(ev), n, ctx->d_items,
                        ctx->d_ranges, (uint32_t)ranges.size(), ctx->d_rec, ctx->d_chunk_flags, ctx->d_tiny, kTinyCap,
                        ctx->d_plan_counters, s);
    CHECK_LAUNCH(1);
    // the pieces of the direct pass: the flagged 32-event pieces, compacted in list order on the device
    const uint32_t nc = (uint32_t)((n + 31) / 32);
    J.n_pieces = 0;
    CU(cudaMemsetAsync(ctx->d_chunk_flags + nc, 0, sizeof(uint32_t), s));
    ctx->launches += launch_exclusive_scan_u32(ctx->d_chunk_flags, ctx->d_chunk_pos, ctx->d_chunk_tmp, nc + 1, s);
    launch_compact_flags(ctx->d_chunk_flags, ctx->d_chunk_pos, nc, ctx->d_chunk_list, s);
    CHECK_LAUNCH(1);
    CU(cudaMemcpyAsync(&J.n_pieces, ctx->d_chunk_pos + nc, sizeof(uint32_t), cudaMemcpyDeviceToHost, s));
    J.hc.resize(plan_counter_bytes());
    CU(cudaMemcpyAsync(J.hc.data(), ctx->d_plan_counters, J.hc.size(), cudaMemcpyDeviceToHost, s));
    return TOFMLEM_OK;  // the host vectors of the job stay alive until plan_finish
}

int plan_finish(tofmlem_ctx *ctx) {
    auto &J = ctx->job;
    uint64_t cnt4[5];
    read_plan_counters(J.hc.data(), cnt4);
    if (cnt4[4] > kTinyCap) return TOFMLEM_OK;  // a list made of slivers: not worth a plan (stays inactive)
    ctx->plan.n_tiny = (uint32_t)cnt4[4];
    ctx->plan.valid = true;
    ctx->plan.x1 = J.ev.x1;
    ctx->plan.n = J.n;
    ctx->plan.tile_log2 = ctx->tile_log2;
    ctx->plan.sigma = ctx->sigma;
    ctx->plan.trunc = ctx->trunc_sigmas;
    ctx->plan.brick = J.p.brick;
    ctx->plan.n_items = (uint32_t)J.items.size();
    ctx->plan.max_item_events = 0;
    for (const TileItem &it : J.items)
        if (it.count + it.count2 > ctx->plan.max_item_events) ctx->plan.max_item_events = it.count + it.count2;
    ctx->plan.n_strag = (uint32_t)cnt4[2];
    ctx->plan.valid_events = cnt4[0];
    ctx->plan.tile_events = cnt4[1];
    ctx->plan.direct_events = J.n - cnt4[1];
    ctx->plan.visits = cnt4[3];
    ctx->plan.direct_valid = cnt4[0] - cnt4[1] - cnt4[4];
    ctx->plan.n_pieces = J.n_pieces;
    return TOFMLEM_OK;
}

}  // namespace

int tofmlem_plan_events(tofmlem_ctx *ctx, const tofmlem_events *ev, uint64_t n) {
    if (!ctx) return TOFMLEM_EINVAL;
    int rc = plan_begin(ctx, ev, n);
    if (rc) return rc < 0 ? rc : TOFMLEM_OK;
    CU(cudaStreamSynchronize(ctx->stream));
    rc = plan_build(ctx);
    if (rc) return rc;
    CU(cudaStreamSynchronize(ctx->stream));
    return plan_finish(ctx);
}

int tofmlem_plan_info(const tofmlem_ctx *ctx, tofmlem_plan *h_out) {
    if (!ctx || !h_out) return TOFMLEM_EINVAL;
    h_out->active = ctx->plan.valid ? 1 : 0;
    h_out->sorted = ctx->plan.sorted;
    h_out->n_tile_items = ctx->plan.n_items;
    h_out->n_direct_chunks = ctx->plan.n_pieces;
    h_out->n_tile_events = ctx->plan.tile_events;
    h_out->n_direct_events = ctx->plan.direct_events;
    h_out->n_stragglers = ctx->plan.n_strag;
    return TOFMLEM_OK;
}

uint32_t tofmlem_num_bins(const tofmlem_ctx *ctx) { return ctx ? num_bins(ctx) : 0u; }

int tofmlem_bin_events(tofmlem_ctx *ctx, const tofmlem_events *ev, uint64_t n, uint32_t *d_key, uint32_t *d_perm,
                       uint32_t *d_bin_offsets) {
    if (!ctx) return TOFMLEM_EINVAL;
    if (n == 0) return TOFMLEM_OK;
    if (!ev_ok(ev, false) || !d_key || n > 0xFFFFFFFFull) return fail(ctx, TOFMLEM_EINVAL, "bin_events: bad argument");
    const uint32_t nb = num_bins(ctx);
    const bool sort = d_perm != nullptr;
    // sub-bins only matter for the permutation; the fine histogram must still fit 32-bit indices
    const uint32_t S = sort ? effective_subbins(ctx) : 1u;
    const size_t nfine = (size_t)nb * S + 1;
    int rc = ensure_bin_scratch(ctx, nfine, S > 1 ? n : 0);
    if (rc) return rc;
    SubBin sb;
    sb.S = S;
    const bool tof_window = ctx->tof && !ctx->bin_whole_chords;
    sb.half_window = tof_window ? (float)(ctx->trunc_sigmas * ctx->sigma) : 0.0f;
    {
        // largest visit count of a window: its length times the l1 norm of u / v, plus the first voxel
        const tofmlem_grid &g = ctx->grid;
        const double diag = sqrt(pow(g.nx * (double)g.vx, 2) + pow(g.ny * (double)g.vy, 2) + pow(g.nz * (double)g.vz, 2));
        const double len = tof_window ? fmin(2.0 * sb.half_window, diag) : diag;
        const double vmax = fmin(len * sqrt(1.0 / (g.vx * g.vx) + 1.0 / (g.vy * g.vy) + 1.0 / (g.vz * g.vz)) + 3.0,
                                 (double)g.nx + g.ny + g.nz);
        sb.quantum = S > 2 ? (uint32_t)fmax(1.0, ceil(vmax / (double)(S - 2))) : 1u << 30;
    }
    uint8_t *d_sub = S > 1 ? ctx->d_sub : nullptr;
    CU(cudaMemsetAsync(ctx->d_hist, 0, nfine * sizeof(uint32_t), ctx->stream));
    launch_bin_keys(grid_f32(ctx), ctx->tile_log2, sb, ev_ptrs(ev), n, d_key, d_sub,
                    (sort || d_bin_offsets) ? ctx->d_hist : nullptr, nb, ctx->stream);
    CHECK_LAUNCH(1);
    if (sort || d_bin_offsets) {
        const int k = launch_exclusive_scan_u32(ctx->d_hist, ctx->d_cursor, ctx->d_scan_tmp, (uint32_t)nfine, ctx->stream);
        CHECK_LAUNCH(k);
        if (d_bin_offsets) {
            launch_strided_copy(ctx->d_cursor, S, nb + 1, d_bin_offsets, ctx->stream);
            CHECK_LAUNCH(1);
        }
    }
    if (sort) {
        launch_scatter_perm(d_key, d_sub, S, n, nb, ctx->d_cursor, d_perm, ctx->stream);
        CHECK_LAUNCH(1);
    }
    return TOFMLEM_OK;
}

static int gather_events_impl(tofmlem_ctx *ctx, const tofmlem_events *in, const uint32_t *d_perm, uint64_t n,
                              const tofmlem_events_mut *out, bool full_permutation, const char *who) {
    if (!ctx) return TOFMLEM_EINVAL;
    if (n == 0) return TOFMLEM_OK;
    if (!ev_ok(in, false) || !d_perm || !out || !out->x1 || !out->y1 || !out->z1 || !out->x2 || !out->y2 || !out->z2)
        return fail(ctx, TOFMLEM_EINVAL, who);
    const float *src[7] = {in->x1, in->y1, in->z1, in->x2, in->y2, in->z2, in->dt};
    float *dst[7] = {out->x1, out->y1, out->z1, out->x2, out->y2, out->z2, out->dt};
    for (int f = 0; f < 7; ++f)
        if (src[f] && dst[f] && src[f] == dst[f]) return fail(ctx, TOFMLEM_EINVAL, who);
    // A permutation of 0..n-1 reads every source event once: interleave the members into 32-byte records (scratch
    // kept by the context until tofmlem_destroy), gather one sector per event instead of one per member
    // (measured at 146 M events: 19.5 -> 5.2 ms).
    if (full_permutation && (src[6] != nullptr) == (dst[6] != nullptr)) {
        if (ensure_pack(ctx, n)) {  // else not enough memory for the records: member-by-member gathers below
            launch_gather_packed(ev_ptrs(in), d_perm, n, ctx->d_pack, dst, ctx->stream);
            CHECK_LAUNCH(2);
            return TOFMLEM_OK;
        }
    }
    for (int f = 0; f < 7; ++f) {
        if (!src[f] || !dst[f]) continue;
        launch_gather(src[f], d_perm, n, dst[f], ctx->stream);
        CHECK_LAUNCH(1);
    }
    return TOFMLEM_OK;
}

int tofmlem_gather_events(tofmlem_ctx *ctx, const tofmlem_events *in, const uint32_t *d_perm, uint64_t n,
                          const tofmlem_events_mut *out) {
    return gather_events_impl(ctx, in, d_perm, n, out, false, "gather_events: bad argument");
}

int tofmlem_permute_events(tofmlem_ctx *ctx, const tofmlem_events *in, const uint32_t *d_perm, uint64_t n,
                           const tofmlem_events_mut *out) {
    return gather_events_impl(ctx, in, d_perm, n, out, true, "permute_events: bad argument");
}

int tofmlem_region_zbounds(const tofmlem_ctx *ctx, int n_regions, float *h_zbounds) {
    if (!ctx || !h_zbounds || n_regions < 1 || n_regions > kMaxRegions) return TOFMLEM_EINVAL;
    default_zbounds(ctx, n_regions, h_zbounds);
    return TOFMLEM_OK;
}

static int split_impl(tofmlem_ctx *ctx, const tofmlem_events *ev, uint64_t n, int n_regions, const float *h_zbounds,
                      bool overlap, int32_t *d_region, uint32_t *d_perm, uint64_t perm_capacity, uint64_t *h_counts) {
    if (!ctx) return TOFMLEM_EINVAL;
    if ((n && !ev_ok(ev, false)) || n_regions < 1 || n_regions > kMaxRegions || (n && !d_region) || !h_counts ||
        n > 0xFFFFFFFFull)
        return fail(ctx, TOFMLEM_EINVAL, "split_regions: bad argument");
    if (overlap && !ctx->tof) return fail(ctx, TOFMLEM_EUNSUPPORTED, "split_regions_overlap needs a TOF context");
    RegionBounds rb;
    rb.n_regions = n_regions;
    if (h_zbounds) {
        for (int j = 0; j <= n_regions; ++j) rb.zb[j] = h_zbounds[j];
        for (int j = 0; j < n_regions; ++j)
            if (!(rb.zb[j] <= rb.zb[j + 1])) return fail(ctx, TOFMLEM_EINVAL, "split_regions: bounds not ascending");
    } else {
        default_zbounds(ctx, n_regions, rb.zb);
    }
    unsigned long long *counts = ctx->d_rcounts, *cursor = ctx->d_rcounts + (kMaxRegions + 1);
    CU(cudaMemsetAsync(counts, 0, 2 * (kMaxRegions + 1) * sizeof(unsigned long long), ctx->stream));
    if (n) {
        if (overlap)
            launch_region_spans(ev_ptrs(ev), n, rb, (float)(ctx->trunc_sigmas * ctx->sigma), d_region, counts, ctx->stream);
        else
            launch_region_ids(ev_ptrs(ev), n, rb, d_region, counts, ctx->stream);
        CHECK_LAUNCH(1);
    }
    unsigned long long h[kMaxRegions + 1];
    CU(cudaMemcpyAsync(h, counts, (n_regions + 1) * sizeof(unsigned long long), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    unsigned long long total = 0;
    for (int r = 0; r < n_regions; ++r) {
        h_counts[r] = h[r];
        total += h[r];
    }
    if (d_perm && n) {
        if (total + h[n_regions] > perm_capacity)
            return fail(ctx, TOFMLEM_EINVAL, "split_regions: the permutation does not fit its buffer");
        unsigned long long start[kMaxRegions + 1];
        unsigned long long run = 0;
        for (int r = 0; r <= n_regions; ++r) {
            start[r] = run;
            run += h[r];
        }
        CU(cudaMemcpyAsync(cursor, start, (n_regions + 1) * sizeof(unsigned long long), cudaMemcpyHostToDevice,
                           ctx->stream));
        if (overlap)
            launch_region_span_scatter(d_region, n, n_regions, cursor, d_perm, ctx->stream);
        else
            launch_region_scatter(d_region, n, n_regions, cursor, d_perm, ctx->stream);
        CHECK_LAUNCH(1);
        CU(cudaStreamSynchronize(ctx->stream));  // `start` lives on this stack frame
    }
    return TOFMLEM_OK;
}

int tofmlem_split_regions(tofmlem_ctx *ctx, const tofmlem_events *ev, uint64_t n, int n_regions,
                          const float *h_zbounds, int32_t *d_region, uint32_t *d_perm, uint64_t *h_counts) {
    return split_impl(ctx, ev, n, n_regions, h_zbounds, false, d_region, d_perm, n, h_counts);
}

int tofmlem_split_regions_overlap(tofmlem_ctx *ctx, const tofmlem_events *ev, uint64_t n, int n_regions,
                                  const float *h_zbounds, int32_t *d_span, uint32_t *d_perm, uint64_t perm_capacity,
                                  uint64_t *h_counts) {
    return split_impl(ctx, ev, n, n_regions, h_zbounds, true, d_span, d_perm, perm_capacity, h_counts);
}

int tofmlem_region_grid(const tofmlem_ctx *ctx, int n_regions, const float *h_zbounds, int r, tofmlem_grid *sub,
                        int32_t *z0, int32_t *z1) {
    if (!ctx || !sub || !z0 || !z1 || n_regions < 1 || n_regions > kMaxRegions || r < 0 || r >= n_regions)
        return TOFMLEM_EINVAL;
    const tofmlem_grid &g = ctx->grid;
    int32_t k0, k1;
    if (h_zbounds) {
        k0 = (int32_t)floor(((double)h_zbounds[r] - g.oz) / g.vz + 1e-4);
        k1 = (int32_t)ceil(((double)h_zbounds[r + 1] - g.oz) / g.vz - 1e-4);
    } else {
        std::vector<int32_t> k;
        default_region_slices(g.nz, n_regions, k);
        k0 = k[r];
        k1 = k[r + 1];
    }
    // R12: the window's half-width + the shell; reading R27 (overlap): the WHOLE window of an event centred up to one
    // half-width outside the core must fit, so twice the half-width
    const int32_t margin = ctx->region_overlap < 0 ? 0 :  // (internal: the bare core)
        (int32_t)ceil(((ctx->region_overlap ? 2.0 : 1.0) * ctx->trunc_sigmas * ctx->sigma + ctx->shell_mm) / (double)g.vz);
    int32_t a = k0 - (r > 0 ? margin : 0), b = k1 + (r < n_regions - 1 ? margin : 0);
    if (a < 0) a = 0;
    if (b > g.nz) b = g.nz;
    if (b <= a) return TOFMLEM_EINVAL;
    *sub = g;
    sub->nz = b - a;
    sub->oz = (float)((double)g.oz + (double)a * (double)g.vz);
    *z0 = a;
    *z1 = b;
    return TOFMLEM_OK;
}

int tofmlem_reconstruct_regions(tofmlem_ctx *ctx, const tofmlem_events *ev, uint64_t n, int n_regions,
                                const float *h_zbounds, float *d_image_out, const float *d_sens, int iters) {
    if (!ctx) return TOFMLEM_EINVAL;
    if (!ev_ok(ev, ctx->tof) || !d_image_out || !d_sens || iters < 0 || n == 0 || n > 0xFFFFFFFFull ||
        n_regions < 1 || n_regions > kMaxRegions)
        return fail(ctx, TOFMLEM_EINVAL, "reconstruct_regions: bad argument");
    cudaStream_t s = ctx->stream;
    const size_t slice = (size_t)ctx->grid.nx * ctx->grid.ny;
    const bool overlap = ctx->region_overlap != 0 && ctx->tof;
    // capacity of the per-region event lists: with overlapping membership (R27) an event may sit in two lists
    const uint64_t stride = ((overlap ? 2 * n : n) + 3) & ~3ull;
    std::vector<uint64_t> counts(n_regions);
    int rc = TOFMLEM_OK;
#define RCU(call)                                          \
    do {                                                   \
        cudaError_t e_ = (call);                           \
        if (e_ != cudaSuccess) {                           \
            rc = cuda_fail(ctx, e_, #call);                \
            cudaDeviceSynchronize();                       \
            free_region_cache(ctx);                        \
            return rc;                                     \
        }                                                  \
    } while (0)
#define RRC(call)                      \
    do {                               \
        rc = (call);                   \
        if (rc != TOFMLEM_OK) {        \
            cudaDeviceSynchronize();   \
            free_region_cache(ctx);    \
            return rc;                 \
        }                              \
    } while (0)
    if (ctx->rg_cap < stride) {  // event scratch is kept by the context: repeated calls do not allocate 64 B per event again
        cudaFree(ctx->d_rg_region);
        cudaFree(ctx->d_rg_perm);
        cudaFree(ctx->d_rg_sorted);
        cudaFree(ctx->d_rg_binned);
        ctx->d_rg_region = nullptr;
        ctx->d_rg_perm = nullptr;
        ctx->d_rg_sorted = ctx->d_rg_binned = nullptr;
        ctx->rg_cap = 0;
        RCU(cudaMalloc(&ctx->d_rg_region, stride * sizeof(int32_t)));
        RCU(cudaMalloc(&ctx->d_rg_perm, stride * sizeof(uint32_t)));
        RCU(cudaMalloc(&ctx->d_rg_sorted, 7 * stride * sizeof(float)));
        RCU(cudaMalloc(&ctx->d_rg_binned, 7 * stride * sizeof(float)));
        ctx->rg_cap = stride;
    }
    int32_t *d_region = ctx->d_rg_region;
    uint32_t *d_perm = ctx->d_rg_perm;
    float *d_sorted = ctx->d_rg_sorted, *d_binned = ctx->d_rg_binned;
    // ---- sub-contexts, streams, events and region images: built once per (bounds, TOF kernel, shell), then reused
    std::vector<float> zb(n_regions + 1);
    if (h_zbounds) zb.assign(h_zbounds, h_zbounds + n_regions + 1);
    else default_zbounds(ctx, n_regions, zb.data());
    auto &C = ctx->rgc;
    const double shell_key = ctx->shell_mm + (overlap ? 1e9 : 0.0);  // the margin rule is part of the cache key
    if (C.zb != zb || C.sigma != ctx->sigma || C.trunc != ctx->trunc_sigmas || C.shell != shell_key) {
        RCU(cudaStreamSynchronize(s));
        free_region_cache(ctx);
        C.subs.assign(n_regions, nullptr);
        C.streams.assign(n_regions, nullptr);
        C.done.assign(n_regions, nullptr);
        C.images.assign(n_regions, nullptr);
        C.z0.assign(n_regions, 0);
        C.z1.assign(n_regions, 0);
        RCU(cudaEventCreateWithFlags(&C.ready, cudaEventDisableTiming));
        for (int r = 0; r < n_regions; ++r) {
            tofmlem_grid sub;
            RRC(tofmlem_region_grid(ctx, n_regions, h_zbounds, r, &sub, &C.z0[r], &C.z1[r]));
            RCU(cudaStreamCreateWithFlags(&C.streams[r], cudaStreamNonBlocking));
            RCU(cudaEventCreateWithFlags(&C.done[r], cudaEventDisableTiming));
            RRC(tofmlem_create(&ctx->scanner, &sub, ctx->tof ? (float)(ctx->sigma / sigma_from_fwhm(1.0)) : 0.0f,
                               C.streams[r], &C.subs[r]));
            RCU(cudaMalloc(&C.images[r], C.subs[r]->nvox * sizeof(float)));
            RRC(ensure_corr(C.subs[r]));
        }
        C.zb = zb;
        C.sigma = ctx->sigma;
        C.trunc = ctx->trunc_sigmas;
        C.shell = shell_key;
    }
    RRC(split_impl(ctx, ev, n, n_regions, h_zbounds, overlap, d_region, d_perm, stride, counts.data()));
    uint64_t n_list = 0;  // entries of the region-sorted list (= valid events, with multiplicity under R27)
    for (int r = 0; r < n_regions; ++r) n_list += counts[r];
    tofmlem_events_mut sorted{d_sorted, d_sorted + stride, d_sorted + 2 * stride, d_sorted + 3 * stride,
                              d_sorted + 4 * stride, d_sorted + 5 * stride, ev->dt ? d_sorted + 6 * stride : nullptr};
    if (overlap) {
        if (n_list) RRC(tofmlem_gather_events(ctx, ev, d_perm, n_list, &sorted));
    } else {
        RRC(tofmlem_permute_events(ctx, ev, d_perm, n, &sorted));
    }
    launch_max_nonneg(d_sens, ctx->nvox, ctx->d_max, s);
    ctx->launches += 1;
    RCU(cudaMemsetAsync(d_image_out, 0, ctx->nvox * sizeof(float), s));
    RCU(cudaEventRecord(C.ready, s));
    // scratch of the per-region binning, sized before any region stream runs (no allocation between the launches)
    {
        uint64_t cmax = 0;
        for (int r = 0; r < n_regions; ++r) cmax = counts[r] > cmax ? counts[r] : cmax;
        for (int r = 0; r < n_regions; ++r) {
            tofmlem_ctx *sc = C.subs[r];
            sc->sigma = ctx->sigma;
            sc->trunc_sigmas = ctx->trunc_sigmas;
            sc->sens_floor_rel = ctx->sens_floor_rel;
            sc->projector = ctx->projector;
            sc->samples_k = ctx->samples_k;
            sc->median = ctx->median;
            sc->corr_bricks = ctx->corr_bricks;
            sc->em_variant = ctx->em_variant;
            sc->cache_share = ctx->cache_share;
            sc->tile_log2 = ctx->tile_log2;
            sc->subbins = ctx->subbins;
            sc->cta_interleave = ctx->cta_interleave;
            sc->tile_min_events = ctx->tile_min_events;
            sc->tile_max_events = ctx->tile_max_events;
            sc->tile_min_items = ctx->tile_min_items;
            sc->l2_persist = ctx->l2_persist;
            sc->tile_check = ctx->tile_check;
            sc->d_max_ext = ctx->d_max;
            sc->launches = 0;
            if (sc->median && !sc->d_tmp_image) RCU(cudaMalloc(&sc->d_tmp_image, sc->nvox * sizeof(float)));
            if (counts[r]) {
                const uint32_t S = effective_subbins(sc);
                RRC(ensure_bin_scratch(sc, (size_t)num_bins(sc) * S + 1, S > 1 ? counts[r] : 0));
            }
        }
        (void)cmax;
    }
    uint64_t off = 0;
    std::vector<tofmlem_events> run_evs(n_regions);
    std::vector<int> planning(n_regions, 0);
    // a plan costs about as much as the four iterations it speeds up by 15 % each (measured at cfg-4: 5 iterations 141.5 ms
    // with plans against 142.3 ms without, 9 iterations 226.9 against 242.6 ms)
    const bool want_plan = (ctx->region_plan == 1 || (ctx->region_plan == 2 && iters >= 6)) && ctx->tof &&
                           ctx->projector == 0 && ctx->em_variant == 0 && iters > 1;
    for (int r = 0; r < n_regions; ++r) {
        tofmlem_ctx *sc = C.subs[r];
        cudaStream_t rs = C.streams[r];
        const uint64_t nv = sc->nvox;
        RCU(cudaStreamWaitEvent(rs, C.ready, 0));
        const float *sens_r = d_sens + (size_t)C.z0[r] * slice;
        launch_mask_init(C.images[r], sens_r, ctx->d_max, (float)ctx->sens_floor_rel, nv, rs);
        sc->launches += 1;
        tofmlem_events sub_ev{sorted.x1 + off, sorted.y1 + off, sorted.z1 + off, sorted.x2 + off, sorted.y2 + off,
                              sorted.z2 + off, sorted.dt ? sorted.dt + off : nullptr};
        // locality binning inside the region (on its own grid and stream); the region-id and region-permutation buffers
        // are free again by now (the region streams start after `ready`) and serve as key / permutation scratch
        tofmlem_events_mut bin_ev{d_binned + off, d_binned + stride + off, d_binned + 2 * stride + off,
                                  d_binned + 3 * stride + off, d_binned + 4 * stride + off, d_binned + 5 * stride + off,
                                  sorted.dt ? d_binned + 6 * stride + off : nullptr};
        if (counts[r]) {
            rc = tofmlem_bin_events(sc, &sub_ev, counts[r], reinterpret_cast<uint32_t *>(d_region) + off, d_perm + off, nullptr);
            if (rc == TOFMLEM_OK && !overlap && ctx->pack_cap >= n) {
                // permutation through 32-byte records in the parent's record scratch (free again after the region split)
                float *dst[7] = {bin_ev.x1, bin_ev.y1, bin_ev.z1, bin_ev.x2, bin_ev.y2, bin_ev.z2, bin_ev.dt};
                launch_gather_packed(ev_ptrs(&sub_ev), d_perm + off, counts[r], ctx->d_pack + 8 * off, dst, rs);
                sc->launches += 2;
            } else if (rc == TOFMLEM_OK) {
                rc = tofmlem_gather_events(sc, &sub_ev, d_perm + off, counts[r], &bin_ev);
            }
            if (rc != TOFMLEM_OK) {
                ctx->err = sc->err;
                cudaDeviceSynchronize();
                free_region_cache(ctx);
                return rc;
            }
        }
        run_evs[r] = tofmlem_events{bin_ev.x1, bin_ev.y1, bin_ev.z1, bin_ev.x2, bin_ev.y2, bin_ev.z2, bin_ev.dt};
        // ray records + tiles for the region's own binned list, phase 1 (key histogram -> host, asynchronous)
        planning[r] = 0;
        sc->plan.valid = false;
        if (counts[r] && want_plan) {
            rc = plan_begin(sc, &run_evs[r], counts[r]);
            if (rc < 0) {
                ctx->err = sc->err;
                cudaDeviceSynchronize();
                free_region_cache(ctx);
                return rc;
            }
            planning[r] = rc == 0;
        }
        off += counts[r];
    }
    // phases 2 and 3 of the plans, region by region: while the host waits for one region's stream the others work
    for (int phase = 2; phase <= 3 && want_plan; ++phase)
        for (int r = 0; r < n_regions; ++r) {
            if (!planning[r]) continue;
            tofmlem_ctx *sc = C.subs[r];
            rc = cudaStreamSynchronize(C.streams[r]) == cudaSuccess ? TOFMLEM_OK : TOFMLEM_ECUDA;
            if (rc == TOFMLEM_OK) rc = phase == 2 ? plan_build(sc) : plan_finish(sc);
            if (rc != TOFMLEM_OK) {
                ctx->err = sc->err;
                cudaDeviceSynchronize();
                free_region_cache(ctx);
                return rc;
            }
        }
    for (int r = 0; r < n_regions; ++r) {
        tofmlem_ctx *sc = C.subs[r];
        cudaStream_t rs = C.streams[r];
        const float *sens_r = d_sens + (size_t)C.z0[r] * slice;
        rc = iterate_device(sc, counts[r] ? ev_ptrs(&run_evs[r]) : EventPtrs{}, counts[r], nullptr, C.images[r], sens_r, iters, false);
        if (rc != TOFMLEM_OK) {
            ctx->err = sc->err;
            cudaDeviceSynchronize();
            free_region_cache(ctx);
            return rc;
        }
        RCU(cudaEventRecord(C.done[r], rs));
    }
    // R13: sum of the extended region images, overlapping margins add up.  R27: every region has seen all
    // the events that reach its core, so the cores alone tile the volume (margins discarded).
    for (int r = 0; r < n_regions; ++r) {
        RCU(cudaStreamWaitEvent(s, C.done[r], 0));
        if (overlap) {
            tofmlem_grid sub;
            int32_t a0, a1, k0, k1;
            const int keep = ctx->region_overlap;
            ctx->region_overlap = -1;  // margin 0: the core itself
            rc = tofmlem_region_grid(ctx, n_regions, h_zbounds, r, &sub, &k0, &k1);
            ctx->region_overlap = keep;
            if (rc == TOFMLEM_OK) rc = tofmlem_region_grid(ctx, n_regions, h_zbounds, r, &sub, &a0, &a1);
            RRC(rc);
            RCU(cudaMemcpyAsync(d_image_out + (size_t)k0 * slice, C.images[r] + (size_t)(k0 - a0) * slice,
                                (size_t)(k1 - k0) * slice * sizeof(float), cudaMemcpyDeviceToDevice, s));
            ctx->launches += C.subs[r]->launches;
        } else {
            launch_add(d_image_out + (size_t)C.z0[r] * slice, C.images[r], C.subs[r]->nvox, s);
            ctx->launches += 1 + C.subs[r]->launches;
        }
    }
    RCU(cudaStreamSynchronize(s));
#undef RCU
#undef RRC
    return TOFMLEM_OK;
}

int tofmlem_get_stats(tofmlem_ctx *ctx, tofmlem_stats *h_out) {
    if (!ctx || !h_out) return TOFMLEM_EINVAL;
    DeviceStats h;
    CU(cudaMemcpyAsync(&h, ctx->d_stats, sizeof h, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    h_out->n_valid = h.n_valid;
    h_out->n_skipped = ctx->last_n >= h.n_valid ? ctx->last_n - h.n_valid : 0;
    h_out->visits = h.visits;
    h_out->reductions = h.reds;
    h_out->tile_events = h.tile_events;
    h_out->tile_oob = h.tile_oob;
    h_out->tile_visits = h.tile_visits;
    h_out->sum_image_sens = h.sum_image_sens;
    return TOFMLEM_OK;
}

int tofmlem_probe(tofmlem_ctx *ctx, int kind, float *d_buf, uint64_t n_elems, uint64_t n_ops, float *h_ms) {
    if (!ctx || !d_buf || !h_ms || n_ops == 0) return TOFMLEM_EINVAL;
    // the probes measure the plain L2 / shared-memory rates: no persisting carve-out left over from a fused pass
    if (ctx->l2_ptr) {
        cudaStreamAttrValue attr;
        memset(&attr, 0, sizeof attr);
        cudaStreamSynchronize(ctx->stream);
        cudaStreamSetAttribute(ctx->stream, cudaStreamAttributeAccessPolicyWindow, &attr);
        cudaCtxResetPersistingL2Cache();
        cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, 0);
        cudaGetLastError();
        ctx->l2_ptr = nullptr;  // the next fused pass sets its window again
    }
    const int rc = run_probe(kind, d_buf, n_elems, n_ops, h_ms, ctx->stream);
    if (rc == -1) return fail(ctx, TOFMLEM_EINVAL, "probe: bad kind or size");
    if (rc != 0) return cuda_fail(ctx, cudaGetLastError(), "probe");
    ctx->launches += 2;
    return TOFMLEM_OK;
}

int tofmlem_pass_timing(tofmlem_ctx *ctx, float h_ms[3]) {
    if (!ctx || !h_ms) return TOFMLEM_EINVAL;
    h_ms[0] = h_ms[1] = h_ms[2] = 0.0f;
    if (!ctx->t_have || !ctx->t_ev[0]) return TOFMLEM_OK;
    CU(cudaEventSynchronize(ctx->t_ev[3]));
    for (int k = 0; k < 3; ++k)
        if (ctx->t_have & (1 << k)) CU(cudaEventElapsedTime(&h_ms[k], ctx->t_ev[k], ctx->t_ev[k + 1]));
    return TOFMLEM_OK;
}

const char *tofmlem_last_error(const tofmlem_ctx *ctx) { return ctx ? ctx->err.c_str() : "NULL context"; }

uint64_t tofmlem_launch_count(const tofmlem_ctx *ctx) { return ctx ? ctx->launches : 0; }

}  // extern "C"
