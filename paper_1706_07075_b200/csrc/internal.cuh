// internal.cuh -- declarations shared by the translation units of libtofmlem (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>

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
    int variant;           // fused EM pass: 0 = persistent per-SM queues (default), 1 = grid order
};

struct EventPtrs {
    const float *x1, *y1, *z1, *x2, *y2, *z2, *dt;
};

struct DeviceStats {
    unsigned long long n_valid;
    unsigned long long visits;
    double sum_image_sens;
};

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
void launch_em_correction(const ProjParams &p, bool tof, const EventPtrs &ev, uint64_t n, const float *image,
                          float *corr, bool vec_ok, DeviceStats *stats, unsigned *queues, cudaStream_t s);

// ---- image_ops.cu
void launch_max_nonneg(const float *x, uint64_t n, float *d_max /* zeroed by the call */, cudaStream_t s);
void launch_update(float *image, float *corr, const float *sens, const float *d_max, float floor_rel, uint64_t n,
                   cudaStream_t s);
void launch_mask_init(float *image, const float *sens, const float *d_max, float floor_rel, uint64_t n,
                      cudaStream_t s);
void launch_dot_f64(const float *a, const float *b, uint64_t n, double *d_out /* zeroed by the call */,
                    cudaStream_t s);
void launch_scale(float *x, float a, uint64_t n, cudaStream_t s);
void launch_add(float *dst, const float *src, uint64_t n, cudaStream_t s);

// ---- binning.cu
void launch_bin_keys(const GridF32 &g, int tile_log2, const EventPtrs &ev, uint64_t n, uint32_t *key,
                     uint32_t *hist /* nbins+1, zeroed by caller */, uint32_t nbins, cudaStream_t s);
void launch_exclusive_scan_u32(const uint32_t *in, uint32_t *out, uint32_t *out2 /* optional copy */, uint32_t n,
                               cudaStream_t s);
void launch_scatter_perm(const uint32_t *key, uint64_t n, uint32_t nbins, uint32_t *cursor, uint32_t *perm,
                         cudaStream_t s);
void launch_gather(const float *in, const uint32_t *perm, uint64_t n, float *out, cudaStream_t s);
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

// ---- probe.cu
int run_probe(int kind, float *d_buf, uint64_t n_elems, uint64_t n_ops, float *ms, cudaStream_t s);

}  // namespace tofmlem
