// binning.cu -- locality bin keys, counting sort, gather, and the TOF-assisted region split.
//
// Integer results are bit-exact against the float32 specification F1: every float operation is a
// single IEEE binary32 round-to-nearest operation in a fixed order (explicit __f*_rn intrinsics, so nvcc
// cannot contract them into FMAs).
#include "internal.cuh"

namespace tofmlem {

constexpr int kBlock = 256;
constexpr float kHalfC = 0.149896229f;  // c/2, mm/ps (F1 literal)

__device__ __forceinline__ bool finite_f(float x) { return fabsf(x) <= 3.402823466e+38f; }

// TOF-estimated annihilation point (kernel centre) per F1.  false for an invalid event.
__device__ __forceinline__ bool tof_centre(const EventPtrs &ev, uint64_t e, float c[3], float d[3]) {
    const float x1 = __ldg(ev.x1 + e), y1 = __ldg(ev.y1 + e), z1 = __ldg(ev.z1 + e);
    const float x2 = __ldg(ev.x2 + e), y2 = __ldg(ev.y2 + e), z2 = __ldg(ev.z2 + e);
    const float dt = ev.dt ? __ldg(ev.dt + e) : 0.0f;
    if (!(finite_f(x1) && finite_f(y1) && finite_f(z1) && finite_f(x2) && finite_f(y2) && finite_f(z2) &&
          finite_f(dt)))
        return false;
    const float dx = __fsub_rn(x2, x1), dy = __fsub_rn(y2, y1), dz = __fsub_rn(z2, z1);
    const float xx = __fmul_rn(dx, dx), yy = __fmul_rn(dy, dy), zz = __fmul_rn(dz, dz);
    const float sxy = __fadd_rn(xx, yy);
    const float L2 = __fadd_rn(sxy, zz);
    if (!(L2 > 0.0f) || !finite_f(L2)) return false;
    const float L = __fsqrt_rn(L2);
    const float h = __fmul_rn(kHalfC, dt);
    const float q = __fdiv_rn(h, L);
    const float mx = __fmul_rn(0.5f, __fadd_rn(x1, x2));
    const float my = __fmul_rn(0.5f, __fadd_rn(y1, y2));
    const float mz = __fmul_rn(0.5f, __fadd_rn(z1, z2));
    c[0] = __fadd_rn(mx, __fmul_rn(q, dx));
    c[1] = __fadd_rn(my, __fmul_rn(q, dy));
    c[2] = __fadd_rn(mz, __fmul_rn(q, dz));
    d[0] = dx;
    d[1] = dy;
    d[2] = dz;
    return true;
}

__device__ __forceinline__ int centre_voxel(float c, float o, float v, int n) {
    const float q = __fdiv_rn(__fsub_rn(c, o), v);
    const float f = floorf(q);
    if (!(f >= 0.0f)) return 0;
    if (f >= (float)n) return n - 1;
    return (int)f;
}

__global__ void __launch_bounds__(kBlock) bin_keys_kernel(GridF32 g, int tile_log2, EventPtrs ev, uint64_t n,
                                                          uint32_t *__restrict__ key, uint32_t *__restrict__ hist,
                                                          uint32_t nbins) {
    const uint64_t e = (uint64_t)blockIdx.x * kBlock + threadIdx.x;
    if (e >= n) return;
    const int t = 1 << tile_log2;
    const uint32_t Tx = (uint32_t)((g.nx + t - 1) >> tile_log2), Ty = (uint32_t)((g.ny + t - 1) >> tile_log2),
                   Tz = (uint32_t)((g.nz + t - 1) >> tile_log2);
    float c[3], d[3];
    uint32_t k = 0xFFFFFFFFu;
    if (tof_centre(ev, e, c, d)) {
        const int ix = centre_voxel(c[0], g.ox, g.vx, g.nx);
        const int iy = centre_voxel(c[1], g.oy, g.vy, g.ny);
        const int iz = centre_voxel(c[2], g.oz, g.vz, g.nz);
        const uint32_t tile =
            (((uint32_t)(iz >> tile_log2)) * Ty + (uint32_t)(iy >> tile_log2)) * Tx + (uint32_t)(ix >> tile_log2);
        int a = 0;
        float best = fabsf(d[0]);
        if (fabsf(d[1]) > best) { a = 1; best = fabsf(d[1]); }
        if (fabsf(d[2]) > best) { a = 2; }
        const float da = a == 0 ? d[0] : (a == 1 ? d[1] : d[2]);
        const float db0 = a == 0 ? d[1] : (a == 1 ? d[2] : d[0]);
        const float dc0 = a == 0 ? d[2] : (a == 1 ? d[0] : d[1]);
        const bool neg = da < 0.0f;
        const float db = neg ? -db0 : db0, dc = neg ? -dc0 : dc0;
        const uint32_t dirclass = 4u * (uint32_t)a + 2u * (db < 0.0f ? 1u : 0u) + (dc < 0.0f ? 1u : 0u);
        k = dirclass * (Tx * Ty * Tz) + tile;
    }
    key[e] = k;
    if (hist) atomicAdd(hist + (k < nbins ? k : nbins), 1u);
}

// single-block exclusive scan (n <= a few 10^5 bins): per-thread segments + shared-memory scan of the sums
__global__ void __launch_bounds__(1024) exclusive_scan_kernel(const uint32_t *__restrict__ in,
                                                              uint32_t *__restrict__ out,
                                                              uint32_t *__restrict__ out2, uint32_t n) {
    __shared__ uint32_t sums[1024];
    const uint32_t per = (n + 1023u) / 1024u;
    const uint32_t lo = min(n, threadIdx.x * per), hi = min(n, lo + per);
    uint32_t s = 0;
    for (uint32_t i = lo; i < hi; ++i) s += in[i];
    sums[threadIdx.x] = s;
    __syncthreads();
    for (int off = 1; off < 1024; off <<= 1) {
        uint32_t v = threadIdx.x >= off ? sums[threadIdx.x - off] : 0u;
        __syncthreads();
        sums[threadIdx.x] += v;
        __syncthreads();
    }
    uint32_t run = threadIdx.x ? sums[threadIdx.x - 1] : 0u;
    for (uint32_t i = lo; i < hi; ++i) {
        const uint32_t v = in[i];
        out[i] = run;
        if (out2) out2[i] = run;
        run += v;
    }
}

__global__ void __launch_bounds__(kBlock) scatter_perm_kernel(const uint32_t *__restrict__ key, uint64_t n,
                                                              uint32_t nbins, uint32_t *__restrict__ cursor,
                                                              uint32_t *__restrict__ perm) {
    const uint64_t e = (uint64_t)blockIdx.x * kBlock + threadIdx.x;
    if (e >= n) return;
    const uint32_t k = key[e];
    const uint32_t pos = atomicAdd(cursor + (k < nbins ? k : nbins), 1u);
    perm[pos] = (uint32_t)e;
}

__global__ void __launch_bounds__(kBlock) gather_kernel(const float *__restrict__ in, const uint32_t *__restrict__ perm,
                                                        uint64_t n, float *__restrict__ out) {
    const uint64_t i = (uint64_t)blockIdx.x * kBlock + threadIdx.x;
    if (i < n) out[i] = __ldg(in + __ldg(perm + i));
}

__global__ void __launch_bounds__(kBlock) region_ids_kernel(EventPtrs ev, uint64_t n, RegionBounds rb,
                                                            int32_t *__restrict__ region,
                                                            unsigned long long *__restrict__ counts) {
    __shared__ unsigned int local[kMaxRegions + 1];
    for (int i = threadIdx.x; i <= rb.n_regions; i += kBlock) local[i] = 0;
    __syncthreads();
    const uint64_t e = (uint64_t)blockIdx.x * kBlock + threadIdx.x;
    if (e < n) {
        float c[3], d[3];
        int r = -1;
        if (tof_centre(ev, e, c, d)) {
            r = 0;
            for (int j = 1; j < rb.n_regions; ++j) r += (rb.zb[j] <= c[2]) ? 1 : 0;
        }
        region[e] = r;
        atomicAdd(local + (r < 0 ? rb.n_regions : r), 1u);
    }
    __syncthreads();
    for (int i = threadIdx.x; i <= rb.n_regions; i += kBlock)
        if (local[i]) atomicAdd(counts + i, (unsigned long long)local[i]);
}

// block-aggregated scatter: one global atomic per (block, region)
__global__ void __launch_bounds__(kBlock) region_scatter_kernel(const int32_t *__restrict__ region, uint64_t n,
                                                                int n_regions,
                                                                unsigned long long *__restrict__ cursor,
                                                                uint32_t *__restrict__ perm) {
    __shared__ unsigned int local[kMaxRegions + 1];
    __shared__ unsigned long long base[kMaxRegions + 1];
    for (int i = threadIdx.x; i <= n_regions; i += kBlock) local[i] = 0;
    __syncthreads();
    const uint64_t e = (uint64_t)blockIdx.x * kBlock + threadIdx.x;
    int r = 0;
    unsigned int rank = 0;
    if (e < n) {
        r = region[e];
        if (r < 0) r = n_regions;
        rank = atomicAdd(local + r, 1u);
    }
    __syncthreads();
    for (int i = threadIdx.x; i <= n_regions; i += kBlock)
        if (local[i]) base[i] = atomicAdd(cursor + i, (unsigned long long)local[i]);
    __syncthreads();
    if (e < n) perm[base[r] + rank] = (uint32_t)e;
}

static inline unsigned grid_for(uint64_t n) { return (unsigned)((n + kBlock - 1) / kBlock); }

void launch_bin_keys(const GridF32 &g, int tile_log2, const EventPtrs &ev, uint64_t n, uint32_t *key, uint32_t *hist,
                     uint32_t nbins, cudaStream_t s) {
    if (n) bin_keys_kernel<<<grid_for(n), kBlock, 0, s>>>(g, tile_log2, ev, n, key, hist, nbins);
}

void launch_exclusive_scan_u32(const uint32_t *in, uint32_t *out, uint32_t *out2, uint32_t n, cudaStream_t s) {
    if (n) exclusive_scan_kernel<<<1, 1024, 0, s>>>(in, out, out2, n);
}

void launch_scatter_perm(const uint32_t *key, uint64_t n, uint32_t nbins, uint32_t *cursor, uint32_t *perm,
                         cudaStream_t s) {
    if (n) scatter_perm_kernel<<<grid_for(n), kBlock, 0, s>>>(key, n, nbins, cursor, perm);
}

void launch_gather(const float *in, const uint32_t *perm, uint64_t n, float *out, cudaStream_t s) {
    if (n) gather_kernel<<<grid_for(n), kBlock, 0, s>>>(in, perm, n, out);
}

void launch_region_ids(const EventPtrs &ev, uint64_t n, const RegionBounds &rb, int32_t *region,
                       unsigned long long *counts, cudaStream_t s) {
    if (n) region_ids_kernel<<<grid_for(n), kBlock, 0, s>>>(ev, n, rb, region, counts);
}

void launch_region_scatter(const int32_t *region, uint64_t n, int n_regions, unsigned long long *cursor,
                           uint32_t *perm, cudaStream_t s) {
    if (n) region_scatter_kernel<<<grid_for(n), kBlock, 0, s>>>(region, n, n_regions, cursor, perm);
}

}  // namespace tofmlem
