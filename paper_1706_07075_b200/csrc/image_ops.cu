// image_ops.cu -- element-wise / reduction kernels over the voxel arrays (HBM-bound, 4-wide loads).
//   update (R1, R11): x_j <- mask_j ? x_j * corr_j / sens_j : 0, corr_j <- 0
#include "internal.cuh"

namespace tofmlem {

constexpr int kBlock = 256;
constexpr int kMaxGrid = 148 * 8;

static inline unsigned grid_for(uint64_t work) {
    uint64_t g = (work + kBlock - 1) / kBlock;
    if (g > kMaxGrid) g = kMaxGrid;
    if (g == 0) g = 1;
    return (unsigned)g;
}

__device__ __forceinline__ float warp_max(float v) {
    for (int o = 16; o; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ double warp_sum(double v) {
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// max over non-negative floats (negative and NaN entries count as 0): uint ordering == float ordering
__global__ void __launch_bounds__(kBlock) max_nonneg_kernel(const float *__restrict__ x, uint64_t n, float *d_max) {
    float m = 0.0f;
    const uint64_t stride = (uint64_t)gridDim.x * kBlock;
    for (uint64_t i = (uint64_t)blockIdx.x * kBlock + threadIdx.x; i < n; i += stride) m = fmaxf(m, __ldg(x + i));
    m = warp_max(m);
    __shared__ float sm[kBlock / 32];
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x < 32) {
        m = threadIdx.x < kBlock / 32 ? sm[threadIdx.x] : 0.0f;
        m = warp_max(m);
        if (threadIdx.x == 0) atomicMax(reinterpret_cast<unsigned int *>(d_max), __float_as_uint(m));
    }
}

__device__ __forceinline__ float update_one(float x, float c, float s, float thr) {
    const bool mask = (s >= thr) && (s > 0.0f);
    return mask ? __fdiv_rn(__fmul_rn(x, c), s) : 0.0f;
}

__global__ void __launch_bounds__(kBlock) update_kernel(float *__restrict__ image, float *__restrict__ corr,
                                                        const float *__restrict__ sens,
                                                        const float *__restrict__ d_max, float floor_rel, uint64_t n,
                                                        int vec_ok) {
    const float thr = __fmul_rn(floor_rel, *d_max);
    const uint64_t stride = (uint64_t)gridDim.x * kBlock;
    const uint64_t tid = (uint64_t)blockIdx.x * kBlock + threadIdx.x;
    uint64_t done = 0;
    if (vec_ok) {
        const uint64_t n4 = n >> 2;
        float4 *img4 = reinterpret_cast<float4 *>(image);
        float4 *cor4 = reinterpret_cast<float4 *>(corr);
        const float4 *sen4 = reinterpret_cast<const float4 *>(sens);
        for (uint64_t i = tid; i < n4; i += stride) {
            float4 x = img4[i];
            const float4 c = cor4[i];
            const float4 s = __ldg(sen4 + i);
            x.x = update_one(x.x, c.x, s.x, thr);
            x.y = update_one(x.y, c.y, s.y, thr);
            x.z = update_one(x.z, c.z, s.z, thr);
            x.w = update_one(x.w, c.w, s.w, thr);
            img4[i] = x;
            cor4[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
        done = n4 << 2;
    }
    for (uint64_t i = done + tid; i < n; i += stride) {
        image[i] = update_one(image[i], corr[i], __ldg(sens + i), thr);
        corr[i] = 0.0f;
    }
}

// update with the correction image in the 2x2x1 brick layout (projector.cu, ray_scatter<BRICK>): one thread per
// brick = one float4 of corr, two float2 of image and of sens.
__global__ void __launch_bounds__(kBlock) update_brick_kernel(float *__restrict__ image, float *__restrict__ corr,
                                                              const float *__restrict__ sens,
                                                              const float *__restrict__ d_max, float floor_rel, int nx,
                                                              int ny, int nz) {
    const float thr = __fmul_rn(floor_rel, *d_max);
    const uint64_t hx = (uint64_t)(nx >> 1), hy = (uint64_t)(ny >> 1);
    const uint64_t nb = hx * hy * (uint64_t)nz;
    const uint64_t stride = (uint64_t)gridDim.x * kBlock;
    float4 *cor4 = reinterpret_cast<float4 *>(corr);
    for (uint64_t b = (uint64_t)blockIdx.x * kBlock + threadIdx.x; b < nb; b += stride) {
        const uint64_t bx = b % hx, t = b / hx;
        const uint64_t by = t % hy, z = t / hy;
        const uint64_t lo = (z * (uint64_t)ny + 2 * by) * (uint64_t)nx + 2 * bx, hi = lo + (uint64_t)nx;
        const float4 c = cor4[b];
        float2 x0 = *reinterpret_cast<float2 *>(image + lo), x1 = *reinterpret_cast<float2 *>(image + hi);
        const float2 s0 = __ldg(reinterpret_cast<const float2 *>(sens + lo));
        const float2 s1 = __ldg(reinterpret_cast<const float2 *>(sens + hi));
        x0.x = update_one(x0.x, c.x, s0.x, thr);
        x0.y = update_one(x0.y, c.y, s0.y, thr);
        x1.x = update_one(x1.x, c.z, s1.x, thr);
        x1.y = update_one(x1.y, c.w, s1.y, thr);
        *reinterpret_cast<float2 *>(image + lo) = x0;
        *reinterpret_cast<float2 *>(image + hi) = x1;
        cor4[b] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
}

// Reproducible accumulation (prepared.cu, em_det_kernel): quanta per unit of the correction image, a power of two fixed
// by max(image) alone: a ray through max(image) everywhere contributes ~0.1 / max per voxel -> 2^26 quanta.
__global__ void det_scale_kernel(const float *__restrict__ d_img_max, float *__restrict__ gscale) {
    const float m = *d_img_max;
    int e = 0;
    if (m > 0.0f && m < 3.0e38f) e = ilogbf(0.1f / m);
    e = max(-60, min(60, 26 - e));
    gscale[0] = ldexpf(1.0f, e);
    gscale[1] = ldexpf(1.0f, -e);
}

__global__ void __launch_bounds__(kBlock) update_det_kernel(float *__restrict__ image,
                                                            unsigned long long *__restrict__ corr_q,
                                                            const float *__restrict__ sens,
                                                            const float *__restrict__ d_max, float floor_rel,
                                                            const float *__restrict__ gscale, uint64_t n) {
    const float thr = __fmul_rn(floor_rel, *d_max);
    const double inv_g = (double)gscale[1];
    const uint64_t stride = (uint64_t)gridDim.x * kBlock;
    for (uint64_t i = (uint64_t)blockIdx.x * kBlock + threadIdx.x; i < n; i += stride) {
        const float c = (float)((double)corr_q[i] * inv_g);
        image[i] = update_one(image[i], c, __ldg(sens + i), thr);
        corr_q[i] = 0ull;
    }
}

void launch_det_scale(const float *d_img_max, float *gscale, cudaStream_t s) { det_scale_kernel<<<1, 1, 0, s>>>(d_img_max, gscale); }

void launch_update_det(float *image, unsigned long long *corr_q, const float *sens, const float *d_max, float floor_rel,
                       const float *gscale, uint64_t n, cudaStream_t s) {
    if (n) update_det_kernel<<<grid_for(n), kBlock, 0, s>>>(image, corr_q, sens, d_max, floor_rel, gscale, n);
}

// x0 = mask (the harness' initial image, R15)
__global__ void __launch_bounds__(kBlock) mask_init_kernel(float *__restrict__ image, const float *__restrict__ sens,
                                                           const float *__restrict__ d_max, float floor_rel,
                                                           uint64_t n) {
    const float thr = __fmul_rn(floor_rel, *d_max);
    const uint64_t stride = (uint64_t)gridDim.x * kBlock;
    for (uint64_t i = (uint64_t)blockIdx.x * kBlock + threadIdx.x; i < n; i += stride) {
        const float s = __ldg(sens + i);
        image[i] = ((s >= thr) && (s > 0.0f)) ? 1.0f : 0.0f;
    }
}

__global__ void __launch_bounds__(kBlock) dot_f64_kernel(const float *__restrict__ a, const float *__restrict__ b,
                                                         uint64_t n, double *d_out) {
    double acc = 0.0;
    const uint64_t stride = (uint64_t)gridDim.x * kBlock;
    for (uint64_t i = (uint64_t)blockIdx.x * kBlock + threadIdx.x; i < n; i += stride)
        acc += (double)__ldg(a + i) * (double)__ldg(b + i);
    acc = warp_sum(acc);
    __shared__ double sm[kBlock / 32];
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x < 32) {
        acc = threadIdx.x < kBlock / 32 ? sm[threadIdx.x] : 0.0;
        acc = warp_sum(acc);
        if (threadIdx.x == 0) atomicAdd(d_out, acc);
    }
}

__global__ void __launch_bounds__(kBlock) scale_kernel(float *__restrict__ x, float a, uint64_t n) {
    const uint64_t stride = (uint64_t)gridDim.x * kBlock;
    for (uint64_t i = (uint64_t)blockIdx.x * kBlock + threadIdx.x; i < n; i += stride) x[i] = __fmul_rn(x[i], a);
}

__global__ void __launch_bounds__(kBlock) add_kernel(float *__restrict__ dst, const float *__restrict__ src,
                                                     uint64_t n) {
    const uint64_t stride = (uint64_t)gridDim.x * kBlock;
    for (uint64_t i = (uint64_t)blockIdx.x * kBlock + threadIdx.x; i < n; i += stride) dst[i] += __ldg(src + i);
}

void launch_max_nonneg(const float *x, uint64_t n, float *d_max, cudaStream_t s) {
    cudaMemsetAsync(d_max, 0, sizeof(float), s);
    if (n) max_nonneg_kernel<<<grid_for(n), kBlock, 0, s>>>(x, n, d_max);
}

void launch_update(float *image, float *corr, const float *sens, const float *d_max, float floor_rel, uint64_t n,
                   cudaStream_t s) {
    if (!n) return;
    const int vec_ok = ((reinterpret_cast<uintptr_t>(image) | reinterpret_cast<uintptr_t>(corr) |
                         reinterpret_cast<uintptr_t>(sens)) & 15) == 0;
    update_kernel<<<grid_for(vec_ok ? (n >> 2) + 1 : n), kBlock, 0, s>>>(image, corr, sens, d_max, floor_rel, n,
                                                                         vec_ok);
}

void launch_mask_init(float *image, const float *sens, const float *d_max, float floor_rel, uint64_t n,
                      cudaStream_t s) {
    if (n) mask_init_kernel<<<grid_for(n), kBlock, 0, s>>>(image, sens, d_max, floor_rel, n);
}

void launch_dot_f64(const float *a, const float *b, uint64_t n, double *d_out, cudaStream_t s) {
    cudaMemsetAsync(d_out, 0, sizeof(double), s);
    if (n) dot_f64_kernel<<<grid_for(n), kBlock, 0, s>>>(a, b, n, d_out);
}

void launch_scale(float *x, float a, uint64_t n, cudaStream_t s) {
    if (n) scale_kernel<<<grid_for(n), kBlock, 0, s>>>(x, a, n);
}

void launch_add(float *dst, const float *src, uint64_t n, cudaStream_t s) {
    if (n) add_kernel<<<grid_for(n), kBlock, 0, s>>>(dst, src, n);
}

}  // namespace tofmlem

namespace tofmlem {

// ---------------------------------------------------------------------------------------------------------------
// NEXT-2: 3x3x3 median filter between iterations ("we introduced a median filter between MLEM
// iterations"; the size is not stated -> R23: the 27-voxel cube, edges replicated).  One thread per output voxel:
// 27 loads (neighbouring threads share them through L1) and a forgetful-selection network in registers: keep 15
// values, drop their minimum and maximum (neither can be the median of 27), take in one more value, repeat; the
// last three values' middle one is the 14th smallest of the 27.  The result is one of the inputs, so the filter
// is bit-exact against any correct implementation.
__device__ __forceinline__ void cmpxchg(float &a, float &b) {
    const float lo = fminf(a, b), hi = fmaxf(a, b);
    a = lo;
    b = hi;
}

__global__ void __launch_bounds__(kBlock) median3_kernel(const float *__restrict__ in, float *__restrict__ out, int nx,
                                                         int ny, int nz) {
    const uint64_t nvox = (uint64_t)nx * ny * nz;
    const uint64_t j = (uint64_t)blockIdx.x * kBlock + threadIdx.x;
    if (j >= nvox) return;
    const int x = (int)(j % (uint64_t)nx);
    const uint64_t t = j / (uint64_t)nx;
    const int y = (int)(t % (uint64_t)ny), z = (int)(t / (uint64_t)ny);
    int xo[3], yo[3], zo[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        xo[d] = min(max(x + d - 1, 0), nx - 1);
        yo[d] = min(max(y + d - 1, 0), ny - 1);
        zo[d] = min(max(z + d - 1, 0), nz - 1);
    }
    float v[27];
#pragma unroll
    for (int dz = 0; dz < 3; ++dz)
#pragma unroll
        for (int dy = 0; dy < 3; ++dy) {
            const float *row = in + ((size_t)zo[dz] * ny + yo[dy]) * nx;
#pragma unroll
            for (int dx = 0; dx < 3; ++dx) v[(dz * 3 + dy) * 3 + dx] = __ldg(row + xo[dx]);
        }
    // working set w = v[0..14]; v[15..26] are fed in one per stage
#pragma unroll
    for (int s = 0; s < 13; ++s) {
#pragma unroll
        for (int i = s + 1; i <= 14; ++i) cmpxchg(v[s], v[i]);  // minimum of the active range -> v[s]
#pragma unroll
        for (int i = s + 1; i < 14; ++i) cmpxchg(v[i], v[14]);  // maximum -> v[14]
        if (s < 12) v[14] = v[15 + s];                          // forget both, take the next value in
    }
    out[j] = v[13];
}

void launch_update_brick(float *image, float *corr, const float *sens, const float *d_max, float floor_rel, int nx,
                         int ny, int nz, cudaStream_t s) {
    const uint64_t nb = (uint64_t)(nx >> 1) * (ny >> 1) * nz;
    update_brick_kernel<<<grid_for(nb), kBlock, 0, s>>>(image, corr, sens, d_max, floor_rel, nx, ny, nz);
}

void launch_median3(const float *in, float *out, int nx, int ny, int nz, cudaStream_t s) {
    const uint64_t nvox = (uint64_t)nx * ny * nz;
    median3_kernel<<<(unsigned)((nvox + kBlock - 1) / kBlock), kBlock, 0, s>>>(in, out, nx, ny, nz);
}

// w <- exp(w)  (NEXT-3: attenuation weight from the line integral of mu, R19); accurate expf
__global__ void __launch_bounds__(kBlock) exp_kernel(float *__restrict__ w, uint64_t n) {
    const uint64_t stride = (uint64_t)gridDim.x * kBlock;
    for (uint64_t i = (uint64_t)blockIdx.x * kBlock + threadIdx.x; i < n; i += stride) w[i] = expf(w[i]);
}

void launch_exp(float *w, uint64_t n, cudaStream_t s) {
    if (n) exp_kernel<<<grid_for(n), kBlock, 0, s>>>(w, n);
}

}  // namespace tofmlem
