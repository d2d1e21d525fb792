// projector.cu -- ray-driven TOF projector kernels (forward, backproject, fused EM pass).
//
// System matrix (include/tofmlem.h; R2,R4-R8): a_ej = l_ej * g_sigma(s_mid - s_c), Siddon chords
// clipped to the +-T sigma window around the TOF centre, Gaussian at the clipped
// chord midpoint.  One thread per event:
//   1. ray set-up in fp64 (direction, slab clip against the grid, window, first plane crossings);
//      everything is then expressed in the window-local parameter t = s - s_lo in [0, 6 sigma], which keeps
//      the fp32 walk's rounding at ~4e-6 mm although coordinates reach +-1200 mm;
//   2. incremental voxel walk in fp32: next crossing per axis = fma(k, dt_axis, t0_axis) (no accumulated
//      additions), weight = l * ex2(gauss_a * tm^2).
#include "internal.cuh"

namespace tofmlem {

struct Ray {
    float t_hi, tc;
    float t0x, t0y, t0z;
    float tdx, tdy, tdz;
    int ix, iy, iz;
    int sx, sy, sz;
};

__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ bool finite_f(float x) { return fabsf(x) <= 3.402823466e+38f; }  // false for NaN/Inf

__device__ __forceinline__ void axis_setup(double p1, double u, double s_lo, double o, double v, double iv, int n,
                                           int &i, int &step, float &t0, float &td) {
    const double q = (p1 + u * s_lo - o) * iv;
    const double fl = floor(q);
    int ii = (int)fl;
    if (u < 0.0 && fl == q) ii -= 1;  // sitting exactly on a plane and moving down: the voxel below
    ii = max(0, min(n - 1, ii));
    i = ii;
    if (u == 0.0) {
        step = 0;
        t0 = __int_as_float(0x7f800000);
        td = 0.0f;
    } else {
        const double iu = 1.0 / u;
        const int k = u > 0.0 ? ii + 1 : ii;
        const double sc = (o + (double)k * v - p1) * iu - s_lo;
        step = u > 0.0 ? 1 : -1;
        t0 = (float)fmax(sc, 0.0);
        td = (float)(v * fabs(iu));
    }
}

template <bool TOF>
__device__ __forceinline__ bool ray_setup(const ProjParams &P, float fx1, float fy1, float fz1, float fx2, float fy2,
                                          float fz2, float fdt, Ray &r) {
    if (!(finite_f(fx1) && finite_f(fy1) && finite_f(fz1) && finite_f(fx2) && finite_f(fy2) && finite_f(fz2)))
        return false;
    if (TOF && !finite_f(fdt)) return false;
    const double x1 = fx1, y1 = fy1, z1 = fz1;
    const double dx = (double)fx2 - x1, dy = (double)fy2 - y1, dz = (double)fz2 - z1;
    const double L2 = dx * dx + dy * dy + dz * dz;
    if (!(L2 > 0.0)) return false;
    const double L = sqrt(L2);
    const double iL = 1.0 / L;
    const double ux = dx * iL, uy = dy * iL, uz = dz * iL;
    double s_lo = 0.0, s_hi = L;
    // slab clip against the grid box
    if (ux == 0.0) {
        if (x1 < P.ox || x1 >= P.hx) return false;
    } else {
        const double iu = 1.0 / ux;
        const double a = (P.ox - x1) * iu, b = (P.hx - x1) * iu;
        s_lo = fmax(s_lo, fmin(a, b));
        s_hi = fmin(s_hi, fmax(a, b));
    }
    if (uy == 0.0) {
        if (y1 < P.oy || y1 >= P.hy) return false;
    } else {
        const double iu = 1.0 / uy;
        const double a = (P.oy - y1) * iu, b = (P.hy - y1) * iu;
        s_lo = fmax(s_lo, fmin(a, b));
        s_hi = fmin(s_hi, fmax(a, b));
    }
    if (uz == 0.0) {
        if (z1 < P.oz || z1 >= P.hz) return false;
    } else {
        const double iu = 1.0 / uz;
        const double a = (P.oz - z1) * iu, b = (P.hz - z1) * iu;
        s_lo = fmax(s_lo, fmin(a, b));
        s_hi = fmin(s_hi, fmax(a, b));
    }
    double s_c = 0.0;
    if (TOF) {
        s_c = 0.5 * L + (0.5 * kCmmPerPs) * (double)fdt;
        s_lo = fmax(s_lo, s_c - P.half_window);
        s_hi = fmin(s_hi, s_c + P.half_window);
    }
    if (!(s_hi > s_lo)) return false;
    r.t_hi = (float)(s_hi - s_lo);
    r.tc = (float)(s_c - s_lo);
    axis_setup(x1, ux, s_lo, P.ox, P.vx, P.ivx, P.nx, r.ix, r.sx, r.t0x, r.tdx);
    axis_setup(y1, uy, s_lo, P.oy, P.vy, P.ivy, P.ny, r.iy, r.sy, r.t0y, r.tdy);
    axis_setup(z1, uz, s_lo, P.oz, P.vz, P.ivz, P.nz, r.iz, r.sz, r.t0z, r.tdz);
    return true;
}

// Walk the voxels of the window; visit(flat index, un-normalised weight) for every clipped chord.
template <bool TOF, class Visit>
__device__ __forceinline__ int ray_walk(const ProjParams &P, const Ray &r, Visit &&visit) {
    int ix = r.ix, iy = r.iy, iz = r.iz;
    int idx = (iz * P.ny + iy) * P.nx + ix;
    const int dyi = r.sy * P.nx, dzi = r.sz * P.nx * P.ny;
    float tx = r.t0x, ty = r.t0y, tz = r.t0z;
    float kx = 0.0f, ky = 0.0f, kz = 0.0f;
    float t = 0.0f;
    const float t_hi = r.t_hi;
    int visits = 0;
    while (true) {
        const float tn = fminf(fminf(tx, ty), fminf(tz, t_hi));
        const float l = tn - t;
        float w = l;
        if (TOF) {
            const float tm = fmaf(0.5f, t + tn, -r.tc);
            w = l * ex2_approx(P.gauss_a * tm * tm);
        }
        visit(idx, w);
        ++visits;
        if (tn >= t_hi) break;
        if (tx <= tn) {
            ix += r.sx;
            if ((unsigned)ix >= (unsigned)P.nx) break;
            idx += r.sx;
            kx += 1.0f;
            tx = fmaf(kx, r.tdx, r.t0x);
        }
        if (ty <= tn) {
            iy += r.sy;
            if ((unsigned)iy >= (unsigned)P.ny) break;
            idx += dyi;
            ky += 1.0f;
            ty = fmaf(ky, r.tdy, r.t0y);
        }
        if (tz <= tn) {
            iz += r.sz;
            if ((unsigned)iz >= (unsigned)P.nz) break;
            idx += dzi;
            kz += 1.0f;
            tz = fmaf(kz, r.tdz, r.t0z);
        }
        t = tn;
    }
    return visits;
}

template <bool TOF>
__device__ __forceinline__ bool load_and_setup(const ProjParams &P, const EventPtrs &ev, uint64_t e, Ray &r) {
    const float x1 = __ldg(ev.x1 + e), y1 = __ldg(ev.y1 + e), z1 = __ldg(ev.z1 + e);
    const float x2 = __ldg(ev.x2 + e), y2 = __ldg(ev.y2 + e), z2 = __ldg(ev.z2 + e);
    const float dt = (TOF && ev.dt) ? __ldg(ev.dt + e) : 0.0f;
    return ray_setup<TOF>(P, x1, y1, z1, x2, y2, z2, dt, r);
}

constexpr int kBlock = 256;

template <bool TOF>
__global__ void __launch_bounds__(kBlock) forward_kernel(ProjParams P, EventPtrs ev, uint64_t n,
                                                         const float *__restrict__ image, float *__restrict__ fwd) {
    const uint64_t e = (uint64_t)blockIdx.x * kBlock + threadIdx.x;
    if (e >= n) return;
    Ray r;
    float acc = 0.0f;
    if (load_and_setup<TOF>(P, ev, e, r)) {
        ray_walk<TOF>(P, r, [&](int idx, float w) { acc = fmaf(w, __ldg(image + idx), acc); });
        if (TOF) acc *= P.gauss_norm;
    }
    fwd[e] = acc;
}

template <bool TOF>
__global__ void __launch_bounds__(kBlock) backproject_kernel(ProjParams P, EventPtrs ev, uint64_t n,
                                                             const float *__restrict__ values,
                                                             float *__restrict__ out) {
    const uint64_t e = (uint64_t)blockIdx.x * kBlock + threadIdx.x;
    if (e >= n) return;
    Ray r;
    if (!load_and_setup<TOF>(P, ev, e, r)) return;
    float val = values ? __ldg(values + e) : 1.0f;
    if (TOF) val *= P.gauss_norm;
    if (val == 0.0f) return;
    ray_walk<TOF>(P, r, [&](int idx, float w) { atomicAdd(out + idx, w * val); });
}

// Fused EM pass: walk 1 gathers the image (forward value stays in a register), walk 2 recomputes the
// weights and scatters w / fwd with float32 reductions at L2.
template <bool TOF>
__global__ void __launch_bounds__(kBlock) em_correction_kernel(ProjParams P, EventPtrs ev, uint64_t n,
                                                               const float *__restrict__ image,
                                                               float *__restrict__ corr, DeviceStats *stats) {
    const uint64_t e = (uint64_t)blockIdx.x * kBlock + threadIdx.x;
    Ray r;
    int visits = 0;
    bool valid = false;
    if (e < n && load_and_setup<TOF>(P, ev, e, r)) {
        float acc = 0.0f;
        visits = ray_walk<TOF>(P, r, [&](int idx, float w) { acc = fmaf(w, __ldg(image + idx), acc); });
        if (acc > 0.0f) {  // R9
            valid = true;
            const float rinv = 1.0f / acc;  // the Gaussian normalisation cancels in a_ej / fwd_e
            ray_walk<TOF>(P, r, [&](int idx, float w) { atomicAdd(corr + idx, w * rinv); });
        }
    }
    // per-warp counters -> one atomic per warp
    const unsigned nv = __popc(__ballot_sync(0xffffffffu, valid));
    const unsigned vis = __reduce_add_sync(0xffffffffu, (unsigned)visits);
    if ((threadIdx.x & 31) == 0 && stats) {
        if (nv) atomicAdd(&stats->n_valid, (unsigned long long)nv);
        if (vis) atomicAdd(&stats->visits, (unsigned long long)vis);
    }
}

static inline unsigned grid_for(uint64_t n) { return (unsigned)((n + kBlock - 1) / kBlock); }

void launch_forward(const ProjParams &p, bool tof, const EventPtrs &ev, uint64_t n, const float *image, float *fwd,
                    cudaStream_t s) {
    if (n == 0) return;
    if (tof)
        forward_kernel<true><<<grid_for(n), kBlock, 0, s>>>(p, ev, n, image, fwd);
    else
        forward_kernel<false><<<grid_for(n), kBlock, 0, s>>>(p, ev, n, image, fwd);
}

void launch_backproject(const ProjParams &p, bool tof, const EventPtrs &ev, uint64_t n, const float *values,
                        float *out, cudaStream_t s) {
    if (n == 0) return;
    if (tof)
        backproject_kernel<true><<<grid_for(n), kBlock, 0, s>>>(p, ev, n, values, out);
    else
        backproject_kernel<false><<<grid_for(n), kBlock, 0, s>>>(p, ev, n, values, out);
}

void launch_em_correction(const ProjParams &p, bool tof, const EventPtrs &ev, uint64_t n, const float *image,
                          float *corr, DeviceStats *stats, cudaStream_t s) {
    if (n == 0) return;
    if (tof)
        em_correction_kernel<true><<<grid_for(n), kBlock, 0, s>>>(p, ev, n, image, corr, stats);
    else
        em_correction_kernel<false><<<grid_for(n), kBlock, 0, s>>>(p, ev, n, image, corr, stats);
}

}  // namespace tofmlem
