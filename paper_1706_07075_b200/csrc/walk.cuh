// walk.cuh -- device code shared by the projector kernels (projector.cu, tile.cu): ray set-up in fp64, the
// branch-free fp32 voxel walk, the gather and scatter walks against global memory.  See the header comment of
// projector.cu for the design.
#pragma once
#include <math.h>

#include "internal.cuh"

namespace tofmlem {

struct Ray {
    float t_end, tc;
    float t0x, t0y, t0z;
    float tdx, tdy, tdz;
    int idx;            // flat index of the first voxel
    int dxi, dyi, dzi;  // flat-index increments of a step along each axis, 0 when parallel
    // brick layout of the correction image (2x2x1 voxels per 16-byte group, see ProjParams::brick):
    int bidx;        // brick-layout index of the first voxel
    int bdx0, bdxs;  // x step: increment for the first step, and the sum of the two alternating increments
    int bdy0, bdys;  // y step: likewise
};

__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ bool finite_f(float x) { return fabsf(x) <= 3.402823466e+38f; }  // false for NaN/Inf

__device__ __forceinline__ void red_v4(float *p, float a, float b, float c, float d) {
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}

__device__ __forceinline__ void red_v4_if(bool p, float *ptr, float a, float b, float c, float d) {
    asm volatile(
        "{\n .reg .pred q;\n setp.ne.s32 q, %5, 0;\n @q red.global.add.v4.f32 [%0], {%1, %2, %3, %4};\n}" ::"l"(ptr),
        "f"(a), "f"(b), "f"(c), "f"(d), "r"((int)p)
        : "memory");
}

constexpr float kBigT = 1.0e30f;

// Per-axis set-up; returns the parameter at which the ray leaves the grid through this axis.
__device__ __forceinline__ float axis_setup(double p1, double u, double s_lo, double o, double v, double iv, int n,
                                            int stride, int &i, int &di, float &t0, float &td) {
    const double q = (p1 + u * s_lo - o) * iv;
    const double fl = floor(q);
    int ii = (int)fl;
    if (u < 0.0 && fl == q) ii -= 1;  // sitting exactly on a plane and moving down: the voxel below
    ii = max(0, min(n - 1, ii));
    i = ii;
    if (u == 0.0) {
        di = 0;
        t0 = __int_as_float(0x7f800000);
        td = 0.0f;
        return t0;
    }
    const double iu = 1.0 / u;
    const int k = u > 0.0 ? ii + 1 : ii;
    const double sc = (o + (double)k * v - p1) * iu - s_lo;
    di = u > 0.0 ? stride : -stride;
    t0 = (float)fmax(sc, 0.0);
    td = fminf((float)(v * fabs(iu)), kBigT);
    const int nsteps = u > 0.0 ? n - 1 - ii : ii;
    return nsteps == 0 ? t0 : fmaf((float)nsteps, td, t0);
}

// Slab clip of one axis; false when the ray is parallel to the axis and outside the slab.
__device__ __forceinline__ bool axis_clip(double p1, double u, double lo, double hi, double &s_lo, double &s_hi) {
    if (u == 0.0) return !(p1 < lo || p1 >= hi);
    const double iu = 1.0 / u;
    const double a = (lo - p1) * iu, b = (hi - p1) * iu;
    s_lo = fmax(s_lo, fmin(a, b));
    s_hi = fmin(s_hi, fmax(a, b));
    return true;
}

// What the tile-mode pass (tile.cu) needs beyond the Ray: the first voxel, the TOF centre in continuous voxel
// coordinates and the direction.
struct RayExtra {
    int i[3];     // first voxel of the window
    double cv[3]; // TOF kernel centre, voxel coordinates (p1 + u s_c - o) / v
    double u[3];  // unit direction
};

// Ray set-up in fp64 (comment (1) at the top); false when the event is skipped or its window misses the grid.
template <bool TOF, bool EXTRA = false>
__device__ __forceinline__ bool ray_setup(const ProjParams &P, float fx1, float fy1, float fz1, float fx2, float fy2,
                                          float fz2, float fdt, Ray &r, RayExtra *x = nullptr) {
    if (!(finite_f(fx1) && finite_f(fy1) && finite_f(fz1) && finite_f(fx2) && finite_f(fy2) && finite_f(fz2)))
        return false;
    if (TOF && !finite_f(fdt)) return false;
    constexpr int A = 0, B = 1, C = 2;
    const int nA = P.n[A], nB = P.n[B], nC = P.n[C];
    const double oA = P.o[A], oB = P.o[B], oC = P.o[C];
    const double hA = P.h[A], hB = P.h[B], hC = P.h[C];
    const double vA = P.v[A], vB = P.v[B], vC = P.v[C];
    const double ivA = P.iv[A], ivB = P.iv[B], ivC = P.iv[C];
    const double x1 = fx1, y1 = fy1, z1 = fz1;
    const double dx = (double)fx2 - x1, dy = (double)fy2 - y1, dz = (double)fz2 - z1;
    const double L2 = dx * dx + dy * dy + dz * dz;
    if (!(L2 > 0.0)) return false;
    const double L = sqrt(L2);
    const double iL = 1.0 / L;
    const double ux = dx * iL, uy = dy * iL, uz = dz * iL;
    double s_lo = 0.0, s_hi = L;
    if (!axis_clip(x1, ux, oA, hA, s_lo, s_hi)) return false;
    if (!axis_clip(y1, uy, oB, hB, s_lo, s_hi)) return false;
    if (!axis_clip(z1, uz, oC, hC, s_lo, s_hi)) return false;
    double s_c = 0.0;
    if (TOF) {
        s_c = 0.5 * L + (0.5 * kCmmPerPs) * (double)fdt;
        s_lo = fmax(s_lo, s_c - P.half_window);
        s_hi = fmin(s_hi, s_c + P.half_window);
    }
    if (!(s_hi > s_lo)) return false;
    r.tc = (float)(s_c - s_lo);
    int ia, ib, ic;
    const float ea = axis_setup(x1, ux, s_lo, oA, vA, ivA, nA, 1, ia, r.dxi, r.t0x, r.tdx);
    const float eb = axis_setup(y1, uy, s_lo, oB, vB, ivB, nB, nA, ib, r.dyi, r.t0y, r.tdy);
    const float ec = axis_setup(z1, uz, s_lo, oC, vC, ivC, nC, nA * nB, ic, r.dzi, r.t0z, r.tdz);
    r.t_end = fminf(fminf((float)(s_hi - s_lo), ea), fminf(eb, ec));
    r.idx = (ic * nB + ib) * nA + ia;
    if (EXTRA) {
        x->i[0] = ia; x->i[1] = ib; x->i[2] = ic;
        x->cv[0] = (x1 + ux * s_c - oA) * ivA;
        x->cv[1] = (y1 + uy * s_c - oB) * ivB;
        x->cv[2] = (z1 + uz * s_c - oC) * ivC;
        x->u[0] = ux; x->u[1] = uy; x->u[2] = uz;
    }
    if (P.brick) {
        // index = (brick number) * 4 + (iy & 1) * 2 + (ix & 1): a step in x alternates between +-1 (inside the brick)
        // and +-3 (into the neighbouring brick), a step in y between +-2 and +-(2 nx - 2); z steps are unchanged
        r.bidx = ((ic * (nB >> 1) + (ib >> 1)) * (nA >> 1) + (ia >> 1)) * 4 + ((ib & 1) << 1) + (ia & 1);
        const int xa = r.dxi > 0 ? 1 : (r.dxi < 0 ? -3 : 0), xb = r.dxi > 0 ? 3 : (r.dxi < 0 ? -1 : 0);
        r.bdx0 = (ia & 1) ? xb : xa;
        r.bdxs = xa + xb;
        const int yo = 2 * nA - 2;
        const int ya = r.dyi > 0 ? 2 : (r.dyi < 0 ? -yo : 0), yb = r.dyi > 0 ? yo : (r.dyi < 0 ? -2 : 0);
        r.bdy0 = (ib & 1) ? yb : ya;
        r.bdys = ya + yb;
    }
    return true;
}

// Branch-free incremental walk.  step() returns the un-normalised weight of the current clipped chord and its
// flat voxel index, and advances; `done` is set on the last chord.
template <bool TOF, bool BRICK = false>
struct Walker {
    float tx, ty, tz, kx, ky, kz, t;
    int idx, dxc, dyc;
    __device__ __forceinline__ explicit Walker(const Ray &r)
        : tx(r.t0x), ty(r.t0y), tz(r.t0z), kx(0.f), ky(0.f), kz(0.f), t(0.f), idx(BRICK ? r.bidx : r.idx),
          dxc(BRICK ? r.bdx0 : r.dxi), dyc(BRICK ? r.bdy0 : r.dyi) {}
    __device__ __forceinline__ float step(const ProjParams &P, const Ray &r, int &at, bool &done) {
        const float tn = fminf(fminf(tx, ty), fminf(tz, r.t_end));
        const float l = tn - t;
        float w = l;
        if (TOF) {
            const float tm = fmaf(0.5f, t + tn, -r.tc);
            w = l * ex2_approx(P.gauss_a * tm * tm);
        }
        at = idx;
        done = tn >= r.t_end;
        if (tx <= tn) {
            kx += 1.0f;
            idx += dxc;
            if (BRICK) dxc = r.bdxs - dxc;
        }
        if (ty <= tn) {
            ky += 1.0f;
            idx += dyc;
            if (BRICK) dyc = r.bdys - dyc;
        }
        if (tz <= tn) { kz += 1.0f; idx += r.dzi; }
        tx = fmaf(kx, r.tdx, r.t0x);
        ty = fmaf(ky, r.tdy, r.t0y);
        tz = fmaf(kz, r.tdz, r.t0z);
        t = tn;
        return w;
    }
};

// sum_j w_j image[j] over the window (un-normalised).  Software pipeline of depth kGatherDepth on the gathers: the
// value loaded in one step is consumed kGatherDepth steps later, which hides the L1/L2 latency behind whole steps of
// arithmetic.  Depth 3 was measured (48 registers): 24.01 vs 24.09 ms, no gain -- the pass is not gather-latency-bound.
constexpr int kGatherDepth = 2;

template <bool TOF>
__device__ __forceinline__ float ray_gather(const ProjParams &P, const Ray &r, const float *__restrict__ image,
                                            int &visits) {
    Walker<TOF> wk(r);
    float acc = 0.0f;
    float w[kGatherDepth], v[kGatherDepth];
#pragma unroll
    for (int i = 0; i < kGatherDepth; ++i) w[i] = v[i] = 0.0f;
    int at, n = 0;
    bool done = false;
    while (!done) {
#pragma unroll
        for (int i = 0; i < kGatherDepth; ++i) {
            if (!done) {
                acc = fmaf(w[i], v[i], acc);  // the pair this slot has held for kGatherDepth steps
                w[i] = wk.step(P, r, at, done);
                v[i] = __ldg(image + at);
                ++n;
            }
        }
    }
#pragma unroll
    for (int i = 0; i < kGatherDepth; ++i) acc = fmaf(w[i], v[i], acc);
    visits = n;
    return acc;
}

// out[j] += w_j * scale over the window: float32 reductions at L2, fire and forget.
// VEC: one 16-byte vector reduction per aligned group of 4 voxels (needs a 16-byte aligned `out` whose
// allocation covers whole groups); otherwise one scalar reduction per voxel.
// BRICK (with VEC): `out` is in the brick layout, whose 16-byte groups are 2x2x1 voxels: a line that meets a group meets
// 1.50 of its voxels on average against 1.34 for 4x1x1 groups (Cauchy: 4 * 6 / surface), i.e. 11 % fewer reductions.
template <bool TOF, bool VEC, bool BRICK = false>
__device__ __forceinline__ int ray_scatter(const ProjParams &P, const Ray &r, float *__restrict__ out, float scale) {
    Walker<TOF, BRICK> wk(r);
    int at, reds = 1;
    bool done;
    if (VEC) {
        // The flush is a predicated instruction, not a branch: some lane of a warp flushes in nearly every step
        // (ncu r01b: 97 % of the warp iterations), so a branch only adds its re-convergence overhead.
        int grp = (BRICK ? r.bidx : r.idx) >> 2;
        float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
#pragma unroll 2
        do {
            const float val = wk.step(P, r, at, done) * scale;
            const int g = at >> 2;
            const bool fl = g != grp;
            red_v4_if(fl, out + 4 * (size_t)grp, a0, a1, a2, a3);
            reds += fl;
            grp = g;
            const int sl = at & 3;  // each voxel is met once per ray: plain writes, no accumulation
            a0 = sl == 0 ? val : (fl ? 0.f : a0);
            a1 = sl == 1 ? val : (fl ? 0.f : a1);
            a2 = sl == 2 ? val : (fl ? 0.f : a2);
            a3 = sl == 3 ? val : (fl ? 0.f : a3);
        } while (!done);
        red_v4(out + 4 * (size_t)grp, a0, a1, a2, a3);
    } else {
        reds = 0;
        do {
            const float w = wk.step(P, r, at, done);
            atomicAdd(out + at, w * scale);  // zero-length chords (corner crossings) add +0: harmless, rare
            ++reds;
        } while (!done);
    }
    return reds;
}

}  // namespace tofmlem
