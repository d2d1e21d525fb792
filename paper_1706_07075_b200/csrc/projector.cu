// projector.cu -- ray-driven TOF projector kernels (forward, backproject, fused EM pass).
//
// System matrix (include/tofmlem.h; R2,R4-R8): a_ej = l_ej * g_sigma(s_mid - s_c), Siddon chords
// clipped to the +-T sigma window around the TOF centre, Gaussian at the clipped
// chord midpoint.  One thread per event:
//   1. ray set-up in fp64 (direction, slab clip against the grid, window, first plane crossings);
//      everything is then expressed in the window-local parameter t = s - s_lo in [0, 6 sigma], which keeps
//      the fp32 walk's rounding at ~4e-6 mm although coordinates reach +-1200 mm;
//   2. incremental voxel walk in fp32, branch-free: next crossing per axis = fma(k, dt_axis, t0_axis) (no
//      accumulated additions), weight = l * ex2(gauss_a * tm^2).  The walk ends at
//      t_end = min(window end, grid-exit crossing of each axis evaluated with the SAME fma), so the flat
//      voxel index never leaves the grid and needs no bounds test inside the loop;
//   3. gathers are software-pipelined over two loop stages (the value loaded in one stage is consumed in the
//      next), which hides the L1/L2 latency behind a full stage of arithmetic;
//   4. scatters: a straight line meets each aligned group of 4 consecutive voxels in ONE contiguous run, so
//      the run is collected in registers and sent as one 16-byte `red.global.add.v4.f32` (measured on B200:
//      ~1.9x the rate of scalar reductions and 1.3-1.8x fewer of them);
//   5. CTAs take 256-event chunks of the (locality-binned) list in an interleaved order (`stride` segments
//      advance in parallel): each CTA stays local for its gathers, while the reductions of the ~900
//      co-resident CTAs spread over the whole volume instead of serialising on a few hot L2 sectors
//      (measured: 47.8 -> 35.7 ms per pass at cfg-3).
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

// Ray set-up in fp64 (comment (1) at the top); false when the event is skipped or its window misses the grid.
template <bool TOF>
__device__ __forceinline__ bool ray_setup(const ProjParams &P, float fx1, float fy1, float fz1, float fx2, float fy2,
                                          float fz2, float fdt, Ray &r) {
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


constexpr int kBlock = 256;

template <bool TOF>
__device__ __forceinline__ bool load_and_setup(const ProjParams &P, const EventPtrs &ev, uint64_t e, Ray &r) {
    const float x1 = __ldcs(ev.x1 + e), y1 = __ldcs(ev.y1 + e), z1 = __ldcs(ev.z1 + e);
    const float x2 = __ldcs(ev.x2 + e), y2 = __ldcs(ev.y2 + e), z2 = __ldcs(ev.z2 + e);
    const float dt = (TOF && ev.dt) ? __ldcs(ev.dt + e) : 0.0f;
    return ray_setup<TOF>(P, x1, y1, z1, x2, y2, z2, dt, r);
}

// Event index of this thread under the interleaved chunk order (comment (5) at the top).
__device__ __forceinline__ uint64_t event_index(unsigned stride) {
    if (stride <= 1) return (uint64_t)blockIdx.x * kBlock + threadIdx.x;
    const unsigned rows = gridDim.x / stride;  // the grid is a multiple of stride
    const uint64_t chunk = (uint64_t)(blockIdx.x % stride) * rows + blockIdx.x / stride;
    return chunk * kBlock + threadIdx.x;
}

template <bool TOF>
__global__ void __launch_bounds__(kBlock) forward_kernel(ProjParams P, EventPtrs ev, uint64_t n,
                                                         const float *__restrict__ image, float *__restrict__ fwd) {
    const uint64_t e = (uint64_t)blockIdx.x * kBlock + threadIdx.x;
    if (e >= n) return;
    Ray r;
    float acc = 0.0f;
    if (load_and_setup<TOF>(P, ev, e, r)) {
        int visits;
        acc = ray_gather<TOF>(P, r, image, visits);
        if (TOF) acc *= P.gauss_norm;
    }
    fwd[e] = acc;
}

template <bool TOF, bool VEC>
__global__ void __launch_bounds__(kBlock) backproject_kernel(ProjParams P, EventPtrs ev, uint64_t n,
                                                             const float *__restrict__ values,
                                                             float *__restrict__ out) {
    const uint64_t e = event_index(P.stride);
    if (e >= n) return;
    Ray r;
    if (!load_and_setup<TOF>(P, ev, e, r)) return;
    float val = values ? __ldg(values + e) : 1.0f;
    if (TOF) val *= P.gauss_norm;
    if (val == 0.0f) return;
    ray_scatter<TOF, VEC>(P, r, out, val);
}

// One event of the fused EM pass: walk 1 gathers the image (the forward value stays in a register), walk 2
// recomputes the weights and scatters w / fwd (the Gaussian normalisation cancels in a_ej / fwd_e).
template <bool TOF, bool VEC, bool BRICK>
__device__ __forceinline__ void em_event(const ProjParams &P, const EventPtrs &ev, uint64_t e, uint64_t n,
                                         const float *__restrict__ evw, const float *__restrict__ image,
                                         float *__restrict__ corr, int &visits, bool &valid, int &reds) {
    Ray r;
    visits = 0;
    reds = 0;
    valid = false;
    if (e < n && load_and_setup<TOF>(P, ev, e, r)) {
        const float acc = ray_gather<TOF>(P, r, image, visits);
        if (acc > 0.0f) {  // R9
            valid = true;
            // evw: optional per-event weight (attenuation correction applied to the LOR, R19)
            reds = ray_scatter<TOF, VEC, BRICK>(P, r, corr, (evw ? __ldg(evw + e) : 1.0f) / acc);
        }
    }
}

// Grid-order form: one CTA per 256-event chunk, chunks interleaved (comment (5) at the top).
template <bool TOF, bool VEC, bool BRICK>
__global__ void __launch_bounds__(kBlock) em_correction_kernel(ProjParams P, EventPtrs ev, uint64_t n,
                                                               const float *__restrict__ evw,
                                                               const float *__restrict__ image,
                                                               float *__restrict__ corr, DeviceStats *stats) {
    int visits, reds;
    bool valid;
    em_event<TOF, VEC, BRICK>(P, ev, event_index(P.stride), n, evw, image, corr, visits, valid, reds);
    // per-warp counters -> one atomic per warp
    const unsigned nv = __popc(__ballot_sync(0xffffffffu, valid));
    const unsigned vis = __reduce_add_sync(0xffffffffu, (unsigned)visits);
    const unsigned nr = __reduce_add_sync(0xffffffffu, (unsigned)reds);
    if ((threadIdx.x & 31) == 0 && stats) {
        if (nv) atomicAdd(&stats->n_valid, (unsigned long long)nv);
        if (vis) atomicAdd(&stats->visits, (unsigned long long)vis);
        if (nr) atomicAdd(&stats->reds, (unsigned long long)nr);
    }
}

// Persistent form of the fused pass (the default): the locality-binned event list is cut into `nseg` contiguous
// segments, two per SM; every warp takes 32-event chunks from the queue of the SM it runs on (%smid), so the warps
// resident on an SM work on neighbouring events and share that SM's L1 for their image gathers (the 8 co-resident
// CTAs of the grid-order form come from 8 unrelated places and thrash it), while different SMs reduce into different
// parts of the volume.  A warp whose segment is exhausted moves on to other segments (work stealing; the invalid
// events sorted to the end of the list make the last segments empty).  Measured at cfg-3: 30.2 -> 25.2 ms.
template <bool TOF, bool VEC, bool BRICK>
__global__ void __launch_bounds__(kBlock, 5) em_persistent_kernel(ProjParams P, EventPtrs ev, uint64_t n,
                                                               const float *__restrict__ evw,
                                                               const float *__restrict__ image,
                                                               float *__restrict__ corr, DeviceStats *stats,
                                                               unsigned *queues, unsigned nseg, unsigned per_seg,
                                                               unsigned segs_per_sm) {
    unsigned smid;
    asm("mov.u32 %0, %%smid;" : "=r"(smid));
    const unsigned lane = threadIdx.x & 31u;
    // nseg = segs_per_sm * base segments: the warps of an SM start on segs_per_sm of them (base apart in the list)
    const unsigned base = nseg / segs_per_sm;
    unsigned seg = smid % base + base * ((threadIdx.x >> 5) % segs_per_sm), tries = 0, nv = 0, vis = 0, nr = 0;
    while (true) {
        unsigned c = per_seg;
        if (lane == 0 && *(volatile unsigned *)(queues + seg) < per_seg) c = atomicAdd(queues + seg, 1u);
        c = __shfl_sync(0xffffffffu, c, 0);
        if (c >= per_seg) {
            if (++tries >= nseg) break;
            seg = (seg + 61u) % nseg;  // 61 is prime: visits every segment for any nseg not a multiple of 61
            continue;
        }
        int visits, reds;
        bool valid;
        em_event<TOF, VEC, BRICK>(P, ev, ((uint64_t)seg * per_seg + c) * 32u + lane, n, evw, image, corr, visits, valid,
                                  reds);
        nv += valid;
        vis += visits;
        nr += reds;
    }
    nv = __reduce_add_sync(0xffffffffu, nv);
    vis = __reduce_add_sync(0xffffffffu, vis);
    nr = __reduce_add_sync(0xffffffffu, nr);
    if (lane == 0 && stats) {
        if (nv) atomicAdd(&stats->n_valid, (unsigned long long)nv);
        if (vis) atomicAdd(&stats->visits, (unsigned long long)vis);
        if (nr) atomicAdd(&stats->reds, (unsigned long long)nr);
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Variant 2 of the fused pass: the reductions go through a software WRITE-BACK CACHE in shared memory.
// ncu (profiles/r02_*): after the sub-bin ordering the pass is bound by the request rate of the L2 atomic units (tag
// requests 77 % on average, 92 % on the busiest slice) with the issue slots 64 % busy.  The 1024 events in flight on
// an SM come from one or two locality bins, so they hit the same few thousand voxels over and over: a direct-mapped
// table of (voxel index, partial sum) pairs, 8 bytes each, updated with one 64-bit compare-and-swap, absorbs the
// repeats; only an entry that is displaced (or left at the end) costs a reduction at L2.
constexpr int kCacheLog2 = 14;  // 16384 entries = 128 KB of the SM's shared memory
constexpr unsigned kCacheEmpty = 0xFFFFFFFFu;
constexpr int kCachedBlock = 1024;

__device__ __forceinline__ int cache_add(unsigned long long *cache, float *__restrict__ out, int at, float val) {
    unsigned long long *slot = cache + (at & ((1 << kCacheLog2) - 1));
    unsigned long long old = *slot;
    while (true) {
        const unsigned tag = (unsigned)(old >> 32);
        const float cur = __uint_as_float((unsigned)old);
        const float sum = tag == (unsigned)at ? cur + val : val;
        const unsigned long long upd = ((unsigned long long)(unsigned)at << 32) | __float_as_uint(sum);
        const unsigned long long prev = atomicCAS(slot, old, upd);
        if (prev == old) {
            if (tag != (unsigned)at && tag != kCacheEmpty) {  // displaced entry: write it back
                atomicAdd(out + tag, cur);
                return 1;
            }
            return 0;
        }
        old = prev;
    }
}

template <bool TOF, bool BRICK>
__global__ void __launch_bounds__(kCachedBlock, 1) em_cached_kernel(ProjParams P, EventPtrs ev, uint64_t n,
                                                                    const float *__restrict__ evw,
                                                                    const float *__restrict__ image,
                                                                    float *__restrict__ corr, DeviceStats *stats,
                                                                    unsigned *queues, unsigned nseg, unsigned per_seg) {
    extern __shared__ unsigned long long cache[];
    for (int i = threadIdx.x; i < (1 << kCacheLog2); i += kCachedBlock) cache[i] = (unsigned long long)kCacheEmpty << 32;
    __syncthreads();
    const unsigned lane = threadIdx.x & 31u;
    // the shared-memory atomics and the L2 atomic units are two separate pipes: `cache_share` of every 8 warps reduce
    // through the cache, the others send their 16-byte reductions straight to L2, so that both pipes work in parallel
    const bool use_cache = ((threadIdx.x >> 5) & 7u) < (unsigned)P.cache_share;
    unsigned seg = blockIdx.x % nseg, tries = 0, nv = 0, vis = 0, nr = 0;
    while (true) {
        unsigned c = per_seg;
        if (lane == 0 && *(volatile unsigned *)(queues + seg) < per_seg) c = atomicAdd(queues + seg, 1u);
        c = __shfl_sync(0xffffffffu, c, 0);
        if (c >= per_seg) {
            if (++tries >= nseg) break;
            seg = (seg + 61u) % nseg;
            continue;
        }
        const uint64_t e = ((uint64_t)seg * per_seg + c) * 32u + lane;
        Ray r;
            if (e < n && load_and_setup<TOF>(P, ev, e, r)) {
            int visits;
            const float acc = ray_gather<TOF>(P, r, image, visits);
            vis += visits;
            if (acc > 0.0f) {  // R9
                ++nv;
                const float scale = (evw ? __ldg(evw + e) : 1.0f) / acc;
                if (use_cache) {
                    Walker<TOF, BRICK> wk(r);
                    int at;
                    bool done;
                    do {
                        const float w = wk.step(P, r, at, done);
                        nr += cache_add(cache, corr, at, w * scale);
                    } while (!done);
                } else {
                    nr += ray_scatter<TOF, true, BRICK>(P, r, corr, scale);
                }
            }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < (1 << kCacheLog2); i += kCachedBlock) {
        const unsigned long long v = cache[i];
        if ((unsigned)(v >> 32) != kCacheEmpty) {
            atomicAdd(corr + (unsigned)(v >> 32), __uint_as_float((unsigned)v));
            ++nr;
        }
    }
    nv = __reduce_add_sync(0xffffffffu, nv);
    vis = __reduce_add_sync(0xffffffffu, vis);
    nr = __reduce_add_sync(0xffffffffu, nr);
    if (lane == 0 && stats) {
        if (nv) atomicAdd(&stats->n_valid, (unsigned long long)nv);
        if (vis) atomicAdd(&stats->visits, (unsigned long long)vis);
        if (nr) atomicAdd(&stats->reds, (unsigned long long)nr);
    }
}

template <bool TOF, bool BRICK>
static void launch_em_cached(const ProjParams &p, const EventPtrs &ev, uint64_t n, const float *evw, const float *image,
                             float *corr, DeviceStats *stats, unsigned *queues, cudaStream_t s) {
    static int n_sm = 0;
    const size_t smem = sizeof(unsigned long long) << kCacheLog2;
    if (!n_sm) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
        cudaFuncSetAttribute(em_cached_kernel<TOF, BRICK>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    }
    unsigned nseg = (unsigned)n_sm;
    if (nseg > (unsigned)kMaxQueues) nseg = kMaxQueues;
    if (nseg % 61u == 0) nseg -= 1;
    const uint64_t wchunks = (n + 31) / 32;
    const unsigned per_seg = (unsigned)((wchunks + nseg - 1) / nseg);
    cudaMemsetAsync(queues, 0, nseg * sizeof(unsigned), s);
    em_cached_kernel<TOF, BRICK><<<n_sm, kCachedBlock, smem, s>>>(p, ev, n, evw, image, corr, stats, queues, nseg,
                                                                 per_seg);
}

static inline unsigned grid_for(uint64_t n, unsigned stride) {
    const unsigned nb = (unsigned)((n + kBlock - 1) / kBlock);
    if (stride <= 1) return nb;
    return ((nb + stride - 1) / stride) * stride;
}

void launch_forward(const ProjParams &p, bool tof, const EventPtrs &ev, uint64_t n, const float *image, float *fwd,
                    cudaStream_t s) {
    if (n == 0) return;
    if (tof)
        forward_kernel<true><<<grid_for(n, 1), kBlock, 0, s>>>(p, ev, n, image, fwd);
    else
        forward_kernel<false><<<grid_for(n, 1), kBlock, 0, s>>>(p, ev, n, image, fwd);
}

void launch_backproject(const ProjParams &p, bool tof, const EventPtrs &ev, uint64_t n, const float *values,
                        float *out, bool vec_ok, cudaStream_t s) {
    if (n == 0) return;
    const unsigned g = grid_for(n, p.stride);
    if (tof) {
        if (vec_ok)
            backproject_kernel<true, true><<<g, kBlock, 0, s>>>(p, ev, n, values, out);
        else
            backproject_kernel<true, false><<<g, kBlock, 0, s>>>(p, ev, n, values, out);
    } else {
        if (vec_ok)
            backproject_kernel<false, true><<<g, kBlock, 0, s>>>(p, ev, n, values, out);
        else
            backproject_kernel<false, false><<<g, kBlock, 0, s>>>(p, ev, n, values, out);
    }
}

template <bool TOF, bool VEC, bool BRICK>
static void launch_em(const ProjParams &p, const EventPtrs &ev, uint64_t n, const float *evw, const float *image,
                      float *corr, DeviceStats *stats, unsigned *queues, cudaStream_t s) {
    if (p.variant != 1 && queues) {
        static int n_sm = 0, per_sm = 0;  // per instantiation; one device per process
        if (!n_sm) {
            int dev = 0;
            cudaGetDevice(&dev);
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, em_persistent_kernel<TOF, VEC, BRICK>, kBlock, 0);
            cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
        }
        // Short windows: the warps of an SM spread over several list segments (measured at 146 M events: 300 ps, 1 / 2 /
        // 3 / 4 / 8 segments per SM -> 21.47 / 21.04 / 20.75 / 22.25 / 23.54 ms; 100 ps, 1 / 2 / 3 / 4 -> 11.35 / 9.57 /
        // 9.44 / 9.32 ms).  Long walks (600 ps: 43.3 -> 45.1 ms, non-TOF: 203 -> 218 ms with 2) keep one.
        const double reach = 2.0 * p.half_window * sqrt(p.iv[0] * p.iv[0] + p.iv[1] * p.iv[1] + p.iv[2] * p.iv[2]);
        const unsigned kSegsPerSm = !TOF || reach > 80.0 ? 1u : (reach > 30.0 ? 3u : 4u);  // reach = largest visit count
        unsigned nseg = (unsigned)n_sm * kSegsPerSm;
        if (nseg > (unsigned)kMaxQueues) nseg = (unsigned)kMaxQueues / kSegsPerSm * kSegsPerSm;
        if (nseg % 61u == 0) nseg -= kSegsPerSm;  // the stealing stride 61 must not divide the number of segments
        const uint64_t wchunks = (n + 31) / 32;
        const unsigned per_seg = (unsigned)((wchunks + nseg - 1) / nseg);
        cudaMemsetAsync(queues, 0, nseg * sizeof(unsigned), s);
        em_persistent_kernel<TOF, VEC, BRICK><<<n_sm * (per_sm > 0 ? per_sm : 1), kBlock, 0, s>>>(
            p, ev, n, evw, image, corr, stats, queues, nseg, per_seg, kSegsPerSm);
    } else {
        em_correction_kernel<TOF, VEC, BRICK><<<grid_for(n, p.stride), kBlock, 0, s>>>(p, ev, n, evw, image, corr, stats);
    }
}

void launch_em_correction(const ProjParams &p, bool tof, const EventPtrs &ev, uint64_t n, const float *evw,
                          const float *image, float *corr, bool vec_ok, DeviceStats *stats, unsigned *queues,
                          cudaStream_t s) {
    if (n == 0) return;
    if (p.variant == 2 && queues && vec_ok) {
        if (tof) {
            if (p.brick)
                launch_em_cached<true, true>(p, ev, n, evw, image, corr, stats, queues, s);
            else
                launch_em_cached<true, false>(p, ev, n, evw, image, corr, stats, queues, s);
        } else {
            if (p.brick)
                launch_em_cached<false, true>(p, ev, n, evw, image, corr, stats, queues, s);
            else
                launch_em_cached<false, false>(p, ev, n, evw, image, corr, stats, queues, s);
        }
        return;
    }
    if (p.brick && vec_ok) {  // the brick layout exists only together with the 16-byte reductions
        if (tof)
            launch_em<true, true, true>(p, ev, n, evw, image, corr, stats, queues, s);
        else
            launch_em<false, true, true>(p, ev, n, evw, image, corr, stats, queues, s);
        return;
    }
    if (tof) {
        if (vec_ok)
            launch_em<true, true, false>(p, ev, n, evw, image, corr, stats, queues, s);
        else
            launch_em<true, false, false>(p, ev, n, evw, image, corr, stats, queues, s);
    } else {
        if (vec_ok)
            launch_em<false, true, false>(p, ev, n, evw, image, corr, stats, queues, s);
        else
            launch_em<false, false, false>(p, ev, n, evw, image, corr, stats, queues, s);
    }
}

}  // namespace tofmlem
