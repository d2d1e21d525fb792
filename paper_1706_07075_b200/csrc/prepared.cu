// prepared.cu -- the planned form of the projector: ray records computed once per event list (prepare_rays_kernel),
// the direct fused pass on records (em_planned_kernel: global gathers, 16-byte reductions) and the forward projection
// on records (planned_forward_kernel).  See prepared.cuh for the record and the exact-add walk; tile.cu holds the
// shared-memory tile pass that runs on the same records.
#include <math.h>

#include "internal.cuh"
#include "prepared.cuh"
#include "walk.cuh"

namespace tofmlem {

constexpr int kBlock = 256;

// ---------------------------------------------------------------------------------------------------------------
// Set-up (fp64, once per event).

struct Geo {
    int i[3];        // first voxel of the window
    int nsteps[3];   // plane crossings of each axis between the first voxel and the grid boundary
    int neg[3];      // 1: the axis runs towards lower indices
    int par[3];      // 1: the ray is parallel to the axis
    double t0[3];    // first crossing after the window start, mm relative to the kernel centre
    double td[3];    // crossing period, mm
    double ts, te;   // window, mm relative to the kernel centre
};

// The geometry of ray_setup (walk.cuh) in the record's frame; false when the event is skipped (R9, invalid fields) or
// its window misses the grid.
__device__ bool geometry(const ProjParams &P, float fx1, float fy1, float fz1, float fx2, float fy2, float fz2,
                         float fdt, Geo &g) {
    if (!(finite_f(fx1) && finite_f(fy1) && finite_f(fz1) && finite_f(fx2) && finite_f(fy2) && finite_f(fz2) &&
          finite_f(fdt)))
        return false;
    const double p1[3] = {(double)fx1, (double)fy1, (double)fz1};
    const double d[3] = {(double)fx2 - p1[0], (double)fy2 - p1[1], (double)fz2 - p1[2]};
    const double L2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
    if (!(L2 > 0.0)) return false;
    const double L = sqrt(L2), iL = 1.0 / L;
    double u[3], s_lo = 0.0, s_hi = L;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        u[a] = d[a] * iL;
        if (!axis_clip(p1[a], u[a], P.o[a], P.h[a], s_lo, s_hi)) return false;
    }
    const double s_c = 0.5 * L + (0.5 * kCmmPerPs) * (double)fdt;
    s_lo = fmax(s_lo, s_c - P.half_window);
    s_hi = fmin(s_hi, s_c + P.half_window);
    if (!(s_hi > s_lo)) return false;
    g.ts = s_lo - s_c;
    g.te = s_hi - s_c;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double q = (p1[a] + u[a] * s_lo - P.o[a]) * P.iv[a];
        const double fl = floor(q);
        int ii = (int)fl;
        if (u[a] < 0.0 && fl == q) ii -= 1;  // R21
        ii = max(0, min(P.n[a] - 1, ii));
        g.i[a] = ii;
        g.par[a] = u[a] == 0.0;
        g.neg[a] = u[a] < 0.0;
        if (g.par[a]) {
            g.t0[a] = g.td[a] = 0.0;
            g.nsteps[a] = 0;
        } else {
            const double iu = 1.0 / u[a];
            const int k = u[a] > 0.0 ? ii + 1 : ii;
            g.t0[a] = (P.o[a] + (double)k * P.v[a] - p1[a]) * iu - s_c;
            g.td[a] = P.v[a] * fabs(iu);
            g.nsteps[a] = u[a] > 0.0 ? P.n[a] - 1 - ii : ii;
        }
    }
    return true;
}

struct QRay {
    float ts, te, t0[3], td[3];
};

// Quantisation to multiples of 2^-k in t units (prepared.cuh); false when nothing of the window is left.
__device__ bool quantise(const Geo &g, double qs /* kappa 2^k */, double qi /* 2^-k */, QRay &r) {
    const double ts = rint(g.ts * qs);
    double te = rint(g.te * qs);
    const double big = 1.0e30 * qs;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        if (g.par[a]) {
            r.t0[a] = __int_as_float(0x7f800000);
            r.td[a] = 0.0f;
            continue;
        }
        const double t0 = fmin(fmax(rint(g.t0[a] * qs), ts), big);
        const double td = fmin(fmax(rint(g.td[a] * qs), 1.0), big);
        te = fmin(te, t0 + (double)g.nsteps[a] * td);  // the crossing that would leave the grid
        r.t0[a] = (float)(t0 * qi);
        r.td[a] = (float)(td * qi);
    }
    if (!(te > ts)) return false;
    r.ts = (float)(ts * qi);
    r.te = (float)(te * qi);
    return true;
}

struct PlanCounters {
    unsigned long long n_valid;      // events whose window meets the grid
    unsigned long long n_tile;       // of these: running on a tile
    unsigned long long n_straggler;  // valid events of a tile item that do not fit its tile (they take the direct pass)
    unsigned long long visits;       // voxel visits of one pass (without the kRecTiny events)
    unsigned long long n_tiny;       // kRecTiny events (appended to the tiny list as one-event pieces while it has room)
};

__device__ __forceinline__ int sel3i(int a, int v0, int v1, int v2) { return a == 0 ? v0 : (a == 1 ? v1 : v2); }
__device__ __forceinline__ float sel3f(int a, float v0, float v1, float v2) { return a == 0 ? v0 : (a == 1 ? v1 : v2); }

__global__ void __launch_bounds__(kBlock)
prepare_rays_kernel(ProjParams P, const TileGeom *__restrict__ Gp, int tile_log2, EventPtrs ev, uint64_t n,
                    const TileItem *__restrict__ items, const TileRange *__restrict__ ranges, unsigned n_ranges,
                    double qs, double qi, RecPtrs rec, uint32_t *__restrict__ chunk_flags,
                    uint2 *__restrict__ tiny_list, unsigned tiny_cap, PlanCounters *__restrict__ counters) {
    const uint64_t e = (uint64_t)blockIdx.x * kBlock + threadIdx.x;
    const unsigned lane = threadIdx.x & 31u;
    bool valid = false, tile = false, straggler = false, is_tiny = false;
    unsigned visits = 0;
    if (e < n) {
        // the tile item that holds this event, if any (the items' event ranges, sorted by their first event)
        int item = -1;
        if (n_ranges) {
            unsigned lo = 0, hi = n_ranges;  // largest i with ranges[i].start <= e
            while (hi - lo > 1) {
                const unsigned mid = (lo + hi) >> 1;
                if ((uint64_t)__ldg(&ranges[mid].start) <= e) lo = mid; else hi = mid;
            }
            const uint64_t st = __ldg(&ranges[lo].start);
            if (st <= e && e < st + __ldg(&ranges[lo].count)) item = (int)__ldg(&ranges[lo].item);
        }
        Geo g;
        QRay r;
        valid = geometry(P, __ldg(ev.x1 + e), __ldg(ev.y1 + e), __ldg(ev.z1 + e), __ldg(ev.x2 + e), __ldg(ev.y2 + e),
                         __ldg(ev.z2 + e), __ldg(ev.dt + e), g) &&
                quantise(g, qs, qi, r);
        float4 ra = make_float4(0.f, 0.f, 0.f, 0.f), rb = ra;
        uint4 rc = make_uint4(0u, 0u, 0u, 0u);
        if (valid) {
            const int nx = P.n[0], ny = P.n[1];
            const int idx0 = (g.i[2] * ny + g.i[1]) * nx + g.i[0];
            const bool tiny = r.te - r.ts < (float)(32768.0 * qi);  // prepared.cuh, kRecTiny
            is_tiny = tiny;
            if (item >= 0 && !tiny) {
                // ---- does the window stay inside the bin's tile?  Dry run of the tile walk, every voxel checked.
                const unsigned key = __ldg(&items[item].key);  // the item's FIRST cube: the tile's origin
                const int var = (int)__ldg(&items[item].variant);
                const int T = Gp->T;
                const unsigned Tx = (unsigned)((nx + T - 1) >> tile_log2), Ty = (unsigned)((ny + T - 1) >> tile_log2),
                               Tz = (unsigned)((P.n[2] + T - 1) >> tile_log2);
                const unsigned T3 = Tx * Ty * Tz, D = key / T3, tl = key - D * T3;
                const int a = (int)(D >> 2), f = a == 0 ? 1 : 0, s = a == 2 ? 1 : 2;
                const int sg1 = (D & 2u) ? -1 : 1, sg2 = (D & 1u) ? -1 : 1;  // signs of axes (a+1)%3 and (a+2)%3
                const int sgf = a == 1 ? sg2 : sg1, sgs = a == 1 ? sg1 : sg2;
                const int c0[3] = {(int)(tl % Tx) * T, (int)((tl / Tx) % Ty) * T, (int)(tl / (Tx * Ty)) * T};
                const int RA = Gp->RA[a], PA = Gp->PA[var][a], Wf = Gp->W[var][a][0], Ws = Gp->W[var][a][1],
                          PS = Gp->PS[var][a];
                const signed char *lof = Gp->lo[var][a][0], *los = Gp->lo[var][a][1];
                int p = sel3i(a, g.i[0], g.i[1], g.i[2]) - sel3i(a, c0[0], c0[1], c0[2]) + RA;
                const int rf = sel3i(f, g.i[0], g.i[1], g.i[2]) - sel3i(f, c0[0], c0[1], c0[2]);
                const int rs = sel3i(s, g.i[0], g.i[1], g.i[2]) - sel3i(s, c0[0], c0[1], c0[2]);
                int nf = sgf > 0 ? rf : T - 1 - rf, ns = sgs > 0 ? rs : T - 1 - rs;  // mirrored cell coordinates
                const int da = sel3i(a, g.neg[0], g.neg[1], g.neg[2]) ? -1 : 1;
                const int df = (sel3i(f, g.neg[0], g.neg[1], g.neg[2]) ? -1 : 1) * sgf;
                const int ds = (sel3i(s, g.neg[0], g.neg[1], g.neg[2]) ? -1 : 1) * sgs;
                auto inside = [&]() {
                    return (unsigned)p < (unsigned)PA && (unsigned)(nf - lof[p]) < (unsigned)Wf &&
                           (unsigned)(ns - los[p]) < (unsigned)Ws;
                };
                bool fit = inside();
                const int p0 = p, lf0 = fit ? nf - lof[p] : 0, ls0 = fit ? ns - los[p] : 0;
                // (selects, not r.t0[a]: a run-time index would put the arrays into local memory)
                const float t0a = sel3f(a, r.t0[0], r.t0[1], r.t0[2]), t0f = sel3f(f, r.t0[0], r.t0[1], r.t0[2]),
                            t0s = sel3f(s, r.t0[0], r.t0[1], r.t0[2]);
                const float tda = sel3f(a, r.td[0], r.td[1], r.td[2]), tdf = sel3f(f, r.td[0], r.td[1], r.td[2]),
                            tds = sel3f(s, r.td[0], r.td[1], r.td[2]);
                float ta = t0a, tf = t0f, tsl = t0s;
                unsigned nvis = 1;
                while (fit) {
                    const float tn = min3f(ta, tf, tsl);
                    if (!(tn < r.te)) break;
                    if (ta <= tn) { ta += tda; p += da; }
                    if (tf <= tn) { tf += tdf; nf += df; }
                    if (tsl <= tn) { tsl += tds; ns += ds; }
                    ++nvis;
                    fit = inside();
                }
                if (fit) {
                    tile = true;
                    visits = nvis;
                    ra = make_float4(r.ts, r.te, t0a, t0f);
                    rb = make_float4(t0s, tda, tdf, tds);
                    const unsigned li0 = (unsigned)(p0 * PS + ls0 * Wf + lf0);
                    rc.x = (unsigned)idx0;
                    rc.y = kRecValid | kRecTile | ((unsigned)a << kRecAxisShift) | (da < 0 ? kRecNeg0 : 0u) |
                           (df < 0 ? kRecNeg1 : 0u) | (ds < 0 ? kRecNeg2 : 0u) | ((unsigned)p0 << kRecPlaneShift) |
                           (li0 << kRecLiShift);
                    rc.z = nvis;
                    rc.w = (sel3i(a, g.neg[0], g.neg[1], g.neg[2]) ? 1u : 0u) | (sel3i(f, g.neg[0], g.neg[1], g.neg[2]) ? 2u : 0u) |
                           (sel3i(s, g.neg[0], g.neg[1], g.neg[2]) ? 4u : 0u);  // grid directions
                } else {
                    straggler = true;
                }
            }
            if (!tile) {
                // ---- direct record (x, y, z order); dry run of the walk for the visit and group counts
                int x = g.i[0], y = g.i[1], z = g.i[2];
                const int ix = g.neg[0] ? -1 : 1, iy = g.neg[1] ? -1 : 1, iz = g.neg[2] ? -1 : 1;
                auto group = [&]() {
                    return P.brick ? (z * (ny >> 1) + (y >> 1)) * (nx >> 1) + (x >> 1) : ((z * ny + y) * nx + x) >> 2;
                };
                float tx = r.t0[0], ty = r.t0[1], tz = r.t0[2];
                unsigned nvis = 1, ngrp = 1;
                int grp = group();
                while (true) {
                    const float tn = min3f(tx, ty, tz);
                    if (!(tn < r.te)) break;
                    if (tx <= tn) { tx += r.td[0]; x += ix; }
                    if (ty <= tn) { ty += r.td[1]; y += iy; }
                    if (tz <= tn) { tz += r.td[2]; z += iz; }
                    ++nvis;
                    const int gg = group();
                    ngrp += gg != grp;
                    grp = gg;
                }
                visits = tiny ? 0u : nvis;
                ra = make_float4(r.ts, r.te, r.t0[0], r.t0[1]);
                rb = make_float4(r.t0[2], r.td[0], r.td[1], r.td[2]);
                rc.x = (unsigned)idx0;
                rc.y = kRecValid | (g.neg[0] ? kRecNeg0 : 0u) | (g.neg[1] ? kRecNeg1 : 0u) | (g.neg[2] ? kRecNeg2 : 0u) |
                       ((g.i[0] & 1) ? kRecOddX : 0u) | ((g.i[1] & 1) ? kRecOddY : 0u) | (tiny ? kRecTiny : 0u);
                rc.z = (nvis & 0xFFFFu) | (ngrp << 16);
                rc.w = (unsigned)(((g.i[2] * (ny >> 1) + (g.i[1] >> 1)) * (nx >> 1) + (g.i[0] >> 1)) * 4 +
                                  ((g.i[1] & 1) << 1) + (g.i[0] & 1));  // brick-layout index of the first voxel
            }
        }
        rec.a[e] = ra;
        rec.b[e] = rb;
        rec.c[e] = rc;
    }
    // counters, one atomic per warp; does this 32-event piece hold work for the direct pass on records?
    const unsigned mv = __ballot_sync(0xffffffffu, valid), mt = __ballot_sync(0xffffffffu, tile),
                   ms = __ballot_sync(0xffffffffu, straggler),
                   md = __ballot_sync(0xffffffffu, valid && !tile && !is_tiny);
    const unsigned vis = __reduce_add_sync(0xffffffffu, visits);
    if (lane == 0) {
        if (mv) atomicAdd(&counters->n_valid, (unsigned long long)__popc(mv));
        if (mt) atomicAdd(&counters->n_tile, (unsigned long long)__popc(mt));
        if (vis) atomicAdd(&counters->visits, (unsigned long long)vis);
        if (ms) atomicAdd(&counters->n_straggler, (unsigned long long)__popc(ms));
        if (e - lane < n) chunk_flags[(e - lane) >> 5] = md ? 1u : 0u;
    }
    // the slivers: one-event pieces for the unplanned fused pass (projector.cu)
    const unsigned mt2 = __ballot_sync(0xffffffffu, is_tiny);
    if (mt2) {
        unsigned b2 = 0;
        if (lane == 0) b2 = (unsigned)atomicAdd(&counters->n_tiny, (unsigned long long)__popc(mt2));
        b2 = __shfl_sync(0xffffffffu, b2, 0);
        const unsigned slot = b2 + __popc(mt2 & ((1u << lane) - 1u));
        if (is_tiny && slot < tiny_cap) tiny_list[slot] = make_uint2((unsigned)e, 1u);
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Walks on a record, global memory.

struct RecRay {
    float t, te, tx, ty, tz, dx, dy, dz;
};

__device__ __forceinline__ RecRay rec_ray(const float4 &a, const float4 &b) {
    return RecRay{a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
}

// sum_j w_j image[j] (t units); three steps per trip, each with its own (weight, value) slot: the gather issued in one step
// is consumed three steps later
#define TOFMLEM_GATHER_STEP(WS, VS)                        \
    {                                                      \
        const float tn = min3f(r.tx, r.ty, r.tz);          \
        if (!(tn < r.te)) break;                           \
        const float w = chord_weight(t, tn);               \
        acc = fmaf(WS, VS, acc);                           \
        VS = __ldg(image + idx);                           \
        WS = w;                                            \
        advance_axis(r.tx, idx, tn, r.dx, ix);             \
        advance_axis(r.ty, idx, tn, r.dy, iy);             \
        advance_axis(r.tz, idx, tn, r.dz, iz);             \
        t = tn;                                            \
    }
__device__ __forceinline__ float rec_gather(RecRay r, int idx, int ix, int iy, int iz, const float *__restrict__ image) {
    float acc = 0.f, w0 = 0.f, v0 = 0.f, w1 = 0.f, v1 = 0.f, w2 = 0.f, v2 = 0.f;
    float t = r.t;
    while (true) {
        TOFMLEM_GATHER_STEP(w0, v0)
        TOFMLEM_GATHER_STEP(w1, v1)
        TOFMLEM_GATHER_STEP(w2, v2)
    }
    const float w = chord_weight(t, r.te);
    acc = fmaf(w0, v0, acc);
    acc = fmaf(w1, v1, acc);
    acc = fmaf(w2, v2, acc);
    return fmaf(w, __ldg(image + idx), acc);
}
#undef TOFMLEM_GATHER_STEP

// if (tx <= tn) { tx += dx; idx += inc; inc = sum - inc; }   (brick layout: the index increment of a step alternates)
__device__ __forceinline__ void advance_axis_alt(float &tx, int &idx, int &inc, float tn, float dx, int sum) {
    asm("{\n .reg .pred p;\n setp.le.f32 p, %0, %3;\n @p add.f32 %0, %0, %4;\n @p add.s32 %1, %1, %2;\n"
        " @p sub.s32 %2, %5, %2;\n}"
        : "+f"(tx), "+r"(idx), "+r"(inc)
        : "f"(tn), "f"(dx), "r"(sum));
}

// out[j] += w_j scale, one 16-byte reduction per group of 4 voxels the line meets (walk.cuh, ray_scatter).
// BRICK: `at` runs in the brick layout (x and y increments alternate), else in the flat layout.
template <bool BRICK>
__device__ __forceinline__ void rec_scatter(RecRay r, int at, int ix, int iy, int iz, int sx, int sy,
                                            float *__restrict__ out, float scale) {
    int grp = at >> 2;
    float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
    float t = r.t;
    bool more = true;
#pragma unroll 2
    do {
        float tn = min3f(r.tx, r.ty, r.tz);
        more = tn < r.te;
        tn = more ? tn : r.te;
        const float val = chord_weight(t, tn) * scale;
        const int g = at >> 2;
        const bool fl = g != grp;
        red_v4_if(fl, out + 4 * (size_t)grp, a0, a1, a2, a3);
        grp = g;
        const int sl = at & 3;
        a0 = sl == 0 ? val : (fl ? 0.f : a0);
        a1 = sl == 1 ? val : (fl ? 0.f : a1);
        a2 = sl == 2 ? val : (fl ? 0.f : a2);
        a3 = sl == 3 ? val : (fl ? 0.f : a3);
        if (BRICK) {
            advance_axis_alt(r.tx, at, ix, tn, r.dx, sx);
            advance_axis_alt(r.ty, at, iy, tn, r.dy, sy);
        } else {
            advance_axis(r.tx, at, tn, r.dx, ix);
            advance_axis(r.ty, at, tn, r.dy, iy);
        }
        advance_axis(r.tz, at, tn, r.dz, iz);
        t = tn;
    } while (more);
    red_v4(out + 4 * (size_t)grp, a0, a1, a2, a3);
}

__device__ __forceinline__ void rec_scatter_scalar(RecRay r, int at, int ix, int iy, int iz, float *__restrict__ out,
                                                   float scale) {
    float t = r.t;
    while (true) {
        const float tn = min3f(r.tx, r.ty, r.tz);
        if (!(tn < r.te)) break;
        atomicAdd(out + at, chord_weight(t, tn) * scale);
        advance_axis(r.tx, at, tn, r.dx, ix);
        advance_axis(r.ty, at, tn, r.dy, iy);
        advance_axis(r.tz, at, tn, r.dz, iz);
        t = tn;
    }
    atomicAdd(out + at, chord_weight(t, r.te) * scale);
}

// Grid strides and signs of a record's three axes (tile records are in (a, f, s) order with the grid directions in c.w).
__device__ __forceinline__ void rec_increments(const uint4 &c, int nx, int ny, int &i0, int &i1, int &i2) {
    const unsigned m = c.y;
    if (m & kRecTile) {
        const int a = (int)((m >> kRecAxisShift) & 3u), f = a == 0 ? 1 : 0, s = a == 2 ? 1 : 2;
        const int st[3] = {1, nx, nx * ny};
        i0 = (c.w & 1u) ? -st[a] : st[a];
        i1 = (c.w & 2u) ? -st[f] : st[f];
        i2 = (c.w & 4u) ? -st[s] : st[s];
    } else {
        i0 = (m & kRecNeg0) ? -1 : 1;
        i1 = (m & kRecNeg1) ? -nx : nx;
        i2 = (m & kRecNeg2) ? -nx * ny : nx * ny;
    }
}

// kRecTiny events: the unplanned walk of walk.cuh from the raw event (fp64 set-up, window-local fp32 frame).
__device__ __noinline__ float tiny_forward(const ProjParams &P, const EventPtrs &ev, uint64_t e,
                                           const float *__restrict__ image) {
    Ray r;
    int visits;
    if (!ray_setup<true>(P, __ldg(ev.x1 + e), __ldg(ev.y1 + e), __ldg(ev.z1 + e), __ldg(ev.x2 + e), __ldg(ev.y2 + e),
                         __ldg(ev.z2 + e), __ldg(ev.dt + e), r))
        return 0.0f;
    return ray_gather<true>(P, r, image, visits);  // un-normalised, mm units
}

// Forward projection of a planned list: fwd_e = gauss_norm / kappa * sum_j l_j 2^(-mid_j^2) x_j.
__global__ void __launch_bounds__(kBlock)
planned_forward_kernel(ProjParams P, EventPtrs ev, RecPtrs rec, uint64_t n, int nx, int ny, float out_scale,
                       const float *__restrict__ image, float *__restrict__ fwd) {
    const uint64_t e = (uint64_t)blockIdx.x * kBlock + threadIdx.x;
    if (e >= n) return;
    const uint4 c = __ldg(rec.c + e);
    float v = 0.f;
    if ((c.y & (kRecValid | kRecTile | kRecTiny)) == (kRecValid | kRecTiny)) {
        v = tiny_forward(P, ev, e, image) * P.gauss_norm;
    } else if (c.y & kRecValid) {
        int i0, i1, i2;
        rec_increments(c, nx, ny, i0, i1, i2);
        v = rec_gather(rec_ray(__ldg(rec.a + e), __ldg(rec.b + e)), (int)c.x, i0, i1, i2, image) * out_scale;
    }
    fwd[e] = v;
}

// The direct fused pass on records: persistent, one work queue per list segment, the warps of an SM on neighbouring
// events (em_persistent_kernel of projector.cu explains the scheduling).  `pieces` lists, in ascending order, the 32-event
// pieces of the list that hold anything for this pass (the plan flags them and compacts the flags on the device); inside
// a piece the records say which events run on tiles (skipped here).
template <bool VEC, bool BRICK>
__global__ void __launch_bounds__(kBlock, 5)
em_planned_kernel(RecPtrs rec, uint64_t n, int nx, int ny, const uint32_t *__restrict__ pieces, uint32_t n_pieces,
                  const float *__restrict__ evw, const float *__restrict__ image, float *__restrict__ corr,
                  DeviceStats *stats, unsigned *queues, unsigned nseg, unsigned per_seg, unsigned segs_per_sm) {
    unsigned smid;
    asm("mov.u32 %0, %%smid;" : "=r"(smid));
    const unsigned lane = threadIdx.x & 31u;
    const unsigned base = nseg / segs_per_sm;
    unsigned seg = smid % base + base * ((threadIdx.x >> 5) % segs_per_sm), tries = 0, nv = 0, vis = 0, nr = 0;
    while (true) {
        unsigned c = per_seg;
        if (lane == 0 && *(volatile unsigned *)(queues + seg * kQueueStride) < per_seg)
            c = atomicAdd(queues + seg * kQueueStride, 1u);
        c = __shfl_sync(0xffffffffu, c, 0);
        if (c >= per_seg) {
            if (++tries >= nseg) break;
            seg = (seg + 61u) % nseg;
            continue;
        }
        const uint64_t wc = (uint64_t)seg * per_seg + c;
        if (wc >= n_pieces) continue;
        const uint64_t e = (uint64_t)__ldg(pieces + wc) * 32u + lane;
        if (e >= n) continue;
        const uint4 rc = __ldcs(rec.c + e);
        // tile records never appear in these lists; the slivers (kRecTiny) have their own pass
        if ((rc.y & (kRecValid | kRecTile | kRecTiny)) != kRecValid) continue;
        const RecRay r = rec_ray(__ldcs(rec.a + e), __ldcs(rec.b + e));
        const int i0 = (rc.y & kRecNeg0) ? -1 : 1, i1 = (rc.y & kRecNeg1) ? -nx : nx,
                  i2 = (rc.y & kRecNeg2) ? -nx * ny : nx * ny;
        vis += rc.z & 0xFFFFu;
        const float fw = rec_gather(r, (int)rc.x, i0, i1, i2, image);
        if (!(fw > 0.0f)) continue;  // R9
        ++nv;
        const float scale = (evw ? __ldg(evw + e) : 1.0f) / fw;
        if (VEC) {
            nr += rc.z >> 16;
            if (BRICK) {
                // brick layout: x steps alternate between +-1 and +-3, y steps between +-2 and +-(2 nx - 2) (walk.cuh)
                const bool nxg = rc.y & kRecNeg0, nyg = rc.y & kRecNeg1;
                const int xa = nxg ? -3 : 1, xb = nxg ? -1 : 3, yo = 2 * nx - 2;
                const int ya = nyg ? -yo : 2, yb = nyg ? -2 : yo;
                rec_scatter<true>(r, (int)rc.w, (rc.y & kRecOddX) ? xb : xa, (rc.y & kRecOddY) ? yb : ya, i2, xa + xb,
                                  ya + yb, corr, scale);
            } else {
                rec_scatter<false>(r, (int)rc.x, i0, i1, i2, 0, 0, corr, scale);
            }
        } else {
            nr += rc.z & 0xFFFFu;
            rec_scatter_scalar(r, (int)rc.x, i0, i1, i2, corr, scale);
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

// ---------------------------------------------------------------------------------------------------------------
// Reproducible accumulation (TOFMLEM_OPT_DETERMINISTIC; "This approach always generated an identically
// reconstructed image").  Every contribution w_ej w_e / fwd_e is rounded to an integer number of quanta 1 / G and added
// to a 64-bit integer correction image: integer additions commute, so the image does not depend on the order in which
// the GPU happens to run the events.  The forward value of an event is summed by one thread in walk order (fixed).
// G is a power of two fixed per pass from max(image) alone (image_ops.cu, det_scale_kernel), a contribution is clamped
// to 2^48 quanta (fwd_e below ~2e-7 of what a ray through max(image) would see: the voxel's correction is huge either
// way).  One thread per event on the ray records, every event through this kernel (no tiles: their flush order would
// not matter either, but one code path keeps the mode simple); scalar 64-bit reductions, about 2.5 x the time of the
// default pass.
__global__ void __launch_bounds__(kBlock, 5)
em_det_kernel(RecPtrs rec, uint64_t n, int nx, int ny, const float *__restrict__ evw, const float *__restrict__ image,
              unsigned long long *__restrict__ corr_q, const float *__restrict__ gscale, DeviceStats *stats,
              unsigned *queues, unsigned nseg, unsigned per_seg) {
    unsigned smid;
    asm("mov.u32 %0, %%smid;" : "=r"(smid));
    const unsigned lane = threadIdx.x & 31u;
    const float G = __ldg(gscale);
    const uint64_t n_pieces = (n + 31u) >> 5;
    unsigned seg = smid % nseg, tries = 0, nv = 0, vis = 0;
    while (true) {
        unsigned c = per_seg;
        if (lane == 0 && *(volatile unsigned *)(queues + seg * kQueueStride) < per_seg)
            c = atomicAdd(queues + seg * kQueueStride, 1u);
        c = __shfl_sync(0xffffffffu, c, 0);
        if (c >= per_seg) {
            if (++tries >= nseg) break;
            seg = (seg + 61u) % nseg;
            continue;
        }
        const uint64_t wc = (uint64_t)seg * per_seg + c;
        if (wc >= n_pieces) continue;
        const uint64_t e = wc * 32u + lane;
        if (e >= n) continue;
        const uint4 rc = __ldcs(rec.c + e);
        if (!(rc.y & kRecValid)) continue;
        RecRay r = rec_ray(__ldcs(rec.a + e), __ldcs(rec.b + e));
        int i0, i1, i2;
        rec_increments(rc, nx, ny, i0, i1, i2);
        vis += rc.z & 0xFFFFu;
        const float fw = rec_gather(r, (int)rc.x, i0, i1, i2, image);
        if (!(fw > 0.0f)) continue;  // R9
        ++nv;
        const float sg = (evw ? __ldg(evw + e) : 1.0f) / fw * G;
        auto put = [&](int at, float w) {
            const float q = fminf(w * sg, 281474976710656.0f);  // 2^48
            atomicAdd(corr_q + at, (unsigned long long)__float2ll_rn(q));
        };
        int at = (int)rc.x;
        float t = r.t;
        while (true) {
            const float tn = min3f(r.tx, r.ty, r.tz);
            if (!(tn < r.te)) break;
            put(at, chord_weight(t, tn));
            advance_axis(r.tx, at, tn, r.dx, i0);
            advance_axis(r.ty, at, tn, r.dy, i1);
            advance_axis(r.tz, at, tn, r.dz, i2);
            t = tn;
        }
        put(at, chord_weight(t, r.te));
    }
    nv = __reduce_add_sync(0xffffffffu, nv);
    vis = __reduce_add_sync(0xffffffffu, vis);
    if (lane == 0 && stats) {
        if (nv) atomicAdd(&stats->n_valid, (unsigned long long)nv);
        if (vis) {
            atomicAdd(&stats->visits, (unsigned long long)vis);
            atomicAdd(&stats->reds, (unsigned long long)vis);
        }
    }
}

void launch_em_det(const ProjParams &p, const RecPtrs &rec, uint64_t n, const float *evw, const float *image,
                   unsigned long long *corr_q, const float *gscale, DeviceStats *stats, unsigned *queues, int n_sm,
                   cudaStream_t s) {
    if (n == 0) return;
    int per_sm = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, em_det_kernel, kBlock, 0);
    if (per_sm < 1) per_sm = 1;
    if (n_sm < 1) n_sm = 1;
    unsigned nseg = (unsigned)n_sm;
    if (nseg > (unsigned)kMaxQueues) nseg = (unsigned)kMaxQueues;
    if (nseg % 61u == 0) nseg -= 1;
    const uint64_t n_pieces = (n + 31) / 32;
    const unsigned per_seg = (unsigned)((n_pieces + nseg - 1) / nseg);
    cudaMemsetAsync(queues, 0, (size_t)nseg * kQueueStride * sizeof(unsigned), s);
    em_det_kernel<<<n_sm * per_sm, kBlock, 0, s>>>(rec, n, p.n[0], p.n[1], evw, image, corr_q, gscale, stats, queues, nseg,
                                                   per_seg);
}

// ---------------------------------------------------------------------------------------------------------------
// Host side.

void plan_quantum(const ProjParams &p, double sigma, double &kappa, double &qs, double &qi) {
    kappa = sqrt(1.4426950408889634 / 2.0) / sigma;
    // |t| <= kappa * half_window over the window; the walk also forms t0 + td of crossings beyond t_end, which may round
    int m = 0;
    while (ldexp(1.0, m) < kappa * p.half_window * 1.0001 + 1e-9) ++m;
    const int k = 24 - m;
    qs = kappa * ldexp(1.0, k);
    qi = ldexp(1.0, -k);
}

size_t plan_counter_bytes() { return sizeof(PlanCounters); }

void launch_prepare_rays(const ProjParams &p, double sigma, const TileGeom *d_geom, int tile_log2, const EventPtrs &ev,
                         uint64_t n, const TileItem *items, const TileRange *ranges, uint32_t n_ranges,
                         const RecPtrs &rec, uint32_t *chunk_flags, uint2 *tiny_list, uint32_t tiny_cap, void *d_counters,
                         cudaStream_t s) {
    if (n == 0) return;
    double kappa, qs, qi;
    plan_quantum(p, sigma, kappa, qs, qi);
    cudaMemsetAsync(d_counters, 0, sizeof(PlanCounters), s);
    prepare_rays_kernel<<<(unsigned)((n + kBlock - 1) / kBlock), kBlock, 0, s>>>(
        p, d_geom, tile_log2, ev, n, items, ranges, d_geom ? n_ranges : 0u, qs, qi, rec, chunk_flags, tiny_list, tiny_cap,
        static_cast<PlanCounters *>(d_counters));
}

void read_plan_counters(const void *h, uint64_t out[5]) {
    const PlanCounters *c = static_cast<const PlanCounters *>(h);
    out[0] = c->n_valid;
    out[1] = c->n_tile;
    out[2] = c->n_straggler;
    out[3] = c->visits;
    out[4] = c->n_tiny;
}

void launch_planned_forward(const ProjParams &p, double sigma, const EventPtrs &ev, const RecPtrs &rec, uint64_t n,
                            const float *image, float *fwd, cudaStream_t s) {
    if (n == 0) return;
    double kappa, qs, qi;
    plan_quantum(p, sigma, kappa, qs, qi);
    planned_forward_kernel<<<(unsigned)((n + kBlock - 1) / kBlock), kBlock, 0, s>>>(
        p, ev, rec, n, p.n[0], p.n[1], (float)((double)p.gauss_norm / kappa), image, fwd);
}

template <bool VEC, bool BRICK>
static void launch_planned(const ProjParams &p, const RecPtrs &rec, uint64_t n, const uint32_t *pieces, uint32_t n_pieces,
                           const float *evw, const float *image, float *corr, DeviceStats *stats, unsigned *queues,
                           int n_sm, bool sparse, cudaStream_t s) {
    int per_sm = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, em_planned_kernel<VEC, BRICK>, kBlock, 0);
    if (per_sm < 1) per_sm = 1;
    if (n_sm < 1) n_sm = 1;
    const double reach = 2.0 * p.half_window * sqrt(p.iv[0] * p.iv[0] + p.iv[1] * p.iv[1] + p.iv[2] * p.iv[2]);
    // list segments per SM: as launch_em (projector.cu) measured them for whole lists; when the dense bins run on tiles
    // the pieces left over are the sparse bins, whose warps gain nothing from several segments (measured at cfg-3 with
    // 1 / 2 / 3 / 4 / 6 / 8 segments: 5.05 / 5.12 / 5.28 / 5.26 / 5.80 / 5.86 ms)
    const unsigned segs = sparse ? 1u : (reach > 80.0 ? 1u : (reach > 30.0 ? 3u : 4u));
    unsigned nseg = (unsigned)n_sm * segs;
    if (nseg > (unsigned)kMaxQueues) nseg = (unsigned)kMaxQueues / segs * segs;
    if (nseg % 61u == 0) nseg -= segs;
    const unsigned per_seg = (n_pieces + nseg - 1) / nseg;
    cudaMemsetAsync(queues, 0, (size_t)nseg * kQueueStride * sizeof(unsigned), s);
    em_planned_kernel<VEC, BRICK><<<n_sm * per_sm, kBlock, 0, s>>>(rec, n, p.n[0], p.n[1], pieces, n_pieces, evw, image,
                                                                  corr, stats, queues, nseg, per_seg, segs);
}

void launch_em_planned(const ProjParams &p, const RecPtrs &rec, uint64_t n, const uint32_t *pieces, uint32_t n_pieces,
                       const float *evw, const float *image, float *corr, bool vec_ok, DeviceStats *stats,
                       unsigned *queues, int n_sm, bool sparse, cudaStream_t s) {
    if (n == 0 || n_pieces == 0) return;
    if (p.brick && vec_ok)
        launch_planned<true, true>(p, rec, n, pieces, n_pieces, evw, image, corr, stats, queues, n_sm, sparse, s);
    else if (vec_ok)
        launch_planned<true, false>(p, rec, n, pieces, n_pieces, evw, image, corr, stats, queues, n_sm, sparse, s);
    else
        launch_planned<false, false>(p, rec, n, pieces, n_pieces, evw, image, corr, stats, queues, n_sm, sparse, s);
}

}  // namespace tofmlem
