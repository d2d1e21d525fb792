// warpwalk.cu -- a WARP per LOR for the long chords of the non-TOF passes (sensitivity image a5, attenuation line
// integrals NEXT-3, forward / backprojection / fused pass of a non-TOF context).  BASELINE.json north_star bullet 2: "a
// thread or warp per event chosen by chord length"; PAPER.md:13, :49, :55 (long axial FOV, highly inclined LORs).
//
// A TOF window at 300 ps is ~30 voxels long: one thread walks it (projector.cu, prepared.cu, tile.cu).  A whole chord
// through the 160 x 160 x 640 grid is 100-900 voxels long and random detector pairs put chords of every length side by
// side in a warp: the thread-per-LOR walk runs with 11 of 32 lanes active and sends one reduction request to L2 per 1.2
// voxel visits (ncu r05, sensitivity image).  Here the 32 lanes of a warp take 32 CONSECUTIVE SLABS of one chord along
// its dominant axis a (the slab between the planes a = k and a = k + 1, in voxel units):
//   * inside a slab a line meets at most three voxels (it can cross one plane of each lateral axis f, s, because
//     |df/da|, |ds/da| <= 1): the three clipped pieces are computed in closed form, no loop-carried state;
//   * the image is stored with the dominant axis FASTEST (layout [s][f][a]): neighbouring lanes touch neighbouring
//     words, so the 32 reductions (or gathers) of one instruction fall into the few 32-byte sectors the chord really
//     crosses;
//   * x-dominant LORs use the image as it is; y- and z-dominant LORs use copies / targets stored y-fastest and
//     z-fastest (two transposes of a 65 MB image per call), one kernel launch per class so that only ONE 65 MB target is
//     hot in L2 at a time (three targets at once fall out of L2: DESIGN.md section 10);
//   * the ray set-up stays a thread per LOR (fp64, once per LOR and class); the warp then goes through its 32 LORs one
//     after the other, the set-up results handed over through shared memory.
//
// Arithmetic of a slab (float32, voxel units).  u' = coordinate along a minus the index k0 of the chord's first slab, so
// that a short chord (a clipped corner) keeps its full relative precision; the chord is [u_lo, u_hi] in u', run towards
// +a (a non-TOF LOR has no orientation); slab j covers [j, j + 1].  Per lateral axis the set-up (fp64) gives
//   g(u) = u asf + goff   = number of planes of that axis the ray has crossed at u, plus the fraction of the current
//                           cell behind it (asf = |slope| <= 1; 0 <= g(u_lo) <= 1),
//   the crossings          u = u1 + (m - 1) udf,  m = 1, 2, ...  (u1 = first crossing ahead of u_lo, udf = 1 / asf),
// the cell index bref at u_lo, the direction of the steps and the number mmax of crossings before the ray would leave the
// grid.  In the loop, m = floor(g) taken with one round-down addition of 2^23 (no conversion instruction: the integer
// sits in the mantissa), clamped to mmax (rounding at the exit face must not step out of the grid: the index is always
// valid, whatever the rounding).  Where m differs between the two ends of a slab the crossing lies at u1 + (m - 1) udf --
// from the fp64 crossing sequence, NOT from inverting the rounded g (ill-conditioned for shallow rays).  g is monotone in
// u, so is m; a slab has at most one crossing per lateral axis because asf <= 1.
#include <math.h>

#include "internal.cuh"
#include "walk.cuh"

namespace tofmlem {

namespace {

constexpr int kWBlock = 256;
constexpr int kWWarps = kWBlock / 32;
constexpr float kMagic = 8388608.0f;  // 2^23
constexpr unsigned kMagicBits = 0x4B000000u;
constexpr unsigned kNegF = 1u << 16, kNegS = 1u << 17;  // flags beside the slab count: the axis steps towards lower indices

// image stored with world axis PA fastest: [s][f][a]
template <int PA>
struct AxisOf {
    static constexpr int a = PA, f = PA == 0 ? 1 : 0, s = PA == 2 ? 1 : 2;
};

struct Lateral {
    float asf, goff, u1, udf, tmax;
    int bref;
    bool neg;
};

struct WarpRec {  // 16 words per LOR go through shared memory (see the kernel)
    float u_lo, u_hi;
    Lateral f, s;
    float lpu;      // mm of chord per unit of u
    unsigned base;  // word index of cell (k0, bref_f, bref_s) minus the magic offsets of the two lateral terms
    unsigned nsl;   // index of the last slab (first = 0) | kNegF | kNegS
    int visits;     // voxels the chord meets (slabs + lateral plane crossings); not part of the shared-memory record
};

// One lateral axis.  c: coordinate (cells) at u_lo; sd: its slope per unit u; u_lo_d / u_lo_f: start of the chord in u'.
__device__ __forceinline__ void lateral_setup(double c, double sd, double u_lo_d, float u_lo_f, int n, Lateral &o) {
    c = fmin(fmax(c, 0.0), (double)n * (1.0 - 9.094947017729282e-13));  // [0, n (1 - 2^-40)]
    const int bref = (int)floor(c);  // 0 .. n - 1
    const double frac = c - (double)bref;
    o.bref = bref;
    o.neg = sd < 0.0;
    const double as = fabs(sd);
    if (as == 0.0) {
        o.asf = 0.0f;
        o.goff = 0.0f;
        o.u1 = kBigT;
        o.udf = 0.0f;
        o.tmax = kMagic;
        return;
    }
    const double behind = o.neg ? 1.0 - frac : frac;  // fraction of the cell already behind the ray, (0, 1] or [0, 1)
    o.asf = (float)as;
    o.goff = (float)(behind - u_lo_d * as);
    // g(u_lo) must not be negative (the magic floor would give garbage): -(u_lo asf rounded down) makes it >= 0 exactly
    if (fmaf(u_lo_f, o.asf, o.goff) < 0.0f) o.goff = -__fmul_rd(u_lo_f, o.asf);
    const double inv = 1.0 / as;
    o.u1 = (float)fmin(u_lo_d + (1.0 - behind) * inv, 1.0e30);
    o.udf = (float)fmin(inv, 1.0e30);
    o.tmax = kMagic + (float)(o.neg ? bref : n - 1 - bref);
}

// fp64 set-up of one LOR for the class with dominant axis PA; false when the LOR is invalid, misses the grid or belongs
// to another class (the class test is the same code in all three launches: every LOR is taken by exactly one).
template <int PA>
__device__ __forceinline__ bool warp_ray_setup(const ProjParams &P, float fx1, float fy1, float fz1, float fx2,
                                               float fy2, float fz2, WarpRec &r) {
    if (!(finite_f(fx1) && finite_f(fy1) && finite_f(fz1) && finite_f(fx2) && finite_f(fy2) && finite_f(fz2)))
        return false;
    double px = fx1, py = fy1, pz = fz1;
    const double dx = (double)fx2 - px, dy = (double)fy2 - py, dz = (double)fz2 - pz;
    const double L2 = dx * dx + dy * dy + dz * dz;
    if (!(L2 > 0.0)) return false;
    const double L = sqrt(L2);
    const double iL = 1.0 / L;
    double ux = dx * iL, uy = dy * iL, uz = dz * iL;
    double s_lo = 0.0, s_hi = L;
    if (!axis_clip(px, ux, P.o[0], P.h[0], s_lo, s_hi)) return false;
    if (!axis_clip(py, uy, P.o[1], P.h[1], s_lo, s_hi)) return false;
    if (!axis_clip(pz, uz, P.o[2], P.h[2], s_lo, s_hi)) return false;
    if (!(s_hi > s_lo)) return false;
    const double ex = fabs(ux) * P.iv[0], ey = fabs(uy) * P.iv[1], ez = fabs(uz) * P.iv[2];
    const int cls = (ex >= ey && ex >= ez) ? 0 : (ey >= ez ? 1 : 2);
    if (cls != PA) return false;
    using AX = AxisOf<PA>;
    if ((AX::a == 0 ? ux : (AX::a == 1 ? uy : uz)) < 0.0) {  // run towards +a: start from the other end point
        px = fx2; py = fy2; pz = fz2;
        ux = -ux; uy = -uy; uz = -uz;
        const double t = s_lo;
        s_lo = L - s_hi;
        s_hi = L - t;
    }
    const double pa = AX::a == 0 ? px : (AX::a == 1 ? py : pz), da = AX::a == 0 ? ux : (AX::a == 1 ? uy : uz);
    const double pf = AX::f == 0 ? px : py, df = AX::f == 0 ? ux : uy;
    const double ps = AX::s == 1 ? py : pz, ds = AX::s == 1 ? uy : uz;
    const int na = P.n[AX::a], nf = P.n[AX::f], ns = P.n[AX::s];
    const double ra = da * P.iv[AX::a];  // du / ds > 0
    const double ira = 1.0 / ra;
    const double u_at = (pa + da * s_lo - P.o[AX::a]) * P.iv[AX::a];  // coordinate along a where the chord starts
    const double ua_lo = fmin(fmax(u_at, 0.0), (double)na);
    const double ua_hi = fmin(fmax(u_at + (s_hi - s_lo) * ra, 0.0), (double)na);
    if (!(ua_hi > ua_lo)) return false;
    int k0 = (int)floor(ua_lo);
    k0 = max(0, min(na - 1, k0));
    const double u_lo_d = ua_lo - (double)k0, u_hi_d = ua_hi - (double)k0;  // u' = u - k0
    r.u_lo = (float)u_lo_d;
    r.u_hi = (float)u_hi_d;
    if (!(r.u_hi > r.u_lo)) return false;
    int last = (int)ceilf(r.u_hi) - 1;  // slabs 0 .. last
    last = max(0, min(na - 1 - k0, last));
    // lateral coordinates where the chord starts (s_lo was clipped in mm; ua_lo may have been clamped since)
    const double s_at = s_lo + (ua_lo - u_at) * ira;
    const double cf = (pf + df * s_at - P.o[AX::f]) * P.iv[AX::f];
    const double cs = (ps + ds * s_at - P.o[AX::s]) * P.iv[AX::s];
    lateral_setup(cf, df * P.iv[AX::f] * ira, u_lo_d, r.u_lo, nf, r.f);
    lateral_setup(cs, ds * P.iv[AX::s] * ira, u_lo_d, r.u_lo, ns, r.s);
    r.lpu = (float)ira;
    const unsigned SF = (unsigned)na, SS = (unsigned)na * (unsigned)nf;
    const unsigned dF = r.f.neg ? 0u - SF : SF, dS = r.s.neg ? 0u - SS : SS;
    r.base = (unsigned)r.s.bref * SS + (unsigned)r.f.bref * SF + (unsigned)k0 - kMagicBits * (dF + dS);
    r.nsl = (unsigned)last | (r.f.neg ? kNegF : 0u) | (r.s.neg ? kNegS : 0u);
    const float ge_f = fminf(__fadd_rd(fmaf(r.u_hi, r.f.asf, r.f.goff), kMagic), r.f.tmax) - kMagic;
    const float ge_s = fminf(__fadd_rd(fmaf(r.u_hi, r.s.asf, r.s.goff), kMagic), r.s.tmax) - kMagic;
    const float gb_f = __fadd_rd(fmaf(r.u_lo, r.f.asf, r.f.goff), kMagic) - kMagic;
    const float gb_s = __fadd_rd(fmaf(r.u_lo, r.s.asf, r.s.goff), kMagic) - kMagic;
    r.visits = last + 1 + (int)(ge_f - gb_f) + (int)(ge_s - gb_s);
    return true;
}

struct Slab {
    float l0, l1, l2;     // clipped lengths of the (up to) three pieces, in u units; <= 0: no piece
    unsigned i0, i1, i2;  // their word indices in the [s][f][a] layout
};

// Record as it lies in shared memory:
//   q0 = {u_lo, u_hi, f.asf, f.goff}   q1 = {f.u1, f.udf, f.tmax, s.asf}   q2 = {s.goff, s.u1, s.udf, s.tmax}
//   q3 = {scale, base, nsl, -}
// The pieces of the chord inside slab j (see the header); dF, dS: signed word steps of the two lateral axes.
__device__ __forceinline__ Slab slab_pieces(const float4 &q0, const float4 &q1, const float4 &q2, unsigned base,
                                            float jf, unsigned j, unsigned dF, unsigned dS) {
    const float ua = fmaxf(jf, q0.x), ub = fminf(jf + 1.0f, q0.y);
    const float tfa = fminf(__fadd_rd(fmaf(ua, q0.z, q0.w), kMagic), q1.z);
    const float tfb = fminf(__fadd_rd(fmaf(ub, q0.z, q0.w), kMagic), q1.z);
    const float tsa = fminf(__fadd_rd(fmaf(ua, q1.w, q2.x), kMagic), q2.w);
    const float tsb = fminf(__fadd_rd(fmaf(ub, q1.w, q2.x), kMagic), q2.w);
    const bool xf = tfa != tfb, xs = tsa != tsb;
    float cf = fmaf(tfb - (kMagic + 1.0f), q1.y, q1.x);  // crossing m = floor(g(ub)): u1 + (m - 1) udf
    float cs = fmaf(tsb - (kMagic + 1.0f), q2.z, q2.y);
    cf = xf ? cf : ub;
    cs = xs ? cs : ub;
    cf = fminf(fmaxf(cf, ua), ub);
    cs = fminf(fmaxf(cs, ua), ub);
    const float c1 = fminf(cf, cs), c2 = fmaxf(cf, cs);
    Slab o;
    o.l0 = c1 - ua;
    o.l1 = c2 - c1;
    o.l2 = ub - c2;
    o.i0 = __float_as_uint(tfa) * dF + (__float_as_uint(tsa) * dS + (base + j));
    const unsigned sf = xf ? dF : 0u, ss = xs ? dS : 0u;
    o.i1 = o.i0 + (cf <= cs ? sf : ss);
    o.i2 = o.i0 + sf + ss;
    return o;
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    return v;
}

// The pieces of 32 slabs (32 to 96 voxel visits) are put in CHORD ORDER into the warp's shared-memory buffer and handled 32
// consecutive visits per instruction: the visits of a chord inside one (f, s) row are consecutive words, so an
// instruction costs about one L2 request per row it meets.  Three predicated reductions per lane, piece by piece, would
// send the second and third pieces as requests of their own: 1.3 instead of 0.7 requests per slab for a typical oblique
// ray, and the scatter walk is bound by these requests (sensitivity of 20 M LORs: 15.8 -> 11.5 ms).
// Returns the number of visits now in buf[0 .. total); the caller runs `for (t = lane; t < total; t += 32)` and then
// __syncwarp() before the next call.
__device__ __forceinline__ unsigned compact_pieces(const Slab &p, float scale, unsigned lt, uint2 *buf) {
    const bool h0 = p.l0 > 0.0f, h1 = p.l1 > 0.0f, h2 = p.l2 > 0.0f;
    const unsigned b0 = __ballot_sync(0xffffffffu, h0), b1 = __ballot_sync(0xffffffffu, h1);
    const unsigned b2 = __ballot_sync(0xffffffffu, h2);
    unsigned slot = __popc(b0 & lt) + __popc(b1 & lt) + __popc(b2 & lt);
    if (h0) buf[slot] = make_uint2(p.i0, __float_as_uint(p.l0 * scale));
    slot += h0;
    if (h1) buf[slot] = make_uint2(p.i1, __float_as_uint(p.l1 * scale));
    slot += h1;
    if (h2) buf[slot] = make_uint2(p.i2, __float_as_uint(p.l2 * scale));
    __syncwarp();
    return __popc(b0) + __popc(b1) + __popc(b2);
}

// a predicated load (ptxas otherwise wraps every access in a branch with its convergence barrier)
__device__ __forceinline__ float ldg_if_pos(float l, const float *p) {
    float v;
    asm volatile(
        "{\n .reg .pred q;\n setp.gt.f32 q, %2, 0f00000000;\n mov.f32 %0, 0f00000000;\n @q ld.global.nc.f32 %0, [%1];\n}"
        : "=f"(v)
        : "l"(p), "f"(l));
    return v;
}

// sum over the chord of (piece length, u units) x src; every lane returns its partial sum.  Three predicated loads per
// lane, piece by piece: the chord-order compaction of the scatter walk was measured here too and is SLOWER (attenuation
// weights of 20 M LORs 9.1 -> 19.0 ms; 13.7 ms with the loads of one iteration consumed in the next): the round trip
// through shared memory and its two warp barriers cost more issue slots and latency than the merged requests save.
__device__ __forceinline__ float chord_gather(const float4 &q0, const float4 &q1, const float4 &q2, const float4 &q3,
                                              unsigned lane, unsigned SF, unsigned SS,
                                              const float *__restrict__ src) {
    const unsigned base = __float_as_uint(q3.y), nsl = __float_as_uint(q3.z);
    const unsigned last = nsl & 0xffffu;
    const unsigned dF = (nsl & kNegF) ? 0u - SF : SF, dS = (nsl & kNegS) ? 0u - SS : SS;
    float acc = 0.0f;
    unsigned j = lane;
    float jf = (float)lane;
    for (unsigned jb = 0; jb <= last; jb += 32u, j += 32u, jf += 32.0f) {
        const Slab p = slab_pieces(q0, q1, q2, base, jf, j, dF, dS);
        // a piece that does not exist has l <= 0 (finite) and loads nothing: l * 0 adds nothing
        const float v0 = ldg_if_pos(p.l0, src + p.i0), v1 = ldg_if_pos(p.l1, src + p.i1);
        const float v2 = ldg_if_pos(p.l2, src + p.i2);
        acc = fmaf(p.l0, v0, acc);
        acc = fmaf(p.l1, v1, acc);
        acc = fmaf(p.l2, v2, acc);
    }
    return acc;
}

// dst[j] += scale * (length of the chord in voxel j, u units)
__device__ __forceinline__ void chord_scatter(const float4 &q0, const float4 &q1, const float4 &q2, const float4 &q3,
                                              unsigned lane, unsigned SF, unsigned SS, float *__restrict__ dst,
                                              float scale, uint2 *buf /* 96 entries of this warp */) {
    const unsigned base = __float_as_uint(q3.y), nsl = __float_as_uint(q3.z);
    const unsigned last = nsl & 0xffffu;
    const unsigned dF = (nsl & kNegF) ? 0u - SF : SF, dS = (nsl & kNegS) ? 0u - SS : SS;
    const unsigned lt = (1u << lane) - 1u;
    unsigned j = lane;
    float jf = (float)lane;
    for (unsigned jb = 0; jb <= last; jb += 32u, j += 32u, jf += 32.0f) {
        const unsigned total = compact_pieces(slab_pieces(q0, q1, q2, base, jf, j, dF, dS), scale, lt, buf);
        for (unsigned t = lane; t < total; t += 32u) {
            const uint2 v = buf[t];
            asm volatile("red.global.add.f32 [%0], %1;" ::"l"(dst + v.x), "f"(__uint_as_float(v.y)) : "memory");
        }
        __syncwarp();
    }
}

// MODE 0: dst += values[e] * a_e (backprojection; values NULL = 1)
// MODE 1: fwd[e] = a_e . src (forward projection / line integral, mm x image units)
// MODE 2: fused pass: dst += (w_e / (a_e . src)) a_e, w_e = values[e] (NULL = 1); a forward sum <= 0 adds nothing (R9)
template <int MODE, int PA>
__global__ void __launch_bounds__(kWBlock) warp_walk_kernel(ProjParams P, EventPtrs ev, uint64_t n,
                                                            const float *__restrict__ values,
                                                            const float *__restrict__ src, float *__restrict__ dst,
                                                            float *__restrict__ fwd, DeviceStats *stats) {
    __shared__ float4 recs[kWWarps][32][4];
    __shared__ uint2 sbuf[kWWarps][96];
    using AX = AxisOf<PA>;
    const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint64_t e = ((uint64_t)blockIdx.x * kWWarps + warp) * 32u + lane;
    const unsigned SF = (unsigned)P.n[AX::a], SS = (unsigned)P.n[AX::a] * (unsigned)P.n[AX::f];
    bool mine = false;
    unsigned vis = 0;
    if (e < n) {
        WarpRec r;
        const float x1 = __ldcs(ev.x1 + e), y1 = __ldcs(ev.y1 + e), z1 = __ldcs(ev.z1 + e);
        const float x2 = __ldcs(ev.x2 + e), y2 = __ldcs(ev.y2 + e), z2 = __ldcs(ev.z2 + e);
        mine = warp_ray_setup<PA>(P, x1, y1, z1, x2, y2, z2, r);
        float val = 1.0f;
        if (mine && MODE != 1 && values) val = __ldg(values + e);
        if (MODE == 0 && val == 0.0f) mine = false;
        if (mine) {
            vis = (unsigned)r.visits;
            recs[warp][lane][0] = make_float4(r.u_lo, r.u_hi, r.f.asf, r.f.goff);
            recs[warp][lane][1] = make_float4(r.f.u1, r.f.udf, r.f.tmax, r.s.asf);
            recs[warp][lane][2] = make_float4(r.s.goff, r.s.u1, r.s.udf, r.s.tmax);
            // .x: what the walk multiplies its pieces (u units) with: mm per u, times the value for the backprojection;
            // the fused pass needs w only (a_ej / fwd_e is a ratio of lengths)
            recs[warp][lane][3] = make_float4(MODE == 0 ? r.lpu * val : (MODE == 1 ? r.lpu : val),
                                              __uint_as_float(r.base), __uint_as_float(r.nsl), 0.0f);
        }
    }
    unsigned todo = __ballot_sync(0xffffffffu, mine);
    __syncwarp();
    float my = 0.0f;
    bool ok = false;
    while (todo) {
        const unsigned from = __ffs(todo) - 1;
        todo &= todo - 1;
        const float4 q0 = recs[warp][from][0], q1 = recs[warp][from][1];
        const float4 q2 = recs[warp][from][2], q3 = recs[warp][from][3];
        if (MODE == 0) {
            chord_scatter(q0, q1, q2, q3, lane, SF, SS, dst, q3.x, sbuf[warp]);
        } else {
            const float acc = warp_sum(chord_gather(q0, q1, q2, q3, lane, SF, SS, src));
            if (MODE == 1) {
                if (lane == from) my = acc * q3.x;
            } else if (acc > 0.0f) {
                chord_scatter(q0, q1, q2, q3, lane, SF, SS, dst, q3.x / acc, sbuf[warp]);
                if (lane == from) ok = true;
            }
        }
    }
    if (MODE == 1 && mine) fwd[e] = my;
    if (MODE == 2 && stats) {
        const unsigned nv = __popc(__ballot_sync(0xffffffffu, ok));
        const unsigned v = __reduce_add_sync(0xffffffffu, ok ? vis : 0u);
        if (lane == 0 && nv) {
            atomicAdd(&stats->n_valid, (unsigned long long)nv);
            atomicAdd(&stats->visits, (unsigned long long)v);
            atomicAdd(&stats->reds, (unsigned long long)v);  // one scalar reduction per visit; L2 sees them per sector
        }
    }
}

// Transposes between the grid order [z][y][x] and the layout with world axis PA (1 = y, 2 = z) fastest:
//   PA = 1: T[(z nx + x) ny + y]      PA = 2: T[(y nx + x) nz + z]
// dir 0: T = image (copy);  dir 1: image += T (fold).  One 32 x 32 tile of (x, a) per CTA, third axis c = blockIdx.z.
template <int PA>
__global__ void __launch_bounds__(256) axis_transpose_kernel(int nx, int ny, int nz, float *__restrict__ img,
                                                             float *__restrict__ T, int dir) {
    __shared__ float tile[32][33];
    const int na = PA == 1 ? ny : nz;
    const size_t Wa = PA == 1 ? (size_t)nx : (size_t)nx * ny;  // stride of a in the image
    const size_t Wc = PA == 1 ? (size_t)nx * ny : (size_t)nx;  // stride of c in the image
    const int c = blockIdx.z;
    const int x0 = blockIdx.x * 32, a0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;  // 32 x 8
    const size_t tbase = (size_t)c * nx * na;
    if (dir == 0) {
        for (int j = ty; j < 32; j += 8) {
            const int a = a0 + j, x = x0 + tx;
            if (a < na && x < nx) tile[j][tx] = img[(size_t)c * Wc + (size_t)a * Wa + x];
        }
        __syncthreads();
        for (int j = ty; j < 32; j += 8) {
            const int x = x0 + j, a = a0 + tx;
            if (a < na && x < nx) T[tbase + (size_t)x * na + a] = tile[tx][j];
        }
    } else {
        for (int j = ty; j < 32; j += 8) {
            const int x = x0 + j, a = a0 + tx;
            if (a < na && x < nx) tile[tx][j] = T[tbase + (size_t)x * na + a];
        }
        __syncthreads();
        for (int j = ty; j < 32; j += 8) {
            const int a = a0 + j, x = x0 + tx;
            if (a < na && x < nx) img[(size_t)c * Wc + (size_t)a * Wa + x] += tile[j][tx];
        }
    }
}

void launch_axis_transpose(const ProjParams &p, int pa, float *img, float *T, int dir, cudaStream_t s) {
    const int nx = p.n[0], ny = p.n[1], nz = p.n[2];
    if (pa == 1) {
        const dim3 g((nx + 31) / 32, (ny + 31) / 32, nz);
        axis_transpose_kernel<1><<<g, 256, 0, s>>>(nx, ny, nz, img, T, dir);
    } else {
        const dim3 g((nx + 31) / 32, (nz + 31) / 32, ny);
        axis_transpose_kernel<2><<<g, 256, 0, s>>>(nx, ny, nz, img, T, dir);
    }
}

template <int MODE>
void launch_class(int pa, const ProjParams &p, const EventPtrs &ev, uint64_t n, const float *values, const float *src,
                  float *dst, float *fwd, DeviceStats *stats, cudaStream_t s) {
    const unsigned grid = (unsigned)((n + kWBlock - 1) / kWBlock);
    if (pa == 0)
        warp_walk_kernel<MODE, 0><<<grid, kWBlock, 0, s>>>(p, ev, n, values, src, dst, fwd, stats);
    else if (pa == 1)
        warp_walk_kernel<MODE, 1><<<grid, kWBlock, 0, s>>>(p, ev, n, values, src, dst, fwd, stats);
    else
        warp_walk_kernel<MODE, 2><<<grid, kWBlock, 0, s>>>(p, ev, n, values, src, dst, fwd, stats);
}

}  // namespace

bool warp_walk_ok(const ProjParams &p) {
    // slab indices are packed in 16 bits each; the z dimension of the transposes' launch grid is <= 65535
    return p.n[0] <= 32767 && p.n[1] <= 32767 && p.n[2] <= 32767 && (int64_t)p.n[0] * p.n[1] * p.n[2] < (1ll << 31);
}

// out (grid order, nvox floats) += backprojection of `values` (NULL = 1) along the n LORs.  scratch: 2 nvox floats.
void launch_warp_backproject(const ProjParams &p, const EventPtrs &ev, uint64_t n, const float *values, float *out,
                             float *scratch, cudaStream_t s) {
    if (!n) return;
    const size_t nvox = (size_t)p.n[0] * p.n[1] * p.n[2];
    cudaMemsetAsync(scratch, 0, 2 * nvox * sizeof(float), s);
    launch_class<0>(0, p, ev, n, values, nullptr, out, nullptr, nullptr, s);
    for (int pa = 1; pa <= 2; ++pa) {
        float *T = scratch + (size_t)(pa - 1) * nvox;
        launch_class<0>(pa, p, ev, n, values, nullptr, T, nullptr, nullptr, s);
        launch_axis_transpose(p, pa, out, T, 1, s);
    }
}

// fwd[e] = line integral of `image` along LOR e (mm x image units); 0 for LORs that miss the grid.  scratch: nvox floats.
void launch_warp_forward(const ProjParams &p, const EventPtrs &ev, uint64_t n, const float *image, float *fwd,
                         float *scratch, cudaStream_t s) {
    if (!n) return;
    cudaMemsetAsync(fwd, 0, n * sizeof(float), s);
    launch_class<1>(0, p, ev, n, nullptr, image, nullptr, fwd, nullptr, s);
    for (int pa = 1; pa <= 2; ++pa) {
        launch_axis_transpose(p, pa, const_cast<float *>(image), scratch, 0, s);  // dir 0 only reads the image
        launch_class<1>(pa, p, ev, n, nullptr, scratch, nullptr, fwd, nullptr, s);
    }
}

// Fused pass of a non-TOF context: corr (grid order, accumulated into) += sum_e w_e a_e / (a_e . image).
// scratch: 2 nvox floats (image and target with the class's axis fastest).
void launch_warp_em(const ProjParams &p, const EventPtrs &ev, uint64_t n, const float *evw, const float *image,
                    float *corr, float *scratch, DeviceStats *stats, cudaStream_t s) {
    if (!n) return;
    const size_t nvox = (size_t)p.n[0] * p.n[1] * p.n[2];
    launch_class<2>(0, p, ev, n, evw, image, corr, nullptr, stats, s);
    float *Ti = scratch, *Tc = scratch + nvox;
    for (int pa = 1; pa <= 2; ++pa) {
        launch_axis_transpose(p, pa, const_cast<float *>(image), Ti, 0, s);
        cudaMemsetAsync(Tc, 0, nvox * sizeof(float), s);
        launch_class<2>(pa, p, ev, n, evw, Ti, Tc, nullptr, stats, s);
        launch_axis_transpose(p, pa, corr, Tc, 1, s);
    }
}

}  // namespace tofmlem
