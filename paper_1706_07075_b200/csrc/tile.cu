// tile.cu -- fused EM pass with shared-memory tile accumulation (BASELINE.json north_star bullet 4: "backprojection
// accumulation through ... shared-memory tile accumulation rather than naive global atomics"; the paper's "direct
// technique for voxel filling").
//
// Why: the direct pass (projector.cu) sends one 16-byte reduction to L2 per 1.5 voxel visits and is bound by the rate
// at which an SM can hand requests to the crossbar (ncu r04: 3.6e9 reductions, 0.88 of the measured request rate), and
// its image gathers keep the L1 data pipe 76 % busy with ~27 sectors per warp-wide load.  Events are sorted by
// locality key (direction class x cube of T^3 voxels holding the TOF centre), so the +-3 sigma windows of the events
// of one bin cover a small double cone around the cube (18.5 k voxels at 300 ps / 3.75 mm in the plane-by-plane layout
// below; its bounding box would be 43 k).  A CTA takes a bin ("item") and works in two phases on ONE tile buffer:
//   A. the tile holds the IMAGE values of the cone: every event of the item is walked forward (LDS gathers), its
//      w_e / fwd_e goes to a per-event scratch array and its exponent into a histogram;
//   B. the tile is cleared and becomes the CORRECTION tile: every event is walked again and adds its chord weights
//      with shared-memory integer atomics (fixed point, see the kernel); the tile is then added to the global
//      correction image once.
// One buffer instead of an image/correction pair means three CTAs (items) per SM at cfg-3, which overlap each other's
// barriers, tile loads and flushes.  Bins with few events stay on the direct pass (the plan, api.cu, decides).
//
// Tile layout: plane by plane along the class's dominant axis a; plane p holds a W[0] x W[1] rectangle of the lateral
// axes (f fast, s slow) whose low corner follows the cone (TileGeom::lo, closed-form envelopes + 1 voxel of slack on
// every side).  A step of the walk along f / s moves the tile index by +-1 / +-W[0]; a step along a by
// +-(plane stride - shift of the rectangle), read from a per-plane table in shared memory.  The weights are computed
// by exactly the arithmetic of the direct walk (walk.cuh), so both passes give the same forward values.
//
// The pass runs on the ray records of a planned list (prepared.cuh): the per-event fp64 set-up is done once by
// tofmlem_plan_events, which also DRY-RUNS the walk of every event of a tile item against the item's tile and marks
// the event for the tile only if every voxel of its window lies inside; the few others (the float32 key put them in
// the bin by a rounding, or their centre was clamped to the grid edge) go to the direct pass as stragglers.  The walk
// here therefore needs no bounds test.  The record's exact-add arithmetic makes the dry run and this walk visit the
// same voxels bit for bit.
#include <math.h>
#include <string.h>

#include "internal.cuh"
#include "prepared.cuh"

namespace tofmlem {

size_t tile_smem_bytes(const TileGeom &g) {
    return ((size_t)g.words + 4 * (kTileMaxPlanes + 1) + 8 + 256) * sizeof(float);
}

#ifndef TOFMLEM_TILE_SLACK
#define TOFMLEM_TILE_SLACK 0
#endif
constexpr int kSlack = TOFMLEM_TILE_SLACK;  // voxels of slack around the closed-form envelopes (the plan's dry run decides
                                            // per event anyway; slack only trades tile size against stragglers)

// CTAs per SM by shared memory (1 KB per CTA is reserved by the system), at most 4 (launch_em_tile's configurations)
int tile_ctas_per_sm(size_t tile_bytes, size_t smem_per_sm) {
    const size_t per_sm = smem_per_sm ? smem_per_sm : 233472;
    const int n = (int)(per_sm / (tile_bytes + 1024));
    return n > 4 ? 4 : n;
}

void build_tile_geom(const ProjParams &p, int tile_log2, size_t smem_budget, size_t smem_per_sm, TileGeom &g) {
    memset(&g, 0, sizeof g);
    const int T = 1 << tile_log2;
    g.T = T;
    const double hw = p.half_window;
    if (!(hw > 0.0)) return;
    int words[2] = {0, 0};
    bool fits[2] = {true, true};
    for (int v = 0; v < 2; ++v) {
        const int Ta = (v + 1) * T;  // extent of the item along a
        for (int a = 0; a < 3; ++a) {
            const int lat[2] = {a == 0 ? 1 : 0, a == 2 ? 1 : 2};  // f, s
            const int RA = (int)ceil(hw / p.v[a]) + kSlack;
            const int PA = 2 * RA + Ta;
            if (PA > kTileMaxPlanes) { fits[v] = false; break; }
            g.RA[a] = RA;
            g.PA[v][a] = PA;
            for (int j = 0; j < 2 && fits[v]; ++j) {
                const int b = lat[j];
                const double rho = p.v[a] / p.v[b];                   // largest slope d(voxel b) / d(voxel a) in the class
                const int M = (int)ceil(hw / (sqrt(2.0) * p.v[b]));   // largest lateral excursion: |u_b| <= |u_a| => <= 1/sqrt 2
                int W = 0;
                for (int pl = 0; pl < PA; ++pl) {
                    const int pa = pl - RA;  // plane index relative to the (first) cube
                    const int below = (int)ceil(rho * (double)(Ta - pa));
                    const int above = (int)ceil(rho * (double)(pa + 1));
                    const int lo = pa < Ta ? -(M < below ? M : below) - kSlack : -kSlack;
                    const int hi = pa >= 0 ? (T - 1) + (M < above ? M : above) + kSlack : T - 1 + kSlack;
                    if (lo < -127) { fits[v] = false; break; }
                    g.lo[v][a][j][pl] = (signed char)lo;
                    if (hi - lo + 1 > W) W = hi - lo + 1;
                }
                g.W[v][a][j] = W;
            }
            if (!fits[v]) break;
            int ps = g.W[v][a][0] * g.W[v][a][1];
            if (!(ps & 1)) ++ps;  // odd plane stride: lanes that differ in the plane only hit different banks
            g.PS[v][a] = ps;
            if (PA * ps > words[v]) words[v] = PA * ps;
        }
    }
    if (!fits[0]) return;
    g.words = words[0];
    // at least two items per SM must fit: with one tile per SM its barriers, load and flush are not overlapped by
    // anything (measured at cfg-2, 222 KB tiles: 2.50 ms per pass against 2.02 ms for the direct pass on records)
    g.ok = tile_smem_bytes(g) <= smem_budget && tile_ctas_per_sm(tile_smem_bytes(g), smem_per_sm) >= 2 ? 1 : 0;
    if (g.ok && fits[1]) {
        TileGeom h = g;
        h.words = words[1] > words[0] ? words[1] : words[0];
        if (tile_smem_bytes(h) <= smem_budget &&
            tile_ctas_per_sm(tile_smem_bytes(h), smem_per_sm) == tile_ctas_per_sm(tile_smem_bytes(g), smem_per_sm)) {
            g.pairs = 1;
            g.words = h.words;
        }
    }
}

__device__ __forceinline__ int sel3(int a, int v0, int v1, int v2) { return a == 0 ? v0 : (a == 1 ? v1 : v2); }

// Geometry of the bin a CTA is working on (uniform over the CTA).
struct Residency {
    int a;             // dominant axis; f = (a == 0 ? 1 : 0), s = (a == 2 ? 1 : 2)
    int ca, cf, cs;    // cube origin (voxels) along a, f, s
    int sgf, sgs;      // +1 / -1: the class's rays run towards +f (+s) or -f (-s) while moving towards +a
    int RA, PA, Wf, Ws, PS, T;
};

// flat index of voxel (x, y, z) in the correction image
template <bool BRICK>
__device__ __forceinline__ int corr_index(int x, int y, int z, int nx, int ny) {
    if (BRICK) return ((z * (ny >> 1) + (y >> 1)) * (nx >> 1) + (x >> 1)) * 4 + ((y & 1) << 1) + (x & 1);
    return (z * ny + y) * nx + x;
}

// Visits every word of the bin's tile once: op(tile index, x, y, z) for the words whose voxel lies in the grid,
// op_out(tile index) for the others.  A warp takes whole planes (everything that depends on the plane only is
// warp-uniform), its lanes sweep the plane's W[0] x W[1] rectangle in tile order, which is x-fastest in global memory
// for the classes whose dominant axis is y or z.  (ncu on the first form, rows of 21 words per 32 lanes and two integer
// divisions per row: the tile load and flush were 32 % of the kernel's instructions.)
template <int NT, typename In, typename Out>
__device__ __forceinline__ void for_each_tile_voxel(const Residency &R, const int *__restrict__ lof,
                                                    const int *__restrict__ los, int nx, int ny, int nz, In op,
                                                    Out op_out) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int a = R.a;
    const int na = sel3(a, nx, ny, nz), nf = a == 0 ? ny : nx, ns = a == 2 ? ny : nz;
    const int rect = R.Wf * R.Ws;
    const unsigned magic = 65536u / (unsigned)R.Wf + 1u;  // i / Wf = (i * magic) >> 16 for i < 2^16 / Wf (rect <= 2^11)
    const int bf = R.sgf > 0 ? R.cf : R.cf + R.T - 1, bs = R.sgs > 0 ? R.cs : R.cs + R.T - 1;
    for (int p = warp; p < R.PA; p += NT / 32) {
        const int ia = R.ca + p - R.RA;
        const bool plane_in = ia >= 0 && ia < na;
        const int of = bf + R.sgf * lof[p], os = bs + R.sgs * los[p];  // voxel of the rectangle's corner (0, 0)
        const int base = p * R.PS;
        for (int i = lane; i < rect; i += 32) {
            const int ls = (int)(((unsigned)i * magic) >> 16), lf = i - ls * R.Wf;
            const int i_f = of + R.sgf * lf, is = os + R.sgs * ls;
            if (plane_in && (unsigned)i_f < (unsigned)nf && (unsigned)is < (unsigned)ns) {
                if (a == 0) op(base + i, ia, i_f, is);
                else if (a == 1) op(base + i, i_f, ia, is);
                else op(base + i, i_f, is, ia);
            } else {
                op_out(base + i);
            }
        }
    }
}

// Shared-memory accesses by 32-bit byte address (the walk keeps its tile index as the address itself: no index
// arithmetic per step).
__device__ __forceinline__ float lds_f32(unsigned addr) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ void red_shared_u32(unsigned addr, unsigned v) {
    asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");  // ATOMS.ADD, no loop, no return
}

// if (ta <= tn) { ta += da; li += na; pq += dpq; na = *pq; }: the step along the tile's plane axis.  pq is the ADDRESS of
// the current plane's entry in the increment table; the increment of the NEXT plane change is fetched right away (na),
// so the table look-up is off the critical path.
__device__ __forceinline__ void advance_plane(float &ta, unsigned &li, int &na, unsigned &pq, float tn, float da,
                                              int dpq) {
    asm volatile(
        "{\n .reg .pred p;\n setp.le.f32 p, %0, %4;\n @p add.f32 %0, %0, %5;\n @p add.s32 %1, %1, %2;\n"
        " @p add.s32 %3, %3, %6;\n @p ld.shared.s32 %2, [%3];\n}"
        : "+f"(ta), "+r"(li), "+r"(na), "+r"(pq)
        : "f"(tn), "f"(da), "r"(dpq));
}

__device__ __forceinline__ void advance_addr(float &tx, unsigned &li, float tn, float dx, int inc) {
    asm("{\n .reg .pred p;\n setp.le.f32 p, %0, %2;\n @p add.f32 %0, %0, %3;\n @p add.s32 %1, %1, %4;\n}"
        : "+f"(tx), "+r"(li)
        : "f"(tn), "f"(dx), "r"(inc));
}

// Chord [t, tn] in integer quanta: rint(l * 2^(-mid^2) * scaleS) with log2(scaleS) folded into the exponent (one
// instruction fewer than scaling the weight afterwards), the rounding done by adding 2^23 (FFMA), the integer read off
// the float's mantissa.
__device__ __forceinline__ unsigned chord_quanta(float t, float tn, float lg2_scale) {
    const float l = tn - t;
    const float mid = fmaf(-0.5f, l, tn);
    float g;
    const float q = fmaf(mid, -mid, lg2_scale);
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(g) : "f"(q));
    return __float_as_uint(fmaf(l, g, 8388608.0f)) - 0x4B000000u;
}

// Fixed-point accumulation of the correction tile (see the kernel).
constexpr int kMedianBits = 4;
struct FixedPoint {
    float lmax;  // longest chord a voxel can hold, t units (kappa x voxel diagonal)
    float qmax;  // an event's contributions stay below this many quanta: 2^31 / tile_max_events
    float qmin;  // ... and its longest possible chord is worth at least this many
    int qexp;    // floor(log2(qmax / lmax))
};

// The rare event of a tile item whose w_e / fwd_e does not suit the item's fixed-point scale: float32 reductions into the
// global correction image, one per voxel.  The record is in the tile's (a, f, s) axis order with the grid directions in
// c.w (prepared.cuh); the brick layout index is formed from the flat one per voxel.
template <bool BRICK>
__device__ __noinline__ void scatter_global(float4 ra, float4 rb, uint4 rc, int nx, int ny, float *__restrict__ corr,
                                            float scale) {
    const int a = (int)((rc.y >> kRecAxisShift) & 3u), f = a == 0 ? 1 : 0, s = a == 2 ? 1 : 2;
    const int st[3] = {1, nx, nx * ny};
    const int i0 = (rc.w & 1u) ? -st[a] : st[a], i1 = (rc.w & 2u) ? -st[f] : st[f], i2 = (rc.w & 4u) ? -st[s] : st[s];
    float t = ra.x, t0 = ra.z, t1 = ra.w, t2 = rb.x;
    int at = (int)rc.x;
    auto put = [&](float w) {
        int j = at;
        if (BRICK) {
            const int z = at / (nx * ny), rem = at - z * nx * ny, y = rem / nx, x = rem - y * nx;
            j = ((z * (ny >> 1) + (y >> 1)) * (nx >> 1) + (x >> 1)) * 4 + ((y & 1) << 1) + (x & 1);
        }
        atomicAdd(corr + j, w * scale);
    };
    while (true) {
        const float tn = min3f(t0, t1, t2);
        if (!(tn < ra.y)) break;
        put(chord_weight(t, tn));
        advance_axis(t0, at, tn, rb.y, i0);
        advance_axis(t1, at, tn, rb.z, i1);
        advance_axis(t2, at, tn, rb.w, i2);
        t = tn;
    }
    put(chord_weight(t, ra.y));
}

// CHECK (TOFMLEM_OPT_TILE_CHECK, a debugging aid): every tile access is bounds-tested and violations are counted in
// tofmlem_stats.tile_oob (must stay 0: the plan's dry run has already walked every event against its tile).
//
// Fixed point: shared memory has a native 32-bit integer add (ATOMS.ADD) but no float add -- atomicAdd(float) is a
// compare-and-swap loop whose retries split the warp for the rest of the walk (ncu on the float form: the scatter loop
// ran with 14 of 32 lanes, twice the instructions).  Scale of an item: S, a power of two, puts the MEDIAN of its
// events' w_e / fwd_e (histogram of float exponents, phase A) kMedianBits below fx.qmax = 2^31 / (largest item) quanta
// for the longest possible chord; no contribution exceeds qmax, so no voxel can overflow whatever the item holds.  An
// event whose largest possible contribution would exceed qmax (w_e / fwd_e more than ~16 x the median: a window that
// barely touches activity) or stay below fx.qmin = 1024 quanta (rounding error of a contribution <= 2^-11 of the
// event's longest chord) adds float32 values to the global correction image instead.  Rounding is to nearest.
template <int NT, int NCTA, bool BRICK, bool CHECK>
__global__ void __launch_bounds__(NT, NCTA)
em_tile_kernel(int nx, int ny, int nz, const TileGeom *__restrict__ Gp, int tile_log2, RecPtrs rec,
               const float *__restrict__ evw, const float *__restrict__ image, float *__restrict__ corr,
               DeviceStats *stats, const TileItem *__restrict__ items, unsigned n_items, unsigned *counter,
               FixedPoint fx, float *__restrict__ ev_scale) {
    extern __shared__ __align__(16) float smem[];
    const int words = Gp->words;
    float *tile = smem;
    // plane tables: up[p] = byte increment of a step from plane p to p + 1, dn[p] = from p to p - 1; lof / los
    int *up = reinterpret_cast<int *>(smem + words);
    int *dn = up + (kTileMaxPlanes + 1);
    int *lof = dn + (kTileMaxPlanes + 1);
    int *los = lof + (kTileMaxPlanes + 1);
    unsigned *ctl = reinterpret_cast<unsigned *>(los + (kTileMaxPlanes + 1));  // [0] item, [1] / [2] next chunk of A / B
    unsigned *hist = ctl + 8;  // 256 bins: float exponent of w_e / fwd_e
    const unsigned tid = threadIdx.x, lane = tid & 31u;
    const unsigned tile_addr = (unsigned)__cvta_generic_to_shared(tile);
    const unsigned up_addr = (unsigned)__cvta_generic_to_shared(up), dn_addr = (unsigned)__cvta_generic_to_shared(dn);
    const int T = Gp->T;
    const unsigned Tx = (unsigned)((nx + T - 1) >> tile_log2), Ty = (unsigned)((ny + T - 1) >> tile_log2),
                   Tz = (unsigned)((nz + T - 1) >> tile_log2);
    const unsigned T3 = Tx * Ty * Tz;
    unsigned nv = 0, vis = 0, nr = 0, oob = 0, nt = 0;
    while (true) {
        __syncthreads();  // the previous item's flush has read the tile and the tables
        if (tid == 0) {
            ctl[0] = atomicAdd(counter, 1u);
            ctl[1] = ctl[2] = 0u;
        }
        __syncthreads();
        const unsigned it = ctl[0];
        if (it >= n_items) break;
        const TileItem item = items[it];
        const int var = (int)item.variant;
        const unsigned n_ev = item.count + item.count2;  // a pair item: the second cube's events follow the first's
        Residency R;
        {
            const unsigned D = item.key / T3, tl = item.key - D * T3;
            R.a = (int)(D >> 2);
            const int sg1 = (D & 2u) ? -1 : 1, sg2 = (D & 1u) ? -1 : 1;  // signs of axes (a+1)%3 and (a+2)%3
            // f = lower-numbered lateral axis: a = 0: f = 1 = (a+1)%3; a = 1: f = 0 = (a+2)%3; a = 2: f = 0 = (a+1)%3
            R.sgf = R.a == 1 ? sg2 : sg1;
            R.sgs = R.a == 1 ? sg1 : sg2;
            const int c0x = (int)(tl % Tx) * T, c0y = (int)((tl / Tx) % Ty) * T, c0z = (int)(tl / (Tx * Ty)) * T;
            R.ca = sel3(R.a, c0x, c0y, c0z);
            R.cf = R.a == 0 ? c0y : c0x;
            R.cs = R.a == 2 ? c0y : c0z;
            R.RA = Gp->RA[R.a];
            R.PA = Gp->PA[var][R.a];
            R.Wf = Gp->W[var][R.a][0];
            R.Ws = Gp->W[var][R.a][1];
            R.PS = Gp->PS[var][R.a];
            R.T = T;
        }
        for (unsigned i = tid; i < 256u; i += NT) hist[i] = 0u;
        for (int p = (int)tid; p <= kTileMaxPlanes; p += NT) {
            int l0 = 0, l1 = 0, u = 0, d = 0;
            if (p < R.PA) {
                l0 = Gp->lo[var][R.a][0][p];
                l1 = Gp->lo[var][R.a][1][p];
                if (p + 1 < R.PA)
                    u = 4 * (R.PS - ((int)Gp->lo[var][R.a][0][p + 1] - l0) - R.Wf * ((int)Gp->lo[var][R.a][1][p + 1] - l1));
                if (p > 0)
                    d = -4 * (R.PS - (l0 - (int)Gp->lo[var][R.a][0][p - 1]) - R.Wf * (l1 - (int)Gp->lo[var][R.a][1][p - 1]));
            }
            lof[p] = l0;
            los[p] = l1;
            up[p] = u;
            dn[p] = d;
        }
        __syncthreads();
        // image values of the tile: asynchronous 4-byte copies global -> shared (LDGSTS), all in flight at once
        for_each_tile_voxel<NT>(
            R, lof, los, nx, ny, nz,
            [&](int ti, int x, int y, int z) {
                asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(tile_addr + 4u * (unsigned)ti),
                             "l"(image + ((size_t)(z * ny + y) * nx + x))
                             : "memory");
            },
            [&](int ti) { tile[ti] = 0.0f; });
        asm volatile("cp.async.wait_all;" ::: "memory");
        __syncthreads();

        const unsigned nchunk = (n_ev + 31u) >> 5;
        const int Wf = R.Wf;
        const unsigned tile_bytes = (unsigned)(R.PA * R.PS) * 4u;
        // ---- phase A: forward values from the image tile, 32 events per warp at a time
        while (true) {
            unsigned c = 0;
            if (lane == 0) c = atomicAdd(&ctl[1], 1u);
            c = __shfl_sync(0xffffffffu, c, 0);
            if (c >= nchunk) break;
            const unsigned k = c * 32u + lane;
            if (k >= n_ev) continue;
            const uint64_t e = k < item.count ? (uint64_t)item.start + k : (uint64_t)item.start2 + (k - item.count);
            const uint4 rc = __ldg(rec.c + e);
            float scale = 0.f;
            if ((rc.y & (kRecValid | kRecTile)) == (kRecValid | kRecTile)) {  // the others (stragglers): direct pass
                const float4 ra = __ldg(rec.a + e), rb = __ldg(rec.b + e);
                const float te = ra.y, da = rb.y, df = rb.z, ds = rb.w;
                const bool down = rc.y & kRecNeg0;
                // +-4 by arithmetic on the flag bits: as selects of two constants ptxas turns every use into an
                // add / predicated add / move triple (ncu: 28 instead of 23 instructions per step)
                const int dpq = 4 - (int)((rc.y & kRecNeg0) >> 1);   // kRecNeg0 = 16 -> 8
                const int inc_f = 4 - (int)((rc.y & kRecNeg1) >> 2);  // kRecNeg1 = 32 -> 8
                const int inc_s = (rc.y & kRecNeg2) ? -4 * Wf : 4 * Wf;
                vis += rc.z;
                float t = ra.x, ta = ra.z, tf = ra.w, ts = rb.x;
                unsigned li = tile_addr + (rc.y >> kRecLiShift) * 4u;
                unsigned pq = (down ? dn_addr : up_addr) + ((rc.y >> kRecPlaneShift) & 127u) * 4u;
                int na = (int)__float_as_int(lds_f32(pq));
                // the tile value is loaded at the top of a step and consumed at its end; the nine warps of a scheduler
                // cover the 29 cycles in between (a hand-made one-step pipeline cost three register moves per two steps)
                float accv = 0.f;
                // rc.z = voxel visits of this window, counted by the plan's dry run of this very walk: a counted loop
                // (one test per two steps) instead of comparing every crossing with the window's end
                auto fstep = [&]() {
                    const float tn = min3f(ta, tf, ts);
                    if (CHECK && li - tile_addr >= tile_bytes) { ++oob; li = tile_addr; }
                    const float v = lds_f32(li);
                    const float w = chord_weight(t, tn);
                    advance_plane(ta, li, na, pq, tn, da, dpq);
                    advance_addr(tf, li, tn, df, inc_f);
                    advance_addr(ts, li, tn, ds, inc_s);
                    accv = fmaf(w, v, accv);
                    t = tn;
                };
                int left = (int)rc.z - 1;
                for (; left >= 2; left -= 2) {
                    fstep();
                    fstep();
                }
                if (left) fstep();
                const float w = chord_weight(t, te);
                if (CHECK && li - tile_addr >= tile_bytes) { ++oob; li = tile_addr; }
                const float fw = fmaf(w, lds_f32(li), accv);
                if (fw > 0.0f) {  // R9
                    ++nv;
                    scale = (evw ? __ldg(evw + e) : 1.0f) / fw;
                    atomicAdd(&hist[__float_as_uint(scale) >> 23], 1u);
                }
            }
            ev_scale[e] = scale;
        }
        __syncthreads();
        // ---- the item's scale: bin B = the lowest exponent with at most half of the events above it (the median's bin);
        // S = 2^(qexp - kMedianBits - (B + 1 - 127)).  Every warp computes it.
        float S;
        {
            unsigned cnt[8], mine = 0;
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                cnt[j] = hist[lane * 8u + j];
                mine += cnt[j];
            }
            unsigned incl = mine;  // suffix sum over lanes (this lane and the higher ones)
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const unsigned o = __shfl_down_sync(0xffffffffu, incl, d);
                if (lane + d < 32u) incl += o;
            }
            const unsigned total = __shfl_sync(0xffffffffu, incl, 0);
            const unsigned limit = total >> 1;
            int B = 0;
            unsigned run = incl - mine;  // events strictly above the bin looked at
#pragma unroll
            for (int j = 7; j >= 0; --j) {
                if (run > limit && B == 0) B = (int)(lane * 8u) + j + 1;
                run += cnt[j];
            }
            B = __reduce_max_sync(0xffffffffu, B);
            if (B > 255) B = 255;
            int field = fx.qexp - kMedianBits - B + 253;  // exponent field of S
            field = field < 1 ? 1 : (field > 254 ? 254 : field);
            S = __uint_as_float((unsigned)field << 23);
        }
        for (int i = tid; i < words; i += NT) tile[i] = 0.0f;  // all-zero bits: the integer zero
        __syncthreads();
        // ---- phase B: the same chords again, w_e / fwd_e * chord weight accumulated on the tile in integer quanta
        while (true) {
            unsigned c = 0;
            if (lane == 0) c = atomicAdd(&ctl[2], 1u);
            c = __shfl_sync(0xffffffffu, c, 0);
            if (c >= nchunk) break;
            const unsigned k = c * 32u + lane;
            if (k >= n_ev) continue;
            const uint64_t e = k < item.count ? (uint64_t)item.start + k : (uint64_t)item.start2 + (k - item.count);
            const float scale = ev_scale[e];
            if (!(scale > 0.0f)) continue;
            const uint4 rc = __ldg(rec.c + e);
            const float4 ra = __ldg(rec.a + e), rb = __ldg(rec.b + e);
            const float scaleS = scale * S;
            const float top = scaleS * fx.lmax;  // quanta of the longest possible chord of this event
            float lg2s;
            asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(lg2s) : "f"(scaleS));
            if (top < fx.qmax && top >= fx.qmin) {
                ++nt;
                const float te = ra.y, da = rb.y, df = rb.z, ds = rb.w;
                const bool down = rc.y & kRecNeg0;
                // +-4 by arithmetic on the flag bits: as selects of two constants ptxas turns every use into an
                // add / predicated add / move triple (ncu: 28 instead of 23 instructions per step)
                const int dpq = 4 - (int)((rc.y & kRecNeg0) >> 1);   // kRecNeg0 = 16 -> 8
                const int inc_f = 4 - (int)((rc.y & kRecNeg1) >> 2);  // kRecNeg1 = 32 -> 8
                const int inc_s = (rc.y & kRecNeg2) ? -4 * Wf : 4 * Wf;
                float t = ra.x, ta = ra.z, tf = ra.w, ts = rb.x;
                unsigned li = tile_addr + (rc.y >> kRecLiShift) * 4u;
                unsigned pq = (down ? dn_addr : up_addr) + ((rc.y >> kRecPlaneShift) & 127u) * 4u;
                int na = (int)__float_as_int(lds_f32(pq));
                auto sstep = [&]() {
                    const float tn = min3f(ta, tf, ts);
                    if (CHECK && li - tile_addr >= tile_bytes) { ++oob; li = tile_addr; }
                    red_shared_u32(li, chord_quanta(t, tn, lg2s));
                    advance_plane(ta, li, na, pq, tn, da, dpq);
                    advance_addr(tf, li, tn, df, inc_f);
                    advance_addr(ts, li, tn, ds, inc_s);
                    t = tn;
                };
                int left = (int)rc.z - 1;  // counted like the forward walk
                for (; left >= 2; left -= 2) {
                    sstep();
                    sstep();
                }
                if (left) sstep();
                if (CHECK && li - tile_addr >= tile_bytes) { ++oob; li = tile_addr; }
                red_shared_u32(li, chord_quanta(t, te, lg2s));
            } else {
                nr += rc.z;
                scatter_global<BRICK>(ra, rb, rc, nx, ny, corr, scale);
            }
        }
        __syncthreads();
        // ---- add the tile to the correction image
        const float inv_S = 1.0f / S;
        for_each_tile_voxel<NT>(
            R, lof, los, nx, ny, nz,
            [&](int ti, int x, int y, int z) {
                const unsigned q = __float_as_uint(tile[ti]);
                if (q != 0u) {
                    atomicAdd(corr + corr_index<BRICK>(x, y, z, nx, ny), (float)q * inv_S);
                    ++nr;
                }
            },
            [&](int) {});
    }
    nv = __reduce_add_sync(0xffffffffu, nv);
    vis = __reduce_add_sync(0xffffffffu, vis);
    nr = __reduce_add_sync(0xffffffffu, nr);
    oob = __reduce_add_sync(0xffffffffu, oob);
    nt = __reduce_add_sync(0xffffffffu, nt);
    if (lane == 0 && stats) {
        if (oob) atomicAdd(&stats->tile_oob, (unsigned long long)oob);
        if (nv) atomicAdd(&stats->n_valid, (unsigned long long)nv);
        if (nt) atomicAdd(&stats->tile_events, (unsigned long long)nt);
        if (vis) {
            atomicAdd(&stats->visits, (unsigned long long)vis);
            atomicAdd(&stats->tile_visits, (unsigned long long)vis);
        }
        if (nr) atomicAdd(&stats->reds, (unsigned long long)nr);
    }
}

struct TileLaunch {
    const ProjParams &p;
    const TileGeom *d_geom;
    size_t smem;
    int tile_log2;
    const RecPtrs &rec;
    const float *evw, *image;
    float *corr;
    DeviceStats *stats;
    const TileItem *items;
    uint32_t n_items;
    unsigned *counter;
    int n_sm;
    FixedPoint fx;
    float *ev_scale;
    int cap_ctas;  // > 0: at most this many CTAs per SM (the direct pass shares the SMs)
    cudaStream_t s;
};

template <int NT, int NCTA, bool BRICK, bool CHECK>
static void launch_tile(const TileLaunch &L) {
    auto k = em_tile_kernel<NT, NCTA, BRICK, CHECK>;
    cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.smem);
    cudaFuncSetAttribute(k, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    const uint32_t cap = (uint32_t)L.n_sm * (uint32_t)(L.cap_ctas > 0 && L.cap_ctas < NCTA ? L.cap_ctas : NCTA);
    k<<<L.n_items < cap ? L.n_items : cap, NT, L.smem, L.s>>>(L.p.n[0], L.p.n[1], L.p.n[2], L.d_geom, L.tile_log2, L.rec,
                                                              L.evw, L.image, L.corr, L.stats, L.items, L.n_items,
                                                              L.counter, L.fx, L.ev_scale);
}

template <int NT, int NCTA>
static void launch_tile_cfg(const TileLaunch &L, bool check) {
    if (L.p.brick) {
        if (check) launch_tile<NT, NCTA, true, true>(L); else launch_tile<NT, NCTA, true, false>(L);
    } else {
        if (check) launch_tile<NT, NCTA, false, true>(L); else launch_tile<NT, NCTA, false, false>(L);
    }
}

void launch_em_tile(const ProjParams &p, const TileGeom &g, const TileGeom *d_geom, int tile_log2, const RecPtrs &rec,
                    const float *evw, const float *image, float *corr, DeviceStats *stats, const TileItem *items,
                    uint32_t n_items, unsigned *counter, int n_sm, size_t smem_per_sm, bool check, double sigma,
                    uint32_t max_item_events, float *ev_scale, int cap_ctas, cudaStream_t s) {
    if (n_items == 0) return;
    cudaMemsetAsync(counter, 0, sizeof(unsigned), s);
    FixedPoint fx;
    {
        const double kappa = sqrt(1.4426950408889634 / 2.0) / sigma;
        fx.lmax = (float)(kappa * sqrt(p.v[0] * p.v[0] + p.v[1] * p.v[1] + p.v[2] * p.v[2]) * 1.0001);
        double qmax = 2147483648.0 / (double)(max_item_events < 1 ? 1 : max_item_events);
        if (qmax > 4194304.0) qmax = 4194304.0;  // the float -> integer conversion holds 23 bits
        fx.qmax = (float)qmax;
        fx.qmin = 1024.0f;
        fx.qexp = (int)floor(log2(qmax / (double)fx.lmax));
    }
    const size_t smem = tile_smem_bytes(g);
    const TileLaunch L{p, d_geom, smem, tile_log2, rec, evw, image, corr, stats, items, n_items, counter, n_sm, fx,
                       ev_scale, cap_ctas, s};
    // CTAs per SM by shared memory; threads so that 56 registers fit
    const int ncta = tile_ctas_per_sm(smem, smem_per_sm);
    if (ncta >= 4) launch_tile_cfg<256, 4>(L, check);
    else if (ncta == 3) launch_tile_cfg<384, 3>(L, check);
    else launch_tile_cfg<512, 2>(L, check);  // build_tile_geom admits no tile that fits only once per SM
}

}  // namespace tofmlem
