// tile.cu -- fused EM pass with shared-memory tile accumulation (BASELINE.json north_star bullet 4: "backprojection
// accumulation through ... shared-memory tile accumulation rather than naive global atomics"; the paper's "direct
// technique for voxel filling").
//
// Why: the direct pass (projector.cu) sends one 16-byte reduction to L2 per 1.5 voxel visits and is bound by the rate
// at which an SM can hand requests to the crossbar (ncu r04: 3.6e9 reductions, 0.88 of the measured request rate), and
// its image gathers keep the L1 data pipe 76 % busy with ~27 sectors per warp-wide load.  Events are sorted by
// locality key (direction class x cube of T^3 voxels holding the TOF centre), so the +-3 sigma windows of the events
// of one bin cover a small double cone around the cube (7.8 k voxels at 300 ps / 3.75 mm; its bounding box would be
// 35 k).  One CTA per SM takes a bin, copies the image values of that cone into shared memory, walks all events of
// the bin with both the gathers (LDS) and the accumulation (shared-memory atomics) on the tile, and adds the tile to
// the global correction image once.  Bins with few events stay on the direct pass (the plan, api.cu, decides).
//
// Tile layout: plane by plane along the class's dominant axis a; plane p holds a W[0] x W[1] rectangle of the lateral
// axes (f fast, s slow) whose low corner follows the cone (TileGeom::lo, closed-form envelopes + 1 voxel of slack on
// every side).  A step of the walk along f / s moves the tile index by +-1 / +-W[0]; a step along a by
// +-(plane stride - shift of the rectangle), read from a per-plane table in shared memory.  The weights are computed
// by exactly the arithmetic of the direct walk (walk.cuh), so both passes give the same forward values.
//
// Safety: an event uses the tile only if its TOF centre lies in the bin's cube and its direction in the bin's class,
// checked in fp64 inside the kernel (the envelopes are derived from exactly these two facts), and its first voxel lies
// inside the tile; every other event of the bin (the float32 key put it there by a rounding, or its centre was
// clamped to the grid edge) takes the direct walk.  TOFMLEM_OPT_TILE_CHECK adds a bounds test to every tile access.
#include <math.h>
#include <string.h>

#include "internal.cuh"
#include "walk.cuh"

namespace tofmlem {

constexpr int kTileThreads = 1024;

size_t tile_smem_bytes(const TileGeom &g) {
    return ((size_t)2 * g.words + 3 * kTileMaxPlanes + 8) * sizeof(float);
}

void build_tile_geom(const ProjParams &p, int tile_log2, size_t smem_budget, TileGeom &g) {
    memset(&g, 0, sizeof g);
    const int T = 1 << tile_log2;
    g.T = T;
    const double hw = p.half_window;
    if (!(hw > 0.0)) return;
    int words = 0;
    for (int a = 0; a < 3; ++a) {
        const int lat[2] = {a == 0 ? 1 : 0, a == 2 ? 1 : 2};  // f, s
        const int RA = (int)ceil(hw / p.v[a]) + 1;
        const int PA = 2 * RA + T;
        if (PA > kTileMaxPlanes) return;
        g.RA[a] = RA;
        g.PA[a] = PA;
        for (int j = 0; j < 2; ++j) {
            const int b = lat[j];
            const double rho = p.v[a] / p.v[b];                   // largest slope d(voxel b) / d(voxel a) in the class
            const int M = (int)ceil(hw / (sqrt(2.0) * p.v[b]));   // largest lateral excursion: |u_b| <= |u_a| => <= 1/sqrt 2
            int W = 0;
            for (int pl = 0; pl < PA; ++pl) {
                const int pa = pl - RA;  // plane index relative to the cube
                const int below = (int)ceil(rho * (double)(T - pa));
                const int above = (int)ceil(rho * (double)(pa + 1));
                const int lo = pa < T ? -(M < below ? M : below) - 1 : -1;
                const int hi = pa >= 0 ? (T - 1) + (M < above ? M : above) + 1 : T;
                if (lo < -127) return;
                g.lo[a][j][pl] = (signed char)lo;
                if (hi - lo + 1 > W) W = hi - lo + 1;
            }
            g.W[a][j] = W;
        }
        int ps = g.W[a][0] * g.W[a][1];
        if (!(ps & 1)) ++ps;  // odd plane stride: lanes that differ in the plane only hit different banks
        g.PS[a] = ps;
        if (PA * ps > words) words = PA * ps;
    }
    g.words = words;
    g.ok = tile_smem_bytes(g) <= smem_budget ? 1 : 0;
}

__device__ __forceinline__ int sel3(int a, int v0, int v1, int v2) { return a == 0 ? v0 : (a == 1 ? v1 : v2); }
__device__ __forceinline__ float sel3(int a, float v0, float v1, float v2) { return a == 0 ? v0 : (a == 1 ? v1 : v2); }
__device__ __forceinline__ double sel3(int a, double v0, double v1, double v2) { return a == 0 ? v0 : (a == 1 ? v1 : v2); }

// Geometry of the bin a CTA is working on (uniform over the CTA).
struct Residency {
    int a;             // dominant axis; f = (a == 0 ? 1 : 0), s = (a == 2 ? 1 : 2)
    int ca, cf, cs;    // cube origin (voxels) along a, f, s
    int sgf, sgs;      // +1 / -1: the class's rays run towards +f (+s) or -f (-s) while moving towards +a
    int RA, PA, Wf, Ws, PS, T;
};

// The walk of walk.cuh's Walker on the tile: same crossing arithmetic (so the same weights), tile-local index.
struct TileWalker {
    float ta, tf, ts, ka, kf, ks, t;
    int li, pq;
    __device__ __forceinline__ float step(float gauss_a, float t_end, float tc, float t0a, float t0f, float t0s,
                                          float tda, float tdf, float tds, const int *__restrict__ ainc, int dir_a,
                                          int inc_f, int inc_s, int &at, bool &done) {
        const float tn = fminf(fminf(ta, tf), fminf(ts, t_end));
        const float l = tn - t;
        const float tm = fmaf(0.5f, t + tn, -tc);
        const float w = l * ex2_approx(gauss_a * tm * tm);
        at = li;
        done = tn >= t_end;
        if (ta <= tn) {
            ka += 1.0f;
            li += dir_a * ainc[pq];
            pq += dir_a;
        }
        if (tf <= tn) { kf += 1.0f; li += inc_f; }
        if (ts <= tn) { ks += 1.0f; li += inc_s; }
        ta = fmaf(ka, tda, t0a);
        tf = fmaf(kf, tdf, t0f);
        ts = fmaf(ks, tds, t0s);
        t = tn;
        return w;
    }
};

// flat index of voxel (x, y, z) in the correction image
template <bool BRICK>
__device__ __forceinline__ int corr_index(int x, int y, int z, int nx, int ny) {
    if (BRICK) return ((z * (ny >> 1) + (y >> 1)) * (nx >> 1) + (x >> 1)) * 4 + ((y & 1) << 1) + (x & 1);
    return (z * ny + y) * nx + x;
}

// Visits every word of the bin's tile once, lanes running along x (global memory rows): op(tile index, x, y, z) for
// the words whose voxel lies in the grid, op_out(tile index) for the others.
template <typename In, typename Out>
__device__ __forceinline__ void for_each_tile_voxel(const Residency &R, const int *__restrict__ lof,
                                                    const int *__restrict__ los, int nx, int ny, int nz, In op,
                                                    Out op_out) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int a = R.a;
    const int na = sel3(a, nx, ny, nz), nf = a == 0 ? ny : nx, ns = a == 2 ? ny : nz;
    if (a != 0) {  // f = x: a row of a plane's rectangle is a run of x
        for (int row = warp; row < R.PA * R.Ws; row += kTileThreads / 32) {
            const int p = row / R.Ws, ls = row - p * R.Ws;
            const int ia = R.ca + p - R.RA;
            const int n_s = ls + los[p];
            const int is = R.sgs > 0 ? R.cs + n_s : R.cs + R.T - 1 - n_s;
            const bool row_in = ia >= 0 && ia < na && is >= 0 && is < ns;
            const int lo_f = lof[p];
            for (int lf = lane; lf < R.Wf; lf += 32) {
                const int n_f = lf + lo_f;
                const int i_f = R.sgf > 0 ? R.cf + n_f : R.cf + R.T - 1 - n_f;
                const int ti = p * R.PS + ls * R.Wf + lf;
                if (row_in && i_f >= 0 && i_f < nf) {
                    if (a == 1) op(ti, i_f, ia, is); else op(ti, i_f, is, ia);
                } else {
                    op_out(ti);
                }
            }
        }
    } else {  // a = x: the planes are consecutive in x
        for (int col = warp; col < R.Wf * R.Ws; col += kTileThreads / 32) {
            const int ls = col / R.Wf, lf = col - ls * R.Wf;
            for (int p = lane; p < R.PA; p += 32) {
                const int ia = R.ca + p - R.RA;
                const int n_f = lf + lof[p], n_s = ls + los[p];
                const int i_f = R.sgf > 0 ? R.cf + n_f : R.cf + R.T - 1 - n_f;
                const int is = R.sgs > 0 ? R.cs + n_s : R.cs + R.T - 1 - n_s;
                const int ti = p * R.PS + col;
                if (ia >= 0 && ia < na && i_f >= 0 && i_f < nf && is >= 0 && is < ns) op(ti, ia, i_f, is);
                else op_out(ti);
            }
        }
    }
}

template <bool BRICK, bool CHECK>
__global__ void __launch_bounds__(kTileThreads, 1)
em_tile_kernel(ProjParams P, const TileGeom *__restrict__ Gp, int tile_log2, EventPtrs ev,
               const float *__restrict__ evw, const float *__restrict__ image, float *__restrict__ corr,
               DeviceStats *stats, const TileItem *__restrict__ items, unsigned n_items, unsigned *counter) {
    extern __shared__ __align__(16) float smem[];
    const int words = Gp->words;
    float *img = smem;
    float *acc = smem + words;
    int *ainc = reinterpret_cast<int *>(smem + 2 * words);
    int *lof = ainc + kTileMaxPlanes;
    int *los = lof + kTileMaxPlanes;
    unsigned *ctl = reinterpret_cast<unsigned *>(los + kTileMaxPlanes);  // [0] item, [1] next chunk of the item
    const unsigned tid = threadIdx.x, lane = tid & 31u;
    for (int i = tid; i < words; i += kTileThreads) acc[i] = 0.0f;
    const int nx = P.n[0], ny = P.n[1], nz = P.n[2];
    const int T = Gp->T;
    const unsigned Tx = (unsigned)((nx + T - 1) >> tile_log2), Ty = (unsigned)((ny + T - 1) >> tile_log2),
                   Tz = (unsigned)((nz + T - 1) >> tile_log2);
    const unsigned T3 = Tx * Ty * Tz;
    unsigned nv = 0, vis = 0, nr = 0, nt = 0, oob = 0;
    while (true) {
        if (tid == 0) {
            ctl[0] = atomicAdd(counter, 1u);
            ctl[1] = 0u;
        }
        __syncthreads();
        const unsigned it = ctl[0];
        if (it >= n_items) break;
        const TileItem item = items[it];
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
            R.PA = Gp->PA[R.a];
            R.Wf = Gp->W[R.a][0];
            R.Ws = Gp->W[R.a][1];
            R.PS = Gp->PS[R.a];
            R.T = T;
        }
        if ((int)tid < R.PA) {
            const int l0 = Gp->lo[R.a][0][tid], l1 = Gp->lo[R.a][1][tid];
            lof[tid] = l0;
            los[tid] = l1;
            if ((int)tid + 1 < R.PA)
                ainc[tid] = R.PS - ((int)Gp->lo[R.a][0][tid + 1] - l0) - R.Wf * ((int)Gp->lo[R.a][1][tid + 1] - l1);
        }
        __syncthreads();
        for_each_tile_voxel(
            R, lof, los, nx, ny, nz,
            [&](int ti, int x, int y, int z) { img[ti] = __ldg(image + ((size_t)(z * ny + y) * nx + x)); },
            [&](int ti) { img[ti] = 0.0f; });
        __syncthreads();

        // ---- the events of the bin, 32 per warp at a time
        const int a = R.a;
        const unsigned nchunk = (item.count + 31u) >> 5;
        const int tile_words = R.PA * R.PS;
        while (true) {
            unsigned c = 0;
            if (lane == 0) c = atomicAdd(&ctl[1], 1u);
            c = __shfl_sync(0xffffffffu, c, 0);
            if (c >= nchunk) break;
            const unsigned k = c * 32u + lane;
            if (k >= item.count) continue;
            const uint64_t e = (uint64_t)item.start + k;
            const float x1 = __ldcs(ev.x1 + e), y1 = __ldcs(ev.y1 + e), z1 = __ldcs(ev.z1 + e);
            const float x2 = __ldcs(ev.x2 + e), y2 = __ldcs(ev.y2 + e), z2 = __ldcs(ev.z2 + e);
            const float dt = __ldcs(ev.dt + e);
            Ray r;
            RayExtra X;
            if (!ray_setup<true, true>(P, x1, y1, z1, x2, y2, z2, dt, r, &X)) continue;
            const double ua = sel3(a, X.u[0], X.u[1], X.u[2]);
            const double uf = a == 0 ? X.u[1] : X.u[0], us = a == 2 ? X.u[1] : X.u[2];
            const double qa = sel3(a, X.cv[0], X.cv[1], X.cv[2]) - (double)R.ca;
            const double qf = (a == 0 ? X.cv[1] : X.cv[0]) - (double)R.cf;
            const double qs = (a == 2 ? X.cv[1] : X.cv[2]) - (double)R.cs;
            const double dT = (double)T;
            bool fit = ua != 0.0 && fabs(uf) <= fabs(ua) && fabs(us) <= fabs(ua) &&
                       (R.sgf > 0 ? uf * ua >= 0.0 : uf * ua <= 0.0) && (R.sgs > 0 ? us * ua >= 0.0 : us * ua <= 0.0) &&
                       qa >= 0.0 && qa <= dT && qf >= 0.0 && qf <= dT && qs >= 0.0 && qs <= dT;
            const int ia = sel3(a, X.i[0], X.i[1], X.i[2]);
            const int i_f = a == 0 ? X.i[1] : X.i[0], is = a == 2 ? X.i[1] : X.i[2];
            const int p0 = ia - R.ca + R.RA;
            int li0 = 0;
            if (fit && (unsigned)p0 < (unsigned)R.PA) {
                const int lf0 = (R.sgf > 0 ? i_f - R.cf : T - 1 - (i_f - R.cf)) - lof[p0];
                const int ls0 = (R.sgs > 0 ? is - R.cs : T - 1 - (is - R.cs)) - los[p0];
                fit = (unsigned)lf0 < (unsigned)R.Wf && (unsigned)ls0 < (unsigned)R.Ws;
                li0 = p0 * R.PS + ls0 * R.Wf + lf0;
            } else {
                fit = false;
            }
            const float w_e = evw ? __ldg(evw + e) : 1.0f;
            if (fit) {
                const int dir_a = ua > 0.0 ? 1 : -1;
                const int inc_f = (uf > 0.0 ? 1 : -1) * R.sgf;
                const int inc_s = (us > 0.0 ? 1 : -1) * R.sgs * R.Wf;
                const float t0a = sel3(a, r.t0x, r.t0y, r.t0z), tda = sel3(a, r.tdx, r.tdy, r.tdz);
                const float t0f = a == 0 ? r.t0y : r.t0x, tdf = a == 0 ? r.tdy : r.tdx;
                const float t0s = a == 2 ? r.t0y : r.t0z, tds = a == 2 ? r.tdy : r.tdz;
                const int pq0 = p0 + (dir_a < 0 ? -1 : 0);
                // walk 1: forward value from the image tile (software pipeline of depth 2 on the LDS, as ray_gather)
                TileWalker wk{t0a, t0f, t0s, 0.f, 0.f, 0.f, 0.f, li0, pq0};
                float fw = 0.0f, w0 = 0.f, v0 = 0.f, w1 = 0.f, v1 = 0.f;
                int at, n = 0;
                bool done = false;
                while (!done) {
                    fw = fmaf(w0, v0, fw);
                    w0 = wk.step(P.gauss_a, r.t_end, r.tc, t0a, t0f, t0s, tda, tdf, tds, ainc, dir_a, inc_f, inc_s, at, done);
                    if (CHECK && (unsigned)at >= (unsigned)tile_words) { ++oob; at = 0; w0 = 0.f; }
                    v0 = img[at];
                    ++n;
                    if (!done) {
                        fw = fmaf(w1, v1, fw);
                        w1 = wk.step(P.gauss_a, r.t_end, r.tc, t0a, t0f, t0s, tda, tdf, tds, ainc, dir_a, inc_f, inc_s, at, done);
                        if (CHECK && (unsigned)at >= (unsigned)tile_words) { ++oob; at = 0; w1 = 0.f; }
                        v1 = img[at];
                        ++n;
                    }
                }
                fw = fmaf(w0, v0, fw);
                fw = fmaf(w1, v1, fw);
                vis += n;
                if (fw > 0.0f) {  // R9
                    ++nv;
                    ++nt;
                    const float scale = w_e / fw;
                    TileWalker wb{t0a, t0f, t0s, 0.f, 0.f, 0.f, 0.f, li0, pq0};
                    do {
                        const float w = wb.step(P.gauss_a, r.t_end, r.tc, t0a, t0f, t0s, tda, tdf, tds, ainc, dir_a, inc_f, inc_s, at, done);
                        if (CHECK && (unsigned)at >= (unsigned)tile_words) { ++oob; continue; }
                        atomicAdd(acc + at, w * scale);
                    } while (!done);
                }
            } else {  // the direct walk of projector.cu for the few events of the bin whose window may leave the tile
                int n;
                const float fw = ray_gather<true>(P, r, image, n);
                vis += n;
                if (fw > 0.0f) {
                    ++nv;
                    nr += ray_scatter<true, true, BRICK>(P, r, corr, w_e / fw);
                }
            }
        }
        __syncthreads();
        // ---- add the tile to the correction image and clear it
        for_each_tile_voxel(
            R, lof, los, nx, ny, nz,
            [&](int ti, int x, int y, int z) {
                const float v = acc[ti];
                if (v != 0.0f) {
                    acc[ti] = 0.0f;
                    atomicAdd(corr + corr_index<BRICK>(x, y, z, nx, ny), v);
                    ++nr;
                }
            },
            [&](int) {});
    }
    nv = __reduce_add_sync(0xffffffffu, nv);
    vis = __reduce_add_sync(0xffffffffu, vis);
    nr = __reduce_add_sync(0xffffffffu, nr);
    nt = __reduce_add_sync(0xffffffffu, nt);
    oob = __reduce_add_sync(0xffffffffu, oob);
    if (lane == 0 && stats) {
        if (nv) atomicAdd(&stats->n_valid, (unsigned long long)nv);
        if (vis) atomicAdd(&stats->visits, (unsigned long long)vis);
        if (nr) atomicAdd(&stats->reds, (unsigned long long)nr);
        if (nt) atomicAdd(&stats->tile_events, (unsigned long long)nt);
        if (oob) atomicAdd(&stats->tile_oob, (unsigned long long)oob);
    }
}

template <bool BRICK, bool CHECK>
static void launch_tile(const ProjParams &p, const TileGeom *d_geom, size_t smem, int tile_log2, const EventPtrs &ev,
                        const float *evw, const float *image, float *corr, DeviceStats *stats, const TileItem *items,
                        uint32_t n_items, unsigned *counter, int n_sm, cudaStream_t s) {
    cudaFuncSetAttribute(em_tile_kernel<BRICK, CHECK>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    em_tile_kernel<BRICK, CHECK><<<n_sm, kTileThreads, smem, s>>>(p, d_geom, tile_log2, ev, evw, image, corr, stats,
                                                                 items, n_items, counter);
}

void launch_em_tile(const ProjParams &p, const TileGeom &g, const TileGeom *d_geom, int tile_log2, const EventPtrs &ev,
                    const float *evw, const float *image, float *corr, DeviceStats *stats, const TileItem *items,
                    uint32_t n_items, unsigned *counter, int n_sm, bool check, cudaStream_t s) {
    if (n_items == 0) return;
    cudaMemsetAsync(counter, 0, sizeof(unsigned), s);
    const size_t smem = tile_smem_bytes(g);
    const unsigned grid = (unsigned)(n_items < (uint32_t)n_sm ? n_items : (uint32_t)n_sm);
    if (p.brick) {
        if (check) launch_tile<true, true>(p, d_geom, smem, tile_log2, ev, evw, image, corr, stats, items, n_items, counter, (int)grid, s);
        else launch_tile<true, false>(p, d_geom, smem, tile_log2, ev, evw, image, corr, stats, items, n_items, counter, (int)grid, s);
    } else {
        if (check) launch_tile<false, true>(p, d_geom, smem, tile_log2, ev, evw, image, corr, stats, items, n_items, counter, (int)grid, s);
        else launch_tile<false, false>(p, d_geom, smem, tile_log2, ev, evw, image, corr, stats, items, n_items, counter, (int)grid, s);
    }
}

}  // namespace tofmlem
