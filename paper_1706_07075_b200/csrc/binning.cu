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

// Predicted number of voxel visits of the event's clipped TOF window (float32, a sorting heuristic only: it decides
// the ORDER of events inside a locality bin, which the specification leaves open (R14), never a reported value).
__device__ __forceinline__ int predicted_visits(const GridF32 &g, const SubBin &sb, const EventPtrs &ev, uint64_t e,
                                                const float d[3]) {
    const float p1[3] = {__ldg(ev.x1 + e), __ldg(ev.y1 + e), __ldg(ev.z1 + e)};
    const float dt = ev.dt ? __ldg(ev.dt + e) : 0.0f;
    const float L = sqrtf(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    const float iL = 1.0f / L;
    const float o[3] = {g.ox, g.oy, g.oz}, v[3] = {g.vx, g.vy, g.vz};
    const int n[3] = {g.nx, g.ny, g.nz};
    float u[3], s_lo = 0.0f, s_hi = L;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        u[a] = d[a] * iL;
        const float lo = o[a], hi = o[a] + (float)n[a] * v[a];
        if (u[a] == 0.0f) {
            if (p1[a] < lo || p1[a] >= hi) return 0;
        } else {
            const float iu = 1.0f / u[a];
            const float ta = (lo - p1[a]) * iu, tb = (hi - p1[a]) * iu;
            s_lo = fmaxf(s_lo, fminf(ta, tb));
            s_hi = fminf(s_hi, fmaxf(ta, tb));
        }
    }
    if (sb.half_window > 0.0f) {
        const float s_c = 0.5f * L + kHalfC * dt;
        s_lo = fmaxf(s_lo, s_c - sb.half_window);
        s_hi = fminf(s_hi, s_c + sb.half_window);
    }
    if (!(s_hi > s_lo)) return 0;
    int visits = 1;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const float qa = floorf((p1[a] + u[a] * s_lo - o[a]) / v[a]), qb = floorf((p1[a] + u[a] * s_hi - o[a]) / v[a]);
        visits += (int)fabsf(qb - qa);
    }
    return visits;
}

// Locality key of one event per F1: dirclass * (Tx Ty Tz) + tile of the TOF centre; 0xFFFFFFFF for an invalid event.
// d receives the float32 direction p2 - p1.
__device__ __forceinline__ uint32_t event_key(const GridF32 &g, int tile_log2, uint32_t Tx, uint32_t Ty, uint32_t Tz,
                                              const EventPtrs &ev, uint64_t e, float d[3]) {
    float c[3];
    if (!tof_centre(ev, e, c, d)) return 0xFFFFFFFFu;
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
    return dirclass * (Tx * Ty * Tz) + tile;
}

// key (F1) of every event; with `sub` also the sub-bin (events of one locality bin ordered by predicted visit count,
// so that the 32 events of a warp run loops of nearly equal length) and the histogram of the fine key
// key * sb.S + sub (invalid events: the last fine bin).
__global__ void __launch_bounds__(kBlock) bin_keys_kernel(GridF32 g, int tile_log2, SubBin sb, EventPtrs ev,
                                                          uint64_t n, uint32_t *__restrict__ key,
                                                          uint8_t *__restrict__ sub, uint32_t *__restrict__ hist,
                                                          uint32_t nbins) {
    const uint64_t e = (uint64_t)blockIdx.x * kBlock + threadIdx.x;
    if (e >= n) return;
    const int t = 1 << tile_log2;
    const uint32_t Tx = (uint32_t)((g.nx + t - 1) >> tile_log2), Ty = (uint32_t)((g.ny + t - 1) >> tile_log2),
                   Tz = (uint32_t)((g.nz + t - 1) >> tile_log2);
    float d[3];
    const uint32_t k = event_key(g, tile_log2, Tx, Ty, Tz, ev, e, d);
    uint32_t sbin = 0;
    if (k != 0xFFFFFFFFu && sub) {
        const int vis = predicted_visits(g, sb, ev, e, d);
        sbin = vis <= 0 ? 0u : min(sb.S - 1u, 1u + (uint32_t)vis / sb.quantum);
    }
    key[e] = k;
    if (sub) sub[e] = (uint8_t)sbin;
    if (hist) atomicAdd(hist + (k < nbins ? k * sb.S + sbin : nbins * sb.S), 1u);
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

// Three-kernel exclusive scan for long histograms: chunk sums -> single-block scan of the sums -> per-chunk scan.
constexpr int kScanItems = 8, kScanChunk = kBlock * kScanItems;

__global__ void __launch_bounds__(kBlock) scan_chunk_sums_kernel(const uint32_t *__restrict__ in, uint32_t n,
                                                                 uint32_t *__restrict__ sums) {
    __shared__ uint32_t wsum[kBlock / 32];
    const uint32_t base = blockIdx.x * kScanChunk;
    uint32_t s = 0;
    for (int i = threadIdx.x; i < kScanChunk; i += kBlock)
        if (base + i < n) s += in[base + i];
    s = __reduce_add_sync(0xffffffffu, s);
    if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t t = 0;
        for (int w = 0; w < kBlock / 32; ++w) t += wsum[w];
        sums[blockIdx.x] = t;
    }
}

__global__ void __launch_bounds__(kBlock) scan_chunks_kernel(const uint32_t *__restrict__ in, uint32_t n,
                                                             const uint32_t *__restrict__ chunk_base,
                                                             uint32_t *__restrict__ out) {
    __shared__ uint32_t wsum[kBlock / 32];
    const uint32_t lo = blockIdx.x * kScanChunk + threadIdx.x * kScanItems;
    uint32_t v[kScanItems], s = 0;
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) {
        v[i] = lo + i < n ? in[lo + i] : 0u;
        s += v[i];
    }
    // exclusive prefix of the per-thread sums inside the block
    uint32_t inc = s;
    const unsigned lane = threadIdx.x & 31u;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, inc, off);
        if (lane >= (unsigned)off) inc += t;
    }
    if (lane == 31) wsum[threadIdx.x >> 5] = inc;
    __syncthreads();
    uint32_t run = chunk_base[blockIdx.x] + inc - s;
    for (int w = 0; w < (int)(threadIdx.x >> 5); ++w) run += wsum[w];
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) {
        if (lo + i < n) out[lo + i] = run;
        run += v[i];
    }
}

__global__ void __launch_bounds__(kBlock) scatter_perm_kernel(const uint32_t *__restrict__ key,
                                                              const uint8_t *__restrict__ sub, uint32_t S, uint64_t n,
                                                              uint32_t nbins, uint32_t *__restrict__ cursor,
                                                              uint32_t *__restrict__ perm) {
    const uint64_t e = (uint64_t)blockIdx.x * kBlock + threadIdx.x;
    if (e >= n) return;
    const uint32_t k = key[e];
    const uint32_t pos = atomicAdd(cursor + (k < nbins ? k * S + (sub ? sub[e] : 0u) : nbins * S), 1u);
    perm[pos] = (uint32_t)e;
}

// offsets of the (coarse) locality bins out of the fine-bin offsets: out[k] = fine[k * S], k = 0..nbins
__global__ void __launch_bounds__(kBlock) strided_copy_kernel(const uint32_t *__restrict__ fine, uint32_t S,
                                                              uint32_t count, uint32_t *__restrict__ out) {
    const uint32_t k = blockIdx.x * kBlock + threadIdx.x;
    if (k < count) out[k] = fine[(size_t)k * S];
}

__global__ void __launch_bounds__(kBlock) gather_kernel(const float *__restrict__ in, const uint32_t *__restrict__ perm,
                                                        uint64_t n, float *__restrict__ out) {
    const uint64_t i = (uint64_t)blockIdx.x * kBlock + threadIdx.x;
    if (i < n) out[i] = __ldg(in + __ldg(perm + i));
}

// Permuting seven separate float arrays with 4-byte random reads moves a 32-byte sector per value (8x amplification).
// The packed path first interleaves the seven fields of every event into one 32-byte record (coalesced), then gathers
// whole records -- one sector per event -- and writes the struct-of-arrays result coalesced.
__global__ void __launch_bounds__(kBlock) pack_events_kernel(EventPtrs ev, uint64_t n, float4 *__restrict__ rec) {
    const uint64_t e = (uint64_t)blockIdx.x * kBlock + threadIdx.x;
    if (e >= n) return;
    rec[2 * e] = make_float4(__ldg(ev.x1 + e), __ldg(ev.y1 + e), __ldg(ev.z1 + e), __ldg(ev.x2 + e));
    rec[2 * e + 1] = make_float4(__ldg(ev.y2 + e), __ldg(ev.z2 + e), ev.dt ? __ldg(ev.dt + e) : 0.0f, 0.0f);
}

__global__ void __launch_bounds__(kBlock) gather_packed_kernel(const float4 *__restrict__ rec,
                                                               const uint32_t *__restrict__ perm, uint64_t n,
                                                               float *__restrict__ x1, float *__restrict__ y1,
                                                               float *__restrict__ z1, float *__restrict__ x2,
                                                               float *__restrict__ y2, float *__restrict__ z2,
                                                               float *__restrict__ dt) {
    const uint64_t i = (uint64_t)blockIdx.x * kBlock + threadIdx.x;
    if (i >= n) return;
    uint64_t p = __ldg(perm + i);
    if (p >= n) p = n - 1;  // not a permutation of 0..n-1 (caller error): stay inside the records
    const float4 a = __ldg(rec + 2 * p), b = __ldg(rec + 2 * p + 1);
    x1[i] = a.x;
    y1[i] = a.y;
    z1[i] = a.z;
    x2[i] = a.w;
    y2[i] = b.x;
    z2[i] = b.y;
    if (dt) dt[i] = b.z;
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

// Reading R27 / specification F3: the event belongs to every region whose core the axial extent of its
// +-hw window meets: regions lo..hi, span = lo | hi << 16 (-1 for an invalid event); counts[r] = events whose span
// holds r (counts[n_regions]: invalid events).  One IEEE binary32 RN operation per step, as F1.
__global__ void __launch_bounds__(kBlock) region_spans_kernel(EventPtrs ev, uint64_t n, RegionBounds rb, float hw,
                                                              int32_t *__restrict__ span,
                                                              unsigned long long *__restrict__ counts) {
    __shared__ unsigned int local[kMaxRegions + 1];
    for (int i = threadIdx.x; i <= rb.n_regions; i += kBlock) local[i] = 0;
    __syncthreads();
    const uint64_t e = (uint64_t)blockIdx.x * kBlock + threadIdx.x;
    if (e < n) {
        float c[3], d[3];
        int sp = -1;
        if (tof_centre(ev, e, c, d)) {
            const float xx = __fmul_rn(d[0], d[0]), yy = __fmul_rn(d[1], d[1]), zz = __fmul_rn(d[2], d[2]);
            const float L = __fsqrt_rn(__fadd_rn(__fadd_rn(xx, yy), zz));
            const float hz = __fmul_rn(__fdiv_rn(hw, L), fabsf(d[2]));
            const float zlo = __fsub_rn(c[2], hz), zhi = __fadd_rn(c[2], hz);
            int lo = 0, hi = 0;
            for (int j = 1; j < rb.n_regions; ++j) {
                lo += (rb.zb[j] <= zlo) ? 1 : 0;
                hi += (rb.zb[j] <= zhi) ? 1 : 0;
            }
            sp = lo | (hi << 16);
            for (int r = lo; r <= hi; ++r) atomicAdd(local + r, 1u);
        } else {
            atomicAdd(local + rb.n_regions, 1u);
        }
        span[e] = sp;
    }
    __syncthreads();
    for (int i = threadIdx.x; i <= rb.n_regions; i += kBlock)
        if (local[i]) atomicAdd(counts + i, (unsigned long long)local[i]);
}

// block-aggregated scatter of the spans: the event's index goes to the list of every region of its span
__global__ void __launch_bounds__(kBlock) region_span_scatter_kernel(const int32_t *__restrict__ span, uint64_t n,
                                                                     int n_regions,
                                                                     unsigned long long *__restrict__ cursor,
                                                                     uint32_t *__restrict__ perm) {
    __shared__ unsigned int local[kMaxRegions + 1];
    __shared__ unsigned long long base[kMaxRegions + 1];
    for (int i = threadIdx.x; i <= n_regions; i += kBlock) local[i] = 0;
    __syncthreads();
    const uint64_t e = (uint64_t)blockIdx.x * kBlock + threadIdx.x;
    int lo = 0, hi = -1;
    unsigned int rank[4] = {0, 0, 0, 0};  // a window longer than three cores is not supported (checked by the caller)
    if (e < n) {
        const int sp = span[e];
        if (sp >= 0) {
            lo = sp & 0xFFFF;
            hi = sp >> 16;
            if (hi > lo + 3) hi = lo + 3;
            for (int r = lo; r <= hi; ++r) rank[r - lo] = atomicAdd(local + r, 1u);
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i <= n_regions; i += kBlock)
        if (local[i]) base[i] = atomicAdd(cursor + i, (unsigned long long)local[i]);
    __syncthreads();
    for (int r = lo; r <= hi; ++r) perm[base[r] + rank[r - lo]] = (uint32_t)e;
}

// NEXT-4: TOF-based scatter rejection (PAPER.md:63 Fig. 2, :69-71; reading R24, float32 specification F2 in
// DESIGN.md): keep the event iff the segment {c + u t : |t| <= h} (c = TOF-estimated annihilation point, u = LOR
// direction, h = 1.96 sigma: the 95 % confidence interval) meets the body outline, a union of ellipsoids.  Every
// float operation is one IEEE binary32 RN operation in the order of F2, so the flags are bit-exact.
// Kept events' indices are appended to `perm` (order unspecified) through one atomic per warp.
__global__ void __launch_bounds__(kBlock) scatter_keep_kernel(EventPtrs ev, uint64_t n, EllipsoidSet es, float h,
                                                              uint8_t *__restrict__ keep, uint32_t *__restrict__ perm,
                                                              unsigned long long *__restrict__ counter) {
    const uint64_t e = (uint64_t)blockIdx.x * kBlock + threadIdx.x;
    bool hit = false;
    float c[3], d[3];
    if (e < n && tof_centre(ev, e, c, d)) {
        const float xx = __fmul_rn(d[0], d[0]), yy = __fmul_rn(d[1], d[1]), zz = __fmul_rn(d[2], d[2]);
        const float L = __fsqrt_rn(__fadd_rn(__fadd_rn(xx, yy), zz));
        const float ux = __fdiv_rn(d[0], L), uy = __fdiv_rn(d[1], L), uz = __fdiv_rn(d[2], L);
        for (int k = 0; k < es.n && !hit; ++k) {
            const float *q = es.v + 6 * k;
            const float rx = __fmul_rn(__fsub_rn(c[0], q[0]), q[3]);
            const float ry = __fmul_rn(__fsub_rn(c[1], q[1]), q[4]);
            const float rz = __fmul_rn(__fsub_rn(c[2], q[2]), q[5]);
            const float wx = __fmul_rn(ux, q[3]), wy = __fmul_rn(uy, q[4]), wz = __fmul_rn(uz, q[5]);
            const float A = __fadd_rn(__fadd_rn(__fmul_rn(wx, wx), __fmul_rn(wy, wy)), __fmul_rn(wz, wz));
            const float B = __fadd_rn(__fadd_rn(__fmul_rn(rx, wx), __fmul_rn(ry, wy)), __fmul_rn(rz, wz));
            float t = -__fdiv_rn(B, A);
            t = fminf(fmaxf(t, -h), h);
            const float px = __fadd_rn(rx, __fmul_rn(wx, t));
            const float py = __fadd_rn(ry, __fmul_rn(wy, t));
            const float pz = __fadd_rn(rz, __fmul_rn(wz, t));
            const float Q = __fadd_rn(__fadd_rn(__fmul_rn(px, px), __fmul_rn(py, py)), __fmul_rn(pz, pz));
            hit = Q <= 1.0f;
        }
    }
    if (e < n) keep[e] = hit ? 1 : 0;
    const unsigned m = __ballot_sync(0xffffffffu, hit);
    if (m) {
        const unsigned lane = threadIdx.x & 31u;
        unsigned long long base = 0;
        if (lane == (unsigned)(__ffs(m) - 1)) base = atomicAdd(counter, (unsigned long long)__popc(m));
        base = __shfl_sync(0xffffffffu, base, __ffs(m) - 1);
        if (hit && perm) perm[base + __popc(m & ((1u << lane) - 1u))] = (uint32_t)e;
    }
}

static inline unsigned grid_for(uint64_t n) { return (unsigned)((n + kBlock - 1) / kBlock); }

// Plan of the tile-mode EM pass (tile.cu): histogram of the keys of an event list that is expected to be sorted by
// key already (the output of tofmlem_bin_events + tofmlem_permute_events), and a flag that says whether it is.
__global__ void __launch_bounds__(kBlock) plan_hist_kernel(GridF32 g, int tile_log2, EventPtrs ev, uint64_t n,
                                                           uint32_t *__restrict__ hist, uint32_t nbins,
                                                           unsigned *__restrict__ unsorted) {
    __shared__ uint32_t keys[kBlock + 1];
    const uint64_t e = (uint64_t)blockIdx.x * kBlock + threadIdx.x;
    const int t = 1 << tile_log2;
    const uint32_t Tx = (uint32_t)((g.nx + t - 1) >> tile_log2), Ty = (uint32_t)((g.ny + t - 1) >> tile_log2),
                   Tz = (uint32_t)((g.nz + t - 1) >> tile_log2);
    float d[3];
    uint32_t k = 0xFFFFFFFFu;
    if (e < n) k = event_key(g, tile_log2, Tx, Ty, Tz, ev, e, d);
    keys[threadIdx.x + 1] = k;
    if (threadIdx.x == 0) keys[0] = e > 0 && e < n ? event_key(g, tile_log2, Tx, Ty, Tz, ev, e - 1, d) : 0u;
    __syncthreads();
    if (e >= n) return;
    if (k < keys[threadIdx.x]) *unsorted = 1u;
    // the list is (expected to be) sorted: the lanes of a warp hold one or two keys, so one atomic per distinct key of the
    // warp instead of one per event (which serialise on the same counter: 21 -> ~4 ms at 146 M events)
    const unsigned active = __activemask();
    const unsigned same = __match_any_sync(active, k);
    if (k < nbins && (threadIdx.x & 31u) == (unsigned)(__ffs(same) - 1)) atomicAdd(hist + k, (uint32_t)__popc(same));
}

// Order-preserving compaction: list[pos[i]] = i for every i with flags[i] != 0 (pos = exclusive scan of flags).
__global__ void __launch_bounds__(kBlock) compact_flags_kernel(const uint32_t *__restrict__ flags,
                                                               const uint32_t *__restrict__ pos, uint32_t n,
                                                               uint32_t *__restrict__ list) {
    const uint32_t i = blockIdx.x * kBlock + threadIdx.x;
    if (i < n && flags[i]) list[pos[i]] = i;
}

void launch_compact_flags(const uint32_t *flags, const uint32_t *pos, uint32_t n, uint32_t *list, cudaStream_t s) {
    if (n) compact_flags_kernel<<<(n + kBlock - 1) / kBlock, kBlock, 0, s>>>(flags, pos, n, list);
}

void launch_plan_hist(const GridF32 &g, int tile_log2, const EventPtrs &ev, uint64_t n, uint32_t *hist, uint32_t nbins,
                      unsigned *unsorted, cudaStream_t s) {
    if (n == 0) return;
    plan_hist_kernel<<<(unsigned)((n + kBlock - 1) / kBlock), kBlock, 0, s>>>(g, tile_log2, ev, n, hist, nbins, unsorted);
}

void launch_bin_keys(const GridF32 &g, int tile_log2, const SubBin &sb, const EventPtrs &ev, uint64_t n, uint32_t *key,
                     uint8_t *sub, uint32_t *hist, uint32_t nbins, cudaStream_t s) {
    if (n) bin_keys_kernel<<<grid_for(n), kBlock, 0, s>>>(g, tile_log2, sb, ev, n, key, sub, hist, nbins);
}

uint32_t scan_tmp_elems(uint32_t n) { return 2 * ((n + kScanChunk - 1) / kScanChunk + 1); }

int launch_exclusive_scan_u32(const uint32_t *in, uint32_t *out, uint32_t *tmp, uint32_t n, cudaStream_t s) {
    if (!n) return 0;
    const uint32_t chunks = (n + kScanChunk - 1) / kScanChunk;
    if (chunks <= 4 || !tmp) {
        exclusive_scan_kernel<<<1, 1024, 0, s>>>(in, out, nullptr, n);
        return 1;
    }
    scan_chunk_sums_kernel<<<chunks, kBlock, 0, s>>>(in, n, tmp);
    exclusive_scan_kernel<<<1, 1024, 0, s>>>(tmp, tmp + chunks + 1, nullptr, chunks);
    scan_chunks_kernel<<<chunks, kBlock, 0, s>>>(in, n, tmp + chunks + 1, out);
    return 3;
}

void launch_scatter_perm(const uint32_t *key, const uint8_t *sub, uint32_t S, uint64_t n, uint32_t nbins,
                         uint32_t *cursor, uint32_t *perm, cudaStream_t s) {
    if (n) scatter_perm_kernel<<<grid_for(n), kBlock, 0, s>>>(key, sub, S, n, nbins, cursor, perm);
}

void launch_strided_copy(const uint32_t *fine, uint32_t S, uint32_t count, uint32_t *out, cudaStream_t s) {
    if (count) strided_copy_kernel<<<(count + kBlock - 1) / kBlock, kBlock, 0, s>>>(fine, S, count, out);
}

void launch_gather(const float *in, const uint32_t *perm, uint64_t n, float *out, cudaStream_t s) {
    if (n) gather_kernel<<<grid_for(n), kBlock, 0, s>>>(in, perm, n, out);
}

void launch_gather_packed(const EventPtrs &in, const uint32_t *perm, uint64_t n, float *rec /* 8 n floats */,
                          float *const out[7], cudaStream_t s) {
    if (!n) return;
    pack_events_kernel<<<grid_for(n), kBlock, 0, s>>>(in, n, reinterpret_cast<float4 *>(rec));
    gather_packed_kernel<<<grid_for(n), kBlock, 0, s>>>(reinterpret_cast<const float4 *>(rec), perm, n, out[0], out[1],
                                                        out[2], out[3], out[4], out[5], out[6]);
}

void launch_region_ids(const EventPtrs &ev, uint64_t n, const RegionBounds &rb, int32_t *region,
                       unsigned long long *counts, cudaStream_t s) {
    if (n) region_ids_kernel<<<grid_for(n), kBlock, 0, s>>>(ev, n, rb, region, counts);
}

void launch_region_scatter(const int32_t *region, uint64_t n, int n_regions, unsigned long long *cursor,
                           uint32_t *perm, cudaStream_t s) {
    if (n) region_scatter_kernel<<<grid_for(n), kBlock, 0, s>>>(region, n, n_regions, cursor, perm);
}

void launch_region_spans(const EventPtrs &ev, uint64_t n, const RegionBounds &rb, float hw, int32_t *span,
                         unsigned long long *counts, cudaStream_t s) {
    if (n) region_spans_kernel<<<grid_for(n), kBlock, 0, s>>>(ev, n, rb, hw, span, counts);
}

void launch_region_span_scatter(const int32_t *span, uint64_t n, int n_regions, unsigned long long *cursor,
                                uint32_t *perm, cudaStream_t s) {
    if (n) region_span_scatter_kernel<<<grid_for(n), kBlock, 0, s>>>(span, n, n_regions, cursor, perm);
}

void launch_scatter_keep(const EventPtrs &ev, uint64_t n, const EllipsoidSet &es, float h, uint8_t *keep,
                         uint32_t *perm, unsigned long long *counter, cudaStream_t s) {
    if (n) scatter_keep_kernel<<<grid_for(n), kBlock, 0, s>>>(ev, n, es, h, keep, perm, counter);
}

}  // namespace tofmlem
