// sampled.cu -- the paper's own K-sample TOF kernel (Fig. 3, "variant V").
//
// K samples equally spaced inside the truncated Gaussian (offset_k = -T sigma + k 2 T sigma / (K-1)), Gaussian
// weights normalised to sum to one, centred on the measured time difference; every sample is filled
// into the voxel that contains it ("direct technique for voxel filling").  Samples beyond the LOR's end
// points or outside the grid are dropped (R8).  The paper kept the look-up table of (offset, weight) pairs as an
// array of structs in Fermi constant memory; here it is an array of structs in global memory read
// with a warp-uniform load (every lane reads entry k at the same time, so it is one L1 broadcast per step), which
// also lets contexts with different sigma run concurrently.
//
// One thread per event, constant work per event (no divergence).  The voxel of a sample is an integer decided by
// floating point: it is taken in fp64 with the oracle's expression floor((p1 + u s - o) / v) (single rounded
// operations, no contraction), evaluated as a multiplication by 1/v and re-done with the exact division only when
// the product is within 1e-9 of an integer (the only case where the two can differ).
//
// Fast path: that fp64 expression is only evaluated for samples that come close to a voxel plane.  Per axis the
// position of sample k in voxel units is q0 + offset_k * (u / v) with q0 the position of the kernel centre; relative to
// floor(q0) this is a float32 fma whose error is below 1e-5 voxel for any window up to a few hundred voxels, so when
// the float32 value is farther than `guard` = 1e-4 + 1e-5 |q| from an integer its floor IS the fp64 decision; otherwise
// (about one sample in a thousand) the exact fp64 path decides.  Results are identical to the all-fp64 kernel.
#include "internal.cuh"

namespace tofmlem {

namespace {

constexpr int kBlock = 256;

__device__ __forceinline__ bool finite_f(float x) { return fabsf(x) <= 3.402823466e+38f; }

struct SampledRay {
    double p1[3], u[3];
    double s_c, L;
    int base[3];   // floor of the kernel centre's position in voxel units, per axis
    float f0[3];   // its fractional part
    float du[3];   // u / v: voxels per mm along the LOR
    float guard;   // fast path: distance from a voxel plane (voxels) below which the fp64 expression decides
    int k0, k1;    // samples k0 <= k < k1 lie between the LOR's end points (the others are dropped, R8)
};

__device__ __forceinline__ bool sampled_setup(const EventPtrs &ev, uint64_t e, SampledRay &r) {
    const float x1 = __ldcs(ev.x1 + e), y1 = __ldcs(ev.y1 + e), z1 = __ldcs(ev.z1 + e);
    const float x2 = __ldcs(ev.x2 + e), y2 = __ldcs(ev.y2 + e), z2 = __ldcs(ev.z2 + e);
    const float dt = ev.dt ? __ldcs(ev.dt + e) : 0.0f;
    if (!(finite_f(x1) && finite_f(y1) && finite_f(z1) && finite_f(x2) && finite_f(y2) && finite_f(z2) && finite_f(dt)))
        return false;
    r.p1[0] = x1;
    r.p1[1] = y1;
    r.p1[2] = z1;
    const double dx = __dsub_rn((double)x2, r.p1[0]), dy = __dsub_rn((double)y2, r.p1[1]),
                 dz = __dsub_rn((double)z2, r.p1[2]);
    const double L2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
    if (!(L2 > 0.0)) return false;
    r.L = __dsqrt_rn(L2);
    r.u[0] = __ddiv_rn(dx, r.L);
    r.u[1] = __ddiv_rn(dy, r.L);
    r.u[2] = __ddiv_rn(dz, r.L);
    // s_c = 0.5 L + 0.5 c dt  ("centered in the coincidence time difference"; R22)
    r.s_c = __dadd_rn(__dmul_rn(0.5, r.L), __dmul_rn(__dmul_rn(0.5, kCmmPerPs), (double)dt));
    return true;
}

// voxel index along one axis of the point p1 + u s, or -1 when outside [0, n)
__device__ __forceinline__ int sample_voxel(double p1, double u, double s, double o, double v, double iv, int n) {
    const double t = __dsub_rn(__dadd_rn(p1, __dmul_rn(u, s)), o);
    double q = __dmul_rn(t, iv);
    if (fabs(q - rint(q)) <= 1e-9 * fmax(1.0, fabs(q))) q = __ddiv_rn(t, v);  // near a voxel plane: the exact quotient
    const double f = floor(q);
    if (!(f >= 0.0) || f >= (double)n) return -1;
    return (int)f;
}

__device__ __forceinline__ void sampled_fast_setup(const ProjParams &P, const SampleLutEntry *__restrict__ lut, int K,
                                                   SampledRay &r) {
    float span = 0.0f;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double q0 = ((r.p1[a] + r.u[a] * r.s_c) - P.o[a]) * P.iv[a];
        const double fl = floor(q0);
        // a centre far outside the grid cannot produce an in-grid sample through the fast path: clamp the base so that
        // the int conversion is defined; such samples fail the bounds test either way
        r.base[a] = (int)fmax(-1.0e9, fmin(1.0e9, fl));
        r.f0[a] = (float)(q0 - fl);
        r.du[a] = (float)(r.u[a] * P.iv[a]);
        span = fmaxf(span, fabsf(r.du[a]));
    }
    // |q| <= 1 + half window * |du|: the float32 error of the fma is below 1e-5 voxel per 100 voxels of |q|
    r.guard = 1.0e-4f + 1.0e-5f * (1.0f + (float)P.half_window * span);
    // The offsets increase with k, so the samples between the end points (0 <= s_c + offset_k <= L, evaluated in
    // fp64 exactly as the per-sample test would be) form one interval [k0, k1): found by scanning from both ends
    // (no iteration at all unless the kernel centre is within 3 sigma of a detector).
    int k0 = 0, k1 = K;
    while (k0 < K) {
        const double s = __dadd_rn(r.s_c, lut[k0].offset);
        if (!(s < 0.0 || s > r.L)) break;
        ++k0;
    }
    while (k1 > k0) {
        const double s = __dadd_rn(r.s_c, lut[k1 - 1].offset);
        if (!(s < 0.0 || s > r.L)) break;
        --k1;
    }
    r.k0 = k0;
    r.k1 = k1;
}

// voxel index along one axis through the float32 fast path; falls back to the exact fp64 decision near a voxel plane
__device__ __forceinline__ int sample_voxel_fast(const ProjParams &P, const SampledRay &r, int a, float off, double s) {
    const float qf = fmaf(off, r.du[a], r.f0[a]);
    const int fl = __float2int_rd(qf);
    const float d = qf - (float)fl;  // distance to the voxel plane below, in voxels
    if (fminf(d, 1.0f - d) < r.guard || !(fabsf(qf) < 1.0e6f))
        return sample_voxel(r.p1[a], r.u[a], s, P.o[a], P.v[a], P.iv[a], P.n[a]);
    const int i = r.base[a] + fl;
    return (unsigned)i < (unsigned)P.n[a] ? i : -1;
}

// flat voxel index of sample k, or -1 when the sample is dropped
// (for k0 <= k < k1; the end-point test was done by sampled_fast_setup)
__device__ __forceinline__ int sample_index(const ProjParams &P, const SampledRay &r, const SampleLutEntry &l) {
    const double s = __dadd_rn(r.s_c, l.offset);  // only used by the fp64 fallback
    const int ix = sample_voxel_fast(P, r, 0, l.offset_f, s);
    const int iy = sample_voxel_fast(P, r, 1, l.offset_f, s);
    const int iz = sample_voxel_fast(P, r, 2, l.offset_f, s);
    if ((ix | iy | iz) < 0) return -1;
    return (iz * P.n[1] + iy) * P.n[0] + ix;
}

__global__ void __launch_bounds__(kBlock) sampled_forward_kernel(ProjParams P, const SampleLutEntry *__restrict__ lut,
                                                                 int K, EventPtrs ev, uint64_t n,
                                                                 const float *__restrict__ image,
                                                                 float *__restrict__ fwd) {
    const uint64_t e = (uint64_t)blockIdx.x * kBlock + threadIdx.x;
    if (e >= n) return;
    SampledRay r;
    float acc = 0.0f;
    if (sampled_setup(ev, e, r)) {
        sampled_fast_setup(P, lut, K, r);
        for (int k = r.k0; k < r.k1; ++k) {
            const SampleLutEntry s = lut[k];
            const int j = sample_index(P, r, s);
            if (j >= 0) acc = fmaf(s.weight, __ldg(image + j), acc);
        }
    }
    fwd[e] = acc;
}

__global__ void __launch_bounds__(kBlock) sampled_backproject_kernel(ProjParams P,
                                                                     const SampleLutEntry *__restrict__ lut, int K,
                                                                     EventPtrs ev, uint64_t n,
                                                                     const float *__restrict__ values,
                                                                     float *__restrict__ out) {
    const uint64_t e = (uint64_t)blockIdx.x * kBlock + threadIdx.x;
    if (e >= n) return;
    SampledRay r;
    if (!sampled_setup(ev, e, r)) return;
    sampled_fast_setup(P, lut, K, r);
    const float val = values ? __ldg(values + e) : 1.0f;
    if (val == 0.0f) return;
    for (int k = r.k0; k < r.k1; ++k) {
        const SampleLutEntry s = lut[k];
        const int j = sample_index(P, r, s);
        if (j >= 0) atomicAdd(out + j, s.weight * val);
    }
}

// Fused EM pass of one event: pass 1 gathers (the forward value stays in a register) and keeps the voxel index of
// each of the first kSampleCache samples in shared memory; pass 2 replays them (samples beyond the cache are recomputed)
// and scatters evw * w_k / fwd.  Consecutive samples of one event often fall into the same voxel (the sample spacing
// 6 sigma/(K-1) = 3.7 mm at 300 ps, K = 32 is about one 3.75 mm voxel): equal neighbours are merged into one reduction.
// (Merging further into 16-byte reductions on a brick layout was measured: 3.64e9 -> 2.90e9 reductions but 28.0 ->
// 30.0 ms at K = 32 -- this pass is bound by its instruction count, not by the L2 atomic units.)
constexpr int kSampleCache = 32;

__device__ __forceinline__ void sampled_em_event(const ProjParams &P, const SampleLutEntry *__restrict__ lut, int K,
                                                 const EventPtrs &ev, uint64_t e, uint64_t n,
                                                 const float *__restrict__ evw, const float *__restrict__ image,
                                                 float *__restrict__ corr, int (*jcache)[kBlock], unsigned &visits,
                                                 unsigned &reds, bool &valid) {
    SampledRay r;
    valid = false;
    visits = reds = 0;
    if (e < n && sampled_setup(ev, e, r)) {
        sampled_fast_setup(P, lut, K, r);
        float acc = 0.0f;
        for (int k = r.k0; k < r.k1; ++k) {
            const SampleLutEntry s = lut[k];
            const int j = sample_index(P, r, s);
            if (k < kSampleCache) jcache[k][threadIdx.x] = j;
            if (j >= 0) {
                acc = fmaf(s.weight, __ldg(image + j), acc);
                ++visits;
            }
        }
        if (acc > 0.0f) {  // R9
            valid = true;
            const float scale = (evw ? __ldg(evw + e) : 1.0f) / acc;
            int pend = -1;
            float pw = 0.0f;
            for (int k = r.k0; k < r.k1; ++k) {
                const int j = k < kSampleCache ? jcache[k][threadIdx.x] : sample_index(P, r, lut[k]);
                if (j < 0) continue;
                if (j != pend) {
                    if (pend >= 0) {
                        atomicAdd(corr + pend, pw * scale);
                        ++reds;
                    }
                    pend = j;
                    pw = 0.0f;
                }
                pw += lut[k].weight;
            }
            if (pend >= 0) {
                atomicAdd(corr + pend, pw * scale);
                ++reds;
            }
        }
    }
}

// Persistent scheduling as in projector.cu's em_persistent_kernel: the (locality-binned) list is cut into one segment
// per SM, every warp takes 32-event chunks from the queue of the SM it runs on and steals from other segments when
// its own is exhausted, so that co-resident warps share L1 while different SMs reduce into different parts of the
// volume.
__global__ void __launch_bounds__(kBlock) sampled_em_kernel(ProjParams P, const SampleLutEntry *__restrict__ lut, int K,
                                                            EventPtrs ev, uint64_t n, const float *__restrict__ evw,
                                                            const float *__restrict__ image, float *__restrict__ corr,
                                                            DeviceStats *stats, unsigned *queues, unsigned nseg,
                                                            unsigned per_seg, unsigned segs_per_sm) {
    __shared__ int jcache[kSampleCache][kBlock];  // voxel index of sample k of this thread's event (thread-private column)
    unsigned smid;
    asm("mov.u32 %0, %%smid;" : "=r"(smid));
    const unsigned lane = threadIdx.x & 31u;
    const unsigned base = nseg / segs_per_sm;  // the warps of an SM start on segs_per_sm segments, base apart
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
        unsigned visits, reds;
        bool valid;
        sampled_em_event(P, lut, K, ev, ((uint64_t)seg * per_seg + c) * 32u + lane, n, evw, image, corr, jcache, visits,
                         reds, valid);
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

inline unsigned grid_for(uint64_t n) { return (unsigned)((n + kBlock - 1) / kBlock); }

}  // namespace

void launch_sampled_forward(const ProjParams &p, const SampleLutEntry *lut, int K, const EventPtrs &ev, uint64_t n,
                            const float *image, float *fwd, cudaStream_t s) {
    if (n) sampled_forward_kernel<<<grid_for(n), kBlock, 0, s>>>(p, lut, K, ev, n, image, fwd);
}

void launch_sampled_backproject(const ProjParams &p, const SampleLutEntry *lut, int K, const EventPtrs &ev, uint64_t n,
                                const float *values, float *out, cudaStream_t s) {
    if (n) sampled_backproject_kernel<<<grid_for(n), kBlock, 0, s>>>(p, lut, K, ev, n, values, out);
}

void launch_sampled_em(const ProjParams &p, const SampleLutEntry *lut, int K, const EventPtrs &ev, uint64_t n,
                       const float *evw, const float *image, float *corr, DeviceStats *stats, unsigned *queues,
                       cudaStream_t s) {
    if (!n) return;
    int per_sm = 0, n_sm = p.n_sm;  // the context's device (tofmlem_create); occupancy asked per launch, no cached state
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, sampled_em_kernel, kBlock, 0);
    if (n_sm < 1) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    }
    constexpr unsigned kSegsPerSm = 2;  // measured 1 / 2 / 3 / 4: 27.8 / 24.1 / 24.3 / 24.6 ms at K = 32's persistent pass for short windows
    unsigned nseg = (unsigned)n_sm * kSegsPerSm;
    if (nseg > (unsigned)kMaxQueues) nseg = (unsigned)kMaxQueues / kSegsPerSm * kSegsPerSm;
    if (nseg % 61u == 0) nseg -= kSegsPerSm;
    const uint64_t wchunks = (n + 31) / 32;
    const unsigned per_seg = (unsigned)((wchunks + nseg - 1) / nseg);
    cudaMemsetAsync(queues, 0, (size_t)nseg * kQueueStride * sizeof(unsigned), s);
    sampled_em_kernel<<<n_sm * (per_sm > 0 ? per_sm : 1), kBlock, 0, s>>>(p, lut, K, ev, n, evw, image, corr, stats,
                                                                        queues, nseg, per_seg, kSegsPerSm);
}

}  // namespace tofmlem
