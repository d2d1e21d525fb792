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
#include "internal.cuh"

namespace tofmlem {

namespace {

constexpr int kBlock = 256;

__device__ __forceinline__ bool finite_f(float x) { return fabsf(x) <= 3.402823466e+38f; }

struct SampledRay {
    double p1[3], u[3];
    double s_c, L;
};

__device__ __forceinline__ bool sampled_setup(const EventPtrs &ev, uint64_t e, SampledRay &r) {
    const float x1 = __ldg(ev.x1 + e), y1 = __ldg(ev.y1 + e), z1 = __ldg(ev.z1 + e);
    const float x2 = __ldg(ev.x2 + e), y2 = __ldg(ev.y2 + e), z2 = __ldg(ev.z2 + e);
    const float dt = ev.dt ? __ldg(ev.dt + e) : 0.0f;
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

// flat voxel index of sample k, or -1 when the sample is dropped
__device__ __forceinline__ int sample_index(const ProjParams &P, const SampledRay &r, double offset) {
    const double s = __dadd_rn(r.s_c, offset);
    if (s < 0.0 || s > r.L) return -1;
    const int ix = sample_voxel(r.p1[0], r.u[0], s, P.o[0], P.v[0], P.iv[0], P.n[0]);
    const int iy = sample_voxel(r.p1[1], r.u[1], s, P.o[1], P.v[1], P.iv[1], P.n[1]);
    const int iz = sample_voxel(r.p1[2], r.u[2], s, P.o[2], P.v[2], P.iv[2], P.n[2]);
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
        for (int k = 0; k < K; ++k) {
            const SampleLutEntry s = lut[k];
            const int j = sample_index(P, r, s.offset);
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
    const float val = values ? __ldg(values + e) : 1.0f;
    if (val == 0.0f) return;
    for (int k = 0; k < K; ++k) {
        const SampleLutEntry s = lut[k];
        const int j = sample_index(P, r, s.offset);
        if (j >= 0) atomicAdd(out + j, s.weight * val);
    }
}

// Fused EM pass: pass 1 gathers (the forward value stays in a register), pass 2 recomputes the sample voxels and
// scatters evw * w_k / fwd.  Consecutive samples of one event often fall into the same voxel (the sample spacing
// 6 sigma/(K-1) = 3.7 mm at 300 ps, K = 32 is about one 3.75 mm voxel): equal neighbours are merged into one
// reduction.
__global__ void __launch_bounds__(kBlock) sampled_em_kernel(ProjParams P, const SampleLutEntry *__restrict__ lut, int K,
                                                            EventPtrs ev, uint64_t n, const float *__restrict__ evw,
                                                            const float *__restrict__ image, float *__restrict__ corr,
                                                            DeviceStats *stats) {
    const uint64_t e = (uint64_t)blockIdx.x * kBlock + threadIdx.x;
    SampledRay r;
    bool valid = false;
    unsigned visits = 0, reds = 0;
    if (e < n && sampled_setup(ev, e, r)) {
        float acc = 0.0f;
        for (int k = 0; k < K; ++k) {
            const SampleLutEntry s = lut[k];
            const int j = sample_index(P, r, s.offset);
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
            for (int k = 0; k < K; ++k) {
                const SampleLutEntry s = lut[k];
                const int j = sample_index(P, r, s.offset);
                if (j < 0) continue;
                if (j != pend) {
                    if (pend >= 0) {
                        atomicAdd(corr + pend, pw * scale);
                        ++reds;
                    }
                    pend = j;
                    pw = 0.0f;
                }
                pw += s.weight;
            }
            if (pend >= 0) {
                atomicAdd(corr + pend, pw * scale);
                ++reds;
            }
        }
    }
    const unsigned nv = __popc(__ballot_sync(0xffffffffu, valid));
    const unsigned vis = __reduce_add_sync(0xffffffffu, visits);
    const unsigned nr = __reduce_add_sync(0xffffffffu, reds);
    if ((threadIdx.x & 31) == 0 && stats) {
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
                       const float *evw, const float *image, float *corr, DeviceStats *stats, cudaStream_t s) {
    if (n) sampled_em_kernel<<<grid_for(n), kBlock, 0, s>>>(p, lut, K, ev, n, evw, image, corr, stats);
}

}  // namespace tofmlem
