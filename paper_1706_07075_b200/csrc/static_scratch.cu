// static_scratch.cu -- tofmlem_em_correction_static: the fused forward+back EM pass (include/tofmlem.h, R1, R9) for
// callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).
// No context, no allocation: the only scratch the pass needs -- the work-queue counters of the persistent kernel -- lives
// in a file-scope __device__ array that every GPU which loads the library holds until exit (kStaticQueues * 4 bytes).
//
// The kernel is a variant of em_persistent_kernel (projector.cu) on the same device code (walk.cuh: fp64 ray set-up,
// branch-free fp32 walk, 16-byte reductions): per-SM work queues over the event list in the order given, correction
// image in GRID order (no bricks: there is no context to remember a layout).
//
// The array's name is a host-side stand-in in host code, not a device address: the address comes from
// cudaGetSymbolAddress, asked once per device with that device current, and is what the kernel and the memset get.
// All calls share the array: the counters are cleared on the caller's stream before every launch, and two calls that
// overlap on the GPU (different streams, no dependency between them) RACE on it -- the caller serialises them.
#include <math.h>

#include <mutex>
#include <string>

#include "internal.cuh"
#include "walk.cuh"

namespace tofmlem {

namespace {

constexpr int kSBlock = 256;
constexpr unsigned kStaticQueues = TOFMLEM_STATIC_MAX_QUEUES;
constexpr int kMaxDevices = 64;

static __device__ __align__(256) unsigned g_static_queues[kStaticQueues];

std::mutex g_mutex;
unsigned *g_queue_ptr[kMaxDevices];  // device address of g_static_queues on device d (NULL: not asked yet)
int g_n_sm[kMaxDevices];
thread_local std::string g_err;

int sfail(int code, const std::string &what) {
    g_err = what;
    return code;
}

template <bool TOF, bool VEC>
__global__ void __launch_bounds__(kSBlock, 5) em_static_kernel(ProjParams P, EventPtrs ev, uint64_t n,
                                                              const float *__restrict__ image,
                                                              float *__restrict__ corr, unsigned *queues,
                                                              unsigned nseg, unsigned per_seg, unsigned segs_per_sm) {
    unsigned smid;
    asm("mov.u32 %0, %%smid;" : "=r"(smid));
    const unsigned lane = threadIdx.x & 31u;
    const unsigned base = nseg / segs_per_sm;
    unsigned seg = smid % base + base * ((threadIdx.x >> 5) % segs_per_sm), tries = 0;
    while (true) {
        unsigned c = per_seg;
        if (lane == 0 && *(volatile unsigned *)(queues + seg) < per_seg) c = atomicAdd(queues + seg, 1u);
        c = __shfl_sync(0xffffffffu, c, 0);
        if (c >= per_seg) {
            if (++tries >= nseg) break;
            seg = (seg + 61u) % nseg;  // work stealing; nseg is never a multiple of 61 (see the launch)
            continue;
        }
        const uint64_t e = ((uint64_t)seg * per_seg + c) * 32u + lane;
        if (e >= n) continue;
        Ray r;
        const float x1 = __ldcs(ev.x1 + e), y1 = __ldcs(ev.y1 + e), z1 = __ldcs(ev.z1 + e);
        const float x2 = __ldcs(ev.x2 + e), y2 = __ldcs(ev.y2 + e), z2 = __ldcs(ev.z2 + e);
        const float dt = (TOF && ev.dt) ? __ldcs(ev.dt + e) : 0.0f;
        if (!ray_setup<TOF>(P, x1, y1, z1, x2, y2, z2, dt, r)) continue;
        int visits;
        const float acc = ray_gather<TOF>(P, r, image, visits);
        if (acc > 0.0f) ray_scatter<TOF, VEC, false>(P, r, corr, 1.0f / acc);  // R9
    }
}

template <bool TOF, bool VEC>
cudaError_t launch_static(const ProjParams &p, const EventPtrs &ev, uint64_t n, const float *image, float *corr,
                          unsigned *queues, int n_sm, unsigned segs, cudaStream_t s) {
    int per_sm = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, em_static_kernel<TOF, VEC>, kSBlock, 0);
    if (e != cudaSuccess) return e;
    unsigned nseg = (unsigned)n_sm * segs;
    if (nseg > segs && nseg % 61u == 0) nseg -= segs;
    const uint64_t pieces = (n + 31) / 32;
    const unsigned per_seg = (unsigned)((pieces + nseg - 1) / nseg);
    e = cudaMemsetAsync(queues, 0, nseg * sizeof(unsigned), s);  // the array keeps the last call's counters
    if (e != cudaSuccess) return e;
    const unsigned grid = (unsigned)n_sm * (unsigned)(per_sm > 0 ? per_sm : 1);
    em_static_kernel<TOF, VEC><<<grid, kSBlock, 0, s>>>(p, ev, n, image, corr, queues, nseg, per_seg, segs);
    return cudaGetLastError();
}

}  // namespace

}  // namespace tofmlem

using namespace tofmlem;

extern "C" const char *tofmlem_static_error(void) { return g_err.c_str(); }

extern "C" int tofmlem_em_correction_static(const tofmlem_grid *grid, double tof_fwhm_ps, double trunc_sigmas,
                                            const tofmlem_events *ev, uint64_t n, const float *d_image, float *d_corr,
                                            int queues_per_sm, void *cuda_stream) {
    if (!grid || !ev || !d_image || !d_corr) return sfail(TOFMLEM_EINVAL, "em_correction_static: NULL argument");
    if (!ev->x1 || !ev->y1 || !ev->z1 || !ev->x2 || !ev->y2 || !ev->z2)
        return sfail(TOFMLEM_EINVAL, "em_correction_static: NULL event array");
    const bool tof = tof_fwhm_ps > 0.0;
    if (!isfinite(tof_fwhm_ps) || tof_fwhm_ps < 0.0) return sfail(TOFMLEM_EINVAL, "em_correction_static: bad tof_fwhm_ps");
    if (tof && !ev->dt) return sfail(TOFMLEM_EINVAL, "em_correction_static: a TOF pass needs dt");
    if (tof && !(trunc_sigmas > 0.0 && isfinite(trunc_sigmas)))
        return sfail(TOFMLEM_EINVAL, "em_correction_static: trunc_sigmas must be > 0");
    if (grid->nx < 1 || grid->ny < 1 || grid->nz < 1 || !(grid->vx > 0.f) || !(grid->vy > 0.f) || !(grid->vz > 0.f) ||
        (int64_t)grid->nx * grid->ny * grid->nz >= (1ll << 31))
        return sfail(TOFMLEM_EINVAL, "em_correction_static: bad grid");
    if (n > 0xFFFFFFFFull) return sfail(TOFMLEM_EINVAL, "em_correction_static: more than 2^32 - 1 events");
    if (queues_per_sm < 0 || queues_per_sm > 8) return sfail(TOFMLEM_EINVAL, "em_correction_static: queues_per_sm in 0..8");
    if (n == 0) return TOFMLEM_OK;

    // once per device, with that device current: the device address of the scratch array and the SM count
    int dev = 0;
    cudaError_t ce = cudaGetDevice(&dev);
    if (ce != cudaSuccess) return sfail(TOFMLEM_ECUDA, cudaGetErrorString(ce));
    if (dev < 0 || dev >= kMaxDevices) return sfail(TOFMLEM_EUNSUPPORTED, "em_correction_static: device ordinal >= 64");
    unsigned *queues = nullptr;
    int n_sm = 0;
    {
        std::lock_guard<std::mutex> lock(g_mutex);
        if (!g_queue_ptr[dev]) {
            unsigned *ptr = nullptr;
            ce = cudaGetSymbolAddress((void **)&ptr, g_static_queues);
            if (ce != cudaSuccess || !ptr) {
                cudaGetLastError();
                return sfail(TOFMLEM_ECUDA, std::string("em_correction_static: cudaGetSymbolAddress: ") +
                                                cudaGetErrorString(ce));
            }
            int sm = 0;
            ce = cudaDeviceGetAttribute(&sm, cudaDevAttrMultiProcessorCount, dev);
            if (ce != cudaSuccess || sm < 1) return sfail(TOFMLEM_ECUDA, "em_correction_static: no SM count");
            g_n_sm[dev] = sm;
            g_queue_ptr[dev] = ptr;
        }
        queues = g_queue_ptr[dev];
        n_sm = g_n_sm[dev];
    }

    ProjParams p;
    p.n[0] = grid->nx; p.n[1] = grid->ny; p.n[2] = grid->nz;
    p.v[0] = grid->vx; p.v[1] = grid->vy; p.v[2] = grid->vz;
    p.o[0] = grid->ox; p.o[1] = grid->oy; p.o[2] = grid->oz;
    for (int a = 0; a < 3; ++a) {
        p.iv[a] = 1.0 / p.v[a];
        p.h[a] = p.o[a] + p.n[a] * p.v[a];
    }
    p.half_window = 0.0;
    p.gauss_a = 0.0f;
    p.gauss_norm = 1.0f;
    if (tof) {
        const double sigma = kCmmPerPs * tof_fwhm_ps / (2.0 * 2.0 * sqrt(2.0 * log(2.0)));
        p.half_window = trunc_sigmas * sigma;
        p.gauss_a = (float)(-1.4426950408889634 / (2.0 * sigma * sigma));
        p.gauss_norm = (float)(1.0 / (sigma * sqrt(2.0 * M_PI)));
    }
    p.stride = 1;
    p.variant = 0;
    p.cache_share = 0;
    p.brick = 0;
    p.n_sm = n_sm;

    // queues per SM: as the context path chooses them (short windows spread the warps of an SM over several segments)
    unsigned segs = (unsigned)queues_per_sm;
    if (segs == 0) {
        const double reach = 2.0 * p.half_window * sqrt(p.iv[0] * p.iv[0] + p.iv[1] * p.iv[1] + p.iv[2] * p.iv[2]);
        segs = !tof || reach > 80.0 ? 1u : (reach > 30.0 ? 3u : 4u);
    }
    if ((uint64_t)n_sm * segs > kStaticQueues)
        return sfail(TOFMLEM_EINVAL, "em_correction_static: " + std::to_string(n_sm) + " SMs x " + std::to_string(segs) +
                                         " queues per SM exceed the static scratch of " +
                                         std::to_string(kStaticQueues) + " work queues (TOFMLEM_STATIC_MAX_QUEUES)");

    const int64_t nvox = (int64_t)grid->nx * grid->ny * grid->nz;
    const bool vec = (nvox & 3) == 0 && (reinterpret_cast<uintptr_t>(d_corr) & 15) == 0;
    const EventPtrs e{ev->x1, ev->y1, ev->z1, ev->x2, ev->y2, ev->z2, tof ? ev->dt : nullptr};
    cudaStream_t s = (cudaStream_t)cuda_stream;
    if (tof)
        ce = vec ? launch_static<true, true>(p, e, n, d_image, d_corr, queues, n_sm, segs, s)
                 : launch_static<true, false>(p, e, n, d_image, d_corr, queues, n_sm, segs, s);
    else
        ce = vec ? launch_static<false, true>(p, e, n, d_image, d_corr, queues, n_sm, segs, s)
                 : launch_static<false, false>(p, e, n, d_image, d_corr, queues, n_sm, segs, s);
    if (ce != cudaSuccess) return sfail(TOFMLEM_ECUDA, std::string("em_correction_static: ") + cudaGetErrorString(ce));
    return TOFMLEM_OK;
}
