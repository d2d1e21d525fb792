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
#include "walk.cuh"

namespace tofmlem {

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
// segments, `segs_per_sm` (1, 3 or 4, see launch_em) per SM; every warp takes 32-event chunks from the queue of the SM it
// runs on (%smid), so the warps resident on an SM (5 CTAs of 256 threads) work on neighbouring events and share that
// SM's L1 for their image gathers (the co-resident CTAs of the grid-order form come from unrelated places and thrash
// it), while different SMs reduce into different
// parts of the volume.  A warp whose segment is exhausted moves on to other segments (work stealing; the invalid
// events sorted to the end of the list make the last segments empty).  Measured at cfg-3: 30.2 -> 25.2 ms.
template <bool TOF, bool VEC, bool BRICK>
__global__ void __launch_bounds__(kBlock, 5) em_persistent_kernel(ProjParams P, EventPtrs ev, uint64_t n,
                                                               const float *__restrict__ evw,
                                                               const float *__restrict__ image,
                                                               float *__restrict__ corr, DeviceStats *stats,
                                                               unsigned *queues, unsigned nseg, unsigned per_seg,
                                                               unsigned segs_per_sm,
                                                               const uint2 *__restrict__ chunks, unsigned n_chunks,
                                                               unsigned gather) {
    unsigned smid;
    asm("mov.u32 %0, %%smid;" : "=r"(smid));
    const unsigned lane = threadIdx.x & 31u;
    // nseg = segs_per_sm * base segments: the warps of an SM start on segs_per_sm of them (base apart in the list)
    const unsigned base = nseg / segs_per_sm;
    unsigned seg = smid % base + base * ((threadIdx.x >> 5) % segs_per_sm), tries = 0, nv = 0, vis = 0, nr = 0;
    while (true) {
        unsigned c = per_seg;
        if (lane == 0 && *(volatile unsigned *)(queues + seg * kQueueStride) < per_seg)
            c = atomicAdd(queues + seg * kQueueStride, 1u);
        c = __shfl_sync(0xffffffffu, c, 0);
        if (c >= per_seg) {
            if (++tries >= nseg) break;
            seg = (seg + 61u) % nseg;  // 61 is prime: visits every segment for any nseg not a multiple of 61
            continue;
        }
        int visits, reds;
        bool valid;
        const uint64_t wc = (uint64_t)seg * per_seg + c;  // index of the warp's 32-event piece
        uint64_t e = wc * 32u + lane;
        if (chunks && gather) {  // a list of single events: 32 of them per warp, a lane each
            const uint64_t k = wc * 32u + lane;
            e = k < n_chunks ? (uint64_t)__ldg(chunks + k).x : n;
        } else if (chunks) {  // the pieces come from a list (the events the tile-mode pass leaves over)
            e = n;
            if (wc < n_chunks) {
                const uint2 ch = __ldg(chunks + wc);
                if (lane < ch.y) e = (uint64_t)ch.x + lane;
            }
        }
        em_event<TOF, VEC, BRICK>(P, ev, e, n, evw, image, corr, visits, valid, reds);
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
        if (lane == 0 && *(volatile unsigned *)(queues + seg * kQueueStride) < per_seg)
            c = atomicAdd(queues + seg * kQueueStride, 1u);
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
    const size_t smem = sizeof(unsigned long long) << kCacheLog2;
    int dev = 0, n_sm = p.n_sm;
    if (n_sm < 1) {
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    }
    cudaFuncSetAttribute(em_cached_kernel<TOF, BRICK>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    unsigned nseg = (unsigned)n_sm;
    if (nseg > (unsigned)kMaxQueues) nseg = kMaxQueues;
    if (nseg % 61u == 0) nseg -= 1;
    const uint64_t wchunks = (n + 31) / 32;
    const unsigned per_seg = (unsigned)((wchunks + nseg - 1) / nseg);
    cudaMemsetAsync(queues, 0, (size_t)nseg * kQueueStride * sizeof(unsigned), s);
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
                      float *corr, DeviceStats *stats, unsigned *queues, cudaStream_t s, const uint2 *chunks = nullptr,
                      uint32_t n_chunks = 0, bool gather = false) {
    if ((p.variant != 1 || chunks) && queues) {
        // SM count of the context's device (queried in tofmlem_create) and resident CTAs per SM of THIS instantiation on
        // the current device (a host-side table look-up in the runtime: asked on every launch, no cached state)
        int per_sm = 0, n_sm = p.n_sm;
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, em_persistent_kernel<TOF, VEC, BRICK>, kBlock, 0);
        if (n_sm < 1) {
            int dev = 0;
            cudaGetDevice(&dev);
            cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
        }
        // Short windows: the warps of an SM spread over several list segments (measured at 146 M events: 300 ps, 1 / 2 /
        // 3 / 4 / 8 segments per SM -> 21.47 / 21.04 / 20.75 / 22.25 / 23.54 ms; 100 ps, 1 / 2 / 3 / 4 -> 11.35 / 9.57 /
        // 9.44 / 9.32 ms).  Long walks (600 ps: 43.3 -> 45.1 ms, non-TOF: 203 -> 218 ms with 2) keep one.
        const double reach = 2.0 * p.half_window * sqrt(p.iv[0] * p.iv[0] + p.iv[1] * p.iv[1] + p.iv[2] * p.iv[2]);
        const unsigned kSegsPerSm = !TOF || reach > 80.0 ? 1u : (reach > 30.0 ? 3u : 4u);  // reach = largest visit count
        unsigned segs = kSegsPerSm;
        unsigned nseg = (unsigned)n_sm * segs;
        unsigned grid = (unsigned)n_sm * (unsigned)(per_sm > 0 ? per_sm : 1);
        const uint64_t wchunks = chunks ? (gather ? ((uint64_t)n_chunks + 31) / 32 : (uint64_t)n_chunks) : (n + 31) / 32;
        if (wchunks < 8ull * nseg) {
            // a short list (the sliver windows of a planned list: a few thousand one-event pieces): a few queues and CTAs
            // only -- a full-size launch spends 0.26 ms polling 444 empty queues
            segs = 1;
            nseg = (unsigned)((wchunks + 7) / 8);
            if (nseg > (unsigned)n_sm) nseg = (unsigned)n_sm;
            if (nseg < 1) nseg = 1;
            const unsigned want = (unsigned)((wchunks * 32 + kBlock - 1) / kBlock);
            if (want < grid) grid = want < 1 ? 1 : want;
        }
        if (nseg > (unsigned)kMaxQueues) nseg = (unsigned)kMaxQueues / segs * segs;
        if (nseg > segs && nseg % 61u == 0) nseg -= segs;  // the stealing stride 61 must not divide the number of segments
        const unsigned per_seg = (unsigned)((wchunks + nseg - 1) / nseg);
        cudaMemsetAsync(queues, 0, (size_t)nseg * kQueueStride * sizeof(unsigned), s);
        em_persistent_kernel<TOF, VEC, BRICK><<<grid, kBlock, 0, s>>>(
            p, ev, n, evw, image, corr, stats, queues, nseg, per_seg, segs, chunks, n_chunks, gather ? 1u : 0u);
    } else {
        em_correction_kernel<TOF, VEC, BRICK><<<grid_for(n, p.stride), kBlock, 0, s>>>(p, ev, n, evw, image, corr, stats);
    }
}

void launch_em_correction(const ProjParams &p, bool tof, const EventPtrs &ev, uint64_t n, const float *evw,
                          const float *image, float *corr, bool vec_ok, DeviceStats *stats, unsigned *queues,
                          cudaStream_t s) {
    launch_em_correction_chunks(p, tof, ev, n, nullptr, 0, evw, image, corr, vec_ok, stats, queues, s, false);
}

void launch_em_correction_chunks(const ProjParams &p, bool tof, const EventPtrs &ev, uint64_t n, const uint2 *chunks,
                                 uint32_t n_chunks, const float *evw, const float *image, float *corr, bool vec_ok,
                                 DeviceStats *stats, unsigned *queues, cudaStream_t s, bool gather) {
    if (n == 0 || (chunks && n_chunks == 0)) return;
    if (p.variant == 2 && queues && vec_ok && !chunks) {
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
            launch_em<true, true, true>(p, ev, n, evw, image, corr, stats, queues, s, chunks, n_chunks, gather);
        else
            launch_em<false, true, true>(p, ev, n, evw, image, corr, stats, queues, s, chunks, n_chunks, gather);
        return;
    }
    if (tof) {
        if (vec_ok)
            launch_em<true, true, false>(p, ev, n, evw, image, corr, stats, queues, s, chunks, n_chunks, gather);
        else
            launch_em<true, false, false>(p, ev, n, evw, image, corr, stats, queues, s, chunks, n_chunks, gather);
    } else {
        if (vec_ok)
            launch_em<false, true, false>(p, ev, n, evw, image, corr, stats, queues, s, chunks, n_chunks, gather);
        else
            launch_em<false, false, false>(p, ev, n, evw, image, corr, stats, queues, s, chunks, n_chunks, gather);
    }
}

}  // namespace tofmlem
