// probe.cu -- micro-benchmarks that MEASURE the roofline denominators of the projector on this GPU:
// float32 reductions (RED.ADD.F32) and 4-byte gathers against an L2-resident array, with warp lanes
// hitting (a) unrelated random voxels, (b) 32 consecutive voxels of a random row.  bench.py runs them
// live beside the timed kernel (BASELINE.json north_star: "achieved fraction of the atomic- and
// L2-bandwidth roofline", measured, not assumed).
#include "internal.cuh"

namespace tofmlem {

__device__ __forceinline__ uint32_t mix32(uint32_t x) {
    x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
    return x;
}

// kind: 0 random RED, 1 row-coalesced RED, 2 random gather, 3 row-coalesced gather,
//       4 random 8-byte vector RED (red.global.add.v2.f32), 5 random 16-byte vector RED (v4)
template <int KIND>
__global__ void __launch_bounds__(256) probe_kernel(float *buf, uint32_t n, int ops, float *sink) {
    const uint32_t tid = blockIdx.x * 256u + threadIdx.x;
    const uint32_t lane = threadIdx.x & 31u, warp = tid >> 5;
    float acc = 0.0f;
    constexpr bool kRow = KIND == 1 || KIND == 3;  // lanes of a warp on 32 consecutive elements of a random row
    uint32_t h = mix32((kRow ? warp : tid) * 2654435761u + 12345u);
#pragma unroll 4
    for (int i = 0; i < ops; ++i) {
        h = mix32(h + 0x9e3779b9u);
        uint32_t a;
        if (kRow)
            a = ((h % (n >> 5)) << 5) + lane;
        else
            a = h % n;
        if (KIND < 2)
            atomicAdd(buf + a, 1.0f);  // result unused: RED.E.ADD.F32
        else if (KIND == 4)
            asm volatile("red.global.add.v2.f32 [%0], {%1, %1};" ::"l"(buf + (a & ~1u)), "f"(1.0f) : "memory");
        else if (KIND == 5)
            asm volatile("red.global.add.v4.f32 [%0], {%1, %1, %1, %1};" ::"l"(buf + (a & ~3u)), "f"(1.0f) : "memory");
        else
            acc += __ldg(buf + a);
    }
    if ((KIND == 2 || KIND == 3) && acc == 123.456f) *sink = acc;
}

// kind 6 / 7: random 32-bit integer adds (ATOMS.ADD, what tile.cu accumulates with) / random 4-byte loads (LDS) on a
// 72 KB shared-memory tile, three CTAs of 384 threads per SM as the tile pass runs: the denominators of its roofline.
template <int KIND>
__global__ void __launch_bounds__(384, 3) smem_probe_kernel(int ops, float *sink) {
    extern __shared__ unsigned tile[];
    constexpr unsigned kWords = 18432;
    for (unsigned i = threadIdx.x; i < kWords; i += 384) tile[i] = i;
    __syncthreads();
    uint32_t h = mix32((blockIdx.x * 384u + threadIdx.x) * 2654435761u + 777u);
    unsigned acc = 0;
#pragma unroll 4
    for (int i = 0; i < ops; ++i) {
        h = mix32(h + 0x9e3779b9u);
        const unsigned a = h % kWords;
        if (KIND == 6) atomicAdd(&tile[a], 1u);
        else acc += tile[a];
    }
    if (KIND == 7 && acc == 0x12345678u) *sink = 1.0f;
}

int run_probe(int kind, float *d_buf, uint64_t n_elems, uint64_t n_ops, float *ms, cudaStream_t s) {
    if (n_elems < 64 || n_elems > 0xFFFFFFFFull) return -1;
    const bool smem = kind == 6 || kind == 7;
    int n_sm = 148;
    {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    }
    const int blocks = smem ? n_sm * 3 : n_sm * 16;
    const uint64_t threads = (uint64_t)blocks * (smem ? 384 : 256);
    if (smem) {
        cudaFuncSetAttribute(smem_probe_kernel<6>, cudaFuncAttributeMaxDynamicSharedMemorySize, 18432 * 4);
        cudaFuncSetAttribute(smem_probe_kernel<7>, cudaFuncAttributeMaxDynamicSharedMemorySize, 18432 * 4);
    }
    const int ops = (int)((n_ops + threads - 1) / threads);
    float *sink = d_buf;  // never written in practice
    cudaEvent_t a, b;
    cudaEventCreate(&a);
    cudaEventCreate(&b);
    for (int rep = 0; rep < 2; ++rep) {  // first pass warms L2
        cudaEventRecord(a, s);
        switch (kind) {
            case 0: probe_kernel<0><<<blocks, 256, 0, s>>>(d_buf, (uint32_t)n_elems, ops, sink); break;
            case 1: probe_kernel<1><<<blocks, 256, 0, s>>>(d_buf, (uint32_t)n_elems, ops, sink); break;
            case 2: probe_kernel<2><<<blocks, 256, 0, s>>>(d_buf, (uint32_t)n_elems, ops, sink); break;
            case 3: probe_kernel<3><<<blocks, 256, 0, s>>>(d_buf, (uint32_t)n_elems, ops, sink); break;
            case 4: probe_kernel<4><<<blocks, 256, 0, s>>>(d_buf, (uint32_t)n_elems, ops, sink); break;
            case 5: probe_kernel<5><<<blocks, 256, 0, s>>>(d_buf, (uint32_t)n_elems, ops, sink); break;
            case 6: smem_probe_kernel<6><<<blocks, 384, 18432 * 4, s>>>(ops, sink); break;
            case 7: smem_probe_kernel<7><<<blocks, 384, 18432 * 4, s>>>(ops, sink); break;
            default: cudaEventDestroy(a); cudaEventDestroy(b); return -1;
        }
        cudaEventRecord(b, s);
    }
    cudaError_t e = cudaEventSynchronize(b);
    if (e == cudaSuccess) e = cudaEventElapsedTime(ms, a, b);
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    if (e != cudaSuccess) return -3;
    // report per-op time basis: caller divides ops*threads by ms
    *ms = *ms * (float)((double)n_ops / ((double)ops * (double)threads));
    return 0;
}

}  // namespace tofmlem
