// prepared.cuh -- ray records of a PLANNED event list and the exact-add voxel walk that runs on them (prepared.cu,
// tile.cu).  BASELINE.json north_star bullet 3: "a fused forward+backprojection kernel that recomputes or caches the
// weights" -- what is cached here is the ray set-up (the fp64 part of every event), once per data set.
//
// Why: the fused pass of projector.cu redoes the fp64 ray set-up of every event in every iteration (393 M fp64
// instructions per pass at cfg-3, a third of the instruction stream at 100 ps) and spends 27 (gather) / 46 (scatter)
// SASS instructions per voxel visit, with the integer/compare pipe 62 % busy (ncu r04).  tofmlem_plan_events
// computes, once, a 48-byte record per event; the per-iteration kernels only load it and walk.
//
// Record (three 16-byte arrays, SoA, in event order):
//   a = {t_start, t_end, t0[0], t0[1]}   b = {t0[2], td[0], td[1], td[2]}   c = {idx0, meta, counts, 0}
// Ray parameter: t = kappa * (s - s_c), s = distance from end point 1 (mm), s_c = TOF kernel centre (R22),
// kappa = sqrt(log2(e) / 2) / sigma, so that the un-normalised chord weight is  l * 2^(-mid^2)  with l and mid in t
// units (the constant factor kappa cancels in a_ej / fwd_e; forward values are rescaled once per event).
// Every field is a multiple of the quantum q = 2^-k, k chosen such that |t| <= 2^(24-k) over the window: then the
// walk's  t_axis += td_axis  is EXACT in float32 (no accumulated rounding, the walker and the set-up agree bit for bit
// on every crossing), and the grid-exit crossing t0 + nsteps * td computed by the set-up in fp64 is the very number the
// walker would reach -- t_end is clipped to it, so the voxel index cannot leave the grid and the loop needs no bounds
// test.  Cost: td carries a rounding of <= q/2 (2.7e-6 mm at 300 ps), i.e. the k-th crossing of an axis is displaced by
// <= k q/2 (<= 8e-5 mm over the 30 crossings of a 300 ps window at 3.75 mm, 2e-5 of a chord), far inside the 1e-4
// forward tolerance (tests/test_gpu_parity_full.py compares the planned forward values with the oracle).
//   t0[i]: first crossing of axis i after t_start (+inf when the ray is parallel to the axis), td[i]: crossing period.
//   Axis order: x, y, z for events of the direct pass; (a, f, s) = (dominant axis of the bin's class, fast, slow
//   lateral axis) for events that run on a shared-memory tile (meta bit kRecTile).
//   idx0: flat index (z*ny + y)*nx + x of the first voxel.  counts: voxel visits | 16-byte groups of the correction
//   image met << 16 (both walks are deterministic, so the statistics of a pass are sums of these).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tofmlem {

constexpr unsigned kRecValid = 1u;        // the window meets the grid
constexpr unsigned kRecTile = 2u;         // runs on the shared-memory tile of its bin (else: direct pass)
constexpr unsigned kRecAxisShift = 2;     // bits 2-3: dominant axis a of the bin's class (tile events)
constexpr unsigned kRecNeg0 = 1u << 4;    // axis 0 / 1 / 2 (in the record's axis order) runs towards lower indices
constexpr unsigned kRecNeg1 = 1u << 5;    //   (tile events: in the tile's mirrored coordinates)
constexpr unsigned kRecNeg2 = 1u << 6;
constexpr unsigned kRecOddX = 1u << 7;    // first voxel has odd ix / iy (brick layout of the correction image)
constexpr unsigned kRecOddY = 1u << 8;
constexpr unsigned kRecTiny = 1u << 9;    // direct records only: the window is shorter than 2^15 quanta -- its two ends
                                          // carry a rounding of one quantum each, more than 1e-4 of such a sliver, so the
                                          // kernels walk this event from the raw fields with the fp64 set-up of walk.cuh
constexpr unsigned kRecPlaneShift = 9;    // bits 9-15: plane of the first voxel in the tile (tile events)
constexpr unsigned kRecLiShift = 16;      // bits 16-31: tile-local word index of the first voxel (tile events)

struct RecPtrs {
    float4 *a, *b;
    uint4 *c;
};

__device__ __forceinline__ float min3f(float a, float b, float c) {
    float d;
    asm("min.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c));  // FMNMX3 (sm_100)
    return d;
}

__device__ __forceinline__ float ex2_neg_sq(float mid) {
    float y;
    const float q = mid * -mid;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(q));
    return y;
}

// if (tx <= tn) { tx += dx; idx += ix; }   as two predicated instructions (ptxas otherwise builds SEL + IADD3 chains)
__device__ __forceinline__ void advance_axis(float &tx, int &idx, float tn, float dx, int ix) {
    asm("{\n .reg .pred p;\n setp.le.f32 p, %0, %2;\n @p add.f32 %0, %0, %3;\n @p add.s32 %1, %1, %4;\n}"
        : "+f"(tx), "+r"(idx)
        : "f"(tn), "f"(dx), "r"(ix));
}

// un-normalised weight of the chord [t, tn] (t units): length x 2^(-midpoint^2)
__device__ __forceinline__ float chord_weight(float t, float tn) {
    const float l = tn - t;
    const float mid = fmaf(-0.5f, l, tn);
    return l * ex2_neg_sq(mid);
}

}  // namespace tofmlem
