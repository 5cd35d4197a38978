// Issue-rate probe for the "alu" roofline: the medians are fp32 min/max selection networks, so
// the peak they are rated against is the rate at which an SM issues FMNMX / FMNMX3.  bench.py measures it in the same
// run through lacosmic_probe_minmax_rate and prints it beside the figure derived from the unit counts.
// Register-only kernel: 8 dependent chains per thread (ILP 8), alternating min and max stages, written as volatile
// inline PTX so that nothing is folded away at compile time (cuobjdump: 128 FMNMX / FMNMX3 in the loop body).
#pragma once
#include "common.cuh"

namespace lac {

constexpr int PROBE_STAGES_PER_ITER = 16;   // 8 min + 8 max stages per loop iteration
constexpr int PROBE_THREADS = 1024;
constexpr int PROBE_CTAS_PER_SM = 2;

// volatile: the compiler may neither fold nor merge these (min/max lattices simplify aggressively otherwise)
__device__ __forceinline__ float vmin2(float a, float b) { float r; asm volatile("min.f32 %0, %1, %2;" : "=f"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ float vmax2(float a, float b) { float r; asm volatile("max.f32 %0, %1, %2;" : "=f"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ float vmin3(float a, float b, float c) { float r; asm volatile("min.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c)); return r; }
__device__ __forceinline__ float vmax3(float a, float b, float c) { float r; asm volatile("max.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c)); return r; }

template <int KIND>   // 0: two-input FMNMX, 1: three-input FMNMX3
__global__ void __launch_bounds__(PROBE_THREADS, PROBE_CTAS_PER_SM)
k_probe_minmax(float* __restrict__ sink, int iters, float seed) {
    float a[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) a[k] = seed * (float)(threadIdx.x * 8 + k + 1) + (float)((threadIdx.x * 7 + k * 13) & 31);
    const float lo = seed, hi = seed * 3.0f;
#pragma unroll 1
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int s = 0; s < PROBE_STAGES_PER_ITER / 2; ++s) {
#pragma unroll
            for (int k = 0; k < 8; ++k) a[k] = KIND == 0 ? vmin2(a[k], hi) : vmin3(a[k], hi, a[(k + 1) & 7]);
#pragma unroll
            for (int k = 0; k < 8; ++k) a[k] = KIND == 0 ? vmax2(a[k], lo) : vmax3(a[k], lo, a[(k + 3) & 7]);
        }
    }
    float r = 0.0f;
#pragma unroll
    for (int k = 0; k < 8; ++k) r += a[k];
    if (r == 12345.678f) sink[0] = r;   // keeps the chains alive; practically never true
}

}  // namespace lac
