// Exact median selection in registers (true, non-separable k x k median: PAPER.md:23,64).
#pragma once
#include "common.cuh"

namespace lac {

// Forgetful selection: keep a working set of N/2+2 values, repeatedly drop its minimum and its
// maximum (neither can be the median of what is left) and take in one unseen value, until three
// values remain.  All indices are compile-time constants after unrolling, so v[] lives in
// registers.  Exact for any input, ties included.
template <int N>
__device__ __forceinline__ float median_forgetful(float (&v)[N]) {
    constexpr int M = N / 2, S0 = M + 2;
#pragma unroll
    for (int i = 0; i <= N - S0; ++i) {
        const int lo = i, hi = S0 - 1, s = hi - lo + 1;
#pragma unroll
        for (int j = 0; j < s / 2; ++j) ce(v[lo + j], v[hi - j]);
#pragma unroll
        for (int j = 1; j < (s + 1) / 2; ++j) ce(v[lo], v[lo + j]);
#pragma unroll
        for (int j = 1; j < (s + 1) / 2; ++j) ce(v[hi - j], v[hi]);
        if (i < N - S0) v[hi] = v[S0 + i];
    }
    return v[N - S0 + 1];
}

// 3x3 median from three column-sorted triples is cheaper, but the plain 9-input version is kept
// as the building block shared by every tile shape.
__device__ __forceinline__ float median9(float (&v)[9]) { return median_forgetful<9>(v); }

}  // namespace lac
