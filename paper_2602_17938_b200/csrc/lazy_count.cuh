// Threshold test of S' = S - med5(S) by counting (see lazy.cuh for the argument): shared by the candidate
// evaluation (lazy.cuh) and the fused growth kernel (grow.cuh).
#pragma once
#include "common.cuh"

namespace lac {

__device__ __forceinline__ float4 ldg4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }

// #{25 taps v of S around pixel p : fsub(Sc, v) > thr} for thr = sigclip (c1) and siglow (c2).
// Interior pixels (window inside the frame): each window row is read as two 16-byte aligned vectors that
// cover it, the test is evaluated on all 8 values and the 5 of the window are selected by a shift.
__device__ __forceinline__ void count_sp_interior(const float* __restrict__ S, int p, int w, float sigclip,
                                                  float siglow, int& c1, int& c2) {
    const float sc = __ldg(S + p);
    c1 = 0;
    c2 = 0;
#pragma unroll
    for (int r = 0; r < 5; ++r) {
        const int base = p + (r - 2) * w - 2, b = base & ~3, sh = base - b;
        const float4 a0 = ldg4(S + b), a1 = ldg4(S + b + 4);
        const float e[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
        uint32_t m1 = 0, m2 = 0;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const float sp = __fsub_rn(sc, e[k]);
            m1 |= (uint32_t)(sp > sigclip) << k;
            m2 |= (uint32_t)(sp > siglow) << k;
        }
        c1 += __popc((m1 >> sh) & 31u);
        c2 += __popc((m2 >> sh) & 31u);
    }
}

// any pixel: clamped scalar taps (R3)
__device__ __forceinline__ void count_sp_clamped(const float* __restrict__ S, int y, int x, int h, int w,
                                                 float sigclip, float siglow, int& c1, int& c2) {
    const float sc = __ldg(S + (size_t)y * w + x);
    int xx[5];
#pragma unroll
    for (int d = 0; d < 5; ++d) xx[d] = clampi(x + d - 2, 0, w - 1);
    c1 = 0;
    c2 = 0;
#pragma unroll
    for (int dy = 0; dy < 5; ++dy) {
        const float* row = S + (size_t)clampi(y + dy - 2, 0, h - 1) * w;
#pragma unroll
        for (int dx = 0; dx < 5; ++dx) {
            const float sp = __fsub_rn(sc, __ldg(row + xx[dx]));
            c1 += sp > sigclip;
            c2 += sp > siglow;
        }
    }
}

__device__ __forceinline__ void count_sp(const float* __restrict__ S, int y, int x, int h, int w, float sigclip,
                                         float siglow, int& c1, int& c2) {
    if (y >= 2 && x >= 2 && x + 2 < w && y + 2 < h && (size_t)(y + 2) * w + x + 6 <= (size_t)h * w)
        count_sp_interior(S, y * w + x, w, sigclip, siglow, c1, c2);
    else
        count_sp_clamped(S, y, x, h, w, sigclip, siglow, c1, c2);
}

}  // namespace lac
