// Threshold test of S' = S - med5(S) by counting (see lazy.cuh for the argument): shared by the candidate
// evaluation (lazy.cuh) and the fused growth kernel (grow.cuh).
#pragma once
#include "common.cuh"

namespace lac {

// #{25 clamped taps v of S around (y, x) : fsub(Sc, v) > thr} for thr = sigclip (c1) and siglow (c2).
// Plain scalar taps: on B200 they beat covering each window row with aligned 16-byte vectors and selecting
// the taps by a shift (fewer bytes per lane and no select chains; measured in k_eval_candidates and
// k_grow_replace).
__device__ __forceinline__ void count_sp(const float* __restrict__ S, int y, int x, int h, int w, float sigclip,
                                         float siglow, int& c1, int& c2) {
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

}  // namespace lac
