// R26: the separable median -- the approximation PAPER.md:29,37 argues AGAINST -- as a COMPARISON
// path only (lacosmic_run_sepmed_compare, lacosmic_sepmedfilt).  The product path never runs these kernels.  Plain
// one-thread-per-pixel passes: the point of this path is the difference in the masks, not its speed.
#pragma once
#include "common.cuh"

namespace lac {

// middle element of K values (K in {3, 5, 7}): odd-even transposition sort
template <int K>
__device__ __forceinline__ float mid_of(float (&v)[K]) {
#pragma unroll
    for (int r = 0; r < K; ++r)
#pragma unroll
        for (int j = r & 1; j + 1 < K; j += 2) ce(v[j], v[j + 1]);
    return v[K / 2];
}

// one 1-D pass of the separable median: ROW: out[y][x] = mid{in<y, x+d>}, else out[y][x] = mid{in<y+d, x>}, |d| <= K/2
template <int K, bool ROW>
__global__ void __launch_bounds__(256)
k_sepmed_pass(const float* __restrict__ in, float* __restrict__ out, int h, int w) {
    const size_t i = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (i >= (size_t)h * w) return;
    const int y = (int)(i / (size_t)w), x = (int)(i - (size_t)y * w);
    float v[K];
#pragma unroll
    for (int d = 0; d < K; ++d) {
        const int yy = ROW ? y : clampi(y + d - K / 2, 0, h - 1), xx = ROW ? clampi(x + d - K / 2, 0, w - 1) : x;
        v[d] = __ldg(in + (size_t)yy * w + xx);
    }
    out[i] = mid_of<K>(v);
}

struct SepGateArgs {
    const float *work, *S, *mS, *m3, *m7;
    uint32_t *G1, *G2, *M1;
    float *dbgSp, *dbgF;
    int h, w, wpr;
    float sigclip, siglow, objlim, satlevel;
};

// a warp per 32-pixel word.  STAGE 0: G1, G2 from S' = S - mS (O3, O5); STAGE 1: M1 = G1 & (L+/F > objlim) with
// F = max(m3 - m7, 0.01) (O4, O5), L+ recomputed from work (O1).
template <int STAGE>
__global__ void __launch_bounds__(256)
k_sep_gates(SepGateArgs a) {
    const int lane = threadIdx.x & 31;
    const size_t word = (size_t)blockIdx.x * 8 + (threadIdx.x >> 5);
    if (word >= (size_t)a.h * a.wpr) return;                    // warp-uniform
    const int y = (int)(word / (size_t)a.wpr), wx = (int)(word - (size_t)y * a.wpr);
    const int x = wx * 32 + lane, h = a.h, w = a.w;
    const bool in = x < w;
    const size_t p = (size_t)y * w + min(x, w - 1);
    if (STAGE == 0) {
        const float sp = __fsub_rn(a.S[p], a.mS[p]);
        const bool ok = in && (a.work[p] < a.satlevel);
        const uint32_t g1 = __ballot_sync(0xffffffffu, ok && sp > a.sigclip);
        const uint32_t g2 = __ballot_sync(0xffffffffu, ok && sp > a.siglow);
        if (in && a.dbgSp) a.dbgSp[p] = sp;
        if (lane == 0) {
            a.G1[word] = g1;
            a.G2[word] = g2;
        }
    } else {
        const float d = __fsub_rn(a.m3[p], a.m7[p]);
        const float f = d > 0.01f ? d : 0.01f;
        const int xc = min(x, w - 1);
        const float* row = a.work + (size_t)y * w;
        const float lp = lplus_px(row[xc], a.work[(size_t)max(y - 1, 0) * w + xc], a.work[(size_t)min(y + 1, h - 1) * w + xc],
                                  row[max(xc - 1, 0)], row[min(xc + 1, w - 1)]);
        const bool g1 = in && ((a.G1[word] >> lane) & 1u);
        const uint32_t m1 = __ballot_sync(0xffffffffu, g1 && (__fdiv_rn(lp, f) > a.objlim));
        if (in && a.dbgF) a.dbgF[p] = f;
        if (lane == 0) a.M1[word] = m1;
    }
}

}  // namespace lac
