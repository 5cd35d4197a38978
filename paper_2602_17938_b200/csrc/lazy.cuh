// Exact lazy evaluation of steps (3b)-(6) over compacted pixel lists ("lazy path").
//
// The dense reference kernels (kernels.cuh) evaluate med5(S), med3, med7 at every pixel.  The results
// of the iteration only depend on them through threshold tests, and a threshold test of a median needs
// no selection: for a monotone predicate P and an odd multiset X with median m,
//     P non-decreasing:  P(m)  <=>  #{x in X : P(x)} >= (|X|+1)/2
//     P non-increasing:  P(m)  <=>  #{x in X : P(x)} >= (|X|+1)/2
// (the elements satisfying P form an upper / lower set of the sorted order, which contains the middle
// element iff it has at least (|X|+1)/2 members).  Every fp32 operation of O3-O5 is monotone under
// round-to-nearest, so with the SAME operations as the dense path:
//   G(thr)  = S' > thr,  S' = fsub(S, med5(S)):         Q(v) = fsub(S, v) > thr          non-increasing in v
//             => G(thr) <=> #{25 taps v of S : Q(v)} >= 13
//   M1 test = fdiv(Lp, max(fsub(m3, med7(m3 plane)), 0.01)) > objlim:
//             P(v) = fdiv(Lp, max(fsub(m3, v), 0.01)) > objlim                            non-decreasing in v
//             => test <=> #{49 taps u of the m3 plane : P(u)} >= 25, and each u = med3x3(work) at the
//                tap, so P(u) <=> #{9 taps v of work : P(v)} >= 5.
// Since S >= +0 everywhere (Lp >= 0, N > 0), med5(S) >= 0 and S' <= S: S' > thr implies S > thr, so the
// tests are only evaluated on the pixels the dense k_noise_S pass flags in A1 = ok & (S > sigclip) and
// A2 = ok & (S > siglow).  Masks, counts and cleaned frames are identical to the dense path.
#pragma once
#include "common.cuh"

namespace lac {

// 3x3 dilation of one word of a bit-plane (outside the frame = 0), neighbours loaded directly
__device__ __forceinline__ uint32_t dil3_word(const uint32_t* __restrict__ in, int y, int wx, int h, int wpr) {
    uint32_t vl = 0, vc = 0, vr = 0;
    for (int yy = max(y - 1, 0); yy <= min(y + 1, h - 1); ++yy) {
        const uint32_t* row = in + (size_t)yy * wpr;
        vc |= row[wx];
        if (wx > 0) vl |= row[wx - 1];
        if (wx + 1 < wpr) vr |= row[wx + 1];
    }
    return vc | (vc << 1) | (vc >> 1) | (vl >> 31) | (vr << 31);
}

// list <- pixels of A1; zero the words of G1, G2, M1 (they are filled by atomicOr afterwards)
__global__ void __launch_bounds__(256)
k_list_candidates(const uint32_t* __restrict__ A1, uint32_t* __restrict__ G1, uint32_t* __restrict__ G2,
                  uint32_t* __restrict__ M1, int* __restrict__ list, int* __restrict__ nlist, int h, int w,
                  int wpr, const int* prev_count) {
    if (prev_count && *prev_count == 0) return;
    const int wx = blockIdx.x * 32 + (threadIdx.x & 31);
    const int y = blockIdx.y * 8 + (threadIdx.x >> 5);
    uint32_t bits = 0;
    if (wx < wpr && y < h) {
        size_t q = (size_t)y * wpr + wx;
        bits = A1[q];
        G1[q] = 0;
        G2[q] = 0;
        M1[q] = 0;
    }
    block_append(bits, y * w + wx * 32, list, nlist);
}

// list <- pixels of dil3(M2) & A2 & ~A1: the only pixels where G2 is still unknown and needed by O6
__global__ void __launch_bounds__(256)
k_list_neighbours(const uint32_t* __restrict__ M2, const uint32_t* __restrict__ A1,
                  const uint32_t* __restrict__ A2, int* __restrict__ list, int* __restrict__ nlist, int h,
                  int w, int wpr, const int* prev_count) {
    if (prev_count && *prev_count == 0) return;
    const int wx = blockIdx.x * 32 + (threadIdx.x & 31);
    const int y = blockIdx.y * 8 + (threadIdx.x >> 5);
    uint32_t bits = 0;
    if (wx < wpr && y < h) {
        size_t q = (size_t)y * wpr + wx;
        const uint32_t cand = A2[q] & ~A1[q];
        if (cand) bits = dil3_word(M2, y, wx, h, wpr) & cand;
    }
    block_append(bits, y * w + wx * 32, list, nlist);
}

// exact median of 9 (19 compare-exchanges)
__device__ __forceinline__ float med9(float a0, float a1, float a2, float a3, float a4, float a5, float a6,
                                      float a7, float a8) {
    ce(a1, a2); ce(a4, a5); ce(a7, a8);
    ce(a0, a1); ce(a3, a4); ce(a6, a7);
    ce(a1, a2); ce(a4, a5); ce(a7, a8);
    a3 = fmaxf(a0, a3); a5 = fminf(a5, a8);
    ce(a4, a7);
    a6 = fmaxf(a3, a6); a4 = fmaxf(a1, a4); a2 = fminf(a2, a5);
    a4 = fminf(a4, a7);
    ce(a4, a2);
    a4 = fmaxf(a6, a4);
    return fminf(a4, a2);
}

// #{25 clamped taps v of S around (y, x) : fsub(Sc, v) > thr} for thr = sigclip (c1) and siglow (c2)
__device__ __forceinline__ void count_sp(const float* __restrict__ S, int y, int x, int h, int w,
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

struct CandArgs {
    const float* S;
    const float* work;
    uint32_t *G1, *G2, *M1;
    int h, w, wpr;
    float sigclip, siglow, objlim;
};

// One thread per pixel of A1: G1, G2 by counting; where G1 holds, the fine-structure test by counting.
__global__ void __launch_bounds__(128)
k_eval_candidates(CandArgs a, const int* __restrict__ list, const int* __restrict__ nlist,
                  const int* prev_count) {
    if (prev_count && *prev_count == 0) return;
    const int n = *nlist;
    const int h = a.h, w = a.w;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const int p = list[i];
        const int y = p / w, x = p - y * w;
        int c1, c2;
        count_sp(a.S, y, x, h, w, a.sigclip, a.siglow, c1, c2);
        const uint32_t bit = 1u << (x & 31);
        const size_t q = (size_t)y * a.wpr + (x >> 5);
        if (c2 >= 13) atomicOr(a.G2 + q, bit);
        if (c1 < 13) continue;
        atomicOr(a.G1 + q, bit);
        // fine-structure test.  Virtual 9x9 window V[r][c] = work<y-4+r, x-4+c>; the m3-plane tap (dy, dx)
        // of the 7x7 window is med3x3 centred on the virtual position (cy(dy), cx(dx)) with
        // cy(dy) = clamp(y+dy) - y (R4: the STORED m3 plane is replicated), whose own taps are
        // V[cy+4+-1][cx+4+-1] (R3).
        int xx[9];
#pragma unroll
        for (int c = 0; c < 9; ++c) xx[c] = clampi(x + c - 4, 0, w - 1);
        float ctr[3][3];
#pragma unroll
        for (int r = 0; r < 3; ++r)
#pragma unroll
            for (int c = 0; c < 3; ++c)
                ctr[r][c] = __ldg(a.work + (size_t)clampi(y + r - 1, 0, h - 1) * w + xx[3 + c]);
        const float lp = lplus_px(ctr[1][1], ctr[0][1], ctr[2][1], ctr[1][0], ctr[1][2]);
        const float m3c = med9(ctr[0][0], ctr[0][1], ctr[0][2], ctr[1][0], ctr[1][1], ctr[1][2], ctr[2][0],
                               ctr[2][1], ctr[2][2]);
        uint32_t rows[9];   // bit c of rows[r] = P(V[r][c])
#pragma unroll
        for (int r = 0; r < 9; ++r) {
            const float* row = a.work + (size_t)clampi(y + r - 4, 0, h - 1) * w;
            uint32_t b = 0;
#pragma unroll
            for (int c = 0; c < 9; ++c) {
                const float d = __fsub_rn(m3c, __ldg(row + xx[c]));
                const float f = d > 0.01f ? d : 0.01f;
                b |= (uint32_t)(__fdiv_rn(lp, f) > a.objlim) << c;
            }
            rows[r] = b;
        }
        // ge5[ry] bit rx = (#P in the 3x3 block rows ry..ry+2, columns rx..rx+2) >= 5, bit-sliced adders
        uint32_t ge5[7];
#pragma unroll
        for (int ry = 0; ry < 7; ++ry) {
            const uint32_t b0 = rows[ry], b1 = rows[ry + 1], b2 = rows[ry + 2];
            const uint32_t s0 = b0 ^ b1 ^ b2, s1 = (b0 & b1) | (b2 & (b0 | b1));      // column sums 0..3
            const uint32_t l = s0 ^ (s0 >> 1) ^ (s0 >> 2);
            const uint32_t cl = (s0 & (s0 >> 1)) | ((s0 >> 2) & (s0 | (s0 >> 1)));
            const uint32_t hx = s1 ^ (s1 >> 1) ^ (s1 >> 2);
            const uint32_t ch = (s1 & (s1 >> 1)) | ((s1 >> 2) & (s1 | (s1 >> 1)));
            const uint32_t x1 = cl ^ hx, c1b = cl & hx;                                // total = l + 2 x1 + 4 (c1b + ch)
            const uint32_t y0 = c1b ^ ch, y1 = c1b & ch;
            ge5[ry] = (y1 | (y0 & (x1 | l))) & 0x7fu;
        }
        int cnt = 0;
        if (y >= 3 && y + 3 < h && x >= 3 && x + 3 < w) {
#pragma unroll
            for (int ry = 0; ry < 7; ++ry) cnt += __popc(ge5[ry]);
        } else {   // frame border: taps of the m3 plane repeat (clamped coordinates)
            for (int dy = -3; dy <= 3; ++dy) {
                const int ry = clampi(y + dy, 0, h - 1) - y + 3;
                uint32_t g = 0;
#pragma unroll
                for (int r = 0; r < 7; ++r) g = (r == ry) ? ge5[r] : g;
                for (int dx = -3; dx <= 3; ++dx) cnt += (g >> (clampi(x + dx, 0, w - 1) - x + 3)) & 1u;
            }
        }
        if (cnt >= 25) atomicOr(a.M1 + q, bit);
    }
}

// One thread per pixel of dil3(M2) & A2 & ~A1: G2 by counting.
__global__ void __launch_bounds__(128)
k_eval_neighbours(const float* __restrict__ S, uint32_t* __restrict__ G2, int h, int w, int wpr, float siglow,
                  const int* __restrict__ list, const int* __restrict__ nlist, const int* prev_count) {
    if (prev_count && *prev_count == 0) return;
    const int n = *nlist;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const int p = list[i];
        const int y = p / w, x = p - y * w;
        int c1, c2;
        count_sp(S, y, x, h, w, siglow, siglow, c1, c2);
        if (c2 >= 13) atomicOr(G2 + (size_t)y * wpr + (x >> 5), 1u << (x & 31));
    }
}

}  // namespace lac
