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
#include "kernels.cuh"
#include "lazy_count.cuh"
#include "median_networks.cuh"

namespace lac {

// Incremental evaluation: G1, G2, M1 persist across the iterations of a frame.  A test at pixel p reads
// `work` within 4 px of p (S' : S within 2, each S from work within 2; fine structure: 9x9), so after the
// replacement pass of iteration t-1 rewrote the pixels NEED, only the tests inside R = dil9x9(NEED) can
// change: iteration t clears G1, G2, M1 inside R and re-evaluates the candidates there.

// list <- pixels of A1 & R; clear G1, G2, G2F (grow.cuh), M1 inside R (R = everything when `dirty` is NULL)
__global__ void __launch_bounds__(256)
k_list_candidates(const uint32_t* __restrict__ A1, const uint32_t* __restrict__ dirty, uint32_t* __restrict__ G1,
                  uint32_t* __restrict__ G2, uint32_t* __restrict__ G2F, uint32_t* __restrict__ M1, int* __restrict__ list,
                  int* __restrict__ nlist, uint32_t* __restrict__ Czero, int h, int w, int wpr, int nbx, const int* prev_count) {
    pdl_entry();
    if (prev_count && *prev_count == 0) return;
    const int lane = threadIdx.x & 31, wi = threadIdx.x >> 5;
    const BlockXY bk = block_xy(nbx);
    const int wx = bk.x * 32 + lane, y0 = bk.y * BW_CTA_ROWS + wi * BW_ROWS;
    uint32_t bits[BW_ROWS];
#pragma unroll
    for (int i = 0; i < BW_ROWS; ++i) bits[i] = 0;
    if (wx < wpr && y0 < h) {
        uint32_t reg[BW_ROWS];
        if (dirty) {
            dilate_rows<4>(dirty, y0, wx, h, wpr, reg);
        } else {
#pragma unroll
            for (int i = 0; i < BW_ROWS; ++i) reg[i] = 0xffffffffu;
        }
#pragma unroll
        for (int i = 0; i < BW_ROWS; ++i) {
            const int y = y0 + i;
            if (y >= h) break;
            const size_t q = (size_t)y * wpr + wx;
            const uint32_t r = reg[i];
            if (r == 0) continue;
            bits[i] = A1[q] & r;
            if (r == 0xffffffffu) {
                G1[q] = 0; G2[q] = 0; G2F[q] = 0; M1[q] = 0;
                if (Czero) Czero[q] = 0;   // frame prologue C = 0, fused (t = 0: every word takes this branch)
            } else {
                G1[q] &= ~r; G2[q] &= ~r; G2F[q] &= ~r; M1[q] &= ~r;
            }
        }
    }
    block_append(bits, y0 * w + wx * 32, w, list, nlist);
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

struct CandArgs {
    const float* S;
    const float* work;
    uint32_t *G1, *G2, *M1;
    int h, w, wpr;
    float sigclip, siglow, objlim;
    // R22 (fsmode 1) only: what N at the candidate is made of
    float gain, rn2;
    const float* gain_dev;   // nullable (R21)
    const float* var;        // nullable (R24)
    int* nfine;              // nullable (lacosmic_stats_enable): += candidates that pass G1 and take the fine-structure test
};

// P(v) of the header comment, with exactly the operations of O4/O5.  nn == 0: R7 (num = L+, F in ADU); nn > 0: R22
// (num = S', F divided by the noise nn) -- non-decreasing in v in both forms because num > 0 wherever it is evaluated.
__device__ __forceinline__ bool fine_test(float num, float m3c, float v, float objlim, float nn = 0.0f) {
    float d = __fsub_rn(m3c, v);
    if (nn > 0.0f) d = __fdiv_rn(d, nn);
    const float f = d > 0.01f ? d : 0.01f;
    return __fdiv_rn(num, f) > objlim;
}

// bit k = P(e[k]).  P is non-decreasing in v and (tlo, thi) brackets its switch point: P(v) is false for
// v <= tlo and true for v >= thi (both verified by the caller with fine_test itself); only values strictly
// inside the bracket need the division.  tlo = -inf, thi = +inf evaluates every value exactly.
template <int N>
__device__ __forceinline__ uint32_t fine_bits(const float (&e)[N], float lp, float m3c, float objlim, float tlo,
                                              float thi, float nn = 0.0f) {
    uint32_t m = 0, amb = 0;
#pragma unroll
    for (int k = 0; k < N; ++k) {
        m |= (uint32_t)(e[k] >= thi) << k;
        amb |= (uint32_t)((e[k] > tlo) & (e[k] < thi)) << k;
    }
    if (amb) {
#pragma unroll
        for (int k = 0; k < N; ++k)
            if ((amb >> k) & 1u) m |= (uint32_t)fine_test(lp, m3c, e[k], objlim, nn) << k;
    }
    return m;
}

// rows[r] bit c = P(V[r][c]) for the 9x9 window -> #{7x7 taps of the m3 plane with P} (see k_eval_candidates)
__device__ __forceinline__ int fine_count(const uint32_t (&rows)[9], int y, int x, int h, int w) {
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
    return cnt;
}

// bracket of the switch point of P (see fine_bits); returns false when P is false everywhere
__device__ __forceinline__ bool fine_bracket(float lp, float m3c, float objlim, float& tlo, float& thi) {
    const float INF = __int_as_float(0x7f800000);
    tlo = -INF;
    thi = INF;
    if (!(__fdiv_rn(lp, 0.01f) > objlim)) return false;        // F at its floor is the most favourable case
    const float fs = lp / objlim;                               // F at the switch point, approximately
    const float tau = m3c - fs;
    const float mg = fmaxf(fabsf(m3c), fabsf(fs)) * 9.5367431640625e-07f;   // 2^-20: >= 8 ulp of either term
    const float hi = tau + mg, lo = tau - mg;
    if (fabsf(hi) < INF && fabsf(lo) < INF && fine_test(lp, m3c, hi, objlim) && !fine_test(lp, m3c, lo, objlim)) {
        thi = hi;
        tlo = lo;
    }
    return true;
}

// One thread per listed pixel of A1: G1, G2 by counting; where G1 holds, the fine-structure test by counting.
// Virtual 9x9 window V[r][c] = work<y-4+r, x-4+c>; the m3-plane tap (dy, dx) of the 7x7 window is med3x3
// centred on the virtual position (cy(dy), cx(dx)), cy(dy) = clamp(y+dy) - y (R4: the STORED m3 plane is
// replicated), whose own taps are V[cy+4+-1][cx+4+-1] (R3).
#ifndef LAC_EVAL_MINB
#define LAC_EVAL_MINB 6
#endif
// FS = 1 (R22): the test compares S' = S - med5(S) with objlim * Fn, Fn = F / N: med5(S) and med5(work) (for N) are
// selected exactly at the candidate (25-input network), then the same counting over the 9x9 window decides, every
// tap evaluated with the exact operations (no bracket).
template <int FS>
__global__ void __launch_bounds__(128, LAC_EVAL_MINB)
k_eval_candidates(CandArgs a, const int* __restrict__ list, const int* __restrict__ nlist,
                  const int* prev_count) {
    pdl_entry();
    // the two counters are read together (one round trip, not two dependent ones, in front of the list)
    const int pc = prev_count ? *prev_count : 1;
    const int n0 = *nlist;
    const int n = pc ? n0 : 0;
    const int h = a.h, w = a.w;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const int p = list[i];
        const int y = p / w, x = p - y * w;
        int c1, c2;
        count_sp(a.S, y, x, h, w, a.sigclip, a.siglow, c1, c2);
        const uint32_t bit = 1u << (x & 31);
        const size_t q = (size_t)y * a.wpr + (x >> 5);
        if (c2 >= 13) atomicOr(a.G2 + q, bit);
        if (a.nfine && c1 >= 13) atomicAdd(a.nfine, 1);      // statistics only (off in timed runs)
        if (c1 < 13) continue;
        atomicOr(a.G1 + q, bit);
        uint32_t rows[9];   // bit c of rows[r] = P(V[r][c])
        float tlo, thi;
        {
            int xx[9];
#pragma unroll
            for (int c = 0; c < 9; ++c) xx[c] = clampi(x + c - 4, 0, w - 1);
            float ctr[3][3];
#pragma unroll
            for (int r = 0; r < 3; ++r)
#pragma unroll
                for (int c = 0; c < 3; ++c)
                    ctr[r][c] = __ldg(a.work + (size_t)clampi(y + r - 1, 0, h - 1) * w + xx[3 + c]);
            float lp = lplus_px(ctr[1][1], ctr[0][1], ctr[2][1], ctr[1][0], ctr[1][2]);
            const float m3c = med9(ctr[0][0], ctr[0][1], ctr[0][2], ctr[1][0], ctr[1][1], ctr[1][2], ctr[2][0],
                                   ctr[2][1], ctr[2][2]);
            float nn = 0.0f;
            if (FS == 1) {
                float v[25], srt[25];
#pragma unroll
                for (int dy = 0; dy < 5; ++dy)
#pragma unroll
                    for (int dx = 0; dx < 5; ++dx)
                        v[5 * dy + dx] = __ldg(a.S + (size_t)clampi(y + dy - 2, 0, h - 1) * w + xx[2 + dx]);
                const float sc = v[12];
                sort25(v, srt);
                lp = __fsub_rn(sc, srt[12]);                  // the numerator of R22 is S'
                if (a.var) {
                    nn = noise_from_var(__ldg(a.var + (size_t)y * w + x));
                } else {
#pragma unroll
                    for (int dy = 0; dy < 5; ++dy)
#pragma unroll
                        for (int dx = 0; dx < 5; ++dx)
                            v[5 * dy + dx] = __ldg(a.work + (size_t)clampi(y + dy - 2, 0, h - 1) * w + xx[2 + dx]);
                    sort25(v, srt);
                    nn = noise_px(srt[12], a.gain_dev ? __ldg(a.gain_dev) : a.gain, a.rn2);
                }
                tlo = -__int_as_float(0x7f800000);
                thi = __int_as_float(0x7f800000);
            } else if (!fine_bracket(lp, m3c, a.objlim, tlo, thi)) {
                continue;
            }
#pragma unroll 3
            for (int r = 0; r < 9; ++r) {
                const float* row = a.work + (size_t)clampi(y + r - 4, 0, h - 1) * w;
                float f[9];
#pragma unroll
                for (int c = 0; c < 9; ++c) f[c] = __ldg(row + xx[c]);
                const uint32_t m = fine_bits<9>(f, lp, m3c, a.objlim, tlo, thi, nn);
#pragma unroll
                for (int k = 0; k < 9; ++k) rows[k] = (k == r) ? m : rows[k];
            }
        }
        if (fine_count(rows, y, x, h, w) >= 25) atomicOr(a.M1 + q, bit);
    }
}

// ------------------------------------------------------------------------------------------------
// Incremental steps (1)-(3a) (iterations t >= 1): S, A1, A2 are recomputed only on the listed quads (aligned
// groups of 4 pixels holding a pixel within 2 px of a rewritten one; k_dirty_lists), one quad per thread, with
// the same window network and the same operations as the dense pass (kernels.cuh, noise_S_tile).  The
// pixels of the quad with S > sigclip are appended to the candidate list (one atomic per CTA and round).
__global__ void __launch_bounds__(256, 4)
k_noise_S_quads(const float* __restrict__ work, NoiseArgs a, const int* __restrict__ qlist,
                const int* __restrict__ nq, int* __restrict__ clist, int* __restrict__ nc, const int* prev_count) {
    pdl_entry();
    __shared__ int s_warp[8];
    __shared__ int s_base;
    const int pc = prev_count ? *prev_count : 1;      // read together with the list length: one round trip
    const int n0 = *nq;
    const int n = pc ? n0 : 0, h = a.h, w = a.w;
    const int tid = threadIdx.x, lane = tid & 31, wi = tid >> 5;
    const bool vec = (w & 3) == 0;
    for (int base = blockIdx.x * 256; base < n; base += gridDim.x * 256) {   // uniform trip count per CTA
        const int i = base + tid;
        uint32_t n1 = 0;
        int p = 0;
        if (i < n) {
            p = qlist[i];
            const int y = p / w, x = p - y * w;
            float win[8][5];   // win[c][r] = work<y-2+r, x-2+c>
            if (vec && x >= 4 && x + 8 <= w && y >= 2 && y + 2 < h) {
#pragma unroll
                for (int r = 0; r < 5; ++r) {
                    const float* row = work + (size_t)(y - 2 + r) * w + (x - 4);
                    const float4 q0 = *reinterpret_cast<const float4*>(row);
                    const float4 q1 = *reinterpret_cast<const float4*>(row + 4);
                    const float4 q2 = *reinterpret_cast<const float4*>(row + 8);
                    const float v[12] = {q0.x, q0.y, q0.z, q0.w, q1.x, q1.y, q1.z, q1.w, q2.x, q2.y, q2.z, q2.w};
#pragma unroll
                    for (int c = 0; c < 8; ++c) win[c][r] = v[2 + c];
                }
            } else {
                int xx[8];
#pragma unroll
                for (int c = 0; c < 8; ++c) xx[c] = clampi(x - 2 + c, 0, w - 1);
#pragma unroll
                for (int r = 0; r < 5; ++r) {
                    const float* row = work + (size_t)clampi(y - 2 + r, 0, h - 1) * w;
#pragma unroll
                    for (int c = 0; c < 8; ++c) win[c][r] = row[xx[c]];
                }
            }
            float m5[4], s[4];
            if (a.var) {                                   // R24: N comes from the variance plane, no median
#pragma unroll
                for (int j = 0; j < 4; ++j) m5[j] = __ldg(a.var + (size_t)y * w + min(x + j, w - 1));
            } else {
                median5x5_x4(win, m5);
            }
            uint32_t n2 = 0;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const float lp = lplus_px(win[2 + j][2], win[2 + j][1], win[2 + j][3], win[1 + j][2], win[3 + j][2]);
                const float nn = a.var ? noise_from_var(m5[j])
                                       : noise_px(m5[j], a.gain_dev ? __ldg(a.gain_dev) : a.gain, a.rn2);
                s[j] = fdiv_nn(lp, __fmul_rn(2.0f, nn));
                // threshold tests as sign bits on the FMA pipe (see noise_S_tile)
                const uint32_t ok = (x + j < w) ? sign01(__fsub_rn(win[2 + j][2], a.satlevel)) : 0u;   // R12
                n1 += (ok & sign01(__fsub_rn(a.sigclip, s[j]))) << j;
                n2 += (ok & sign01(__fsub_rn(a.siglow, s[j]))) << j;
            }
            store4(a.S, (size_t)y * w, x, w, s);
            // this thread alone owns its nibble of the A1 / A2 words; the other nibbles change concurrently
            const size_t q = (size_t)y * a.wpr + (x >> 5);
            const int sh = x & 31;
            if (a.nok) {                                   // R23 / R25: never flagged
                const uint32_t nk = (a.nok[q] >> sh) & 0xFu;
                n1 &= ~nk;
                n2 &= ~nk;
            }
            const uint32_t o1 = (a.A1[q] >> sh) & 0xFu, o2 = (a.A2[q] >> sh) & 0xFu;
            if (o1 != n1) atomicXor(a.A1 + q, (o1 ^ n1) << sh);
            if (o2 != n2) atomicXor(a.A2 + q, (o2 ^ n2) << sh);
        }
        const int cnt = __popc(n1);
        int incl = cnt;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int o = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += o;
        }
        if (lane == 31) s_warp[wi] = incl;
        __syncthreads();
        if (tid == 0) {
            int tot = 0;
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const int c = s_warp[k];
                s_warp[k] = tot;
                tot += c;
            }
            s_base = tot ? atomicAdd(nc, tot) : 0;
        }
        __syncthreads();
        int o = s_base + s_warp[wi] + incl - cnt;
#pragma unroll
        for (int j = 0; j < 4; ++j)
            if ((n1 >> j) & 1u) clist[o++] = p + j;
        __syncthreads();   // s_warp / s_base are rewritten in the next round
    }
}

}  // namespace lac
