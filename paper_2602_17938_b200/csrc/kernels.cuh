// sm_100a kernels of the L.A.Cosmic iteration (DESIGN.md section 5 lists each with its roofline).
#pragma once
#include <cuda.h>

#include "common.cuh"
#include "median_networks.cuh"

namespace lac {

constexpr int TW = 128;   // output tile width: 32 lanes x 4 adjacent outputs per thread
constexpr int TH = 16;    // output tile height: 8 warps x 2 rows
constexpr int NT = 256;   // threads per CTA (8 warps)
constexpr int NWARP = NT / 32;

struct GateParams {
    float sigclip, siglow, objlim, satlevel;
};

// Edge-replicate tile load with margins (R3): sm[r][c] = src<y0-MY+r, x0-MX+c>.
template <int MX, int MY, int PITCH, int TILE_H = TH>
__device__ __forceinline__ void load_tile(float* sm, const float* __restrict__ src, int h, int w, int y0,
                                          int x0, int tid) {
    constexpr int SW = TW + 2 * MX, SH = TILE_H + 2 * MY;
    static_assert(PITCH >= SW && PITCH % 4 == 0, "pitch must hold the tile and keep float4 alignment");
    for (int i = tid; i < SW * SH; i += NT) {
        int r = i / SW, c = i - r * SW;
        int yy = clampi(y0 - MY + r, 0, h - 1), xx = clampi(x0 - MX + c, 0, w - 1);
        sm[r * PITCH + c] = __ldg(src + (size_t)yy * w + xx);
    }
}

// K x (K+T-1) register window for T adjacent outputs (T = 4 or 8): in[c][r], c = 0..K+T-2 left to right, r = 0..K-1 top
// to bottom.  `p` points at (top row, the 16-byte aligned column 4 to the left of the first output).
template <int K, int PITCH, int T = 4>
__device__ __forceinline__ void load_window(const float* p, float (&in)[K + T - 1][K]) {
    constexpr int R = K / 2, NV = (T + 8) / 4;      // float4 per row: columns -4 .. T+3
#pragma unroll
    for (int r = 0; r < K; ++r) {
        float v[4 * NV];
#pragma unroll
        for (int q = 0; q < NV; ++q) {
            const float4 a = *reinterpret_cast<const float4*>(p + r * PITCH + 4 * q);
            v[4 * q] = a.x; v[4 * q + 1] = a.y; v[4 * q + 2] = a.z; v[4 * q + 3] = a.w;
        }
#pragma unroll
        for (int cc = 0; cc < K + T - 1; ++cc) in[cc][r] = v[4 - R + cc];
    }
}

template <int K>
__device__ __forceinline__ void median_x4(const float (&in)[K + 3][K], float (&out)[4]);
template <>
__device__ __forceinline__ void median_x4<3>(const float (&in)[6][3], float (&out)[4]) { median3x3_x4(in, out); }
template <>
__device__ __forceinline__ void median_x4<5>(const float (&in)[8][5], float (&out)[4]) { median5x5_x4(in, out); }
template <>
__device__ __forceinline__ void median_x4<7>(const float (&in)[10][7], float (&out)[4]) { median7x7_x4(in, out); }

__device__ __forceinline__ void store4(float* __restrict__ dst, size_t row_off, int x, int w,
                                       const float (&v)[4]) {
    if (x + 3 < w && ((row_off + x) & 3) == 0) {
        *reinterpret_cast<float4*>(dst + row_off + x) = make_float4(v[0], v[1], v[2], v[3]);
    } else {
#pragma unroll
        for (int j = 0; j < 4; ++j)
            if (x + j < w) dst[row_off + x + j] = v[j];
    }
}

template <bool ALIGNED>
__device__ __forceinline__ void store4q(float* __restrict__ dst, size_t row_off, int x, int w, const float (&v)[4]) {
    if (ALIGNED) *reinterpret_cast<float4*>(dst + row_off + x) = make_float4(v[0], v[1], v[2], v[3]);
    else store4(dst, row_off, x, w, v);
}

// ------------------------------------------------------------------------------------------------
// Standalone k x k median (lacosmic_medfilt): same selection networks and tile shape as the fused
// kernels.  Each thread produces 4 adjacent outputs from a (k+3) x k register window.
template <int K>
__global__ void __launch_bounds__(NT) k_medfilt(const float* __restrict__ in, float* __restrict__ out,
                                               int h, int w, int nbx) {
    constexpr int R = K / 2, MX = 4, PITCH = TW + 2 * MX;
    __shared__ __align__(16) float sm[(TH + 2 * R) * PITCH];
    const int tid = threadIdx.x, lane = tid & 31, wi = tid >> 5;
    const BlockXY bk = block_xy(nbx);
    const int x0 = bk.x * TW, y0 = bk.y * TH;
    load_tile<MX, R, PITCH>(sm, in, h, w, y0, x0, tid);
    __syncthreads();
#pragma unroll 1
    for (int ly = wi; ly < TH; ly += NWARP) {
        int y = y0 + ly, x = x0 + 4 * lane;
        if (y >= h || x >= w) continue;
        float win[K + 3][K], o[4];
        load_window<K, PITCH>(sm + ly * PITCH + 4 * lane, win);
        median_x4<K>(win, o);
        store4(out, (size_t)y * w, x, w, o);
    }
}

// Standalone L+ (lacosmic_lplus).
__global__ void __launch_bounds__(NT) k_lplus(const float* __restrict__ in, float* __restrict__ out,
                                             int h, int w, int nbx) {
    const BlockXY bk = block_xy(nbx);
    int x = bk.x * 32 + (threadIdx.x & 31), y = bk.y * 8 + (threadIdx.x >> 5);
    if (x >= w || y >= h) return;
    const float* row = in + (size_t)y * w;
    float c = row[x];
    float U = in[(size_t)max(y - 1, 0) * w + x], D = in[(size_t)min(y + 1, h - 1) * w + x];
    float Lf = row[max(x - 1, 0)], R = row[min(x + 1, w - 1)];
    out[(size_t)y * w + x] = lplus_px(c, U, D, Lf, R);
}

// ------------------------------------------------------------------------------------------------
// K_A: steps (1)-(3a).  work -> L+ (recomputed later, not stored), N = sqrt(gain*med5+rn^2)/gain,
// S = L+/(2N).  Writes S; Lp/N only when a debug plane is requested.
// Tile height 32: 128x64 tiles are 1 % faster for a single frame (0.640 vs 0.647 ms) but their two 38 KB stages x 3 CTAs
// fill the SM's shared memory, and frames in flight on other streams can no longer interleave their kernels
// (configs[3] with 4 frames in flight: 1321 frames/s against 1923 with 128x32 tiles; B200)
#ifndef LAC_NS_TH
#define LAC_NS_TH 32
#endif
constexpr int NS_TH = LAC_NS_TH;   // tile height of the noise/S pass (own constant: its tile is much lighter than K_B's)
// pitch 140 = 128 + 4 (left margin) + 8: the tile needs 136 columns; 140 (35 x 16 bytes) makes consecutive rows start 48
// bytes apart modulo 128, so the 16-byte window loads of a quarter warp (4 octets x 2 rows) hit eight distinct bank groups
constexpr int NS_MX = 4, NS_MY = 2, NS_PITCH = TW + 2 * NS_MX + 4, NS_ROWS = NS_TH + 2 * NS_MY;

struct NoiseArgs {
    float* S;
    float* dbgLp;
    float* dbgN;
    uint32_t *A1, *A2;       // nullable (lazy path): bit-planes ok & (S > sigclip), ok & (S > siglow)
    float* copy_out;         // nullable: also write the input tile here (frame prologue work = img_in fused
                             // into the first pass, which then reads img_in itself)
    int h, w, wpr;
    float gain, rn2, sigclip, siglow, satlevel;
    float* R;                // nullable (R21): also write r = (work - med5) / sqrt(max(med5, 1e-4)) here, and
                             // store med5 itself in the S plane (k_S_from_m5 turns it into S once the gain is known)
    const float* gain_dev;   // nullable (R21): the gain of this iteration, estimated on the device
    int* zero_ptr;           // nullable: the frame's counter block, cleared by the first launch of a frame
    int zero_n;              // (nothing reads or adds to it before the next launch)
    const uint32_t* nok;     // nullable (R23, R25): bit-plane of the pixels that may never be flagged (bad pixels,
                             // extended saturated-star mask); cleared from A1 / A2
    const float* var;        // nullable (R24): variance plane; N = sqrt(max(var, 1e-8)) replaces the noise model
    uint8_t* mask_zero;      // nullable: the frame's uint8 mask, cleared by this pass (k_grow_replace then sets the flagged
                             // pixels directly, and the frame needs no bit-plane -> uint8 expansion at its end)
};

// R24: N from a variance entry
__device__ __forceinline__ float noise_from_var(float v) { return __fsqrt_rn(v > 1e-8f ? v : 1e-8f); }

__device__ __forceinline__ void zero_counters(const NoiseArgs& a) {
    if (a.zero_ptr)
        for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < a.zero_n; i += gridDim.x * blockDim.x) a.zero_ptr[i] = 0;
}

// gather the 4-bit nibbles of the 8 lanes that share a 32-pixel word
__device__ __forceinline__ uint32_t nibbles_to_word(uint32_t nib, int lane) {
    uint32_t v = nib << ((lane & 7) * 4);
    v |= __shfl_xor_sync(0xffffffffu, v, 1);
    v |= __shfl_xor_sync(0xffffffffu, v, 2);
    v |= __shfl_xor_sync(0xffffffffu, v, 4);
    return v;
}

// gather the 8-bit groups of the 4 lanes that share a 32-pixel word
__device__ __forceinline__ uint32_t bytes_to_word(uint32_t b, int lane) {
    uint32_t v = b << ((lane & 3) * 8);
    v |= __shfl_xor_sync(0xffffffffu, v, 1);
    v |= __shfl_xor_sync(0xffffffffu, v, 2);
    return v;
}

// A warp computes one UNIT of 32 x 8 pixels at a time (lane = 4 octets x 8 rows: 8 adjacent outputs per thread from
// a 12 x 5 window, median5x5_x8 -- 69.25 min/max per output against 81.5 with 4 outputs per thread), so that the 4
// lanes of a row assemble whole 32-pixel words of A1 / A2.
constexpr int UW = 32, UH = 8;

// sm: work tile with margins (NS_MX, NS_MY), edge-replicated
// W4: w % 4 == 0 and 16-byte aligned planes (the TMA path): quads are whole and every store is one vector
// CFG >= 0: the nullable outputs are known at compile time (bit 0: copy_out, bit 1: A1 / A2, bit 2: mask_zero, bit 3: the
// residual plane of the gain estimate instead of S; no debug plane, no device-side gain), which takes their tests out of the unit loop; CFG < 0: decided at run time.
// The threshold tests and their packing run on the FMA pipe: for finite a, b the sign of fsub(a, b) is set iff a < b
// (a difference of two floats never rounds to zero unless they are equal: gradual underflow), so
// (s > thr) = sign(thr - s), (c < satlevel) = sign(c - satlevel), and the nibble is a sum of sign bits times 2^j.
template <bool W4, int CFG>
__device__ __forceinline__ void noise_S_tile(const float* sm, const NoiseArgs& a, int x0, int y0, int lane,
                                             int wi) {
    const int lx = lane & 3, lr = lane >> 2;
    const bool has_copy = CFG < 0 ? a.copy_out != nullptr : (CFG & 1) != 0;
    const bool has_A = CFG < 0 ? a.A1 != nullptr : (CFG & 2) != 0;
    const bool has_mz = CFG < 0 ? a.mask_zero != nullptr : (CFG & 4) != 0;
    const bool has_lp = CFG < 0 && a.dbgLp != nullptr, has_n = CFG < 0 && a.dbgN != nullptr;
    const bool has_R = CFG < 0 ? a.R != nullptr : (CFG & 8) != 0;
    // CFG 8 / 9: the residual pass of the gain estimate (R21) -- med5 and the residual are all it writes, so L+, N, S and
    // the threshold tests are not computed at all
    constexpr bool ONLY_R = CFG >= 0 && (CFG & 8) != 0;
    const float gain = (CFG < 0 && a.gain_dev) ? __ldg(a.gain_dev) : a.gain;
    static_assert((TW / UW) * (NS_TH / UH) <= NWARP || NS_TH % UH == 0, "units must tile the tile");
#pragma unroll 1
    for (int u = wi; u < (TW / UW) * (NS_TH / UH); u += NWARP) {
        const int xu = x0 + (u & 3) * UW, lyu = (u >> 2) * UH, yu = y0 + lyu;
        if (yu >= a.h || xu >= a.w) continue;                                            // warp-uniform
        const int ly = lyu + lr, y = y0 + ly, x = xu + 8 * lx;
        uint32_t n1 = 0, n2 = 0;
        if (y < a.h && x < a.w) {
            float win[12][5], m5[8], s[8], lp[8], n[8], ctr[8];
            load_window<5, NS_PITCH, 8>(sm + ly * NS_PITCH + (x - x0), win);
            median5x5_x8(win, m5);
            uint32_t nok = 0;
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                ctr[j] = win[2 + j][2];
                if (ONLY_R) continue;
                lp[j] = lplus_px(win[2 + j][2], win[2 + j][1], win[2 + j][3], win[1 + j][2], win[3 + j][2]);
                n[j] = noise_px(m5[j], gain, a.rn2);
                s[j] = fdiv_nn(lp[j], __fmul_rn(2.0f, n[j]));
                n1 += sign01(__fsub_rn(a.sigclip, s[j])) << j;                            // S > sigclip
                n2 += sign01(__fsub_rn(a.siglow, s[j])) << j;                             // S > siglow
                nok += sign01(__fsub_rn(ctr[j], a.satlevel)) << j;                        // R12: c < satlevel
            }
            // pixels beyond the right edge (the octet straddles it): never flagged, never stored
            const int nin = min(a.w - x, 8);
            nok &= (1u << nin) - 1u;
            n1 &= nok;
            n2 &= nok;
            const size_t ro = (size_t)y * a.w;
            auto put = [&](float* dst, const float (&v)[8]) {
                if (W4) {          // w % 4 == 0: the octet is one or two whole, aligned quads
                    *reinterpret_cast<float4*>(dst + ro + x) = make_float4(v[0], v[1], v[2], v[3]);
                    if (nin == 8) *reinterpret_cast<float4*>(dst + ro + x + 4) = make_float4(v[4], v[5], v[6], v[7]);
                } else {
#pragma unroll
                    for (int j = 0; j < 8; ++j)
                        if (j < nin) dst[ro + x + j] = v[j];
                }
            };
            if (has_R) put(a.S, m5);
            else put(a.S, s);
            if (has_lp) put(a.dbgLp, lp);
            if (has_n) put(a.dbgN, n);
            if (has_copy) put(a.copy_out, ctr);
            if (has_mz) {
                if (W4) {          // the API checks the alignment of the plane
                    *reinterpret_cast<uint32_t*>(a.mask_zero + ro + x) = 0u;
                    if (nin == 8) *reinterpret_cast<uint32_t*>(a.mask_zero + ro + x + 4) = 0u;
                } else {
#pragma unroll
                    for (int j = 0; j < 8; ++j)
                        if (j < nin) a.mask_zero[ro + x + j] = 0;
                }
            }
            if (has_R) {   // R21: residual in units of sqrt(signal)
                float r[8];
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const float m5c = m5[j] > 1e-4f ? m5[j] : 1e-4f;
                    r[j] = __fdiv_rn(__fsub_rn(ctr[j], m5[j]), __fsqrt_rn(m5c));
                }
                put(a.R, r);
            }
        }
        if (has_A) {
            const uint32_t b1 = bytes_to_word(n1, lane), b2 = bytes_to_word(n2, lane);
            if (lx == 0 && y < a.h) {
                size_t q = (size_t)y * a.wpr + (xu >> 5);
                const uint32_t keep = a.nok ? ~a.nok[q] : 0xffffffffu;
                a.A1[q] = b1 & keep;
                a.A2[q] = b2 & keep;
            }
        }
    }
}

// generic path (any w): one tile per CTA, tile loaded with clamped scalar loads
__global__ void __launch_bounds__(NT)
k_noise_S(const float* __restrict__ work, NoiseArgs a, int ntx, const int* prev_count) {
    if (prev_count && *prev_count == 0) return;   // fixed point reached (R17)
    zero_counters(a);
    __shared__ __align__(16) float sm[NS_ROWS * NS_PITCH];
    const int tid = threadIdx.x;
    const int t = blockIdx.x;
    const int ty = t / ntx, tx = t - ty * ntx;
    const int x0 = tx * TW, y0 = ty * NS_TH;
    load_tile<NS_MX, NS_MY, NS_PITCH, NS_TH>(sm, work, a.h, a.w, y0, x0, tid);
    __syncthreads();
    noise_S_tile<false, -1>(sm, a, x0, y0, tid & 31, tid >> 5);
}

// K_B: steps (3b)-(5).  S' = S - med5(S); m3 = med3(work) (tile in shared memory, replicated at the
// frame border as a STORED plane would be, R4); F = max(m3 - med7(m3), 0.01); gates -> bit-planes.
constexpr int FG_AX = 8, FG_AY = 4, FG_PA = TW + 2 * FG_AX, FG_AROWS = TH + 2 * FG_AY;   // work tile
constexpr int FG_BX = 4, FG_BY = 3, FG_PB = TW + 2 * FG_BX, FG_BROWS = TH + 2 * FG_BY;   // m3 tile
constexpr int FG_SX = 4, FG_SY = 2, FG_PS = TW + 2 * FG_SX, FG_SROWS = TH + 2 * FG_SY;   // S tile

struct FineArgs {
    uint32_t *G1, *G2, *M1;
    float *dbgSp, *dbgM3, *dbgF;
    int h, w, wpr;
    GateParams gp;
    const float* N;          // R22 (fsmode 1): the noise plane the noise/S pass stored; null: R7 (L+/F, F in ADU)
    const uint32_t* nok;     // nullable (R23, R25): pixels that may never be flagged
};

// smA / smS: edge-replicated work / S tiles; smB: scratch for the m3 tile.  Contains block barriers.
__device__ __forceinline__ void fine_gates_tile(const float* smA, float* smB, const float* smS,
                                                const FineArgs& a, int x0, int y0, int tid) {
    constexpr int PA = FG_PA, PB = FG_PB, PS = FG_PS, BX = FG_BX, BY = FG_BY, AY = FG_AY;
    constexpr int BH = FG_BROWS, BG = PB / 4;
    const int lane = tid & 31, wi = tid >> 5;
    const int h = a.h, w = a.w;
    // m3 tile: B[r][4g..4g+3] = med3 at frame rows y0-3+r, columns x0-4+4g .. +3
    for (int i = tid; i < BH * BG; i += NT) {
        int r = i / BG, g = i - r * BG;
        float win[6][3], o[4];
        load_window<3, PA>(smA + r * PA + 4 * g, win);
        median3x3_x4(win, o);
        *reinterpret_cast<float4*>(smB + r * PB + 4 * g) = make_float4(o[0], o[1], o[2], o[3]);
    }
    __syncthreads();
    // R4: positions outside the frame take the value of the stored plane's edge, not a median evaluated
    // at virtual coordinates.  Only tiles that touch the frame border have such positions.
    if (y0 - BY < 0 || y0 + TH + BY > h || x0 - BX < 0 || x0 + TW + BX > w) {
        constexpr int NFIX = (BH * PB + NT - 1) / NT;
        float fix[NFIX];
#pragma unroll
        for (int q = 0; q < NFIX; ++q) {
            int i = tid + q * NT;
            if (i < BH * PB) {
                int r = i / PB, c = i - r * PB;
                int cr = clampi(y0 - BY + r, 0, h - 1) - (y0 - BY);
                int cc = clampi(x0 - BX + c, 0, w - 1) - (x0 - BX);
                fix[q] = smB[cr * PB + cc];
            }
        }
        __syncthreads();
#pragma unroll
        for (int q = 0; q < NFIX; ++q) {
            int i = tid + q * NT;
            if (i < BH * PB) smB[i] = fix[q];
        }
        __syncthreads();
    }
#pragma unroll 1
    for (int ly = wi; ly < TH; ly += NWARP) {
        const int y = y0 + ly, x = x0 + 4 * lane;
        uint32_t n1 = 0, n2 = 0, n3 = 0;
        if (y < h && x < w) {
            float sp[4], f[4], m3[4];
            {
                float win[8][5], mS[4];
                load_window<5, PS>(smS + ly * PS + 4 * lane, win);
                median5x5_x4(win, mS);
#pragma unroll
                for (int j = 0; j < 4; ++j) sp[j] = __fsub_rn(win[2 + j][2], mS[j]);
            }
            {
                float win[10][7], m7[4];
                load_window<7, PB>(smB + ly * PB + 4 * lane, win);
                median7x7_x4(win, m7);
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    m3[j] = win[3 + j][3];
                    float d = __fsub_rn(m3[j], m7[j]);
                    if (a.N) d = __fdiv_rn(d, a.N[(size_t)y * w + min(x + j, w - 1)]);   // R22: in units of the noise
                    f[j] = d > 0.01f ? d : 0.01f;
                }
            }
            const float* ac = smA + (ly + AY) * PA + 4 * lane + 4;      // columns x-4 .. x+7 of row y
            const float4 c0 = *reinterpret_cast<const float4*>(ac);
            const float4 c1 = *reinterpret_cast<const float4*>(ac + 4);
            const float4 c2 = *reinterpret_cast<const float4*>(ac + 8);
            const float4 up = *reinterpret_cast<const float4*>(ac - PA + 4);
            const float4 dn = *reinterpret_cast<const float4*>(ac + PA + 4);
            const float ctr[6] = {c0.w, c1.x, c1.y, c1.z, c1.w, c2.x};
            const float u[4] = {up.x, up.y, up.z, up.w}, d4[4] = {dn.x, dn.y, dn.z, dn.w};
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                float lp = lplus_px(ctr[1 + j], u[j], d4[j], ctr[j], ctr[2 + j]);
                bool ok = (x + j < w) && (ctr[1 + j] < a.gp.satlevel);            // R12
                bool g1 = ok && (sp[j] > a.gp.sigclip);
                bool g2 = ok && (sp[j] > a.gp.siglow);
                // R8; R22 compares S' (positive where G1 holds) instead of L+
                bool m1 = g1 && ((a.N ? __fdiv_rn(sp[j], f[j]) : fdiv_nn(lp, f[j])) > a.gp.objlim);
                n1 |= (uint32_t)g1 << j;
                n2 |= (uint32_t)g2 << j;
                n3 |= (uint32_t)m1 << j;
            }
            size_t ro = (size_t)y * w;
            if (a.dbgSp) store4(a.dbgSp, ro, x, w, sp);
            if (a.dbgM3) store4(a.dbgM3, ro, x, w, m3);
            if (a.dbgF) store4(a.dbgF, ro, x, w, f);
        }
        uint32_t b1 = nibbles_to_word(n1, lane), b2 = nibbles_to_word(n2, lane), b3 = nibbles_to_word(n3, lane);
        int wx = (x0 >> 5) + (lane >> 3);
        if ((lane & 7) == 0 && y < h && wx < a.wpr) {
            size_t q = (size_t)y * a.wpr + wx;
            const uint32_t keep = a.nok ? ~a.nok[q] : 0xffffffffu;
            a.G1[q] = b1 & keep;
            a.G2[q] = b2 & keep;
            a.M1[q] = b3 & keep;
        }
    }
}

// generic path (any w): one tile per CTA, tiles loaded with clamped scalar loads
__global__ void __launch_bounds__(NT)
k_fine_gates(const float* __restrict__ work, const float* __restrict__ S, FineArgs a, int nbx,
             const int* prev_count) {
    if (prev_count && *prev_count == 0) return;
    __shared__ __align__(16) float smA[FG_AROWS * FG_PA];
    __shared__ __align__(16) float smB[FG_BROWS * FG_PB];
    __shared__ __align__(16) float smS[FG_SROWS * FG_PS];
    const int tid = threadIdx.x;
    const BlockXY bk = block_xy(nbx);
    const int x0 = bk.x * TW, y0 = bk.y * TH;
    load_tile<FG_AX, FG_AY, FG_PA>(smA, work, a.h, a.w, y0, x0, tid);
    load_tile<FG_SX, FG_SY, FG_PS>(smS, S, a.h, a.w, y0, x0, tid);
    __syncthreads();
    fine_gates_tile(smA, smB, smS, a, x0, y0, tid);
}

// ------------------------------------------------------------------------------------------------
// TMA path (w % 4 == 0): persistent CTAs, each walking tiles t = blockIdx.x, +gridDim.x, ... with a
// two-stage pipeline: one elected thread issues cp.async.bulk.tensor loads of the NEXT tile's boxes
// while all warps run the selection networks on the current one.  TMA fills out-of-frame elements
// with zeros; tiles touching the frame border repair them in shared memory to edge-replicate (R3).
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    } while (!done);
}
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* map, int cx, int cy, uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
        ::"r"(smem_u32(dst)), "l"(reinterpret_cast<uint64_t>(map)), "r"(cx), "r"(cy), "r"(smem_u32(bar)) : "memory");
}

constexpr int NS_STAGE_BYTES = (NS_ROWS * NS_PITCH * 4 + 127) / 128 * 128;   // a stage of the noise/S tile pipeline

// repair a TMA-loaded tile (zeros outside the frame) to edge-replicate; tile origin (ox, oy) in frame coords
template <int ROWS, int PITCH>
__device__ __forceinline__ void replicate_fix(float* sm, int oy, int ox, int h, int w, int tid) {
    for (int i = tid; i < ROWS * PITCH; i += NT) {
        int r = i / PITCH, c = i - r * PITCH;
        int yy = oy + r, xx = ox + c;
        if (yy < 0 || yy >= h || xx < 0 || xx >= w)
            sm[i] = sm[(clampi(yy, 0, h - 1) - oy) * PITCH + (clampi(xx, 0, w - 1) - ox)];
    }
}

#ifndef LAC_NS_MINB
#define LAC_NS_MINB 3
#endif
template <int CFG>
__global__ void __launch_bounds__(NT, LAC_NS_MINB)
k_noise_S_tma(const __grid_constant__ CUtensorMap mapWork, NoiseArgs a, int ntx, int ntiles,
              const int* prev_count, int tile0) {
    pdl_entry();
    if (prev_count && *prev_count == 0) return;
    zero_counters(a);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int TILE_BYTES = NS_ROWS * NS_PITCH * 4;
    auto buf = [&](int st) { return reinterpret_cast<float*>(smem_raw + st * NS_STAGE_BYTES); };
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + 2 * NS_STAGE_BYTES);
    const int tid = threadIdx.x;
    if (tid == 0) {
        mbar_init(&full[0], 1);
        mbar_init(&full[1], 1);
        fence_mbar_init();
    }
    __syncthreads();
    const int nt = ntiles;                                  // this launch: tiles tile0 .. tile0 + ntiles - 1
    auto tile_of = [&](int i) { return tile0 + i; };
    auto issue = [&](int t, int st) {
        int ty = t / ntx, tx = t - ty * ntx;
        mbar_expect_tx(&full[st], TILE_BYTES);
        tma_load_2d(buf(st), &mapWork, tx * TW - NS_MX, ty * NS_TH - NS_MY, &full[st]);
    };
    int i = blockIdx.x;
    if (tid == 0 && i < nt) issue(tile_of(i), 0);
    for (int it = 0; i < nt; i += gridDim.x, ++it) {
        const int st = it & 1;
        if (tid == 0 && i + (int)gridDim.x < nt) issue(tile_of(i + gridDim.x), st ^ 1);
        mbar_wait(&full[st], (it >> 1) & 1);
        const int t = tile_of(i);
        const int ty = t / ntx, tx = t - ty * ntx;
        const int x0 = tx * TW, y0 = ty * NS_TH;
        if (y0 - NS_MY < 0 || y0 + NS_TH + NS_MY > a.h || x0 - NS_MX < 0 || x0 + TW + NS_MX > a.w) {
            replicate_fix<NS_ROWS, NS_PITCH>(buf(st), y0 - NS_MY, x0 - NS_MX, a.h, a.w, tid);
            fence_proxy_async();
            __syncthreads();
        }
        noise_S_tile<true, CFG>(buf(st), a, x0, y0, tid & 31, tid >> 5);
        __syncthreads();   // stage st is free for the load issued at the top of the next iteration
    }
}

constexpr int FG_A_BYTES = FG_AROWS * FG_PA * 4, FG_S_BYTES = FG_SROWS * FG_PS * 4,
              FG_B_BYTES = FG_BROWS * FG_PB * 4;
constexpr int FG_SMEM_BYTES = 2 * FG_A_BYTES + 2 * FG_S_BYTES + FG_B_BYTES + 16;
constexpr int NS_SMEM_BYTES = 2 * NS_STAGE_BYTES + 16;
static_assert(FG_A_BYTES % 128 == 0 && FG_S_BYTES % 128 == 0, "TMA destinations must stay 128-byte aligned");
static_assert(NS_STAGE_BYTES % 128 == 0 && (NS_PITCH * 4) % 16 == 0, "TMA destinations must stay 128-byte aligned");

__global__ void __launch_bounds__(NT)
k_fine_gates_tma(const __grid_constant__ CUtensorMap mapWork, const __grid_constant__ CUtensorMap mapS,
                 FineArgs a, int ntx, int ntiles, const int* prev_count) {
    if (prev_count && *prev_count == 0) return;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    auto bufA = [&](int st) { return reinterpret_cast<float*>(smem_raw + st * FG_A_BYTES); };
    auto bufS = [&](int st) { return reinterpret_cast<float*>(smem_raw + 2 * FG_A_BYTES + st * FG_S_BYTES); };
    float* smB = reinterpret_cast<float*>(smem_raw + 2 * FG_A_BYTES + 2 * FG_S_BYTES);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + 2 * FG_A_BYTES + 2 * FG_S_BYTES + FG_B_BYTES);
    const int tid = threadIdx.x;
    if (tid == 0) {
        mbar_init(&full[0], 1);
        mbar_init(&full[1], 1);
        fence_mbar_init();
    }
    __syncthreads();
    auto issue = [&](int t, int st) {
        int ty = t / ntx, tx = t - ty * ntx;
        mbar_expect_tx(&full[st], FG_A_BYTES + FG_S_BYTES);
        tma_load_2d(bufA(st), &mapWork, tx * TW - FG_AX, ty * TH - FG_AY, &full[st]);
        tma_load_2d(bufS(st), &mapS, tx * TW - FG_SX, ty * TH - FG_SY, &full[st]);
    };
    int t = blockIdx.x;
    if (tid == 0 && t < ntiles) issue(t, 0);
    for (int it = 0; t < ntiles; t += gridDim.x, ++it) {
        const int st = it & 1;
        if (tid == 0 && t + (int)gridDim.x < ntiles) issue(t + gridDim.x, st ^ 1);
        mbar_wait(&full[st], (it >> 1) & 1);
        const int ty = t / ntx, tx = t - ty * ntx;
        const int x0 = tx * TW, y0 = ty * TH;
        if (y0 - FG_AY < 0 || y0 + TH + FG_AY > a.h || x0 - FG_AX < 0 || x0 + TW + FG_AX > a.w) {
            replicate_fix<FG_AROWS, FG_PA>(bufA(st), y0 - FG_AY, x0 - FG_AX, a.h, a.w, tid);
            replicate_fix<FG_SROWS, FG_PS>(bufS(st), y0 - FG_SY, x0 - FG_SX, a.h, a.w, tid);
            fence_proxy_async();
            __syncthreads();
        }
        fine_gates_tile(bufA(st), smB, bufS(st), a, x0, y0, tid);
        __syncthreads();   // stage st and smB are free again
    }
}

// ------------------------------------------------------------------------------------------------
// R21, second half of an iteration with an estimated gain: the S plane holds med5(work) (written by the
// residual pass); turn it into S in place, with L+, N and the A1 / A2 planes, using the gain the selection left
// on the device.  Same operations as noise_S_tile; no median here, so the pass is HBM bound (work and med5
// read, S written).  one_S_px: one pixel.
__device__ __forceinline__ float one_S_px(float c, float U, float D, float Lf, float R, float m5, float gain,
                                          const NoiseArgs& a, bool inframe, int j, uint32_t& n1, uint32_t& n2,
                                          float& lp, float& nn) {
    lp = lplus_px(c, U, D, Lf, R);
    nn = a.var ? noise_from_var(m5) : noise_px(m5, gain, a.rn2);   // R24: the plane holds the variance
    const float s = fdiv_nn(lp, __fmul_rn(2.0f, nn));
    const bool ok = inframe && (c < a.satlevel);                                         // R12
    n1 |= (uint32_t)(ok && s > a.sigclip) << j;
    n2 |= (uint32_t)(ok && s > a.siglow) << j;
    return s;
}

// w % 4 == 0: a warp owns 128 columns x SM5_ROWS rows; lane l keeps the four pixels x0 + 4 l .. + 3 of three
// consecutive rows in registers (sliding down), horizontal neighbours come from the adjacent lanes.
constexpr int SM5_ROWS = 16;
__global__ void __launch_bounds__(256)
k_S_from_m5(const float* __restrict__ work, NoiseArgs a, int nbx, const int* prev_count) {
    if (prev_count && *prev_count == 0) return;
    zero_counters(a);
    const int lane = threadIdx.x & 31, wi = threadIdx.x >> 5;
    const int h = a.h, w = a.w;
    const BlockXY bk = block_xy(nbx);
    const int x = bk.x * 128 + 4 * lane;
    const int ya = (bk.y * 8 + wi) * SM5_ROWS;
    if (ya >= h) return;                          // warp-uniform
    const bool inx = x < w;                       // w % 4 == 0: a quad is inside or outside as a whole
    const int xc = inx ? x : w - 4;               // out-of-frame lanes read a valid quad; results unused
    const float gain = a.gain_dev ? __ldg(a.gain_dev) : a.gain;
    auto ldrow = [&](int y) -> float4 {
        return __ldg(reinterpret_cast<const float4*>(work + (size_t)clampi(y, 0, h - 1) * w + xc));
    };
    float4 up = ldrow(ya - 1), cur = ldrow(ya), dn;
    const int yend = min(ya + SM5_ROWS, h);
    for (int y = ya; y < yend; ++y) {
        dn = ldrow(y + 1);
        const size_t o = (size_t)y * w + xc;
        const float4 m5 = *reinterpret_cast<const float4*>((a.var ? a.var : a.S) + o);
        float lf = __shfl_up_sync(0xffffffffu, cur.w, 1);          // R3: clamped at the frame edge
        float rt = __shfl_down_sync(0xffffffffu, cur.x, 1);
        if (lane == 0) lf = x > 0 ? __ldg(work + (size_t)y * w + x - 1) : cur.x;
        if (x + 4 >= w) rt = cur.w;
        else if (lane == 31) rt = __ldg(work + (size_t)y * w + x + 4);
        uint32_t n1 = 0, n2 = 0;
        float lp[4], nn[4], s[4];
        s[0] = one_S_px(cur.x, up.x, dn.x, lf, cur.y, m5.x, gain, a, inx, 0, n1, n2, lp[0], nn[0]);
        s[1] = one_S_px(cur.y, up.y, dn.y, cur.x, cur.z, m5.y, gain, a, inx, 1, n1, n2, lp[1], nn[1]);
        s[2] = one_S_px(cur.z, up.z, dn.z, cur.y, cur.w, m5.z, gain, a, inx, 2, n1, n2, lp[2], nn[2]);
        s[3] = one_S_px(cur.w, up.w, dn.w, cur.z, rt, m5.w, gain, a, inx, 3, n1, n2, lp[3], nn[3]);
        const uint32_t b1 = nibbles_to_word(n1, lane), b2 = nibbles_to_word(n2, lane);
        if (inx) {
            *reinterpret_cast<float4*>(a.S + o) = make_float4(s[0], s[1], s[2], s[3]);
            if (a.copy_out) *reinterpret_cast<float4*>(a.copy_out + o) = cur;
            if (a.dbgLp) store4(a.dbgLp, (size_t)y * w, x, w, lp);
            if (a.dbgN) store4(a.dbgN, (size_t)y * w, x, w, nn);
            if (a.A1 && (lane & 7) == 0) {
                const size_t q = (size_t)y * a.wpr + (x >> 5);
                const uint32_t keep = a.nok ? ~a.nok[q] : 0xffffffffu;
                a.A1[q] = b1 & keep;
                a.A2[q] = b2 & keep;
            }
        }
        up = cur;
        cur = dn;
    }
}

// any w: one thread per aligned group of 4 pixels, clamped scalar loads
__global__ void __launch_bounds__(256)
k_S_from_m5_generic(const float* __restrict__ work, NoiseArgs a, int nbx, const int* prev_count) {
    if (prev_count && *prev_count == 0) return;
    zero_counters(a);
    const int lane = threadIdx.x & 31, wi = threadIdx.x >> 5;
    const int h = a.h, w = a.w;
    const BlockXY bk = block_xy(nbx);
    const int x = bk.x * 128 + 4 * lane, y = bk.y * 8 + wi;
    if (y >= h) return;                           // warp-uniform
    const float gain = a.gain_dev ? __ldg(a.gain_dev) : a.gain;
    const float* rc = work + (size_t)y * w;
    const float* ru = work + (size_t)max(y - 1, 0) * w;
    const float* rd = work + (size_t)min(y + 1, h - 1) * w;
    float c[6];
#pragma unroll
    for (int k = 0; k < 6; ++k) c[k] = __ldg(rc + clampi(x - 1 + k, 0, w - 1));
    uint32_t n1 = 0, n2 = 0;
    float lp[4], nn[4], s[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int xj = min(x + j, w - 1);
        s[j] = one_S_px(c[1 + j], __ldg(ru + xj), __ldg(rd + xj), c[j], c[2 + j],
                        (a.var ? a.var : a.S)[(size_t)y * w + xj], gain, a, x + j < w, j, n1, n2, lp[j], nn[j]);
    }
    const uint32_t b1 = nibbles_to_word(n1, lane), b2 = nibbles_to_word(n2, lane);
    if (x < w) {
        const float ctr[4] = {c[1], c[2], c[3], c[4]};
        store4(a.S, (size_t)y * w, x, w, s);
        if (a.copy_out) store4(a.copy_out, (size_t)y * w, x, w, ctr);
        if (a.dbgLp) store4(a.dbgLp, (size_t)y * w, x, w, lp);
        if (a.dbgN) store4(a.dbgN, (size_t)y * w, x, w, nn);
        if (a.A1 && (lane & 7) == 0) {
            const size_t q = (size_t)y * a.wpr + (x >> 5);
            const uint32_t keep = a.nok ? ~a.nok[q] : 0xffffffffu;
            a.A1[q] = b1 & keep;
            a.A2[q] = b2 & keep;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Step (6) primitive on bit-planes (lacosmic_dilate3): out = dil3(in), pad bits cleared.  Thread layout of
// common.cuh (8 words of one column of words per thread; the horizontally dilated rows are shared between
// them).  The whole path runs the same word arithmetic inside k_grow_replace (grow.cuh).
__global__ void __launch_bounds__(256)
k_dilate3(const uint32_t* __restrict__ in, uint32_t* __restrict__ out, int h, int w, int wpr, int nbx) {
    const int lane = threadIdx.x & 31, wi = threadIdx.x >> 5;
    const BlockXY bk = block_xy(nbx);
    const int wx = bk.x * 32 + lane, y0 = bk.y * BW_CTA_ROWS + wi * BW_ROWS;
    if (wx >= wpr || y0 >= h) return;
    uint32_t res[BW_ROWS];
    dilate_rows<1>(in, y0, wx, h, wpr, res);
    const int rem = w - wx * 32;
    const uint32_t pad = rem >= 32 ? 0xffffffffu : ((1u << rem) - 1u);
#pragma unroll
    for (int i = 0; i < BW_ROWS; ++i)
        if (y0 + i < h) out[(size_t)(y0 + i) * wpr + wx] = res[i] & pad;
}

// ------------------------------------------------------------------------------------------------
// bit-plane <-> uint8 plane
__global__ void __launch_bounds__(256)
k_unpack_bits(const uint32_t* __restrict__ bits, uint8_t* __restrict__ u8, int h, int w, int wpr,
              const int* __restrict__ counts_src, int* __restrict__ counts_dst, int ncounts) {
    // epilogue of a frame: the per-iteration counts go to the caller's array in the same launch
    if (counts_dst && blockIdx.x == 0 && (int)threadIdx.x < ncounts) counts_dst[threadIdx.x] = counts_src[threadIdx.x];
    // 16 consecutive bytes of the flat uint8 plane per thread, aligned to 16 bytes of the destination (the
    // first thread starts at the first aligned address); a group may straddle two rows when w % 16 != 0
    const unsigned P = (unsigned)h * (unsigned)w;   // h * w < 2^31 (checked at the boundary): 32-bit index math
    const int lead = (int)((16 - (reinterpret_cast<uintptr_t>(u8) & 15)) & 15);
    const unsigned g = blockIdx.x * 256u + threadIdx.x;
    if (g == 0) {                                    // unaligned head of the plane
        for (int p = 0; p < lead && (unsigned)p < P; ++p) {
            const int y = p / w, x = p - y * w;
            u8[p] = (uint8_t)((bits[(size_t)y * wpr + (x >> 5)] >> (x & 31)) & 1u);
        }
    }
    if (g >= (P + 15u) / 16u + 1u) return;
    const unsigned p0 = (unsigned)lead + g * 16u;
    if (p0 >= P) return;
    const int y = (int)(p0 / (unsigned)w), x = (int)(p0 - (unsigned)y * (unsigned)w);
    if (x + 16 <= w && p0 + 16 <= P) {
        const uint32_t* row = bits + (size_t)y * wpr;
        const int wq = x >> 5, sh = x & 31;
        const uint32_t lo = row[wq], hi = (sh > 16 && wq + 1 < wpr) ? row[wq + 1] : 0u;
        const uint32_t half = __funnelshift_r(lo, hi, sh) & 0xffffu;
        uint32_t o[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const uint32_t nib = (half >> (4 * q)) & 0xfu;   // spread 4 bits into 4 bytes (0x01 each): the four
            o[q] = (nib * 0x00204081u) & 0x01010101u;        // shifted copies 0, 7, 14, 21 do not overlap
        }
        *reinterpret_cast<uint4*>(u8 + p0) = make_uint4(o[0], o[1], o[2], o[3]);
    } else {
        for (int j = 0; j < 16 && p0 + j < P; ++j) {
            const unsigned p = p0 + j;
            const int yy = (int)(p / (unsigned)w), xx = (int)(p - (unsigned)yy * (unsigned)w);
            u8[p] = (uint8_t)((bits[(size_t)yy * wpr + (xx >> 5)] >> (xx & 31)) & 1u);
        }
    }
}

__global__ void __launch_bounds__(256)
k_pack_bits(const uint8_t* __restrict__ u8, uint32_t* __restrict__ bits, int h, int w, int wpr, int nbx,
            uint32_t* __restrict__ or_into) {
    const BlockXY bk = block_xy(nbx);
    int x = bk.x * 256 + threadIdx.x, y = bk.y;
    bool b = (x < w) && (u8[(size_t)y * w + x] != 0);
    uint32_t word = __ballot_sync(0xffffffffu, b);
    if ((threadIdx.x & 31) == 0 && (x >> 5) < wpr) {
        bits[(size_t)y * wpr + (x >> 5)] = word;
        if (or_into) or_into[(size_t)y * wpr + (x >> 5)] |= word;      // R23: bad pixels join the never-flag plane
    }
}

// bits = (img >= level) (R25: the saturated pixels of the input frame)
__global__ void __launch_bounds__(256)
k_pack_ge(const float* __restrict__ img, float level, uint32_t* __restrict__ bits, int h, int w, int wpr, int nbx) {
    const BlockXY bk = block_xy(nbx);
    int x = bk.x * 256 + threadIdx.x, y = bk.y;
    bool b = (x < w) && (img[(size_t)y * w + x] >= level);
    uint32_t word = __ballot_sync(0xffffffffu, b);
    if ((threadIdx.x & 31) == 0 && (x >> 5) < wpr) bits[(size_t)y * wpr + (x >> 5)] = word;
}

// R25: core = (med5(img) >= satlevel) from the bit-plane sat = (img >= satlevel): the median of the 25 clamped taps
// reaches the level iff at least 13 of them do.  One thread per word; a word with no saturated pixel within two rows and
// one word of it (almost every word of a frame) is zero without looking at single pixels.
__global__ void __launch_bounds__(256)
k_satcore(const uint32_t* __restrict__ sat, uint32_t* __restrict__ core, int h, int w, int wpr, int nbx) {
    const BlockXY bk = block_xy(nbx);
    const int wx = bk.x * 256 + threadIdx.x, y = bk.y;
    if (wx >= wpr) return;
    const int wl = max(wx - 1, 0), wr = min(wx + 1, wpr - 1);
    uint32_t any = 0;
#pragma unroll
    for (int dy = -2; dy <= 2; ++dy) {
        const uint32_t* row = sat + (size_t)clampi(y + dy, 0, h - 1) * wpr;
        any |= row[wl] | row[wx] | row[wr];
    }
    uint32_t out = 0;
    if (any) {
        for (int b = 0; b < 32; ++b) {
            const int x = wx * 32 + b;
            if (x >= w) break;
            int cnt = 0;
            for (int dy = -2; dy <= 2; ++dy) {
                const uint32_t* row = sat + (size_t)clampi(y + dy, 0, h - 1) * wpr;
                for (int dx = -2; dx <= 2; ++dx) {
                    const int xx = clampi(x + dx, 0, w - 1);
                    cnt += (row[xx >> 5] >> (xx & 31)) & 1u;
                }
            }
            out |= (uint32_t)(cnt >= 13) << b;
        }
    }
    core[(size_t)y * wpr + wx] = out;
}

}  // namespace lac
