// sm_100a kernels of the L.A.Cosmic iteration (DESIGN.md section 5 lists each with its roofline).
#pragma once
#include "common.cuh"
#include "median_select.cuh"

namespace lac {

constexpr int TW = 64;    // output tile width  (two ballot words)
constexpr int TH = 32;    // output tile height
constexpr int NT = 256;   // threads per CTA, laid out 32 x 8
constexpr int PX = TW / 32;
constexpr int PY = TH / 8;

struct GateParams {
    float sigclip, siglow, objlim, satlevel;
};

// median of the K x K window centred at tile-local (r, c) of a shared-memory tile (r, c already
// include the halo offset)
template <int K, int PITCH>
__device__ __forceinline__ float median_window(const float* sm, int r, int c) {
    constexpr int R = K / 2;
    float v[K * K];
#pragma unroll
    for (int dy = 0; dy < K; ++dy)
#pragma unroll
        for (int dx = 0; dx < K; ++dx) v[dy * K + dx] = sm[(r - R + dy) * PITCH + (c - R + dx)];
    return median_forgetful<K * K>(v);
}

// ------------------------------------------------------------------------------------------------
// Standalone k x k median (lacosmic_medfilt; also the dense reference for the fused kernels).
template <int K>
__global__ void __launch_bounds__(NT) k_medfilt(const float* __restrict__ in, float* __restrict__ out,
                                               int h, int w) {
    constexpr int R = K / 2, PITCH = TW + 2 * R + 1;
    __shared__ float sm[(TH + 2 * R) * PITCH];
    const int tid = threadIdx.y * 32 + threadIdx.x;
    const int x0 = blockIdx.x * TW, y0 = blockIdx.y * TH;
    load_tile_clamped<TW, TH, R, PITCH, NT>(sm, in, h, w, y0, x0, tid);
    __syncthreads();
#pragma unroll 1
    for (int j = 0; j < PY; ++j)
#pragma unroll 1
        for (int i = 0; i < PX; ++i) {
            int ly = threadIdx.y + 8 * j, lx = threadIdx.x + 32 * i;
            int y = y0 + ly, x = x0 + lx;
            if (y < h && x < w) out[(size_t)y * w + x] = median_window<K, PITCH>(sm, ly + R, lx + R);
        }
}

// Standalone L+ (lacosmic_lplus).
__global__ void __launch_bounds__(NT) k_lplus(const float* __restrict__ in, float* __restrict__ out,
                                             int h, int w) {
    int x = blockIdx.x * 32 + threadIdx.x, y = blockIdx.y * 8 + threadIdx.y;
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
__global__ void __launch_bounds__(NT)
k_noise_S(const float* __restrict__ work, float* __restrict__ S, float* __restrict__ dbgLp,
          float* __restrict__ dbgN, int h, int w, float gain, float rn2, const int* prev_count) {
    if (prev_count && *prev_count == 0) return;   // fixed point reached (R17)
    constexpr int R = 2, PITCH = TW + 2 * R + 1;
    __shared__ float sm[(TH + 2 * R) * PITCH];
    const int tid = threadIdx.y * 32 + threadIdx.x;
    const int x0 = blockIdx.x * TW, y0 = blockIdx.y * TH;
    load_tile_clamped<TW, TH, R, PITCH, NT>(sm, work, h, w, y0, x0, tid);
    __syncthreads();
#pragma unroll 1
    for (int j = 0; j < PY; ++j)
#pragma unroll 1
        for (int i = 0; i < PX; ++i) {
            int ly = threadIdx.y + 8 * j, lx = threadIdx.x + 32 * i;
            int y = y0 + ly, x = x0 + lx;
            if (y >= h || x >= w) continue;
            int r = ly + R, c = lx + R;
            float m5 = median_window<5, PITCH>(sm, r, c);
            float lp = lplus_px(sm[r * PITCH + c], sm[(r - 1) * PITCH + c], sm[(r + 1) * PITCH + c],
                                sm[r * PITCH + c - 1], sm[r * PITCH + c + 1]);
            float m5c = m5 > 1e-4f ? m5 : 1e-4f;                                  // R5
            float n = __fdiv_rn(__fsqrt_rn(__fadd_rn(__fmul_rn(gain, m5c), rn2)), gain);
            float s = __fdiv_rn(lp, __fmul_rn(2.0f, n));
            size_t p = (size_t)y * w + x;
            S[p] = s;
            if (dbgLp) dbgLp[p] = lp;
            if (dbgN) dbgN[p] = n;
        }
}

// K_B: steps (3b)-(5).  S' = S - med5(S); m3 = med3(work) (tile in shared memory, replicated at the
// frame border as a STORED plane would be, R4); F = max(m3 - med7(m3), 0.01); gates -> bit-planes.
__global__ void __launch_bounds__(NT)
k_fine_gates(const float* __restrict__ work, const float* __restrict__ S, uint32_t* __restrict__ G1,
             uint32_t* __restrict__ G2, uint32_t* __restrict__ M1, float* __restrict__ dbgSp,
             float* __restrict__ dbgM3, float* __restrict__ dbgF, int h, int w, int wpr,
             GateParams gp, const int* prev_count) {
    if (prev_count && *prev_count == 0) return;
    constexpr int RA = 4, PA = TW + 2 * RA + 1;   // work tile, halo 4
    constexpr int RB = 3, PB = TW + 2 * RB + 1;   // m3 tile, halo 3
    constexpr int RS = 2, PS = TW + 2 * RS + 1;   // S tile, halo 2
    __shared__ float smA[(TH + 2 * RA) * PA];
    __shared__ float smB[(TH + 2 * RB) * PB];
    __shared__ float smS[(TH + 2 * RS) * PS];
    const int tid = threadIdx.y * 32 + threadIdx.x;
    const int x0 = blockIdx.x * TW, y0 = blockIdx.y * TH;
    load_tile_clamped<TW, TH, RA, PA, NT>(smA, work, h, w, y0, x0, tid);
    load_tile_clamped<TW, TH, RS, PS, NT>(smS, S, h, w, y0, x0, tid);
    __syncthreads();
    {
        constexpr int BW = TW + 2 * RB, BH = TH + 2 * RB;
        for (int i = tid; i < BW * BH; i += NT) {
            int r = i / BW, c = i - r * BW;
            int cy = clampi(y0 - RB + r, 0, h - 1), cx = clampi(x0 - RB + c, 0, w - 1);
            int ar = cy - (y0 - RA), ac = cx - (x0 - RA);
            smB[r * PB + c] = median_window<3, PA>(smA, ar, ac);
        }
    }
    __syncthreads();
#pragma unroll 1
    for (int j = 0; j < PY; ++j)
#pragma unroll 1
        for (int i = 0; i < PX; ++i) {
            int ly = threadIdx.y + 8 * j, lx = threadIdx.x + 32 * i;
            int y = y0 + ly, x = x0 + lx;
            bool inside = (y < h) && (x < w);
            bool g1 = false, g2 = false, m1 = false;
            if (inside) {
                float s = smS[(ly + RS) * PS + lx + RS];
                float sp = __fsub_rn(s, median_window<5, PS>(smS, ly + RS, lx + RS));
                float m3 = smB[(ly + RB) * PB + lx + RB];
                float f = __fsub_rn(m3, median_window<7, PB>(smB, ly + RB, lx + RB));
                f = f > 0.01f ? f : 0.01f;
                int r = ly + RA, c = lx + RA;
                float ctr = smA[r * PA + c];
                float lp = lplus_px(ctr, smA[(r - 1) * PA + c], smA[(r + 1) * PA + c],
                                    smA[r * PA + c - 1], smA[r * PA + c + 1]);
                bool ok = ctr < gp.satlevel;                                  // R12
                g1 = ok && (sp > gp.sigclip);
                g2 = ok && (sp > gp.siglow);
                m1 = g1 && (__fdiv_rn(lp, f) > gp.objlim);                    // R8
                size_t p = (size_t)y * w + x;
                if (dbgSp) dbgSp[p] = sp;
                if (dbgM3) dbgM3[p] = m3;
                if (dbgF) dbgF[p] = f;
            }
            uint32_t b1 = __ballot_sync(0xffffffffu, g1);
            uint32_t b2 = __ballot_sync(0xffffffffu, g2);
            uint32_t b3 = __ballot_sync(0xffffffffu, m1);
            int wx = (x0 >> 5) + i;
            if (threadIdx.x == 0 && y < h && wx < wpr) {
                size_t q = (size_t)y * wpr + wx;
                G1[q] = b1;
                G2[q] = b2;
                M1[q] = b3;
            }
        }
}

// ------------------------------------------------------------------------------------------------
// Step (6) primitive on bit-planes: out = dil3(in) & gate.  One thread per 32-pixel word; the left
// and right neighbour words come from the adjacent lanes by shuffle (lanes at a warp edge load
// them).  If Cio is given: count += popc(out & ~C); C |= out  (R11).
__global__ void __launch_bounds__(256)
k_dilate_gate(const uint32_t* __restrict__ in, const uint32_t* __restrict__ gate,
              uint32_t* __restrict__ out, uint32_t* __restrict__ Cio, int* __restrict__ count, int h,
              int w, int wpr, const int* prev_count) {
    if (prev_count && *prev_count == 0) return;
    const int lane = threadIdx.x & 31;
    int wx = blockIdx.x * 32 + lane;
    int y = blockIdx.y * 8 + (threadIdx.x >> 5);
    uint32_t v = 0, res = 0;
    bool valid = (wx < wpr) && (y < h);
    if (valid) {
        v = in[(size_t)y * wpr + wx];
        if (y > 0) v |= in[(size_t)(y - 1) * wpr + wx];
        if (y + 1 < h) v |= in[(size_t)(y + 1) * wpr + wx];
    }
    uint32_t vl = __shfl_up_sync(0xffffffffu, v, 1), vr = __shfl_down_sync(0xffffffffu, v, 1);
    if (valid) {
        if (lane == 0) {
            vl = 0;
            if (wx > 0) {
                vl = in[(size_t)y * wpr + wx - 1];
                if (y > 0) vl |= in[(size_t)(y - 1) * wpr + wx - 1];
                if (y + 1 < h) vl |= in[(size_t)(y + 1) * wpr + wx - 1];
            }
        }
        if (lane == 31 || wx + 1 >= wpr) {
            vr = 0;
            if (wx + 1 < wpr) {
                vr = in[(size_t)y * wpr + wx + 1];
                if (y > 0) vr |= in[(size_t)(y - 1) * wpr + wx + 1];
                if (y + 1 < h) vr |= in[(size_t)(y + 1) * wpr + wx + 1];
            }
        }
        res = v | (v << 1) | (v >> 1) | (vl >> 31) | (vr << 31);
        uint32_t g;
        if (gate) g = gate[(size_t)y * wpr + wx];
        else {   // no gate: only clear the pad bits beyond column w-1
            int rem = w - wx * 32;
            g = rem >= 32 ? 0xffffffffu : ((1u << rem) - 1u);
        }
        res &= g;
        out[(size_t)y * wpr + wx] = res;
    }
    if (Cio) {
        int n = 0;
        if (valid) {
            uint32_t c = Cio[(size_t)y * wpr + wx];
            n = __popc(res & ~c);
            if (res & ~c) Cio[(size_t)y * wpr + wx] = c | res;
        }
        n = __reduce_add_sync(0xffffffffu, n);
        if (lane == 0 && n) atomicAdd(count, n);
    }
}

// ------------------------------------------------------------------------------------------------
// Step (7): sparse masked-median replacement.  A warp owns 32 consecutive words of the cumulative
// mask C; the non-empty words are found by ballot and their set bits walked one pixel at a time.
// For a pixel the 25 taps sit on lanes 0..24; each lane ranks its tap among the donors by 25
// shuffles (ties broken by lane so ranks are a permutation), and the lanes holding the middle
// rank(s) supply the median (R13-R16).  Reads only img_in and C, writes only work.
__global__ void __launch_bounds__(256)
k_replace(const float* __restrict__ img, const uint32_t* __restrict__ Cb, float* __restrict__ work,
          int h, int w, int wpr, const int* prev_count) {
    if (prev_count && *prev_count == 0) return;
    const int lane = threadIdx.x & 31;
    const long long nwords = (long long)h * wpr;
    long long base = ((long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5)) * 32;
    if (base >= nwords) return;
    long long mine = base + lane;
    uint32_t cw = mine < nwords ? Cb[mine] : 0u;
    uint32_t nz = __ballot_sync(0xffffffffu, cw != 0u);
    const int dy = lane / 5 - 2, dx = lane % 5 - 2;   // lanes >= 25 idle in the vote
    while (nz) {
        int src = __ffs(nz) - 1;
        nz &= nz - 1;
        uint32_t word = __shfl_sync(0xffffffffu, cw, src);
        long long idx = base + src;
        int y = (int)(idx / wpr), wx = (int)(idx - (long long)y * wpr);
        while (word) {
            int b = __ffs(word) - 1;
            word &= word - 1;
            int x = wx * 32 + b;
            float val = 0.0f;
            bool donor = false;
            if (lane < 25) {
                int yy = clampi(y + dy, 0, h - 1), xx = clampi(x + dx, 0, w - 1);
                val = __ldg(img + (size_t)yy * w + xx);
                donor = !((Cb[(size_t)yy * wpr + (xx >> 5)] >> (xx & 31)) & 1u);
            }
            uint32_t dm = __ballot_sync(0xffffffffu, donor);
            if (dm == 0u) dm = 0x01ffffffu;            // R15: no donor -> all 25 taps
            const int k = __popc(dm);
            int rank = 0;
#pragma unroll
            for (int t = 0; t < 25; ++t) {
                float vt = __shfl_sync(0xffffffffu, val, t);
                bool before = (vt < val) || (vt == val && t < lane);
                rank += (((dm >> t) & 1u) && before) ? 1 : 0;
            }
            bool mineIn = (dm >> lane) & 1u;
            uint32_t hiM = __ballot_sync(0xffffffffu, mineIn && rank == (k >> 1));
            uint32_t loM = __ballot_sync(0xffffffffu, mineIn && rank == (k >> 1) - 1);
            float hi = __shfl_sync(0xffffffffu, val, __ffs(hiM) - 1);
            float lo = __shfl_sync(0xffffffffu, val, (k & 1) ? 0 : __ffs(loM) - 1);
            float r = (k & 1) ? hi : __fmul_rn(__fadd_rn(lo, hi), 0.5f);   // R14
            if (lane == 0) work[(size_t)y * w + x] = r;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// bit-plane <-> uint8 plane
__global__ void __launch_bounds__(256)
k_unpack_bits(const uint32_t* __restrict__ bits, uint8_t* __restrict__ u8, int h, int w, int wpr) {
    int x = blockIdx.x * 256 + threadIdx.x, y = blockIdx.y;
    if (x >= w) return;
    u8[(size_t)y * w + x] = (uint8_t)((bits[(size_t)y * wpr + (x >> 5)] >> (x & 31)) & 1u);
}

__global__ void __launch_bounds__(256)
k_pack_bits(const uint8_t* __restrict__ u8, uint32_t* __restrict__ bits, int h, int w, int wpr) {
    int x = blockIdx.x * 256 + threadIdx.x, y = blockIdx.y;
    bool b = (x < w) && (u8[(size_t)y * w + x] != 0);
    uint32_t word = __ballot_sync(0xffffffffu, b);
    if ((threadIdx.x & 31) == 0 && (x >> 5) < wpr) bits[(size_t)y * wpr + (x >> 5)] = word;
}

}  // namespace lac
