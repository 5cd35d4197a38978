// Common device helpers for the L.A.Cosmic sm_100a kernels.
// No code here is shared with oracle/ (the CPU oracle is an independent C file).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace lac {

__device__ __forceinline__ int clampi(int v, int lo, int hi) { return min(max(v, lo), hi); }

// Programmatic dependent launch (the kernels of a lazy frame are launched with the programmatic-stream-serialization
// attribute): let the NEXT kernel of the stream be scheduled while this one runs, then wait until the PREVIOUS one has
// completed and its writes are visible.  Every thread calls this before its first global access, so the frame's kernels
// still execute in order; what overlaps is the launch and the scheduling of the next grid with the tail of this one.
// Without the attribute both instructions do nothing.
__device__ __forceinline__ void pdl_entry() {
    asm volatile("griddepcontrol.launch_dependents;");
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

// 2-D CTA coordinates out of a 1-D grid of nbx * nby CTAs: gridDim.y stops at 65535, which a tall, narrow frame
// (rows on y) would exceed; gridDim.x reaches 2^31 - 1, enough for every shape the boundary accepts.
struct BlockXY { int x, y; };
__device__ __forceinline__ BlockXY block_xy(int nbx) {
    BlockXY b;
    b.y = (int)(blockIdx.x / (unsigned)nbx);
    b.x = (int)(blockIdx.x - (unsigned)b.y * (unsigned)nbx);
    return b;
}

// compare-exchange: a <- min, b <- max (two FMNMX on the ALU pipe)
__device__ __forceinline__ void ce(float& a, float& b) {
    float t = fminf(a, b);
    b = fmaxf(a, b);
    a = t;
}

// 3-input min / max: one FMNMX3 each on sm_100a
__device__ __forceinline__ float min3(float a, float b, float c) {
    float r;
    asm("min.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));
    return r;
}
__device__ __forceinline__ float max3(float a, float b, float c) {
    float r;
    asm("max.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));
    return r;
}

// exact median of three
__device__ __forceinline__ float med3(float a, float b, float c) {
    return fmaxf(fminf(a, b), fminf(fmaxf(a, b), c));
}

// Edge-replicate tile load (R3): sm[r][c] = src<y0-R+r, x0-R+c>, r < TH+2R, c < TW+2R.
template <int TW, int TH, int R, int PITCH, int NT>
__device__ __forceinline__ void load_tile_clamped(float* sm, const float* __restrict__ src, int h,
                                                  int w, int y0, int x0, int tid) {
    constexpr int SW = TW + 2 * R, SH = TH + 2 * R;
    for (int i = tid; i < SW * SH; i += NT) {
        int r = i / SW, c = i - r * SW;
        int yy = clampi(y0 - R + r, 0, h - 1), xx = clampi(x0 - R + c, 0, w - 1);
        sm[r * PITCH + c] = __ldg(src + (size_t)yy * w + xx);
    }
}

// Step (1), O1: L+ from the centre and its four edge-replicated neighbours.
// Operation order is normative (bit-exact against the oracle); no FMA contraction.
__device__ __forceinline__ float lplus_px(float c, float U, float D, float Lf, float R) {
    float two = __fmul_rn(2.0f, c);
    float a = __fsub_rn(two, __fadd_rn(U, Lf));
    float b = __fsub_rn(two, __fadd_rn(U, R));
    float g = __fsub_rn(two, __fadd_rn(D, Lf));
    float d = __fsub_rn(two, __fadd_rn(D, R));
    a = a > 0.0f ? a : 0.0f;
    b = b > 0.0f ? b : 0.0f;
    g = g > 0.0f ? g : 0.0f;
    d = d > 0.0f ? d : 0.0f;
    return __fmul_rn(__fadd_rn(__fadd_rn(a, b), __fadd_rn(g, d)), 0.25f);
}

// fdiv(num, den) for num >= +0 and den > 0: the value of __fdiv_rn(num, den), but a zero numerator (about 30 %
// of the L+ values) does not take the division's slow path, which the range check of the fast path (FCHK)
// sends it to: +0 / den = +0 for every den > 0, infinity included.  Both callers have den > 0: den = 2N with
// N >= 1e-2 / sqrt(gain) > 0 for every finite positive gain (med5 is floored at 1e-4, R5), and den = F >= 0.01.
__device__ __forceinline__ uint32_t sign01(float v) {   // sign bit as 0 / 1 (IMAD.HI: FMA pipe, not the ALU pipe)
    uint32_t r;
    asm("mul.hi.u32 %0, %1, 2;" : "=r"(r) : "r"(__float_as_uint(v)));
    return r;
}
__device__ __forceinline__ float fdiv_nn(float num, float den) {
    // (measured: doing the zero test and the two selections as FMA-pipe arithmetic saves 3 ALU-pipe instructions per
    // pixel but lengthens the dependent chain in front of the division -- 0.210 vs 0.204 ms for the dense pass)
    const bool z = num == 0.0f;
    const float q = __fdiv_rn(z ? 1.0f : num, den);
    return z ? 0.0f : q;
}

// O2: N = sqrt(gain * max(med5, 1e-4) + rn^2) / gain.  gain == 1 (uniform) skips the multiply and the
// division, which are exact identities then.
__device__ __forceinline__ float noise_px(float m5, float gain, float rn2) {
    const float m5c = m5 > 1e-4f ? m5 : 1e-4f;                                            // R5
    if (gain == 1.0f) return __fsqrt_rn(__fadd_rn(m5c, rn2));
    return __fdiv_rn(__fsqrt_rn(__fadd_rn(__fmul_rn(gain, m5c), rn2)), gain);
}

// ---- block-wide compaction of bit-plane words into a pixel list ------------------------------------
// Bit-plane kernels use 256-thread CTAs (32 lanes x 8 warps); thread (lane, wi) owns NR words of one word
// column (word wx, rows y .. y+NR-1).  All 256 threads must call block_append: it appends the flat pixel
// index p0 + i*w + k of every set bit k of bits[i] (one atomicAdd per CTA: same-address atomics serialise
// in L2, so they are aggregated per CTA).  Contains block barriers; a second call in the same kernel must
// be separated from the first by __syncthreads().
constexpr int BW_ROWS = 8;
constexpr int BW_CTA_ROWS = 64;

template <int NR>
__device__ __forceinline__ void block_append(const uint32_t (&bits)[NR], int p0, int w,
                                             int* __restrict__ list, int* __restrict__ nlist) {
    __shared__ int s_warp[8];
    __shared__ int s_base;
    const int lane = threadIdx.x & 31, wi = threadIdx.x >> 5;
    int n = 0;
#pragma unroll
    for (int i = 0; i < NR; ++i) n += __popc(bits[i]);
    int incl = n;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        int o = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += o;
    }
    if (lane == 31) s_warp[wi] = incl;
    __syncthreads();
    if (threadIdx.x == 0) {
        int tot = 0;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            int c = s_warp[i];
            s_warp[i] = tot;
            tot += c;
        }
        s_base = tot ? atomicAdd(nlist, tot) : 0;
    }
    __syncthreads();
    int base = s_base + s_warp[wi] + incl - n;
#pragma unroll
    for (int i = 0; i < NR; ++i) {
        uint32_t b = bits[i];
        const int pi = p0 + i * w;
        while (b) {
            int k = __ffs(b) - 1;
            b &= b - 1;
            list[base++] = pi + k;
        }
    }
}

// horizontal dilation by R pixels of the word vc given its left / right neighbour words
template <int R>
__device__ __forceinline__ uint32_t hdil(uint32_t vl, uint32_t vc, uint32_t vr) {
    uint32_t o = vc;
#pragma unroll
    for (int k = 1; k <= R; ++k) o |= (vc << k) | (vc >> k) | (vl >> (32 - k)) | (vr << (32 - k));
    return o;
}

// (2R+1) x (2R+1) dilation of a bit-plane at the BW_ROWS words a thread owns (rows y0 .. y0+BW_ROWS-1,
// word column wx; outside the frame = 0): horizontally dilated rows are shared between the outputs
template <int R>
__device__ __forceinline__ void dilate_rows(const uint32_t* __restrict__ in, int y0, int wx, int h, int wpr,
                                            uint32_t (&out)[BW_ROWS]) {
    uint32_t hd[BW_ROWS + 2 * R];
    const int wl = max(wx - 1, 0), wr = min(wx + 1, wpr - 1);
#pragma unroll
    for (int r = 0; r < BW_ROWS + 2 * R; ++r) {
        // branch-free: clamped addresses, masked values (all loads of a thread are in flight together)
        const int yy = y0 - R + r;
        const bool ok = (yy >= 0) & (yy < h);
        const uint32_t* row = in + (size_t)clampi(yy, 0, h - 1) * wpr;
        const uint32_t vl = row[wl], vc = row[wx], vr = row[wr];
        hd[r] = hdil<R>((ok & (wx > 0)) ? vl : 0u, ok ? vc : 0u, (ok & (wx + 1 < wpr)) ? vr : 0u);
    }
#pragma unroll
    for (int i = 0; i < BW_ROWS; ++i) {
        uint32_t o = 0;
#pragma unroll
        for (int r = 0; r <= 2 * R; ++r) o |= hd[i + r];
        out[i] = o;
    }
}

}  // namespace lac
