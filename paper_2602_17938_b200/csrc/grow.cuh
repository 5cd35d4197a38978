// Steps (6)-(7) fused, and the bit-plane pass that opens an incremental iteration.
//
// k_grow_replace: one CTA per 1024 x 32 pixel tile of the bit-planes, staged in shared memory with a halo
// of 4 rows / 1 word, does
//     M2 = dil3(M1) & G1                                   on tile + 3 px
//     G2 where the second growth reads it and it is not known yet (lazy path only)   on tile + 2 px
//     M3 = dil3(M2) & G2,  fresh = M3 & ~C,  C' = C | M3   on tile + 2 px
//     need = dil5x5(fresh) & C'                            on the tile
//     work[p] = masked 5x5 median of img_in around p       for p in need
// Every quantity in the halo is recomputed from the same inputs by the neighbouring CTA (bit arithmetic,
// and a handful of redundant G2 evaluations), so there is no exchange between CTAs and the six launches
// of the unfused sequence (dilate, list, evaluate, dilate, list, replace) become one.  C is double
// buffered (read `Cold`, write `Cnew`) because a neighbour still reads the old plane in its halo.
#pragma once
#include "common.cuh"
#include "lazy_count.cuh"
#include "median_networks.cuh"

namespace lac {

constexpr int GT_W = 32;                      // tile width in 32-px words
constexpr int GT_H = 32;                      // tile height in rows
constexpr int GT_HALO = 4;                    // halo rows (and pixels: one halo word on each side)
constexpr int GS_W = GT_W + 2, GS_H = GT_H + 2 * GT_HALO, GS_N = GS_W * GS_H;
constexpr int G_CAP = 2048;                   // shared pixel list capacity per compaction round

// haloed tile of a bit-plane into shared memory; outside the frame (and for a null plane) = 0
__device__ __forceinline__ void load_bits_tile(uint32_t* sm, const uint32_t* __restrict__ g, int y0, int wx0,
                                               int h, int wpr, int tid) {
    for (int i = tid; i < GS_N; i += 256) {
        const int r = i / GS_W, c = i - r * GS_W;
        const int y = y0 - GT_HALO + r, wx = wx0 - 1 + c;
        const bool ok = (y >= 0) & (y < h) & (wx >= 0) & (wx < wpr);
        uint32_t v = 0;
        if (g) v = g[(size_t)clampi(y, 0, h - 1) * wpr + clampi(wx, 0, wpr - 1)];   // branch-free address
        sm[i] = ok ? v : 0u;
    }
}

// horizontally dilated word (r, c) of a shared tile; words beyond the tile's halo read as 0 (only the
// outer bits of the halo words depend on them, and no result of the own tile depends on those)
template <int R>
__device__ __forceinline__ uint32_t hdil_sm(const uint32_t* sm, int r, int c) {
    const uint32_t* row = sm + r * GS_W;
    return hdil<R>(c > 0 ? row[c - 1] : 0u, row[c], c + 1 < GS_W ? row[c + 1] : 0u);
}

// One compaction round: every thread offers the set bits of its words (code = tile-local word index * 32 +
// bit); up to G_CAP of them are written to s_list, the bits that did not fit stay in `bits` for the next
// round.  Returns the number of entries.  Contains block barriers.
template <int NW>
__device__ __forceinline__ int smem_compact(uint32_t (&bits)[NW], const int (&widx)[NW], int* s_cnt, int* s_list,
                                            int tid) {
    if (tid == 0) *s_cnt = 0;
    __syncthreads();
#pragma unroll
    for (int k = 0; k < NW; ++k) {
        uint32_t b = bits[k];
        if (b) {
            int slot = atomicAdd(s_cnt, __popc(b));
            while (b && slot < G_CAP) {
                const int bit = __ffs(b) - 1;
                b &= b - 1;
                s_list[slot++] = widx[k] * 32 + bit;
            }
            bits[k] = b;
        }
    }
    __syncthreads();
    return min(*s_cnt, G_CAP);
}

struct GrowArgs {
    const uint32_t *M1, *G1;
    uint32_t* G2;                 // lazy path: completed where step (6) reads it (own words rewritten)
    const uint32_t *A1, *A2;      // lazy path: S > sigclip / S > siglow planes; null: G2 is complete
    const uint32_t* Cold;
    uint32_t* Cnew;
    uint32_t* NEED;               // pixels rewritten in `work` by this launch
    uint32_t *M2out, *M3out;      // nullable (debug planes)
    const float* S;
    const float* img;             // img_in: donor values (R13)
    float* work;
    int* count;                   // += |M3 & ~C|
    int h, w, wpr;
    float siglow;
};

__global__ void __launch_bounds__(256)
k_grow_replace(GrowArgs a, const int* prev_count) {
    const int tid = threadIdx.x, lane = tid & 31, wi = tid >> 5;
    const int wx0 = blockIdx.x * GT_W, y0 = blockIdx.y * GT_H;
    const int h = a.h, w = a.w, wpr = a.wpr;
    if (prev_count && *prev_count == 0) {
        // fixed point (R17): nothing changes; carry C over to the plane the next reader expects
        for (int i = tid; i < GT_W * GT_H; i += 256) {
            const int y = y0 + i / GT_W, wx = wx0 + i % GT_W;
            if (y < h && wx < wpr) a.Cnew[(size_t)y * wpr + wx] = a.Cold[(size_t)y * wpr + wx];
        }
        return;
    }
    __shared__ uint32_t sA[GS_N];    // M1, then D = dil3(M2)
    __shared__ uint32_t sB[GS_N];    // G1, then M2
    __shared__ uint32_t sC[GS_N];    // C, then C'
    __shared__ uint32_t sG2[GS_N];
    __shared__ uint32_t sN[GS_N];    // A1, then fresh
    __shared__ uint32_t sA2[GS_N];
    __shared__ int s_list[G_CAP];
    __shared__ int s_cnt;
    __shared__ int s_red[8];
    const bool lazy = a.A2 != nullptr;
    load_bits_tile(sA, a.M1, y0, wx0, h, wpr, tid);
    load_bits_tile(sB, a.G1, y0, wx0, h, wpr, tid);
    load_bits_tile(sC, a.Cold, y0, wx0, h, wpr, tid);
    load_bits_tile(sG2, a.G2, y0, wx0, h, wpr, tid);
    if (lazy) {
        load_bits_tile(sN, a.A1, y0, wx0, h, wpr, tid);
        load_bits_tile(sA2, a.A2, y0, wx0, h, wpr, tid);
    }
    __syncthreads();
    // M2 = dil3(M1) & G1 on rows 1 .. GS_H-2 (in place of G1: each element is read by its writer only)
    for (int i = tid + GS_W; i < GS_N - GS_W; i += 256) {
        const int r = i / GS_W, c = i - r * GS_W;
        sB[i] = (hdil_sm<1>(sA, r - 1, c) | hdil_sm<1>(sA, r, c) | hdil_sm<1>(sA, r + 1, c)) & sB[i];
    }
    __syncthreads();
    // D = dil3(M2) on rows 2 .. GS_H-3 (over M1, which is dead); pixels whose G2 is still unknown
    constexpr int NWD = ((GS_H - 4) * GS_W + 255) / 256;
    uint32_t nb[NWD];
    int nbw[NWD];
#pragma unroll
    for (int k = 0; k < NWD; ++k) {
        const int i = 2 * GS_W + tid + k * 256;
        nb[k] = 0;
        nbw[k] = i;
        if (i < GS_N - 2 * GS_W) {
            const int r = i / GS_W, c = i - r * GS_W;
            const uint32_t d = hdil_sm<1>(sB, r - 1, c) | hdil_sm<1>(sB, r, c) | hdil_sm<1>(sB, r + 1, c);
            sA[i] = d;
            if (lazy) {
                // only within 2 px of the own tile: the neighbouring CTAs evaluate the rest
                const uint32_t keep = c == 0 ? 0xC0000000u : c == GS_W - 1 ? 0x00000003u : 0xffffffffu;
                nb[k] = d & sA2[i] & ~sN[i] & ~sG2[i] & keep;
            }
        }
    }
    if (lazy) {
        // G2 = (S' > siglow) at those pixels, by counting (lazy_count.cuh); rounds of at most G_CAP pixels
        for (;;) {
            const int n = smem_compact(nb, nbw, &s_cnt, s_list, tid);
            for (int i = tid; i < n; i += 256) {
                const int code = s_list[i], wd = code >> 5, bit = code & 31;
                const int r = wd / GS_W, c = wd - r * GS_W;
                const int y = y0 - GT_HALO + r, x = (wx0 - 1 + c) * 32 + bit;
                int c1, c2;
                count_sp(a.S, y, x, h, w, a.siglow, a.siglow, c1, c2);
                if (c2 >= 13) atomicOr(&sG2[wd], 1u << bit);
            }
            bool more = false;
#pragma unroll
            for (int k = 0; k < NWD; ++k) more |= nb[k] != 0;
            if (!__syncthreads_or(more)) break;
        }
    } else {
        __syncthreads();
    }
    // M3 = D & G2; fresh = M3 & ~C; C' = C | M3 on rows 2 .. GS_H-3
    int nfresh = 0;
    for (int i = 2 * GS_W + tid; i < GS_N - 2 * GS_W; i += 256) {
        const int r = i / GS_W, c = i - r * GS_W;
        const uint32_t m3 = sA[i] & sG2[i], cold = sC[i], fresh = m3 & ~cold;
        sC[i] = cold | m3;
        sN[i] = fresh;
        const int y = y0 - GT_HALO + r, wx = wx0 - 1 + c;
        if (r >= GT_HALO && r < GT_HALO + GT_H && c >= 1 && c <= GT_W && y < h && wx < wpr) {
            const size_t q = (size_t)y * wpr + wx;
            a.Cnew[q] = cold | m3;
            if (lazy) a.G2[q] = sG2[i];
            if (a.M2out) a.M2out[q] = sB[i];
            if (a.M3out) a.M3out[q] = m3;
            nfresh += __popc(fresh);
        }
    }
    nfresh = __reduce_add_sync(0xffffffffu, nfresh);
    if (lane == 0) s_red[wi] = nfresh;
    __syncthreads();
    if (tid == 0) {
        int tot = 0;
#pragma unroll
        for (int k = 0; k < 8; ++k) tot += s_red[k];
        if (tot) atomicAdd(a.count, tot);
    }
    // need = dil5x5(fresh) & C' on the own tile: thread (lane, wi) owns rows 4 wi .. 4 wi + 3 of column lane
    constexpr int NWN = GT_H / 8;
    uint32_t need[NWN];
    int needw[NWN];
    {
        const int c = 1 + lane, r0 = GT_HALO + wi * NWN;
        uint32_t hd[NWN + 4];
#pragma unroll
        for (int k = 0; k < NWN + 4; ++k) hd[k] = hdil_sm<2>(sN, r0 - 2 + k, c);
#pragma unroll
        for (int k = 0; k < NWN; ++k) {
            const int i = (r0 + k) * GS_W + c, y = y0 + wi * NWN + k, wx = wx0 + lane;
            need[k] = (hd[k] | hd[k + 1] | hd[k + 2] | hd[k + 3] | hd[k + 4]) & sC[i];
            needw[k] = i;
            if (y < h && wx < wpr) a.NEED[(size_t)y * wpr + wx] = need[k];
            else need[k] = 0;
        }
    }
    // step (7) at those pixels: 25 clamped taps of img_in, +inf where the tap's pixel is in C', 25-input
    // sorting network, middle element(s) of the k donors (R13-R16)
    const float INF = __int_as_float(0x7f800000);
    for (;;) {
        const int n = smem_compact(need, needw, &s_cnt, s_list, tid);
        for (int i = tid; i < n; i += 256) {
            const int code = s_list[i], wd = code >> 5, bit = code & 31;
            const int r = wd / GS_W, c = wd - r * GS_W;
            const int y = y0 - GT_HALO + r, x = (wx0 - 1 + c) * 32 + bit;
            int xx[5], yy[5];
#pragma unroll
            for (int d = 0; d < 5; ++d) {
                xx[d] = clampi(x + d - 2, 0, w - 1);
                yy[d] = clampi(y + d - 2, 0, h - 1);
            }
            uint32_t donors = 0;   // bit (5 dy + dx): the (clamped) tap is NOT in C'
#pragma unroll
            for (int dy = 0; dy < 5; ++dy) {
                const uint32_t* row = sC + (yy[dy] - (y0 - GT_HALO)) * GS_W - (wx0 - 1);
                const int wl = xx[0] >> 5, wr = xx[4] >> 5;
                const uint32_t cl = row[wl], cr = row[wr];
#pragma unroll
                for (int dx = 0; dx < 5; ++dx) {
                    const uint32_t word = (xx[dx] >> 5) == wl ? cl : cr;
                    donors |= (((word >> (xx[dx] & 31)) & 1u) ^ 1u) << (5 * dy + dx);
                }
            }
            if (donors == 0u) donors = 0x01ffffffu;            // R15: no donor -> all 25 taps
            const int k = __popc(donors);
            float v[25], s[25];
#pragma unroll
            for (int dy = 0; dy < 5; ++dy)
#pragma unroll
                for (int dx = 0; dx < 5; ++dx) {
                    const float t = __ldg(a.img + (size_t)yy[dy] * w + xx[dx]);
                    v[5 * dy + dx] = ((donors >> (5 * dy + dx)) & 1u) ? t : INF;
                }
            sort25(v, s);
            const int ihi = k >> 1, ilo = (k - 1) >> 1;
            float lo = s[0], hi = s[0];
#pragma unroll
            for (int q = 1; q < 25; ++q) {
                lo = (q == ilo) ? s[q] : lo;
                hi = (q == ihi) ? s[q] : hi;
            }
            a.work[(size_t)y * w + x] = (k & 1) ? hi : __fmul_rn(__fadd_rn(lo, hi), 0.5f);   // R14
        }
        bool more = false;
#pragma unroll
        for (int k = 0; k < NWN; ++k) more |= need[k] != 0;
        if (!__syncthreads_or(more)) break;
    }
}

// ------------------------------------------------------------------------------------------------
// Opening pass of an incremental iteration (lazy path, t >= 1).  NEED = the pixels the previous
// k_grow_replace rewrote in `work`.
//   D5 = dil5x5(NEED): the pixels whose S changes (med5 window; L+ needs 1 px).  Their aligned 4-pixel
//        groups ("quads") go to qlist for k_noise_S_quads, which also re-lists the candidates among them.
//   R  = dil9x9(NEED) | quads: the pixels whose tests (3b)-(5) can change (S' reads S within 2 px, the fine
//        structure test reads work within 4 px).  G1, G2, M1 are cleared inside R and the pixels of A1 in R
//        outside the quads (their A1 is unchanged) go to the candidate list.
__global__ void __launch_bounds__(256)
k_dirty_lists(const uint32_t* __restrict__ NEED, const uint32_t* __restrict__ A1, uint32_t* __restrict__ G1,
              uint32_t* __restrict__ G2, uint32_t* __restrict__ M1, int* __restrict__ qlist, int* __restrict__ nq,
              int* __restrict__ clist, int* __restrict__ nc, int h, int w, int wpr, const int* prev_count) {
    if (prev_count && *prev_count == 0) return;
    __shared__ uint32_t sN[GS_N];
    const int tid = threadIdx.x, lane = tid & 31, wi = tid >> 5;
    const int wx0 = blockIdx.x * GT_W, y0 = blockIdx.y * GT_H;
    load_bits_tile(sN, NEED, y0, wx0, h, wpr, tid);
    __syncthreads();
    constexpr int NR = GT_H / 8;
    const int c = 1 + lane, r0 = GT_HALO + wi * NR, wx = wx0 + lane, yb = y0 + wi * NR;
    uint32_t h2[NR + 8], h4[NR + 8];
#pragma unroll
    for (int k = 0; k < NR + 8; ++k) {
        const uint32_t* row = sN + (r0 - 4 + k) * GS_W;
        const uint32_t vl = row[c - 1], vc = row[c], vr = row[c + 1];
        h2[k] = hdil<2>(vl, vc, vr);
        h4[k] = hdil<4>(vl, vc, vr);
    }
    uint32_t quads[NR], cand[NR];
    const int rem = w - wx * 32;
    const uint32_t valid = rem >= 32 ? 0xffffffffu : rem > 0 ? ((1u << rem) - 1u) : 0u;
#pragma unroll
    for (int k = 0; k < NR; ++k) {
        quads[k] = 0;
        cand[k] = 0;
        const int y = yb + k;
        if (y < h && wx < wpr) {
            uint32_t d5 = 0, r9 = 0;
#pragma unroll
            for (int d = 2; d <= 6; ++d) d5 |= h2[k + d];
#pragma unroll
            for (int d = 0; d <= 8; ++d) r9 |= h4[k + d];
            d5 &= valid;
            uint32_t t = d5 | (d5 >> 1);
            t |= t >> 2;
            t &= 0x11111111u;                       // bit 4j: quad j of this word holds a pixel of D5
            const uint32_t dq = t * 0xFu;           // all four pixels of those quads
            const uint32_t R = (r9 | dq) & valid;
            quads[k] = t;
            if (R) {
                const size_t q = (size_t)y * wpr + wx;
                cand[k] = A1[q] & R & ~dq;
                if (R == 0xffffffffu) {
                    G1[q] = 0; G2[q] = 0; M1[q] = 0;
                } else {
                    G1[q] &= ~R; G2[q] &= ~R; M1[q] &= ~R;
                }
            }
        }
    }
    block_append<NR>(quads, yb * w + wx * 32, w, qlist, nq);
    __syncthreads();
    block_append<NR>(cand, yb * w + wx * 32, w, clist, nc);
}

}  // namespace lac
