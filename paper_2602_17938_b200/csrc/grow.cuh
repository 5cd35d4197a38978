// Steps (6)-(7) fused, and the bit-plane pass that opens an incremental iteration.
//
// Both kernels are WARP-AUTONOMOUS: a warp owns a strip of 30 words x WG_R = 4 rows (960 x 4 pixels) of the
// bit-planes, lane l holds word column wx0 - 1 + l (lanes 0 and 31 are the horizontal halo) of every row it
// needs in registers, horizontal neighbours come from warp shuffles, and everything in the halo is
// recomputed from the same inputs by the neighbouring warp (bit arithmetic, plus a handful of redundant G2
// evaluations).  There is no exchange between warps, no block barrier and no staging of whole planes.
//
// k_grow_replace, per warp:
//     M2 = dil3(M1) & G1                                   on strip + 3 px      (G1 read only under dil3(M1))
//     G2 where the second growth reads it and it is not known yet (lazy path)   on strip + 2 px
//     M3 = dil3(M2) & G2,  fresh = M3 & ~C,  C' = C | M3   on strip + 2 px
//     need = dil5x5(fresh) & C'                            on the strip
//     work[p] = masked 5x5 median of img_in around p       for p in need
// so the six launches of the unfused sequence (dilate, list, evaluate, dilate, list, replace) become one.
// C is double buffered (read `Cold`, write `Cnew`) because a neighbour still reads the old plane in its halo.
#pragma once
#include "common.cuh"
#include "lazy_count.cuh"
#include "median_networks.cuh"

namespace lac {

constexpr int WG_OWN = 30;                    // own word columns of a warp (lanes 1..30)
#ifndef LAC_WG_R
#define LAC_WG_R 4
#endif
constexpr int WG_R = LAC_WG_R;                // own rows of a warp
#ifndef LAC_WG_WARPS
#define LAC_WG_WARPS 8
#endif
constexpr int WG_WARPS = LAC_WG_WARPS;        // warps per CTA, stacked vertically
constexpr int WG_J = WG_R + 8;                // register rows: y = ya - 4 + j, j < WG_J
constexpr int WG_LCAP = 128;                  // per-warp pixel list capacity of one round
constexpr unsigned FULL = 0xffffffffu;

// horizontal dilation of a row held one word per lane.  Lanes 0 / 31 have no outer neighbour (the shuffle hands them
// their own word): that only spoils their outer R bits per stage -- at most 4 bits over the three chained stages of
// k_grow_replace, 4 in k_dirty_lists -- and the own columns (lanes 1..30) only ever read the INNER 4 bits of a halo word.
template <int R>
__device__ __forceinline__ uint32_t hdil_w(uint32_t v, int lane) {
    const uint32_t vl = __shfl_up_sync(FULL, v, 1), vr = __shfl_down_sync(FULL, v, 1);
    uint32_t o = v;
#pragma unroll
    for (int k = 1; k <= R; ++k) o |= __funnelshift_l(vl, v, k) | __funnelshift_r(v, vr, k);
    return o;
}

// Warp-cooperative loop over every set bit of bits[J0..J1) of every lane: the bits are compacted into the
// warp's shared list (rounds of at most WG_LCAP) and handed out one per lane: f(j, source lane, bit).
template <int J0, int J1, class F>
__device__ __forceinline__ void warp_for_each_bit(uint32_t (&bits)[WG_J], int* s_list, int lane, F f) {
    for (;;) {
        int n = 0;
#pragma unroll
        for (int j = J0; j < J1; ++j) n += __popc(bits[j]);
        int incl = n;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int o = __shfl_up_sync(FULL, incl, d);
            if (lane >= d) incl += o;
        }
        const int total = __shfl_sync(FULL, incl, 31);
        if (total == 0) break;
        int off = incl - n;
#pragma unroll
        for (int j = J0; j < J1; ++j) {
            uint32_t b = bits[j];
            while (b && off < WG_LCAP) {
                const int bit = __ffs(b) - 1;
                b &= b - 1;
                s_list[off++] = (j << 10) | (lane << 5) | bit;
            }
            bits[j] = b;
        }
        __syncwarp();
        const int m = min(total, WG_LCAP);
        for (int i = lane; i < m; i += 32) {
            const int code = s_list[i];
            f(code >> 10, (code >> 5) & 31, code & 31);
        }
        __syncwarp();
    }
}

struct GrowArgs {
    const uint32_t *M1, *G1;
    uint32_t* G2;                 // lazy path: completed where step (6) reads it
    uint32_t* G2F;                // lazy path: pixels (outside A1) whose G2 was evaluated and is false.  A bit
                                  // of G2 or of G2F is conclusive on its own, so a neighbouring warp may read
                                  // either plane before or after the owner's update
    const uint32_t *A1, *A2;      // lazy path: S > sigclip / S > siglow planes; null: G2 is complete
    const uint32_t* Cold;
    uint32_t* Cnew;
    uint32_t* NEED;               // pixels rewritten in `work` by this launch
    uint32_t *M2out, *M3out;      // nullable (debug planes)
    const float* S;
    const float* img;             // img_in: donor values (R13)
    float* work;
    int* count;                   // += |M3 & ~C|
    int incremental;              // t >= 1 of the lazy path: M1 holds this iteration's new detections only
    int h, w, wpr;
    float siglow;
    int nbx;                      // strips per row of strips = CTAs per row of CTAs (1-D grid, block_xy)
    const uint32_t* donx;         // nullable (R23): bad pixels, never donors of the replacement
    int* nneed;                   // nullable (lacosmic_stats_enable): += pixels whose replacement value is (re)computed
    uint8_t* mask_u8;             // nullable: the frame's uint8 mask (cleared by the first pass): every pixel whose
                                  // replacement is computed is in C', so it is set here
};

#ifndef LAC_GROW_MINB
#define LAC_GROW_MINB 3
#endif
__global__ void __launch_bounds__(32 * WG_WARPS, LAC_GROW_MINB)
k_grow_replace(GrowArgs a, const int* prev_count) {
    pdl_entry();
    const int lane = threadIdx.x & 31, wi = threadIdx.x >> 5;
    const int h = a.h, w = a.w, wpr = a.wpr;
    const BlockXY bk = block_xy(a.nbx);
    const int wxh = bk.x * WG_OWN - 1;                       // word column of lane 0
    const int wx = wxh + lane;
    const int ya = (bk.y * WG_WARPS + wi) * WG_R;             // first own row
    if (ya >= h) return;                                      // warp-uniform; the kernel has no block barrier
    const bool colok = wx >= 0 && wx < wpr;
    const bool own = lane >= 1 && lane <= WG_OWN && colok;
    __shared__ uint32_t s_plane_all[WG_WARPS][(WG_R + 4) * 32];   // G2, then C', rows ya-2 .. ya+WG_R+1
    __shared__ int s_list_all[WG_WARPS][WG_LCAP];
    uint32_t* s_plane = s_plane_all[wi];
    int* s_list = s_list_all[wi];
    // word (row j, this lane's column) of a plane sits at base + j * wpr; rows / columns outside the frame read as 0
    // (predicated loads: the address is never formed into an access there)
    const int base = (ya - 4) * wpr + wx;
    auto rowok = [&](int j) -> bool { return colok && (unsigned)(ya - 4 + j) < (unsigned)h; };
    // one pointer per plane at the strip's first register row, one offset per row shared by all planes (half of this
    // kernel's instructions used to be 64-bit address arithmetic, one chain per access)
    const uint32_t *const pM1 = a.M1 + base, *const pG1 = a.G1 + base, *const pCo = a.Cold + base;
    const uint32_t *const pA1 = a.A1 ? a.A1 + base : nullptr, *const pA2 = a.A2 ? a.A2 + base : nullptr;
    uint32_t *const pG2 = a.G2 + base, *const pG2F = a.G2F + base, *const pCn = a.Cnew + base, *const pNE = a.NEED + base;
    int ro[WG_J];
#pragma unroll
    for (int j = 0; j < WG_J; ++j) ro[j] = j * wpr;
    auto qof = [&](int j) -> int { return base + j * wpr; };
    const int pc = prev_count ? *prev_count : 1;             // tested below, after the M1 loads have been issued
    const bool lazy = a.A2 != nullptr;
    // M1 first.  In an incremental iteration (t >= 1) M1 only holds the new detections of this iteration, so most
    // strips see none within their 16 rows: then M2 = M3 = 0, nothing is fresh and nothing needs a replacement --
    // the strip carries C over and is done after 24 words instead of the ~100 of all planes (the bit-plane
    // traffic of all strips at once, not the arithmetic, is what these launches cost).
    uint32_t m1[WG_J];
    bool anym1 = false;
#pragma unroll
    for (int j = 0; j < WG_J; ++j) {
        m1[j] = rowok(j) ? pM1[ro[j]] : 0u;
        anym1 |= m1[j] != 0;
    }
    if (pc == 0) {
        // fixed point (R17): nothing changes; carry C over to the plane the next reader expects
#pragma unroll
        for (int j = 4; j < 4 + WG_R; ++j)
            if (own && ya - 4 + j < h) pCn[ro[j]] = pCo[ro[j]];
        return;
    }
    if (a.incremental && !__any_sync(FULL, anym1)) {
#pragma unroll
        for (int j = 4; j < 4 + WG_R; ++j)
            if (own && ya - 4 + j < h) {
                pCn[ro[j]] = pCo[ro[j]];
                pNE[ro[j]] = 0u;
            }
        return;
    }
    // every other word the strip can need, requested together (independent loads, one round trip), row by row so
    // that one offset and one predicate serve all planes of a row
    uint32_t m2[WG_J], g2[WG_J], nbm[WG_J], cold[WG_J];
    {
        uint32_t g1[WG_J];
#pragma unroll
        for (int j = 1; j < WG_J - 1; ++j) {
            const bool ok = rowok(j);
            const int q = ro[j];
            g1[j] = ok ? pG1[q] : 0u;
            if (j >= 2 && j < WG_J - 2) {
                g2[j] = ok ? pG2[q] : 0u;
                cold[j] = ok ? pCo[q] : 0u;
                nbm[j] = (lazy && ok) ? (pA2[q] & ~pA1[q] & ~pG2F[q]) : 0u;
            }
        }
        // ---- M2 = dil3(M1) & G1, rows 1 .. WG_J-2
#pragma unroll
        for (int j = 0; j < WG_J; ++j) m1[j] = hdil_w<1>(m1[j], lane);
        m2[0] = m2[WG_J - 1] = 0;
#pragma unroll
        for (int j = 1; j < WG_J - 1; ++j) m2[j] = (m1[j - 1] | m1[j] | m1[j + 1]) & g1[j];
    }
    // ---- D = dil3(M2), rows 2 .. WG_J-3
    uint32_t d[WG_J];
    {
        uint32_t hm[WG_J];
#pragma unroll
        for (int j = 1; j < WG_J - 1; ++j) hm[j] = hdil_w<1>(m2[j], lane);
#pragma unroll
        for (int j = 2; j < WG_J - 2; ++j) d[j] = hm[j - 1] | hm[j] | hm[j + 1];
    }
    if (lazy) {
        // pixels under D whose G2 = (S' > siglow) is not known yet: evaluate by counting (lazy_count.cuh).
        // Only within 2 px of the own columns: the neighbouring warps evaluate the rest.
        const uint32_t keep = lane == 0 ? 0xC0000000u : lane == 31 ? 0x00000003u : 0xffffffffu;
        uint32_t nb[WG_J];
        bool any = false;
#pragma unroll
        for (int j = 2; j < WG_J - 2; ++j) {
            nb[j] = d[j] & nbm[j] & ~g2[j] & keep;
            any |= nb[j] != 0;
        }
        if (__any_sync(FULL, any)) {
#pragma unroll
            for (int j = 2; j < WG_J - 2; ++j) s_plane[(j - 2) * 32 + lane] = g2[j];
            __syncwarp();
            uint32_t todo[WG_J];
#pragma unroll
            for (int j = 0; j < WG_J; ++j) todo[j] = (j >= 2 && j < WG_J - 2) ? nb[j] : 0u;
            warp_for_each_bit<2, WG_J - 2>(todo, s_list, lane, [&](int j, int sl, int bit) {
                const int y = ya - 4 + j, x = (wxh + sl) * 32 + bit;
                int c1, c2;
                count_sp(a.S, y, x, h, w, a.siglow, a.siglow, c1, c2);
                if (c2 >= 13) atomicOr(&s_plane[(j - 2) * 32 + sl], 1u << bit);
            });
#pragma unroll
            for (int j = 2; j < WG_J - 2; ++j) g2[j] = s_plane[(j - 2) * 32 + lane];
            __syncwarp();
            // remember the evaluations of the own words
#pragma unroll
            for (int j = 4; j < 4 + WG_R; ++j)
                if (nb[j] && own && ya - 4 + j < h) {
                    pG2[ro[j]] = g2[j];
                    pG2F[ro[j]] |= nb[j] & ~g2[j];
                }
        }
    }
    // ---- M3 = D & G2; fresh = M3 & ~C; C' = C | M3, rows 2 .. WG_J-3
    uint32_t cn[WG_J], fresh[WG_J];
    int nfresh = 0;
    bool anyfresh = false;
#pragma unroll
    for (int j = 2; j < WG_J - 2; ++j) {
        const uint32_t m3 = d[j] & g2[j];
        fresh[j] = m3 & ~cold[j];
        cn[j] = cold[j] | m3;
        anyfresh |= fresh[j] != 0;
        if (j >= 4 && j < 4 + WG_R && own && ya - 4 + j < h) {
            pCn[ro[j]] = cn[j];
            if (a.M2out) a.M2out[qof(j)] = m2[j];
            if (a.M3out) a.M3out[qof(j)] = m3;
            nfresh += __popc(fresh[j]);
        }
    }
    nfresh = __reduce_add_sync(FULL, nfresh);
    if (lane == 0 && nfresh) atomicAdd(a.count, nfresh);
    // ---- need = dil5x5(fresh) & C' on the own words
    uint32_t need[WG_J];
#pragma unroll
    for (int j = 0; j < WG_J; ++j) need[j] = 0;
    if (__any_sync(FULL, anyfresh)) {
        uint32_t hf[WG_J];
#pragma unroll
        for (int j = 2; j < WG_J - 2; ++j) hf[j] = hdil_w<2>(fresh[j], lane);
#pragma unroll
        for (int j = 4; j < 4 + WG_R; ++j)
            if (own && ya - 4 + j < h) need[j] = (hf[j - 2] | hf[j - 1] | hf[j] | hf[j + 1] | hf[j + 2]) & cn[j];
    }
#pragma unroll
    for (int j = 4; j < 4 + WG_R; ++j)
        if (own && ya - 4 + j < h) pNE[ro[j]] = need[j];
    bool anyneed = false;
#pragma unroll
    for (int j = 4; j < 4 + WG_R; ++j) anyneed |= need[j] != 0;
    if (!__any_sync(FULL, anyneed)) return;
    if (a.nneed) {                                            // statistics only (off in timed runs)
        int nn = 0;
#pragma unroll
        for (int j = 4; j < 4 + WG_R; ++j) nn += __popc(need[j]);
        nn = __reduce_add_sync(FULL, nn);
        if (lane == 0) atomicAdd(a.nneed, nn);
    }
    // ---- step (7) at those pixels: 25 clamped taps of img_in, +inf where the tap's pixel is in C', 25-input
    // sorting network, middle element(s) of the k donors (R13-R16)
    // s_plane: the pixels that are no donors = C' (R13), plus the bad pixels (R23)
#pragma unroll
    for (int j = 2; j < WG_J - 2; ++j) s_plane[(j - 2) * 32 + lane] = cn[j] | ((a.donx && rowok(j)) ? a.donx[qof(j)] : 0u);
    __syncwarp();
    const float INF = __int_as_float(0x7f800000);
    warp_for_each_bit<4, 4 + WG_R>(need, s_list, lane, [&](int j, int sl, int bit) {
        const int y = ya - 4 + j, x = (wxh + sl) * 32 + bit;
        int xx[5], yy[5];
#pragma unroll
        for (int t = 0; t < 5; ++t) {
            xx[t] = clampi(x + t - 2, 0, w - 1);
            yy[t] = clampi(y + t - 2, 0, h - 1);
        }
        uint32_t donors = 0;   // bit (5 dy + dx): the (clamped) tap is NOT in C'
#pragma unroll
        for (int dy = 0; dy < 5; ++dy) {
            const uint32_t* row = s_plane + (yy[dy] - (ya - 2)) * 32 - wxh;
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
        if (a.mask_u8) a.mask_u8[(size_t)y * w + x] = 1;
    });
}

// ------------------------------------------------------------------------------------------------
// warp-aggregated append of the set bits of bits[J0..J1) (pixel index p0 + (j - J0) * w + bit) to a global
// list: one atomicAdd per warp that has something to append
template <int J0, int J1>
__device__ __forceinline__ void warp_append(const uint32_t (&bits)[WG_J], int p0, int w, int* __restrict__ list,
                                            int* __restrict__ nlist, int lane) {
    int n = 0;
#pragma unroll
    for (int j = J0; j < J1; ++j) n += __popc(bits[j]);
    int incl = n;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int o = __shfl_up_sync(FULL, incl, d);
        if (lane >= d) incl += o;
    }
    const int total = __shfl_sync(FULL, incl, 31);
    if (total == 0) return;
    int base = 0;
    if (lane == 31) base = atomicAdd(nlist, total);
    int off = __shfl_sync(FULL, base, 31) + incl - n;
#pragma unroll
    for (int j = J0; j < J1; ++j) {
        uint32_t b = bits[j];
        const int pj = p0 + (j - J0) * w;
        while (b) {
            const int bit = __ffs(b) - 1;
            b &= b - 1;
            list[off++] = pj + bit;
        }
    }
}

// Opening pass of an incremental iteration (lazy path, t >= 1).  NEED = the pixels the previous
// k_grow_replace rewrote in `work`.
//   D5 = dil5x5(NEED): the pixels whose S changes (med5 window; L+ needs 1 px).  Their aligned 4-pixel
//        groups ("quads") go to qlist for k_noise_S_quads, which also re-lists the candidates among them.
//   R  = dil9x9(NEED) | quads: the pixels whose tests (3b)-(5) can change (S' reads S within 2 px, the fine
//        structure test reads work within 4 px).  G1, G2, G2F, M1 are cleared inside R and the pixels of A1 in
//        R outside the quads (their A1 is unchanged) go to the candidate list.
// Same warp-autonomous layout as k_grow_replace.
#ifndef LAC_DIRTY_MINB
#define LAC_DIRTY_MINB 2
#endif
__global__ void __launch_bounds__(32 * WG_WARPS, LAC_DIRTY_MINB)
k_dirty_lists(const uint32_t* __restrict__ NEED, const uint32_t* __restrict__ A1, uint32_t* __restrict__ G1,
              uint32_t* __restrict__ G2, uint32_t* __restrict__ G2F, uint32_t* __restrict__ M1,
              int* __restrict__ qlist, int* __restrict__ nq, int* __restrict__ clist, int* __restrict__ nc,
              int h, int w, int wpr, int nbx, const int* prev_count) {
    pdl_entry();
    const int pc = prev_count ? *prev_count : 1;             // tested below, after the NEED loads have been issued
    const int lane = threadIdx.x & 31, wi = threadIdx.x >> 5;
    const BlockXY bk = block_xy(nbx);
    const int wx = bk.x * WG_OWN - 1 + lane;
    const int ya = (bk.y * WG_WARPS + wi) * WG_R;
    if (ya >= h) return;                                      // warp-uniform; no block barrier in this kernel
    const bool colok = wx >= 0 && wx < wpr;
    const bool own = lane >= 1 && lane <= WG_OWN && colok;
    const int base = (ya - 4) * wpr + wx;           // word (row ya - 4 + j, this lane's column) = base + j * wpr
    // one pointer per plane at the strip's first register row, one offset per row shared by all planes
    const uint32_t *const pNE = NEED + base, *const pA1 = A1 + base;
    uint32_t *const pG1 = G1 + base, *const pG2 = G2 + base, *const pG2F = G2F + base, *const pM1 = M1 + base;
    int ro[WG_J];
#pragma unroll
    for (int j = 0; j < WG_J; ++j) ro[j] = j * wpr;
    uint32_t h2[WG_J], h4[WG_J];
    bool any = false;
#pragma unroll
    for (int j = 0; j < WG_J; ++j) {
        h2[j] = (colok && (unsigned)(ya - 4 + j) < (unsigned)h) ? pNE[ro[j]] : 0u;
        any |= h2[j] != 0;
    }
    if (pc == 0 || !__any_sync(FULL, any)) return;            // fixed point (R17), or nothing was rewritten near this strip
#pragma unroll
    for (int j = 0; j < WG_J; ++j) {
        // (halo lanes 0 / 31 have no outer neighbour: see hdil_w)
        const uint32_t vl = __shfl_up_sync(FULL, h2[j], 1), vc = h2[j], vr = __shfl_down_sync(FULL, h2[j], 1);
        uint32_t o2 = vc;
#pragma unroll
        for (int k = 1; k <= 2; ++k) o2 |= __funnelshift_l(vl, vc, k) | __funnelshift_r(vc, vr, k);
        uint32_t o4 = o2;
#pragma unroll
        for (int k = 3; k <= 4; ++k) o4 |= __funnelshift_l(vl, vc, k) | __funnelshift_r(vc, vr, k);
        h2[j] = o2;
        h4[j] = o4;
    }
    uint32_t quads[WG_J], cand[WG_J], Rr[WG_R], dqr[WG_R];
    const int rem = w - wx * 32;
    const uint32_t valid = rem >= 32 ? 0xffffffffu : rem > 0 ? ((1u << rem) - 1u) : 0u;
#pragma unroll
    for (int j = 0; j < WG_J; ++j) quads[j] = cand[j] = 0;
#pragma unroll
    for (int k = 0; k < WG_R; ++k) {
        const int j = k + 4;
        Rr[k] = dqr[k] = 0;
        if (own && ya + k < h) {
            uint32_t d5 = 0, r9 = 0;
#pragma unroll
            for (int d = -2; d <= 2; ++d) d5 |= h2[j + d];
#pragma unroll
            for (int d = -4; d <= 4; ++d) r9 |= h4[j + d];
            d5 &= valid;
            uint32_t t = d5 | (d5 >> 1);
            t |= t >> 2;
            t &= 0x11111111u;                       // bit 4k: quad k of this word holds a pixel of D5
            dqr[k] = t * 0xFu;                      // all four pixels of those quads
            Rr[k] = (r9 | dqr[k]) & valid;
            quads[j] = t;
        }
    }
    // the gate planes are only read (and rewritten) in the words that hold a pixel of R: late iterations touch a
    // few words per strip, and the bit-plane traffic of all strips at once is what this launch costs
    uint32_t a1[WG_R], g1[WG_R], g2[WG_R], g2f[WG_R], m1[WG_R];
#pragma unroll
    for (int k = 0; k < WG_R; ++k) {
        const bool rd = Rr[k] != 0;
        const int q = ro[4 + k];
        a1[k] = rd ? pA1[q] : 0u; g1[k] = rd ? pG1[q] : 0u; g2[k] = rd ? pG2[q] : 0u;
        g2f[k] = rd ? pG2F[q] : 0u; m1[k] = rd ? pM1[q] : 0u;
    }
#pragma unroll
    for (int k = 0; k < WG_R; ++k) {
        const uint32_t R = Rr[k];
        if (R) {
            const int q = ro[4 + k];
            cand[k + 4] = a1[k] & R & ~dqr[k];
            if (g1[k] & R) pG1[q] = g1[k] & ~R;
            if (g2[k] & R) pG2[q] = g2[k] & ~R;
            if (g2f[k] & R) pG2F[q] = g2f[k] & ~R;
            if (m1[k] & R) pM1[q] = m1[k] & ~R;
        }
    }
    const int p0 = ya * w + wx * 32;
    warp_append<4, 4 + WG_R>(quads, p0, w, qlist, nq, lane);
    warp_append<4, 4 + WG_R>(cand, p0, w, clist, nc, lane);
}

}  // namespace lac
