// Gain estimation, fast path (reading R21, section 5.3): the sigma clipping of select.cuh -- three
// rounds of { c = element of rank (n-1)/2 of r over the kept set, d = element of the same rank of |r - c| } --
// with TWO reads of the residual plane instead of eighteen.  The answer is the same element, bit for bit:
//
//   k_selz_init     a strided sample of 128 residuals gives a rough centre and scale (its median and MAD); they
//                   only place a grid of 4096 value-linear buckets over the plane's values (any grid gives the same
//                   answer).
//   k_selz_hist     read 1: exact counts of every bucket (shared-memory histograms).  The CTA that finishes last
//                   PLANS: from the cumulative counts it follows the three rounds at bucket resolution and marks
//                   five ZONES of buckets -- Z0 around the centres, Z- / Z+ around c -/+ d, OUT- / OUT+ beyond
//                   the clipping bounds -- wide enough to hold every value a round can select or compare with.
//   k_selz_compact  read 2: the residuals of Z0 go to one list (1-2 % of the plane), those of Z- and Z+ to a second
//                   one (about 5 %), those of OUT- and OUT+ to a third one together with their med5 (about 2 %).
//   k_selz_resolve  one cluster of 16 CTAs runs the three rounds EXACTLY on the lists: the pixels outside the
//                   zones only enter through their counts, which the histogram holds exactly; every selection is
//                   a radix selection over a list.  Every step checks that what it selected lies inside its zone
//                   (the first and last floats of a bucket are found by bisection on the bucket function, so the
//                   bounds are exact): if a check fails -- a frame of few distinct values, a plan that missed -- the
//                   state says so and k_sel_rounds (select.cuh: the eighteen radix passes as one cooperative launch,
//                   which otherwise returns at once) does the rounds over the plane.
// The typical signal (rank (n-1)/2 of max(med5, 1e-4) over the kept set) rides along: a second grid over max(med5,
// 1e-4), its counts in k_selz_hist, ONE zone ZM around the positions the wanted element can have among all pixels
// (every pixel outside the kept interval is in an OUT zone, so the position is known to within their number),
// compacted in k_selz_compact and selected in k_selz_resolve as the zone list MINUS the OUT entries outside the kept
// interval; the gain formula follows there.  If that fails, k_sel_rounds selects it by three radix passes over the med5
// plane (the listed pixels outside the kept interval subtracted from the histograms).
#pragma once
#include <cooperative_groups.h>

#include "common.cuh"
#include "select.cuh"

namespace lac {

namespace cg = cooperative_groups;

#ifndef LAC_SELZ_NB
#define LAC_SELZ_NB 4096
#endif
constexpr int SELZ_NB = LAC_SELZ_NB;          // buckets
constexpr int SELZ_SAMPLE = 128;
constexpr int SELZ_IT = 1024;                 // threads of k_selz_init (the first SELZ_SAMPLE sample, all clear the histograms)
constexpr int SELZ_HT = 1024;                 // threads per CTA of k_selz_hist
#ifndef LAC_SELZ_CLUSTER
#define LAC_SELZ_CLUSTER 16
#endif
constexpr int SELZ_CLUSTER = LAC_SELZ_CLUSTER;   // CTAs of k_selz_resolve (16 needs the non-portable cluster size opt-in)
constexpr int SELZ_RT = 1024;                 // its threads per CTA
constexpr int SELZ_BUF = 2048;                // staging entries per list and CTA of k_selz_compact
constexpr int SELZ_UNROLL = 8;                // list entries a thread of k_selz_resolve has in flight

struct SelZone {
    float base, scale;                        // bucket(r) = clamp(floor((r - base) * scale), 0, SELZ_NB - 1)
    int z0lo, z0hi, zmlo, zmhi, zplo, zphi;   // bucket ranges (inclusive) of Z0, Z-, Z+
    int omhi, oplo;                           // OUT- = [0, omhi], OUT+ = [oplo, SELZ_NB - 1]
    uint32_t below_z0;                        // values in buckets < z0lo
    uint32_t cnt_z0, cnt_zm, cnt_zp;          // values in the zones
    uint32_t inner;                           // values in buckets zmhi + 1 .. zplo - 1 (Z0 included)
    uint32_t cnt_om, cnt_op;
    uint32_t npx;
    uint32_t n0, n1, no;                      // list cursors of k_selz_compact (Z0; Z- and Z+; OUT)
    uint32_t nscr[2];                         // cursors of the resolve kernel's scratch list (used alternately)
    uint32_t ok;                              // 1: plan made, lists fit; the resolve kernel may run
    uint32_t done;                            // 1: k_selz_resolve finished the three rounds (0: the radix passes run)
    uint32_t why;                             // diagnostic: where the fast path stopped (0 = it did not)
    uint32_t nzero;                           // residuals that are exactly +0 (a pixel that is the median of its own window:
                                              // 4 % of a frame).  Inside Z0 they are counted, not listed.
    uint32_t nneg0;                           // negative residuals in the bucket of 0: when a centre's rank inside that bucket
                                              // falls on the zeros, the centre is +0 without a selection (the usual case)
    // the typical signal: a second grid over max(med5, 1e-4) and one zone ZM around its median
    float mbase, mscale;
    int m5lo, m5hi;                           // bucket range of ZM
    uint32_t below_m5, cnt_m5;                // values in buckets < m5lo; in ZM
    uint32_t nm;                              // list cursor
    uint32_t mok;                             // 1: grid and zone made, the list fits
    uint32_t mdone;                           // 1: k_selz_resolve selected the typical signal and wrote the gain
};

// capacities of the five lists inside `words` 32-bit words of storage
struct SelzLists {
    float* z0;
    float* z1;
    float2* o;
    float* zm;
    uint32_t* scr;
    uint32_t cap0, cap1, capo, capm, capscr;
};
__host__ __device__ inline SelzLists selz_carve(void* base, size_t words) {
    SelzLists l;
    const size_t e = (words / 20) & ~(size_t)1;      // a twentieth, even
    l.z0 = (float*)base;                 l.cap0 = (uint32_t)(3 * e);
    l.z1 = l.z0 + 3 * e;                 l.cap1 = (uint32_t)(4 * e);
    l.o = (float2*)(l.z1 + 4 * e);       l.capo = (uint32_t)(3 * e);
    l.zm = l.z1 + 10 * e;                l.capm = (uint32_t)(4 * e);
    l.scr = (uint32_t*)(l.z1 + 14 * e);  l.capscr = (uint32_t)(3 * e);
    return l;
}

__device__ __forceinline__ int selz_bucket(float r, float base, float scale) {
    return min(max(__float2int_rd(__fmul_rn(__fsub_rn(r, base), scale)), 0), SELZ_NB - 1);
}

// One CTA of SELZ_IT threads: all clear the histograms; the first SELZ_SAMPLE take a strided sample of the two planes and
// place the two bucket grids by its medians and MADs (rank counting: thread i counts the sample values below its own).
__global__ void __launch_bounds__(SELZ_IT)
k_selz_init(const float* __restrict__ R, const float* __restrict__ M5, size_t npx, SelState* st, SelZone* zn, uint32_t* hist,
            uint32_t* histz, uint32_t* histm, int force_classic, const int* prev_count) {
    if (prev_count && *prev_count == 0) return;
    __shared__ __align__(16) uint32_t k[SELZ_SAMPLE];
    __shared__ uint32_t s_res[4];
    const int tid = threadIdx.x;
    for (int i = tid; i < SEL_BINS; i += SELZ_IT) hist[i] = 0;
    for (int i = tid; i < SELZ_NB; i += SELZ_IT) { histz[i] = 0; histm[i] = 0; }
    const uint32_t ns = (uint32_t)(npx < SELZ_SAMPLE ? npx : SELZ_SAMPLE);
    float v = 0.0f, vm = 1e-4f;
    bool valid = false;
    if ((uint32_t)tid < ns) {
        // groups of 32 values 61 apart (few pages to touch), the groups spread over the plane
        const size_t grp = npx / (SELZ_SAMPLE / 32), step = grp / 32 < 61 ? grp / 32 : 61;
        const size_t i = npx < SELZ_SAMPLE ? (size_t)tid : (size_t)(tid >> 5) * grp + (size_t)(tid & 31) * step;
        v = R[i];
        valid = v == v;                                   // NaN (caller error) is left out of the sample
        vm = M5[i];
        vm = vm > 1e-4f ? vm : 1e-4f;
    }
    const uint32_t nv = (uint32_t)__syncthreads_count(valid);
    if (tid == 0) s_res[0] = s_res[1] = s_res[2] = s_res[3] = 0x80000000u;      // key of +0
    // ranks of two keys among the valid keys of their arrays (ties by index); invalid entries hold the largest key and
    // sort last.  One loop for both: the residual and max(med5, 1e-4) at the sampled pixels.
    __shared__ __align__(16) uint32_t k2[SELZ_SAMPLE];
    auto rank_of2 = [&](uint32_t mine, uint32_t mine2, uint32_t& rk, uint32_t& rk2) {
        if (tid < SELZ_SAMPLE) { k[tid] = mine; k2[tid] = mine2; }
        __syncthreads();
        rk = rk2 = 0;
#pragma unroll 4
        for (int j = 0; j < (tid < SELZ_SAMPLE ? SELZ_SAMPLE : 0); j += 4) {
            const uint4 o = *reinterpret_cast<const uint4*>(k + j), p = *reinterpret_cast<const uint4*>(k2 + j);
            rk += (o.x < mine || (o.x == mine && j < tid)) ? 1u : 0u;
            rk += (o.y < mine || (o.y == mine && j + 1 < tid)) ? 1u : 0u;
            rk += (o.z < mine || (o.z == mine && j + 2 < tid)) ? 1u : 0u;
            rk += (o.w < mine || (o.w == mine && j + 3 < tid)) ? 1u : 0u;
            rk2 += (p.x < mine2 || (p.x == mine2 && j < tid)) ? 1u : 0u;
            rk2 += (p.y < mine2 || (p.y == mine2 && j + 1 < tid)) ? 1u : 0u;
            rk2 += (p.z < mine2 || (p.z == mine2 && j + 2 < tid)) ? 1u : 0u;
            rk2 += (p.w < mine2 || (p.w == mine2 && j + 3 < tid)) ? 1u : 0u;
        }
        __syncthreads();
    };
    const uint32_t want = nv ? (nv - 1u) / 2u : 0u;
    uint32_t ra, rb;
    const uint32_t key0 = valid ? sel_key(v) : 0xffffffffu;
    const uint32_t key2 = valid ? (__float_as_uint(vm) | 0x80000000u) : 0xffffffffu;
    rank_of2(key0, key2, ra, rb);
    if (ra == want && valid) s_res[0] = key0;
    if (rb == want && valid) s_res[2] = key2;
    __syncthreads();
    const float c0 = sel_unkey(s_res[0]);
    const float cm = __uint_as_float(s_res[2] & 0x7fffffffu);
    const uint32_t key1 = valid ? (__float_as_uint(fabsf(v - c0)) | 0x80000000u) : 0xffffffffu;
    const uint32_t key3 = valid ? (__float_as_uint(fabsf(vm - cm)) | 0x80000000u) : 0xffffffffu;
    rank_of2(key1, key3, ra, rb);
    if (ra == want && valid) s_res[1] = key1;
    if (rb == want && valid) s_res[3] = key3;
    __syncthreads();
    if (tid == 0) {
        st->lo = -__int_as_float(0x7f800000);
        st->hi = __int_as_float(0x7f800000);
        st->c = 0.0f;
        st->s = 0.0f;
        st->prefix = 0;
        st->kth = 0;
        st->n = 0;
        st->ticket = 0;
        const float INF = __int_as_float(0x7f800000);
        const float d0 = __uint_as_float(s_res[1] & 0x7fffffffu);
        const float s0 = 1.4826f * d0;
        const float base = c0 - 8.0f * s0, scale = (float)SELZ_NB / (16.0f * s0);
        SelZone z;
        z.base = base;
        z.scale = scale;
        z.z0lo = z.z0hi = z.zmlo = z.zmhi = z.zplo = z.zphi = z.omhi = z.oplo = 0;
        z.below_z0 = z.cnt_z0 = z.cnt_zm = z.cnt_zp = z.inner = z.cnt_om = z.cnt_op = 0;
        z.npx = (uint32_t)npx;
        z.n0 = z.n1 = z.no = z.nscr[0] = z.nscr[1] = 0;
        // a usable grid: positive finite scale, finite base
        z.ok = (!force_classic && nv > 0 && s0 > 0.0f && s0 < INF && scale > 0.0f && scale < INF && fabsf(base) < INF) ? 1u : 0u;
        z.done = 0;
        z.why = z.ok ? 0u : 1u;                             // 1: switched off, or no usable bucket grid
        z.nzero = z.nneg0 = 0;
        const float sm0 = 1.4826f * __uint_as_float(s_res[3] & 0x7fffffffu);
        z.mbase = cm - 8.0f * sm0;
        z.mscale = (float)SELZ_NB / (16.0f * sm0);
        z.m5lo = z.m5hi = 0;
        z.below_m5 = z.cnt_m5 = z.nm = 0;
        z.mok = (z.ok && sm0 > 0.0f && sm0 < INF && z.mscale > 0.0f && z.mscale < INF && fabsf(z.mbase) < INF) ? 1u : 0u;
        z.mdone = 0;
        *zn = z;
    }
}

// ---- read 1: bucket counts, then the plan ---------------------------------------------------------
// cum: SELZ_NB + 1 words of shared memory, cum[b] = values in buckets < b
__device__ __forceinline__ int selz_bucket_of_rank(const uint32_t* cum, uint32_t g) {   // largest b with cum[b] <= g
    int lo = 0, hi = SELZ_NB;                 // invariant: cum[lo] <= g < cum[hi] (cum[SELZ_NB] = total > g)
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (cum[mid] <= g) lo = mid; else hi = mid;
    }
    return lo;
}

// The plan, by one thread.  It follows the three rounds with bucket ranges in place of intervals; all it has to
// get right is that the zones are wide enough -- k_selz_resolve checks every use.
__device__ void selz_plan(const uint32_t* cum, SelZone* zn, SelzLists cap) {
    int a = 0, b = SELZ_NB - 1;               // kept bucket range of the round
    int bmin = SELZ_NB, bmax = -1, pmin = SELZ_NB, pmax = -1, qmin = SELZ_NB, qmax = -1;
    float outl = -1e30f, outh = 1e30f, extmin = 1e30f;
    bool ok = true;
    uint32_t why = 2;                         // 2: a round of the plan found nothing
    for (int j = 0; j < SEL_ROUNDS && ok; ++j) {
        const uint32_t n = cum[b + 1] - cum[a];
        if (n == 0) { ok = false; break; }
        const uint32_t k = (n - 1u) / 2u;
        const int bj = selz_bucket_of_rank(cum, cum[a] + k);
        // smallest m with (values of [bj - m, bj + m] inside the kept range) >= k + 1
        int mlo = -1, mhi = SELZ_NB;          // count(mlo) < k + 1 <= count(mhi)
        while (mhi - mlo > 1) {
            const int mid = (mlo + mhi) >> 1;
            const uint32_t cnt = cum[min(bj + mid, b) + 1] - cum[max(bj - mid, a)];
            if (cnt >= k + 1u) mhi = mid; else mlo = mid;
        }
        const int mj = mhi;
        const float ext = 7.413f * (float)mj;                       // 5 * 1.4826 * d, in buckets
        bmin = min(bmin, bj); bmax = max(bmax, bj);
        pmin = min(pmin, bj + mj); pmax = max(pmax, bj + mj);
        qmin = min(qmin, bj - mj); qmax = max(qmax, bj - mj);
        outl = fmaxf(outl, (float)bj - ext);
        outh = fminf(outh, (float)bj + ext);
        extmin = fminf(extmin, ext);
        a = max(a, min((int)ceilf((float)bj - ext), SELZ_NB - 1));
        b = min(b, max((int)floorf((float)bj + ext), 0));
        if (a > b) ok = false;
    }
    SelZone z = *zn;
    z.nzero = __ldcg(&zn->nzero);             // (summed by the other CTAs; this CTA's L1 may hold the line from before)
    z.nneg0 = __ldcg(&zn->nneg0);
    if (ok) {
        const int mo = 10 + (int)(0.03f * extmin);
        z.z0lo = bmin - 3; z.z0hi = bmax + 3;
        z.zmlo = qmin - 4; z.zmhi = qmax + 4;
        z.zplo = pmin - 4; z.zphi = pmax + 4;
        z.omhi = (int)ceilf(outl) + mo;
        z.oplo = (int)floorf(outh) - mo;
        ok = z.omhi >= 0 && z.omhi < z.zmlo && z.zmhi < z.z0lo && z.z0hi < z.zplo && z.zphi < z.oplo && z.oplo <= SELZ_NB - 1;
        why = 3;                              // 3: the zones overlap or leave the grid
    }
    if (ok) {
        z.below_z0 = cum[z.z0lo];
        z.cnt_z0 = cum[z.z0hi + 1] - cum[z.z0lo];
        z.cnt_zm = cum[z.zmhi + 1] - cum[z.zmlo];
        z.cnt_zp = cum[z.zphi + 1] - cum[z.zplo];
        z.inner = cum[z.zplo] - cum[z.zmhi + 1];
        z.cnt_om = cum[z.omhi + 1];
        z.cnt_op = cum[SELZ_NB] - cum[z.oplo];
        const int bzero = selz_bucket(0.0f, z.base, z.scale);
        const uint32_t listed0 = z.cnt_z0 - ((bzero >= z.z0lo && bzero <= z.z0hi) ? z.nzero : 0u);
        ok = listed0 <= cap.cap0 && (unsigned long long)z.cnt_zm + z.cnt_zp <= cap.cap1 &&
             (unsigned long long)z.cnt_om + z.cnt_op <= cap.capo;
        why = 4;                              // 4: a list does not fit
    }
    z.ok = ok ? 1u : 0u;
    z.why = ok ? 0u : why;
    z.n0 = z.n1 = z.no = z.nscr[0] = z.nscr[1] = 0;
    *zn = z;
}

// cumulative counts of a global histogram into cum[0 .. SELZ_NB] (shared memory), by the first 256 threads of the CTA;
// scan: 256 words of shared memory.  Contains block barriers (all threads call).
__device__ __forceinline__ void selz_cumulate(const uint32_t* hist_g, uint32_t* cum, uint32_t* scan) {
    constexpr int PER = SELZ_NB / 256;
    uint32_t loc[PER], sum = 0;
    if (threadIdx.x < 256) {
#pragma unroll
        for (int i = 0; i < PER; ++i) {
            loc[i] = __ldcg(hist_g + threadIdx.x * PER + i);
            sum += loc[i];
        }
        scan[threadIdx.x] = sum;
    }
    __syncthreads();
    if (threadIdx.x == 0) {                   // 256 partial sums: one thread
        uint32_t acc = 0;
        for (int i = 0; i < 256; ++i) { acc += scan[i]; scan[i] = acc; }
    }
    __syncthreads();
    if (threadIdx.x < 256) {
        uint32_t acc = scan[threadIdx.x] - sum;
#pragma unroll
        for (int i = 0; i < PER; ++i) {
            cum[threadIdx.x * PER + i] = acc;
            acc += loc[i];
        }
        if (threadIdx.x == 255) cum[SELZ_NB] = acc;
    }
    __syncthreads();
}

// The zone of the typical signal, by one thread, after selz_plan.  The wanted element has rank (n3 - 1) / 2 among the
// kept pixels, n3 = npx - (excluded pixels), and every excluded pixel is in an OUT zone: among ALL pixels its position
// lies in [(npx - nout - 1) / 2, (npx - 1) / 2 + nout].
__device__ void selz_plan_m(const uint32_t* cum, SelZone* zn, SelzLists cap) {
    SelZone z = *zn;
    bool ok = z.ok && z.mok;
    if (ok) {
        const uint32_t nout = z.cnt_om + z.cnt_op;
        ok = nout < z.npx;
        if (ok) {
            const uint32_t glo = (z.npx - nout - 1u) / 2u;
            const unsigned long long gh = (unsigned long long)(z.npx - 1u) / 2u + nout;
            const uint32_t ghi = gh < z.npx ? (uint32_t)gh : z.npx - 1u;
            z.m5lo = max(selz_bucket_of_rank(cum, glo) - 1, 0);
            z.m5hi = min(selz_bucket_of_rank(cum, ghi) + 1, SELZ_NB - 1);
            z.below_m5 = cum[z.m5lo];
            z.cnt_m5 = cum[z.m5hi + 1] - cum[z.m5lo];
            ok = z.cnt_m5 <= cap.capm;
        }
    }
    z.mok = ok ? 1u : 0u;
    z.nm = 0;
    *zn = z;
}

__global__ void __launch_bounds__(SELZ_HT)
k_selz_hist(const float* __restrict__ R, const float* __restrict__ M5, size_t npx, SelState* st, SelZone* zn, uint32_t* histz,
            uint32_t* histm, void* lists, size_t list_words, const int* prev_count) {
    if (prev_count && *prev_count == 0) return;
    if (!zn->ok) return;
    __shared__ uint32_t sh[SELZ_NB + 1], shm[SELZ_NB + 1];
    for (int i = threadIdx.x; i < SELZ_NB; i += SELZ_HT) sh[i] = shm[i] = 0;
    __syncthreads();
    const float base = zn->base, scale = zn->scale, mbase = zn->mbase, mscale = zn->mscale;
    const bool wm = zn->mok != 0;             // also the grid of the typical signal
    const int bzero = selz_bucket(0.0f, base, scale);
    uint32_t nzero = 0, nneg0 = 0;
    auto visit = [&](float r, float m5, bool ok, size_t) {
        if (ok) {
            const int b = selz_bucket(r, base, scale);
            atomicAdd(&sh[b], 1u);
            if (b == bzero) {
                const uint32_t u = __float_as_uint(r);
                nzero += u == 0u ? 1u : 0u;
                nneg0 += u >> 31;
            }
            if (wm) atomicAdd(&shm[selz_bucket(m5 > 1e-4f ? m5 : 1e-4f, mbase, mscale)], 1u);
        }
    };
    if (wm) sel_visit_plane<true, SELZ_HT>(R, M5, npx, visit);
    else sel_visit_plane<false, SELZ_HT>(R, nullptr, npx, visit);
    nzero = __reduce_add_sync(0xffffffffu, nzero);
    nneg0 = __reduce_add_sync(0xffffffffu, nneg0);
    if ((threadIdx.x & 31) == 0 && nzero) atomicAdd(&zn->nzero, nzero);
    if ((threadIdx.x & 31) == 0 && nneg0) atomicAdd(&zn->nneg0, nneg0);
    __syncthreads();
    for (int i = threadIdx.x; i < SELZ_NB; i += SELZ_HT) {
        if (sh[i]) atomicAdd(&histz[i], sh[i]);
        if (wm && shm[i]) atomicAdd(&histm[i], shm[i]);
    }
    __shared__ bool s_last;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = atomicAdd(&st->ticket, 1u) == gridDim.x - 1;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    // cumulative counts (the histograms stay in global memory: k_selz_resolve reads single buckets of the first)
    __shared__ uint32_t scan[256];
    selz_cumulate(histz, sh, scan);
    if (wm) selz_cumulate(histm, shm, scan);
    if (threadIdx.x == 0) {
        selz_plan(sh, zn, selz_carve(lists, list_words));
        selz_plan_m(shm, zn, selz_carve(lists, list_words));
        st->ticket = 0;
    }
}

// zone id of a bucket: 0 none, 1 Z-, 2 Z0, 3 Z+, 4 OUT-, 5 OUT+
__device__ __forceinline__ uint32_t selz_zone_of(const SelZone& z, int b) {
    if (b <= z.omhi) return 4;
    if (b >= z.oplo) return 5;
    if (b >= z.z0lo && b <= z.z0hi) return 2;
    if (b >= z.zmlo && b <= z.zmhi) return 1;
    if (b >= z.zplo && b <= z.zphi) return 3;
    return 0;
}

// ---- read 2: the zones' values -> lists (any order) -----------------------------------------------
// A thread classifies 16 values at a time (zone id of a bucket from a table in shared memory); a warp then takes its
// slots in the CTA's staging with one atomic per list, and the CTA appends its staging with one global atomic per list
// at the end.  What does not fit the staging (a chunk that is all zone) takes slots of the list directly.  The
// residuals +0 of Z0 are not listed (SelZone::nzero).
__global__ void __launch_bounds__(256)
k_selz_compact(const float* __restrict__ R, const float* __restrict__ M5, size_t npx, SelZone* zn, void* lists,
               size_t list_words, const int* prev_count) {
    if (prev_count && *prev_count == 0) return;
    if (!zn->ok) return;
    __shared__ float s_0[SELZ_BUF], s_1[SELZ_BUF];
    __shared__ float2 s_o[SELZ_BUF];
    __shared__ uint8_t s_cls[SELZ_NB];        // list of a bucket: 0 none, 1 Z0, 2 Z- / Z+, 3 OUT
    __shared__ float s_m[SELZ_BUF];           // max(med5, 1e-4) of the pixels in ZM
    __shared__ uint32_t s_n[4], s_b[4];
    const SelzLists L = selz_carve(lists, list_words);
    const SelZone z = *zn;
    for (int i = threadIdx.x; i < SELZ_NB; i += 256) {
        const uint32_t zid = selz_zone_of(z, i);
        s_cls[i] = (uint8_t)(zid == 2 ? 1 : (zid == 1 || zid == 3) ? 2 : zid >= 4 ? 3 : 0);
    }
    if (threadIdx.x < 4) s_n[threadIdx.x] = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31;
    const float base = z.base, scale = z.scale, mbase = z.mbase, mscale = z.mscale;
    const bool wm = z.mok != 0;               // the list of the typical signal's zone too (reads the med5 plane as well)
    const int m5lo = z.m5lo, m5w = z.m5hi - z.m5lo;
    auto putm = [&](uint32_t p, float m5c) {
        if (p < SELZ_BUF) s_m[p] = m5c; else L.zm[atomicAdd(&zn->nm, 1u)] = m5c;
    };
    auto put = [&](uint32_t cls, uint32_t p, float r, size_t idx) {
        if (cls == 1) { if (p < SELZ_BUF) s_0[p] = r; else L.z0[atomicAdd(&zn->n0, 1u)] = r; }
        else if (cls == 2) { if (p < SELZ_BUF) s_1[p] = r; else L.z1[atomicAdd(&zn->n1, 1u)] = r; }
        else {
            const float2 e = make_float2(r, M5[idx]);
            if (p < SELZ_BUF) s_o[p] = e; else L.o[atomicAdd(&zn->no, 1u)] = e;
        }
    };
    const size_t nvec = npx / 4;
    for (size_t b0 = (size_t)blockIdx.x * 1024; b0 < nvec; b0 += (size_t)gridDim.x * 1024) {
        float v[16], mv[16];
        bool okv[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const size_t i = b0 + u * 256 + threadIdx.x;
            okv[u] = i < nvec;
            const float4 q = okv[u] ? __ldg(reinterpret_cast<const float4*>(R) + i) : make_float4(0.f, 0.f, 0.f, 0.f);
            v[4 * u] = q.x; v[4 * u + 1] = q.y; v[4 * u + 2] = q.z; v[4 * u + 3] = q.w;
            const float4 m = (wm && okv[u]) ? __ldg(reinterpret_cast<const float4*>(M5) + i) : make_float4(0.f, 0.f, 0.f, 0.f);
            mv[4 * u] = m.x; mv[4 * u + 1] = m.y; mv[4 * u + 2] = m.z; mv[4 * u + 3] = m.w;
        }
        uint32_t mbits = 0;                   // values whose med5 lies in ZM
        if (wm) {
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                mv[e] = mv[e] > 1e-4f ? mv[e] : 1e-4f;
                const uint32_t in = (uint32_t)(selz_bucket(mv[e], mbase, mscale) - m5lo) <= (uint32_t)m5w ? 1u : 0u;
                mbits |= (okv[e >> 2] ? in : 0u) << e;
            }
        }
        uint32_t codes = 0;                   // 2 bits per value: its list
#pragma unroll
        for (int e = 0; e < 16; ++e) {
            uint32_t cls = okv[e >> 2] ? s_cls[selz_bucket(v[e], base, scale)] : 0u;
            if (cls == 1 && __float_as_uint(v[e]) == 0u) cls = 0;
            codes |= cls << (2 * e);
        }
        // entries of this thread per list: fields equal to 1, 2, 3
        const uint32_t lo1 = codes & 0x55555555u, hi1 = (codes >> 1) & 0x55555555u;
        const uint32_t c0 = __popc(lo1 & ~hi1), c1 = __popc(hi1 & ~lo1), co = __popc(lo1 & hi1);
        if (__ballot_sync(0xffffffffu, (codes | mbits) != 0u) == 0) continue;
        // inclusive prefix sums over the warp (at most 16 x 32 = 512 entries per list: two lists share a word)
        const uint32_t own_a = c0 | (c1 << 16), own_b = co | ((uint32_t)__popc(mbits) << 16);
        uint32_t inc_a = own_a, inc_b = own_b;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t oa = __shfl_up_sync(0xffffffffu, inc_a, d), ob = __shfl_up_sync(0xffffffffu, inc_b, d);
            if (lane >= d) { inc_a += oa; inc_b += ob; }
        }
        uint32_t base0 = 0, base1 = 0, baseo = 0, basem = 0;
        if (lane == 31) {
            const uint32_t t0 = inc_a & 0xffffu, t1 = inc_a >> 16, to = inc_b & 0xffffu, tm = inc_b >> 16;
            if (t0) base0 = atomicAdd(&s_n[0], t0);
            if (t1) base1 = atomicAdd(&s_n[1], t1);
            if (to) baseo = atomicAdd(&s_n[2], to);
            if (tm) basem = atomicAdd(&s_n[3], tm);
        }
        const uint32_t ex_a = inc_a - own_a, ex_b = inc_b - own_b;
        uint32_t p0 = __shfl_sync(0xffffffffu, base0, 31) + (ex_a & 0xffffu);
        uint32_t p1 = __shfl_sync(0xffffffffu, base1, 31) + (ex_a >> 16);
        uint32_t po = __shfl_sync(0xffffffffu, baseo, 31) + (ex_b & 0xffffu);
        uint32_t pm = __shfl_sync(0xffffffffu, basem, 31) + (ex_b >> 16);
        while (mbits) {
            const int e = __ffs(mbits) - 1;
            mbits &= mbits - 1;
            float m = mv[0];
#pragma unroll
            for (int q = 1; q < 16; ++q) m = (e == q) ? mv[q] : m;
            putm(pm++, m);
        }
        uint32_t rem = codes;                 // (a thread has one hit in 16 values on average: loop over the hits)
        while (rem) {
            const int e = (__ffs(rem) - 1) >> 1;
            const uint32_t cls = (rem >> (2 * e)) & 3u;
            rem &= ~(3u << (2 * e));
            float r = v[0];
#pragma unroll
            for (int q = 1; q < 16; ++q) r = (e == q) ? v[q] : r;
            const size_t idx = 4 * (b0 + (size_t)(e >> 2) * 256 + threadIdx.x) + (e & 3);
            put(cls, cls == 1 ? p0++ : cls == 2 ? p1++ : po++, r, idx);
        }
    }
    if (blockIdx.x == 0) {                    // the last npx % 4 values: straight to the lists
        const size_t t = nvec * 4 + threadIdx.x;
        if (t < npx) {
            const float r = R[t];
            uint32_t cls = s_cls[selz_bucket(r, base, scale)];
            if (cls == 1 && __float_as_uint(r) == 0u) cls = 0;
            if (cls) put(cls, SELZ_BUF, r, t);
            if (wm) {
                const float m = M5[t] > 1e-4f ? M5[t] : 1e-4f;
                if ((uint32_t)(selz_bucket(m, mbase, mscale) - m5lo) <= (uint32_t)m5w) putm(SELZ_BUF, m);
            }
        }
    }
    __syncthreads();
    if (threadIdx.x < 4) {
        const uint32_t n = min(s_n[threadIdx.x], (uint32_t)SELZ_BUF);
        s_n[threadIdx.x] = n;
        uint32_t* cur = threadIdx.x == 0 ? &zn->n0 : threadIdx.x == 1 ? &zn->n1 : threadIdx.x == 2 ? &zn->no : &zn->nm;
        s_b[threadIdx.x] = n ? atomicAdd(cur, n) : 0u;
    }
    __syncthreads();
    for (uint32_t i = threadIdx.x; i < s_n[0]; i += 256) L.z0[s_b[0] + i] = s_0[i];
    for (uint32_t i = threadIdx.x; i < s_n[1]; i += 256) L.z1[s_b[1] + i] = s_1[i];
    for (uint32_t i = threadIdx.x; i < s_n[2]; i += 256) L.o[s_b[2] + i] = s_o[i];
    for (uint32_t i = threadIdx.x; i < s_n[3]; i += 256) L.zm[s_b[3] + i] = s_m[i];
}

// ---- the three rounds on the lists ----------------------------------------------------------------
struct SelzShared {
    uint32_t hist[SEL_BINS];
    uint32_t red[2][32];
    uint32_t bc[2][4];            // CTA 0: what a pick or a finished selection hands to the cluster (double buffered)
    uint32_t loc[4];              // CTA 0: the same inside its own passes
    uint32_t sums[2][2];          // per CTA: its part of the two counts of a round (double buffered)
    uint32_t edge[12];            // bucket edges as keys
};

// Every thread of the cluster visits its share of list[0..n): f(value, valid) is called the same number of times by
// all threads (votes are safe), SELZ_UNROLL loads in flight per thread.
template <class T, class F>
__device__ __forceinline__ void selz_for_each(cg::cluster_group& cl, const T* __restrict__ list, uint32_t n, F f) {
    const uint32_t gtid = cl.block_rank() * SELZ_RT + threadIdx.x, gn = SELZ_CLUSTER * SELZ_RT;
    if (n == 0) return;
    for (uint32_t b0 = 0; b0 < n; b0 += gn * SELZ_UNROLL) {
        T v[SELZ_UNROLL];
        bool ok[SELZ_UNROLL];
#pragma unroll
        for (int u = 0; u < SELZ_UNROLL; ++u) {
            const uint32_t i = b0 + u * gn + gtid;
            ok[u] = i < n;
            v[u] = __ldcg(list + (ok[u] ? i : 0u));      // (n > 0 here: entry 0 exists)
        }
#pragma unroll
        for (int u = 0; u < SELZ_UNROLL; ++u) f(v[u], ok[u]);
    }
}

// All SELZ_RT threads of ONE CTA: the digit that holds rank kth among 2048 digit totals, two per thread (t0: digit
// 2 tid, t1: digit 2 tid + 1).  out[0] = digit, out[1] = rank inside it, out[2] = its members; visible to the CTA on return.
__device__ __forceinline__ void selz_pick(SelzShared* sm, uint32_t t0, uint32_t t1, uint32_t kth, uint32_t* out) {
    const uint32_t sum = t0 + t1;
    uint32_t incl = sum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t o = __shfl_up_sync(0xffffffffu, incl, d);
        if ((threadIdx.x & 31) >= d) incl += o;
    }
    if ((threadIdx.x & 31) == 31) sm->red[0][threadIdx.x >> 5] = incl;
    __syncthreads();
    uint32_t woff = 0;
    for (int w = 0; w < (int)(threadIdx.x >> 5); ++w) woff += sm->red[0][w];
    incl += woff;
    const uint32_t excl = incl - sum;
    if (kth >= excl && kth < incl) {
        const uint32_t hi1 = kth >= excl + t0 ? 1u : 0u;
        out[0] = 2 * threadIdx.x + hi1;
        out[1] = kth - excl - (hi1 ? t0 : 0u);
        out[2] = hi1 ? t1 : t0;
    }
    __syncthreads();
}

// Radix selection on the cluster over the keys keyfn(list[i]) inside [klo, khi]: returns the key of rank `kth` among
// them (the caller guarantees that there are more than kth).  A pass histograms 11 bits of the remaining key range on
// all CTAs; as soon as the digit that holds the rank has at most `capscr` members, they are copied to the scratch
// list and CTA 0 finishes the selection over those alone (block barriers only: a cluster barrier with its fences costs
// about as much as a pass over the list).  `vcount` further elements of key `vkey` take part without being in the
// list (the residuals +0 of Z0).  par, cpar: the caller's counters of broadcasts and scratch uses (the same in all threads).
template <class T, class KF>
__device__ __forceinline__ uint32_t selz_select(cg::cluster_group& cl, SelzShared* sm, const T* __restrict__ list, uint32_t n,
                                                uint32_t klo, uint32_t khi, uint32_t kth, uint32_t* scr, uint32_t capscr,
                                                uint32_t* scr_cursor, uint32_t vkey, uint32_t vcount, int& par, int& cpar,
                                                KF keyfn) {
    const bool lead = cl.block_rank() == 0;
    const SelzShared* lsm = cl.map_shared_rank(sm, 0);
    while (khi > klo) {
        const uint32_t span = khi - klo;
        const int bits = 32 - __clz(span);
        const int shift = bits > 11 ? bits - 11 : 0;
        for (int i = threadIdx.x; i < SEL_BINS; i += SELZ_RT) sm->hist[i] = 0;
        __syncthreads();
        // (plain shared-memory atomics: the keys of a pass spread over the digits unless the list is all ties)
        selz_for_each(cl, list, n, [&](T e, bool ok) {
            const uint32_t dk = keyfn(e) - klo;
            if (ok && dk <= span) atomicAdd(&sm->hist[dk >> shift], 1u);
        });
        cl.sync();
        if (lead) {
            uint32_t t2[2];
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                uint32_t t = 0;
                for (int r = 0; r < SELZ_CLUSTER; ++r) t += cl.map_shared_rank(sm, r)->hist[2 * threadIdx.x + u];
                if (vcount && vkey - klo <= span && ((vkey - klo) >> shift) == 2u * threadIdx.x + u) t += vcount;
                t2[u] = t;
            }
            selz_pick(sm, t2[0], t2[1], kth, sm->bc[par & 1]);
        }
        cl.sync();
        const uint32_t digit = lsm->bc[par & 1][0], members = lsm->bc[par & 1][2];
        kth = lsm->bc[par & 1][1];
        ++par;
        klo += digit << shift;
        const uint32_t nhi = shift ? klo + ((1u << shift) - 1u) : klo;
        khi = nhi < khi ? nhi : khi;
        if (khi == klo) break;
        const bool vin = vcount && vkey >= klo && vkey <= khi;
        const uint32_t listed = members - (vin ? vcount : 0u);
        if (listed > capscr) continue;                    // (a list of ties) another pass over the whole list
        // copy the candidates; CTA 0 finishes over them
        uint32_t* cur = scr_cursor + (cpar & 1);
        if (lead && threadIdx.x == 0) scr_cursor[(cpar + 1) & 1] = 0;   // the other cursor, for the next use
        ++cpar;
        {
            const uint32_t nspan = khi - klo;
            selz_for_each(cl, list, n, [&](T e, bool ok) {
                const uint32_t k = keyfn(e);
                const bool v = ok && k - klo <= nspan;
                const unsigned m = __ballot_sync(0xffffffffu, v);
                if (m) {
                    const int lane = threadIdx.x & 31;
                    uint32_t b = 0;
                    if (lane == 0) b = atomicAdd(cur, (uint32_t)__popc(m));
                    b = __shfl_sync(0xffffffffu, b, 0);
                    if (v) scr[b + __popc(m & ((1u << lane) - 1u))] = k;
                }
            });
        }
        __threadfence();
        cl.sync();
        if (lead) {
            while (khi > klo) {
                const uint32_t sp2 = khi - klo;
                const int b2 = 32 - __clz(sp2);
                const int sh2 = b2 > 11 ? b2 - 11 : 0;
                for (int i = threadIdx.x; i < SEL_BINS; i += SELZ_RT) sm->hist[i] = 0;
                __syncthreads();
                for (uint32_t i = threadIdx.x; i < listed; i += SELZ_RT) {
                    const uint32_t dk = __ldcg(scr + i) - klo;
                    if (dk <= sp2) atomicAdd(&sm->hist[dk >> sh2], 1u);
                }
                __syncthreads();
                uint32_t t0 = sm->hist[2 * threadIdx.x], t1 = sm->hist[2 * threadIdx.x + 1];
                if (vin && vkey - klo <= sp2) {
                    const uint32_t vd = (vkey - klo) >> sh2;
                    if (vd == 2u * threadIdx.x) t0 += vcount;
                    if (vd == 2u * threadIdx.x + 1u) t1 += vcount;
                }
                selz_pick(sm, t0, t1, kth, sm->loc);
                kth = sm->loc[1];
                klo += sm->loc[0] << sh2;
                const uint32_t h2 = sh2 ? klo + ((1u << sh2) - 1u) : klo;
                khi = h2 < khi ? h2 : khi;
                __syncthreads();                         // loc and hist are rewritten by the next pass
            }
            if (threadIdx.x == 0) sm->bc[par & 1][0] = klo;
        }
        cl.sync();
        klo = khi = lsm->bc[par & 1][0];
        ++par;
    }
    return klo;
}

// smallest key k in [key(-inf), key(+inf)] with bucket(unkey(k)) >= b (the bucket is non-decreasing in the key there);
// b in 1 .. SELZ_NB (b = SELZ_NB: one past key(+inf))
__device__ __forceinline__ uint32_t selz_edge_key(int b, float base, float scale) {
    uint32_t lo = 0x007fffffu, hi = 0xff800000u;        // bucket(lo) = 0 < b
    if (b >= SELZ_NB || selz_bucket(sel_unkey(hi), base, scale) < b) return hi + 1u;
    while (hi - lo > 1u) {                               // invariant: bucket(lo) < b <= bucket(hi)
        const uint32_t mid = lo + ((hi - lo) >> 1);
        if (selz_bucket(sel_unkey(mid), base, scale) >= b) hi = mid; else lo = mid;
    }
    return hi;
}

// the same for the grid of max(med5, 1e-4) (positive values: key = bits | 0x80000000): smallest key with bucket >= b
__device__ __forceinline__ uint32_t selz_edge_key_m(int b, float base, float scale) {
    uint32_t lo = 0x80000000u, hi = 0xff800000u;        // +0 (below every value: they are >= 1e-4) .. +inf
    if (selz_bucket(__uint_as_float(lo & 0x7fffffffu), base, scale) >= b) return lo;
    if (b >= SELZ_NB || selz_bucket(__uint_as_float(hi & 0x7fffffffu), base, scale) < b) return hi + 1u;
    while (hi - lo > 1u) {                               // invariant: bucket(lo) < b <= bucket(hi)
        const uint32_t mid = lo + ((hi - lo) >> 1);
        if (selz_bucket(__uint_as_float(mid & 0x7fffffffu), base, scale) >= b) hi = mid; else lo = mid;
    }
    return hi;
}

// Radix selection on the cluster over the multiset { keys of `add` } minus { keyfn_sub of the entries of `sub` it accepts }
// inside [klo, khi]: the key of rank kth (the caller guarantees more than kth members).  No scratch list: two or
// three passes over the lists.
template <class KS>
__device__ __forceinline__ uint32_t selz_select_sub(cg::cluster_group& cl, SelzShared* sm, const float* __restrict__ add, uint32_t nadd,
                                                    const float2* __restrict__ sub, uint32_t nsub, uint32_t klo, uint32_t khi,
                                                    uint32_t kth, int& par, KS keyfn_sub) {
    const bool lead = cl.block_rank() == 0;
    const SelzShared* lsm = cl.map_shared_rank(sm, 0);
    while (khi > klo) {
        const uint32_t span = khi - klo;
        const int bits = 32 - __clz(span);
        const int shift = bits > 11 ? bits - 11 : 0;
        for (int i = threadIdx.x; i < SEL_BINS; i += SELZ_RT) sm->hist[i] = 0;
        __syncthreads();
        selz_for_each(cl, add, nadd, [&](float v, bool ok) {
            const uint32_t dk = (__float_as_uint(v) | 0x80000000u) - klo;
            if (ok && dk <= span) atomicAdd(&sm->hist[dk >> shift], 1u);
        });
        selz_for_each(cl, sub, nsub, [&](float2 e, bool ok) {
            uint32_t k = 0;
            if (ok && keyfn_sub(e, k) && k - klo <= span) atomicSub(&sm->hist[(k - klo) >> shift], 1u);   // (wraps; the sum is exact)
        });
        cl.sync();
        if (lead) {
            uint32_t t2[2];
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                uint32_t t = 0;
                for (int r = 0; r < SELZ_CLUSTER; ++r) t += cl.map_shared_rank(sm, r)->hist[2 * threadIdx.x + u];
                t2[u] = t;
            }
            selz_pick(sm, t2[0], t2[1], kth, sm->bc[par & 1]);
        }
        cl.sync();
        const uint32_t digit = lsm->bc[par & 1][0];
        kth = lsm->bc[par & 1][1];
        ++par;
        klo += digit << shift;
        const uint32_t nhi = shift ? klo + ((1u << shift) - 1u) : klo;
        khi = nhi < khi ? nhi : khi;
    }
    return klo;
}

__global__ void __cluster_dims__(SELZ_CLUSTER, 1, 1) __launch_bounds__(SELZ_RT)
k_selz_resolve(SelState* st, SelZone* zn, const uint32_t* __restrict__ histz, void* lists, size_t list_words,
               float rn2, float* gain_out, float* stats, const int* prev_count) {
    float* const path_out = stats ? stats + 6 : nullptr;
    if (prev_count && *prev_count == 0) return;
    if (!zn->ok) {
        if (path_out && blockIdx.x == 0 && threadIdx.x == 0) *path_out = 0.0f;
        return;
    }
    cg::cluster_group cl = cg::this_cluster();
    __shared__ SelzShared sm_;
    SelzShared* sm = &sm_;
    const SelZone z = *zn;
    const SelzLists L = selz_carve(lists, list_words);
    const int bzero = selz_bucket(0.0f, z.base, z.scale);
    const uint32_t vzero = (bzero >= z.z0lo && bzero <= z.z0hi) ? z.nzero : 0u;    // the residuals +0 of Z0: counted, not listed
    const uint32_t n0 = z.cnt_z0 - vzero, n1 = z.cnt_zm + z.cnt_zp, no = z.cnt_om + z.cnt_op;
    const float INF = __int_as_float(0x7f800000);
    const float base = z.base, scale = z.scale;
    // first and last float of what lies between the zones, exactly (bisection on the bucket function, one thread each):
    //   every value outside OUT- / OUT+ is in [e_keep_lo, e_keep_hi];
    //   every value between Z- and Z+ is in [e_in_lo, e_in_hi]; every value beyond them is <= e_out_lo or >= e_out_hi
    if (threadIdx.x < 6) {
        const int eb[6] = {z.omhi + 1, z.oplo, z.zmhi + 1, z.zplo, z.zmlo, z.zphi + 1};
        sm->edge[threadIdx.x] = selz_edge_key(eb[threadIdx.x], base, scale);
    }
    __syncthreads();
    const float e_keep_lo = sel_unkey(sm->edge[0]), e_keep_hi = sel_unkey(sm->edge[1] - 1u);
    const float e_in_lo = sel_unkey(sm->edge[2]), e_in_hi = sel_unkey(sm->edge[3] - 1u);
    const float e_out_lo = sel_unkey(sm->edge[4] - 1u), e_out_hi = sel_unkey(sm->edge[5]);

    float lo = -INF, hi = INF, c = 0.0f, s = 0.0f, lo0 = -INF, hi0 = INF;
    uint32_t nkept = 0, why = 0;
    int par = 0, cpar = 0;
    bool ok = true;
    for (int j = 0; j < SEL_ROUNDS && ok; ++j) {
        // the kept set: everything except the OUT values outside [lo, hi] (NaN counts as below)
        uint32_t nl = 0, nh = 0;
        selz_for_each(cl, L.o, no, [&](float2 e, bool v) {
            nl += (v && !(e.x >= lo)) ? 1u : 0u;
            nh += (v && e.x > hi) ? 1u : 0u;
        });
        nl = __reduce_add_sync(0xffffffffu, nl);
        nh = __reduce_add_sync(0xffffffffu, nh);
        if ((threadIdx.x & 31) == 0) { sm->red[0][threadIdx.x >> 5] = nl; sm->red[1][threadIdx.x >> 5] = nh; }
        __syncthreads();
        if (threadIdx.x < 2) {
            uint32_t t = 0;
            for (int i = 0; i < SELZ_RT / 32; ++i) t += sm->red[threadIdx.x][i];
            sm->sums[j & 1][threadIdx.x] = t;
        }
        cl.sync();
        uint32_t nlow = 0, nhigh = 0;
        for (int r = 0; r < SELZ_CLUSTER; ++r) {
            const SelzShared* o = cl.map_shared_rank(sm, r);
            nlow += o->sums[j & 1][0];
            nhigh += o->sums[j & 1][1];
        }
        // every value outside the OUT zones must be kept
        ok = (lo == -INF || lo <= e_keep_lo) && (hi == INF || hi >= e_keep_hi) && nlow + nhigh < z.npx;
        why = 10 * (j + 1) + 1;                          // the clipping bounds left the OUT zones
        if (!ok) break;
        const uint32_t n = z.npx - nlow - nhigh;
        lo0 = lo; hi0 = hi; nkept = n;
        const uint32_t k = (n - 1u) / 2u;
        const uint32_t g = k + nlow;                     // rank among all values
        ok = g >= z.below_z0 && g - z.below_z0 < z.cnt_z0;
        why = 10 * (j + 1) + 2;                          // the centre left Z0
        if (!ok) break;
        // centre: the bucket of Z0 that holds rank g, then a selection among its members
        uint32_t acc = z.below_z0;
        int bq = z.z0lo;
        for (; bq < z.z0hi; ++bq) {
            const uint32_t hq = __ldcg(histz + bq);
            if (g < acc + hq) break;
            acc += hq;
        }
        if (vzero && bq == bzero && g - acc >= z.nneg0 && g - acc - z.nneg0 < vzero) {
            c = 0.0f;                                    // the rank falls on the residuals +0 of that bucket
        } else {
            __syncthreads();
            if (threadIdx.x < 2) sm->edge[6 + threadIdx.x] = selz_edge_key(bq + threadIdx.x, base, scale);
            __syncthreads();
            const uint32_t kclo = sm->edge[6], kchi = sm->edge[7] - 1u;
            const uint32_t kc = selz_select(cl, sm, L.z0, n0, kclo, kchi, g - acc, L.scr, L.capscr, zn->nscr, 0x80000000u, vzero,
                                            par, cpar, [&](float r) -> uint32_t { return sel_key(r); });
            c = sel_unkey(kc);
        }
        // MAD: rank k of |r - c| over the kept set.  With c between Z- and Z+, every value between them is at
        // most vin away from c and every kept value beyond them at least vout; if the element of rank k - inner of
        // V = { |r - c| : r in Z- or Z+ } lies in [vin, vout], it is the element of rank k of all.
        ok = k >= z.inner && k - z.inner < n1 && c >= e_in_lo && c <= e_in_hi;
        why = 10 * (j + 1) + 3;                          // the rank of the MAD left Z- / Z+
        if (!ok) break;
        const float vin = fmaxf(fabsf(__fsub_rn(e_in_lo, c)), fabsf(__fsub_rn(e_in_hi, c)));
        const float vout = fminf(fabsf(__fsub_rn(e_out_lo, c)), fabsf(__fsub_rn(e_out_hi, c)));
        // (all of V lies between the nearer inner edge and the farther outer edge)
        const float vmin = fminf(fabsf(__fsub_rn(e_in_lo, c)), fabsf(__fsub_rn(e_in_hi, c)));
        const float vmax = fmaxf(fabsf(__fsub_rn(e_out_lo, c)), fabsf(__fsub_rn(e_out_hi, c)));
        const uint32_t kd = selz_select(cl, sm, L.z1, n1, __float_as_uint(vmin) | 0x80000000u, __float_as_uint(vmax) | 0x80000000u,
                                        k - z.inner, L.scr, L.capscr, zn->nscr, 0u, 0u, par, cpar,
                                        [&](float r) -> uint32_t { return __float_as_uint(fabsf(__fsub_rn(r, c))) | 0x80000000u; });
        const float d = __uint_as_float(kd & 0x7fffffffu);
        ok = d >= vin && d <= vout;
        why = 10 * (j + 1) + 4;                          // the MAD left Z- / Z+
        if (!ok) break;
        s = __fmul_rn(1.4826f, d);
        if (j < SEL_ROUNDS - 1) {
            const float five_s = __fmul_rn(5.0f, s);
            const float nlo = __fsub_rn(c, five_s), nhi = __fadd_rn(c, five_s);
            lo = nlo > lo ? nlo : lo;
            hi = nhi < hi ? nhi : hi;
        }
    }
    // The typical signal: rank (n - 1) / 2 of max(med5, 1e-4) over the kept pixels = all pixels minus the OUT entries
    // outside the interval the last round started from.  Everything outside ZM enters through the exact bucket counts.
    bool mok = ok && z.mok;
    float mt = 0.0f;
    if (mok) {
        const float mbase = z.mbase, mscale = z.mscale;
        uint32_t nb = 0, nin = 0;                 // excluded pixels below ZM / inside ZM
        selz_for_each(cl, L.o, no, [&](float2 e, bool v) {
            if (v && !(e.x >= lo0 && e.x <= hi0)) {
                const int bm = selz_bucket(e.y > 1e-4f ? e.y : 1e-4f, mbase, mscale);
                nb += bm < z.m5lo ? 1u : 0u;
                nin += (bm >= z.m5lo && bm <= z.m5hi) ? 1u : 0u;
            }
        });
        nb = __reduce_add_sync(0xffffffffu, nb);
        nin = __reduce_add_sync(0xffffffffu, nin);
        __syncthreads();
        if ((threadIdx.x & 31) == 0) { sm->red[0][threadIdx.x >> 5] = nb; sm->red[1][threadIdx.x >> 5] = nin; }
        __syncthreads();
        if (threadIdx.x < 2) {
            uint32_t t = 0;
            for (int i = 0; i < SELZ_RT / 32; ++i) t += sm->red[threadIdx.x][i];
            sm->sums[1][threadIdx.x] = t;         // (slot 1 was last used by round 1; round 2 used slot 0)
        }
        cl.sync();
        uint32_t xb = 0, xin = 0;
        for (int r = 0; r < SELZ_CLUSTER; ++r) {
            const SelzShared* o = cl.map_shared_rank(sm, r);
            xb += o->sums[1][0];
            xin += o->sums[1][1];
        }
        const uint32_t k3 = (nkept - 1u) / 2u;
        const uint32_t kept_below = z.below_m5 - xb;
        mok = xb <= z.below_m5 && xin <= z.cnt_m5 && k3 >= kept_below && k3 - kept_below < z.cnt_m5 - xin;
        if (mok) {
            __syncthreads();
            if (threadIdx.x < 2) sm->edge[8 + threadIdx.x] = selz_edge_key_m(threadIdx.x == 0 ? z.m5lo : z.m5hi + 1, mbase, mscale);
            __syncthreads();
            const uint32_t km = selz_select_sub(cl, sm, L.zm, z.cnt_m5, L.o, no, sm->edge[8], sm->edge[9] - 1u, k3 - kept_below, par,
                                                [&](float2 e, uint32_t& key) {
                if (e.x >= lo0 && e.x <= hi0) return false;
                const float m = e.y > 1e-4f ? e.y : 1e-4f;
                const int bm = selz_bucket(m, mbase, mscale);
                key = __float_as_uint(m) | 0x80000000u;
                return bm >= z.m5lo && bm <= z.m5hi;
            });
            mt = __uint_as_float(km & 0x7fffffffu);
        }
    }
    cl.sync();                                            // nobody leaves while its shared memory may still be read
    if (cl.block_rank() == 0 && threadIdx.x == 0) {
        if (ok) {
            st->c = c; st->s = s; st->lo = lo0; st->hi = hi0; st->n = nkept;
            st->prefix = 0; st->kth = 0;
        }
        zn->done = ok ? 1u : 0u;
        zn->why = ok ? 0u : why;
        zn->mdone = mok ? 1u : 0u;
        if (path_out) *path_out = ok ? 1.0f : 0.0f;
        if (mok) {
            // sigma^2 gain^2 - gain - rn^2 / mt = 0, positive root, in the oracle's operation order (as sel_pick<2, 2>)
            const float s2 = __fmul_rn(s, s);
            const float aa = __fdiv_rn(__fmul_rn(__fmul_rn(4.0f, s2), rn2), mt);
            const float g = __fdiv_rn(__fadd_rn(1.0f, __fsqrt_rn(__fadd_rn(1.0f, aa))), __fmul_rn(2.0f, s2));
            *gain_out = (s > 0.0f && s < INF && g > 0.0f && g < INF) ? g : 1.0f;
            if (stats) {
                stats[0] = c; stats[1] = s; stats[2] = lo0; stats[3] = hi0; stats[4] = (float)nkept;
                stats[5] = mt;
            }
        }
    }
}

}  // namespace lac
