// Gain estimation when no gain is supplied (reading R21; "sigma_clip"):
// sigma clipping of the residual plane r = (work - med5) / sqrt(med5) made of SELECTION only, so the
// result does not depend on the order in which pixels are visited and equals the CPU oracle bit for bit.
//
// An element of given rank is found by a three-pass radix selection over an order-preserving 32-bit key of
// the value (11 + 11 + 10 bits): every pass histograms one digit of the keys that match the digits already
// fixed (shared-memory histogram per CTA, flushed with atomics); the CTA that finishes last (atomic ticket)
// then walks the 2048 counts to the bucket holding the wanted rank, so a pass is one launch.  One round of
// the clipping is two selections over the kept set K = { lo <= r <= hi }: the centre c (rank (n-1)/2 of r)
// and the MAD d (same rank of |r - c|).  A last selection gives the typical signal mt (same rank of max(med5,
// 1e-4) over the set the last round kept), and the gain follows from the noise model (R21).
#pragma once
#include <cooperative_groups.h>

#include "common.cuh"

namespace lac {

constexpr int SEL_BINS = 2048;
constexpr int SEL_ROUNDS = 3;

struct SelState {
    float lo, hi;          // interval the current round started from
    float c, s;            // centre and 1.4826 * MAD of the current round
    uint32_t prefix;       // key digits fixed so far
    uint32_t kth;          // wanted rank among the keys that match `prefix`
    uint32_t n;            // |K| of the current round
    uint32_t ticket;       // CTAs of the running pass that have flushed their histogram
};

// order-preserving key: ascending keys <=> ascending floats (a total order that refines the float order:
// -0 sorts directly below +0, so an element of given rank has the right VALUE; NaNs fall outside
// [key(-inf), key(+inf)])
__device__ __forceinline__ uint32_t sel_key(float v) {
    const uint32_t u = __float_as_uint(v);
    return u ^ ((uint32_t)((int32_t)u >> 31) | 0x80000000u);
}
__device__ __forceinline__ float sel_unkey(uint32_t k) {
    return __uint_as_float((k & 0x80000000u) ? (k & 0x7fffffffu) : ~k);
}

// inclusive prefix sums over the 256 threads of a CTA (scan: 256 words of shared memory); returns this thread's
__device__ __forceinline__ uint32_t sel_scan256(uint32_t sum, uint32_t* scan) {
    const int tid = threadIdx.x;
    scan[tid] = sum;
    __syncthreads();
    for (int d = 1; d < 256; d <<= 1) {
        const uint32_t v = tid >= d ? scan[tid - d] : 0u;
        __syncthreads();
        scan[tid] += v;
        __syncthreads();
    }
    return scan[tid];
}

// Visits the plane R (and M5 when WITH_M5) in chunks of 16 values per thread of an NT-thread CTA: f(r, m5, valid, index) is
// called by ALL threads of the CTA the same number of times (valid = false past the end), so f may use warp votes.
template <bool WITH_M5, int NT, class F>
__device__ __forceinline__ void sel_visit_plane(const float* __restrict__ R, const float* __restrict__ M5, size_t npx, F f) {
    const size_t nvec = npx / 4;
    const float4 zero4 = make_float4(0.f, 0.f, 0.f, 0.f);
    for (size_t b0 = (size_t)blockIdx.x * (4 * NT); b0 < nvec; b0 += (size_t)gridDim.x * (4 * NT)) {
        float4 q[4], m[4];
        bool ok[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {     // four independent 16-byte loads in flight per thread
            const size_t i = b0 + u * NT + threadIdx.x;
            ok[u] = i < nvec;
            q[u] = ok[u] ? __ldg(reinterpret_cast<const float4*>(R) + i) : zero4;
            m[u] = (WITH_M5 && ok[u]) ? __ldg(reinterpret_cast<const float4*>(M5) + i) : zero4;
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const size_t i4 = 4 * (b0 + u * NT + threadIdx.x);
            f(q[u].x, m[u].x, ok[u], i4); f(q[u].y, m[u].y, ok[u], i4 + 1); f(q[u].z, m[u].z, ok[u], i4 + 2);
            f(q[u].w, m[u].w, ok[u], i4 + 3);
        }
    }
    if (blockIdx.x == 0) {                // the last npx % 4 values
        const size_t t = nvec * 4 + threadIdx.x;
        const bool ok = t < npx;
        f(ok ? R[t] : 0.0f, (WITH_M5 && ok) ? M5[t] : 0.0f, ok, t);
    }
}

// shared-memory histogram increment with the warp's votes for the leader's bucket combined into one atomic
// (values that are smooth over the frame, or a list of equal keys, put a whole warp on one address).  All 32
// lanes call.
__device__ __forceinline__ void sel_hist_add(uint32_t* sh, bool valid, uint32_t bin) {
    const unsigned m = __ballot_sync(0xffffffffu, valid);
    if (m == 0) return;
    const int lane = threadIdx.x & 31, leader = __ffs(m) - 1;
    const uint32_t b0 = __shfl_sync(0xffffffffu, bin, leader);
    const unsigned same = __ballot_sync(0xffffffffu, valid && bin == b0);
    if (lane == leader) atomicAdd(&sh[b0], (uint32_t)__popc(same));
    else if (valid && bin != b0) atomicAdd(&sh[bin], 1u);
}

__global__ void k_sel_init(SelState* st, uint32_t* hist, const int* prev_count) {
    if (prev_count && *prev_count == 0) return;
    for (int i = threadIdx.x; i < SEL_BINS; i += blockDim.x) hist[i] = 0;
    if (threadIdx.x == 0) {
        st->lo = -__int_as_float(0x7f800000);
        st->hi = __int_as_float(0x7f800000);
        st->c = 0.0f;
        st->s = 0.0f;
        st->prefix = 0;
        st->kth = 0;
        st->n = 0;
        st->ticket = 0;
    }
}

// Executed by the last CTA of a pass (256 threads; `scan` is 256 words of shared memory): find the bucket
// holding rank kth, fix its digit, clear the histogram.  After the last pass of MODE 0 the selected value is
// the centre c; after the last pass of MODE 1 it is the MAD d: s = 1.4826 d and the next round's interval
// follow with exactly the oracle's operations; the `last` round writes the gain instead (and the statistics
// {c, s, lo, hi, kept} of the round when stats is given).
template <int MODE, int PASS>
__device__ __forceinline__ void sel_pick(SelState* st, uint32_t* hist, uint32_t* scan, int last, float rn2,
                                         float* gain_out, float* stats) {
    const int tid = threadIdx.x;
    constexpr int PER = SEL_BINS / 256;
    uint32_t loc[PER], sum = 0;
#pragma unroll
    for (int i = 0; i < PER; ++i) {
        loc[i] = __ldcg(hist + tid * PER + i);
        sum += loc[i];
        hist[tid * PER + i] = 0;
    }
    scan[tid] = sum;
    __syncthreads();
    for (int d = 1; d < 256; d <<= 1) {   // inclusive prefix sums of the 256 group totals
        const uint32_t v = tid >= d ? scan[tid - d] : 0u;
        __syncthreads();
        scan[tid] += v;
        __syncthreads();
    }
    const uint32_t incl = scan[tid], excl = incl - sum, n = scan[255];
    const uint32_t kth = PASS == 0 ? (n - 1u) / 2u : __ldcg(&st->kth);
    if (kth >= excl && kth < incl) {      // exactly one thread: the group that holds the rank
        uint32_t acc = excl;
        int i = 0;
        while (i < PER - 1 && acc + loc[i] <= kth) acc += loc[i++];
        const uint32_t digit = (uint32_t)(tid * PER + i);
        const uint32_t prefix = PASS == 0 ? digit : PASS == 1 ? ((__ldcg(&st->prefix) << 11) | digit) : ((__ldcg(&st->prefix) << 10) | digit);
        if (PASS == 0) st->n = n;
        st->kth = kth - acc;
        st->prefix = prefix;
        if (PASS == 2) {
            const float v = sel_unkey(prefix);
            if (MODE == 0) {
                st->c = v;
            } else if (MODE == 1) {
                const float s = __fmul_rn(1.4826f, v);
                const float five_s = __fmul_rn(5.0f, s);
                const float cc = __ldcg(&st->c), olo = __ldcg(&st->lo), ohi = __ldcg(&st->hi);
                const float nlo = __fsub_rn(cc, five_s), nhi = __fadd_rn(cc, five_s);
                st->s = s;
                if (!last) {   // the next round starts from the intersection
                    st->lo = nlo > olo ? nlo : olo;
                    st->hi = nhi < ohi ? nhi : ohi;
                }
            } else {
                // v = mt, the typical signal.  sigma^2 gain^2 - gain - rn^2/mt = 0, positive root, in the
                // oracle's operation order
                const float s = __ldcg(&st->s);
                const float s2 = __fmul_rn(s, s);
                const float a = __fdiv_rn(__fmul_rn(__fmul_rn(4.0f, s2), rn2), v);
                const float g = __fdiv_rn(__fadd_rn(1.0f, __fsqrt_rn(__fadd_rn(1.0f, a))), __fmul_rn(2.0f, s2));
                const float INF = __int_as_float(0x7f800000);
                *gain_out = (s > 0.0f && s < INF && g > 0.0f && g < INF) ? g : 1.0f;
                if (stats) {
                    stats[0] = __ldcg(&st->c); stats[1] = s; stats[2] = __ldcg(&st->lo); stats[3] = __ldcg(&st->hi); stats[4] = (float)__ldcg(&st->n);
                    stats[5] = v;
                }
            }
            st->prefix = 0;
        }
    }
}

// MODE 0: value = r; MODE 1: value = |r - c|; MODE 2: value = max(med5, 1e-4) (plane M5), all over the kept
// set lo <= r <= hi.  PASS 0/1/2: key bits 31..21 / 20..10 / 9..0.
// sh: SEL_BINS words of shared memory; fast (MODE 2 only): the three rounds were resolved on the zone lists
// (selectz.cuh) and the typical signal is selected over ALL pixels of the med5 plane minus the listed pixels outside
// the kept interval (every such pixel is in the OUT list), so that the residual plane is not read again.
template <int MODE, int PASS>
__device__ __forceinline__ void sel_hist_pass(const float* __restrict__ R, const float* __restrict__ M5, size_t npx, SelState* st,
                                              uint32_t* hist, int last, float rn2, float* gain_out, float* stats, bool fast,
                                              const uint32_t* zno, const float2* __restrict__ olist, uint32_t* sh) {
    for (int i = threadIdx.x; i < SEL_BINS; i += 256) sh[i] = 0;
    __syncthreads();
    // (the state is read past the L1: inside k_sel_rounds it was written by another CTA of the same launch)
    const float lo = __ldcg(&st->lo), hi = __ldcg(&st->hi), c = __ldcg(&st->c);
    const uint32_t st_prefix = __ldcg(&st->prefix);
    // keys under the digits already fixed form one range; MODE 0 intersects it with the kept interval, which
    // is a key range too (the key is monotone), so a value costs one key and one unsigned range check
    constexpr int SHIFT = PASS == 0 ? 21 : PASS == 1 ? 10 : 0;
    constexpr uint32_t MASK = PASS == 2 ? 0x3ffu : 0x7ffu;
    uint32_t klo = 0u, khi = 0xffffffffu;
    if (PASS == 1) { klo = st_prefix << 21; khi = klo | 0x1fffffu; }
    if (PASS == 2) { klo = st_prefix << 10; khi = klo | 0x3ffu; }
    if (MODE == 0) {
        klo = max(klo, sel_key(lo));
        khi = min(khi, sel_key(hi));
    }
    const bool none = klo > khi;                    // empty intersection (cannot hold the wanted rank)
    const uint32_t span = khi - klo;
    auto visit = [&](float r, float m5) {
        uint32_t k;
        if (MODE == 0) {
            k = sel_key(r);
        } else {
            if (!(MODE == 2 && fast) && !(r >= lo && r <= hi)) return;
            const float v = MODE == 1 ? fabsf(__fsub_rn(r, c)) : (m5 > 1e-4f ? m5 : 1e-4f);
            k = __float_as_uint(v) | 0x80000000u;   // non-negative value
        }
        if (!none && k - klo <= span) atomicAdd(&sh[(k >> SHIFT) & MASK], 1u);
    };
    const size_t nvec = npx / 4;
    const size_t stride = (size_t)gridDim.x * 256, end = nvec;
    size_t i = (size_t)blockIdx.x * 256 + threadIdx.x;
    const float4 zero4 = make_float4(0.f, 0.f, 0.f, 0.f);
    const bool one = MODE == 2 && fast;             // only the med5 plane is read
    const float* P0 = one ? M5 : R;
    for (; i + 3 * stride < end; i += 4 * stride) {   // four independent 16-byte loads in flight per thread
        float4 q[4], m[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            q[u] = __ldg(reinterpret_cast<const float4*>(P0) + i + u * stride);
            m[u] = (MODE == 2 && !one) ? __ldg(reinterpret_cast<const float4*>(M5) + i + u * stride) : MODE == 2 ? q[u] : zero4;
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            visit(q[u].x, m[u].x); visit(q[u].y, m[u].y); visit(q[u].z, m[u].z); visit(q[u].w, m[u].w);
        }
    }
    for (; i < end; i += stride) {
        const float4 q = __ldg(reinterpret_cast<const float4*>(P0) + i);
        const float4 m = (MODE == 2 && !one) ? __ldg(reinterpret_cast<const float4*>(M5) + i) : MODE == 2 ? q : zero4;
        visit(q.x, m.x); visit(q.y, m.y); visit(q.z, m.z); visit(q.w, m.w);
    }
    if (blockIdx.x == 0 && threadIdx.x < (int)(npx - nvec * 4)) {
        const size_t t = nvec * 4 + threadIdx.x;
        visit(P0[t], MODE == 2 ? M5[t] : 0.0f);
    }
    if (one) {                                      // take the listed pixels outside the kept interval out again
        const uint32_t no = *zno;
        for (uint32_t j = blockIdx.x * 256 + threadIdx.x; j < no; j += gridDim.x * 256) {
            const float2 e = olist[j];
            if (e.x >= lo && e.x <= hi) continue;
            const float v = e.y > 1e-4f ? e.y : 1e-4f;
            const uint32_t k = __float_as_uint(v) | 0x80000000u;
            if (!none && k - klo <= span) atomicSub(&sh[(k >> SHIFT) & MASK], 1u);   // (wraps; the global sum is exact)
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < SEL_BINS; i += 256)
        if (sh[i]) atomicAdd(&hist[i], sh[i]);
    // the CTA that flushes last picks the bucket (threadFenceReduction pattern)
    __shared__ bool s_last;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = atomicAdd(&st->ticket, 1u) == gridDim.x - 1;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    sel_pick<MODE, PASS>(st, hist, sh, last, rn2, gain_out, stats);
    if (threadIdx.x == 0) st->ticket = 0;
}

// The selections by radix passes over the planes, as ONE cooperative launch (grid barriers between the passes): the
// path of the frames the fast path of selectz.cuh does not fit -- the three clipping rounds (eighteen passes) when
// *zdone is 0, the typical signal and the gain (three passes) when *zmdone is 0.  Returns at once when that path has
// done both, which is why it is one launch and not twenty-one.
__global__ void __launch_bounds__(256)
k_sel_rounds(const float* __restrict__ R, const float* __restrict__ M5, size_t npx, SelState* st, uint32_t* hist, float rn2,
             float* gain_out, float* stats, const int* prev_count, const uint32_t* zdone, const uint32_t* zmdone,
             const uint32_t* zno, const float2* __restrict__ olist) {
    if (prev_count && *prev_count == 0) {          // fixed point (R17): same image, same estimate
        if (blockIdx.x == 0 && threadIdx.x == 0) *gain_out = gain_out[-1];
        return;
    }
    const bool fast = zdone && *zdone;
    if (fast && zmdone && *zmdone) return;
    cooperative_groups::grid_group grid = cooperative_groups::this_grid();
    __shared__ uint32_t sh[SEL_BINS];
    if (!fast) {
        for (int j = 0; j < SEL_ROUNDS; ++j) {
            const int last = j == SEL_ROUNDS - 1;
            sel_hist_pass<0, 0>(R, M5, npx, st, hist, 0, rn2, gain_out, stats, false, zno, olist, sh); grid.sync();
            sel_hist_pass<0, 1>(R, M5, npx, st, hist, 0, rn2, gain_out, stats, false, zno, olist, sh); grid.sync();
            sel_hist_pass<0, 2>(R, M5, npx, st, hist, 0, rn2, gain_out, stats, false, zno, olist, sh); grid.sync();
            sel_hist_pass<1, 0>(R, M5, npx, st, hist, 0, rn2, gain_out, stats, false, zno, olist, sh); grid.sync();
            sel_hist_pass<1, 1>(R, M5, npx, st, hist, 0, rn2, gain_out, stats, false, zno, olist, sh); grid.sync();
            sel_hist_pass<1, 2>(R, M5, npx, st, hist, last, rn2, gain_out, stats, false, zno, olist, sh); grid.sync();
        }
    }
    // typical signal over the set the last round kept, then the gain (fast: over the med5 plane alone, the listed
    // pixels outside the kept interval subtracted)
    sel_hist_pass<2, 0>(R, M5, npx, st, hist, 1, rn2, gain_out, stats, fast, zno, olist, sh); grid.sync();
    sel_hist_pass<2, 1>(R, M5, npx, st, hist, 1, rn2, gain_out, stats, fast, zno, olist, sh); grid.sync();
    sel_hist_pass<2, 2>(R, M5, npx, st, hist, 1, rn2, gain_out, stats, fast, zno, olist, sh);
}

}  // namespace lac
