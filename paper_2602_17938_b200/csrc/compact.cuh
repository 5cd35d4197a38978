// Sparse result of a frame (lacosmic_run_host_sparse): the flagged pixels of the final mask as a list of flat
// indices in ascending order with their replacement values.  Three small launches: popcount per block of
// 1024 mask words, exclusive scan of the block sums (one CTA), ordered emission.
#pragma once
#include "common.cuh"

namespace lac {

constexpr int CP_WORDS_PER_THREAD = 4;
constexpr int CP_WORDS_PER_CTA = 256 * CP_WORDS_PER_THREAD;

__device__ __forceinline__ int cta_exclusive_scan_256(int v, int* s_warp, int& total) {
    const int lane = threadIdx.x & 31, wi = threadIdx.x >> 5;
    int incl = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int o = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += o;
    }
    if (lane == 31) s_warp[wi] = incl;
    __syncthreads();
    int base = 0, tot = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const int c = s_warp[k];
        if (k < wi) base += c;
        tot += c;
    }
    __syncthreads();
    total = tot;
    return base + incl - v;
}

__global__ void __launch_bounds__(256)
k_popc_blocks(const uint32_t* __restrict__ bits, int nwords, int* __restrict__ blocksum) {
    __shared__ int s_warp[8];
    const int w0 = blockIdx.x * CP_WORDS_PER_CTA + threadIdx.x * CP_WORDS_PER_THREAD;
    int n = 0;
#pragma unroll
    for (int k = 0; k < CP_WORDS_PER_THREAD; ++k)
        if (w0 + k < nwords) n += __popc(bits[w0 + k]);
    int total;
    cta_exclusive_scan_256(n, s_warp, total);
    if (threadIdx.x == 0) blocksum[blockIdx.x] = total;
}

// in place: blocksum[b] <- sum of blocksum[0..b-1]; blocksum[nblocks] <- grand total.  One CTA of 256 threads.
__global__ void __launch_bounds__(256)
k_scan_blocks(int* __restrict__ blocksum, int nblocks) {
    __shared__ int s_warp[8];
    __shared__ int s_carry;
    if (threadIdx.x == 0) s_carry = 0;
    __syncthreads();
    for (int b0 = 0; b0 < nblocks; b0 += 256) {
        const int b = b0 + threadIdx.x;
        const int v = b < nblocks ? blocksum[b] : 0;
        int total;
        const int excl = cta_exclusive_scan_256(v, s_warp, total);
        const int carry = s_carry;
        if (b < nblocks) blocksum[b] = carry + excl;
        __syncthreads();
        if (threadIdx.x == 0) s_carry = carry + total;
        __syncthreads();
    }
    if (threadIdx.x == 0) blocksum[nblocks] = s_carry;
}

__global__ void __launch_bounds__(256)
k_emit_flagged(const uint32_t* __restrict__ bits, int nwords, const int* __restrict__ blocksum,
               const float* __restrict__ clean, int32_t* __restrict__ idx, float* __restrict__ val, int cap, int w,
               int wpr) {
    __shared__ int s_warp[8];
    const int w0 = blockIdx.x * CP_WORDS_PER_CTA + threadIdx.x * CP_WORDS_PER_THREAD;
    uint32_t b[CP_WORDS_PER_THREAD];
    int n = 0;
#pragma unroll
    for (int k = 0; k < CP_WORDS_PER_THREAD; ++k) {
        b[k] = w0 + k < nwords ? bits[w0 + k] : 0u;
        n += __popc(b[k]);
    }
    int total;
    int pos = blocksum[blockIdx.x] + cta_exclusive_scan_256(n, s_warp, total);
#pragma unroll
    for (int k = 0; k < CP_WORDS_PER_THREAD; ++k) {
        uint32_t m = b[k];
        const int wi = w0 + k, y = wi / wpr, wx = wi - y * wpr;
        const int p0 = y * w + wx * 32;
        while (m) {
            const int bit = __ffs(m) - 1;
            m &= m - 1;
            if (pos < cap) {
                idx[pos] = p0 + bit;
                val[pos] = clean[p0 + bit];
            }
            ++pos;
        }
    }
}

}  // namespace lac
