// =============================================================================
// iqa_candidates.cuh -- candidate extraction over the IQA matrices: the
// "finder" output.  The paper gives no decision rule (it shows the matrices and says the finders
// localise "transients to tiles"), so the rule is the plainest one (R17):
//   below_kernel     tiles whose value is < a threshold, listed in ascending tile index
//   bottom_k_kernel  the k tiles of lowest value, ascending by (value, tile index)
// One CTA per matrix (a batch of pairs / the comparisons of a series gives several matrices).
// Everything is integer / comparison work on the fp32 values as they are: results are exact and
// deterministic (the only atomics are integer histogram counts, which commute).
//   order key   u = bits(v + 0.0f) (so -0 == +0), flipped so that unsigned order == float order;
//               NaN (never produced: C2, C > 0) sorts last
//   bottom-k    radix select (4 passes of 8 bits) finds the k-th smallest key and how many of its
//               equals belong to the answer; an ordered compaction gathers the k selected
//               (key, index) pairs in index order into shared memory; a bitonic sort orders them
// =============================================================================
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "iqa_kernels.cuh"

namespace iqa {

constexpr int kCandThreads = 256;
constexpr int kCandPerThread = 4;
constexpr int kCandChunk = kCandThreads * kCandPerThread;
constexpr int kMaxBottomK = 1024;

__device__ __forceinline__ uint32_t order_key(float v) {
    if (v != v) return 0xffffffffu;                         // NaN last
    const uint32_t u = __float_as_uint(v + 0.0f);           // -0 -> +0
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

// Exclusive scan of one int per thread over the CTA (256 threads); returns the offset of this
// thread and the CTA total.  `warp_tot` is shared scratch of kCandThreads / 32 ints.
__device__ __forceinline__ int block_exclusive_scan(int c, int* warp_tot, int& total) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int inc = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    __syncthreads();                                        // previous use of warp_tot is over
    if (lane == 31) warp_tot[w] = inc;
    __syncthreads();
    int base = 0, tot = 0;
#pragma unroll
    for (int i = 0; i < kCandThreads / 32; ++i) {
        const int t = warp_tot[i];
        if (i < w) base += t;
        tot += t;
    }
    total = tot;
    return base + inc - c;
}

// values [n_maps][n]; indices [n_maps][capacity] (ascending tile index, first `capacity` only);
// counts [n_maps] = number of tiles below the threshold (may exceed capacity).
__global__ void __launch_bounds__(kCandThreads)
below_kernel(const float* __restrict__ values, int n, float threshold, int* __restrict__ indices, int capacity,
             int* __restrict__ counts) {
    __shared__ int warp_tot[kCandThreads / 32];
    pdl_prologue();
    const float* v = values + (size_t)blockIdx.x * n;
    int* out = indices + (size_t)blockIdx.x * capacity;
    int base = 0;
    for (int c0 = 0; c0 < n; c0 += kCandChunk) {
        const int i0 = c0 + threadIdx.x * kCandPerThread;
        bool f[kCandPerThread];
        int c = 0;
#pragma unroll
        for (int j = 0; j < kCandPerThread; ++j) {
            f[j] = (i0 + j < n) && (v[i0 + j] < threshold);
            c += f[j];
        }
        int total;
        int pos = base + block_exclusive_scan(c, warp_tot, total);
#pragma unroll
        for (int j = 0; j < kCandPerThread; ++j)
            if (f[j]) {
                if (pos < capacity) out[pos] = i0 + j;
                ++pos;
            }
        base += total;
    }
    if (threadIdx.x == 0) counts[blockIdx.x] = base;
}

// values [n_maps][n]; indices [n_maps][k], vals [n_maps][k] (nullable).  Entries beyond
// min(k, n) are filled with index -1 and value +Inf.  k <= kMaxBottomK.
__global__ void __launch_bounds__(kCandThreads)
bottom_k_kernel(const float* __restrict__ values, int n, int k, int* __restrict__ indices, float* __restrict__ vals) {
    __shared__ int hist[256];
    __shared__ int warp_tot[kCandThreads / 32];
    __shared__ uint32_t s_prefix;
    __shared__ int s_rank;
    __shared__ unsigned long long keys[kMaxBottomK];
    pdl_prologue();
    const float* v = values + (size_t)blockIdx.x * n;
    const int kk = k < n ? k : n;                           // entries that exist
    const int tid = threadIdx.x;

    // ---- radix select: the kk-th smallest order key (rank counts from 1) ----
    uint32_t prefix = 0, mask = 0;
    int rank = kk;
    for (int shift = 24; shift >= 0 && kk > 0; shift -= 8) {
        hist[tid] = 0;
        __syncthreads();
        for (int i = tid; i < n; i += kCandThreads) {
            const uint32_t u = order_key(v[i]);
            if ((u & mask) == prefix) atomicAdd(&hist[(u >> shift) & 255u], 1);
        }
        __syncthreads();
        if (tid == 0) {
            int cum = 0, b = 0;
            for (; b < 255; ++b) {
                if (cum + hist[b] >= rank) break;
                cum += hist[b];
            }
            s_prefix = prefix | ((uint32_t)b << shift);
            s_rank = rank - cum;
        }
        __syncthreads();
        prefix = s_prefix;
        rank = s_rank;
        mask |= 255u << shift;
        __syncthreads();
    }
    const uint32_t pivot = prefix;                          // key of the kk-th smallest value
    const int take_eq = rank;                               // how many tiles equal to it belong to the answer

    // ---- ordered compaction of the selected (key, index) pairs into shared memory ----
    int base = 0, eq_seen = 0;
    for (int c0 = 0; c0 < n && kk > 0; c0 += kCandChunk) {
        const int i0 = c0 + tid * kCandPerThread;
        uint32_t u[kCandPerThread];
        bool eq[kCandPerThread];
        int ce = 0;
#pragma unroll
        for (int j = 0; j < kCandPerThread; ++j) {
            u[j] = i0 + j < n ? order_key(v[i0 + j]) : 0xffffffffu;
            eq[j] = (i0 + j < n) && u[j] == pivot;
            ce += eq[j];
        }
        int tot_e;
        int erank = eq_seen + block_exclusive_scan(ce, warp_tot, tot_e);
        bool sel[kCandPerThread];
        int cs = 0;
#pragma unroll
        for (int j = 0; j < kCandPerThread; ++j) {
            sel[j] = (i0 + j < n) && (u[j] < pivot || (eq[j] && erank < take_eq));
            erank += eq[j];
            cs += sel[j];
        }
        int tot_s;
        int pos = base + block_exclusive_scan(cs, warp_tot, tot_s);
#pragma unroll
        for (int j = 0; j < kCandPerThread; ++j)
            if (sel[j]) keys[pos++] = ((unsigned long long)u[j] << 32) | (uint32_t)(i0 + j);
        base += tot_s;
        eq_seen += tot_e;
    }
    // base == kk here.  Pad to a power of two and sort ascending by (key, index).
    int P = 1;
    while (P < kk) P <<= 1;
    for (int i = kk + tid; i < P; i += kCandThreads) keys[i] = ~0ull;
    __syncthreads();
    for (int size = 2; size <= P; size <<= 1)
        for (int stride = size >> 1; stride > 0; stride >>= 1) {
            for (int i = tid; i < P / 2; i += kCandThreads) {
                const int lo = 2 * i - (i & (stride - 1));  // index with the `stride` bit clear
                const int hi = lo + stride;
                const bool up = (lo & size) == 0;
                const unsigned long long a = keys[lo], b = keys[hi];
                if ((a > b) == up) { keys[lo] = b; keys[hi] = a; }
            }
            __syncthreads();
        }
    int* out_i = indices + (size_t)blockIdx.x * k;
    float* out_v = vals ? vals + (size_t)blockIdx.x * k : nullptr;
    for (int i = tid; i < k; i += kCandThreads) {
        if (i < kk) {
            const int idx = (int)(uint32_t)keys[i];
            out_i[i] = idx;
            if (out_v) out_v[i] = v[idx];
        } else {
            out_i[i] = -1;
            if (out_v) out_v[i] = __int_as_float(0x7f800000);
        }
    }
}

}  // namespace iqa
