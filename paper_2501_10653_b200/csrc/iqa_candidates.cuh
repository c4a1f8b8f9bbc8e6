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
//   bottom-k    radix select (8-bit digits, starting below the bits ALL keys share) finds the k-th smallest
//               key and how many of its equals belong to the answer; an ordered compaction gathers the k selected
//               (key, index) pairs in index order into shared memory; a bitonic sort orders them
// =============================================================================
#pragma once
#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "iqa_kernels.cuh"

namespace iqa {

constexpr int kCandThreads = 1024;     // at most: one CTA per matrix, as many threads as the matrix has 16-tile runs
constexpr int kCandPerThread = 16;

// Threads of the CTA for a matrix of n tiles: a power of two in [64, 1024] covering n / 16 (a small matrix must
// not pay for 32 warps walking through the whole kernel).
inline int cand_threads(int n) {
    int t = 64;
    while (t < kCandThreads && t * kCandPerThread < n) t <<= 1;
    return t;
}
constexpr int kMaxBottomK = 1024;

__device__ __forceinline__ uint32_t order_key(float v) {
    if (v != v) return 0xffffffffu;                         // NaN last
    const uint32_t u = __float_as_uint(v + 0.0f);           // -0 -> +0
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

// Exclusive scan of one int per thread over the CTA (blockDim.x threads); returns the offset of this
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
    // every warp scans the (at most 32) warp totals itself: lane l holds warp l's total
    const int nw = (int)(blockDim.x >> 5);
    const int t = lane < nw ? warp_tot[lane] : 0;
    int tinc = t;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int q = __shfl_up_sync(0xffffffffu, tinc, o);
        if (lane >= o) tinc += q;
    }
    total = __shfl_sync(0xffffffffu, tinc, 31);
    const int base = __shfl_sync(0xffffffffu, tinc - t, w);
    return base + inc - c;
}

// The kCandPerThread = 16 consecutive values [i0, i0 + 16) of a matrix of n values; positions >= n read as `fill`.
// Four 128-bit loads when the run is whole and 16-byte aligned (a warp then touches 2 KiB with 4 instructions instead of 16).
__device__ __forceinline__ void load_run16(const float* __restrict__ v, int i0, int n, float fill, float (&f)[kCandPerThread]) {
    if (i0 + kCandPerThread <= n && (((uintptr_t)(v + i0)) & 15u) == 0) {
        const float4* q = reinterpret_cast<const float4*>(v + i0);
#pragma unroll
        for (int j = 0; j < kCandPerThread / 4; ++j) {
            const float4 a = __ldg(q + j);
            f[4 * j] = a.x; f[4 * j + 1] = a.y; f[4 * j + 2] = a.z; f[4 * j + 3] = a.w;
        }
    } else {
#pragma unroll
        for (int j = 0; j < kCandPerThread; ++j) f[j] = i0 + j < n ? v[i0 + j] : fill;
    }
}

// ---- 64-bit (order key, tile index) pairs: unique, and their unsigned order is the (value, index) order -------------
__device__ __forceinline__ unsigned long long key64(uint32_t u, int idx) { return ((unsigned long long)u << 32) | (uint32_t)idx; }
__device__ __forceinline__ unsigned long long umin64(unsigned long long a, unsigned long long b) { return a < b ? a : b; }
__device__ __forceinline__ unsigned long long umax64(unsigned long long a, unsigned long long b) { return a < b ? b : a; }
// One key per lane -> ascending by lane (bitonic network over shuffles, 15 compare-exchange steps).
__device__ __forceinline__ unsigned long long warp_sort32(unsigned long long x, int lane) {
#pragma unroll
    for (int size = 2; size <= 32; size <<= 1)
#pragma unroll
        for (int stride = size >> 1; stride > 0; stride >>= 1) {
            const unsigned long long y = __shfl_xor_sync(0xffffffffu, x, stride);
            const bool keep_min = ((lane & stride) == 0) == ((lane & size) == 0);
            x = keep_min ? umin64(x, y) : umax64(x, y);
        }
    return x;
}
// x: this warp's ascending list (one key per lane); other_rev: lane i holds element 31 - i of another ascending list.
// Returns the 32 smallest of the 64 keys, ascending by lane (bitonic merge).
__device__ __forceinline__ unsigned long long warp_merge_low32(unsigned long long x, unsigned long long other_rev, int lane) {
    x = umin64(x, other_rev);
#pragma unroll
    for (int stride = 16; stride > 0; stride >>= 1) {
        const unsigned long long y = __shfl_xor_sync(0xffffffffu, x, stride);
        x = (lane & stride) == 0 ? umin64(x, y) : umax64(x, y);
    }
    return x;
}
// Ascending bitonic sort of keys[0, P) in shared memory, P a power of two: by the first warp alone when P <= 64 (no CTA
// barrier per step), by the whole CTA otherwise.  Ends with a CTA barrier.
__device__ __forceinline__ void sort_keys_shared(unsigned long long* keys, int P) {
    const int tid = threadIdx.x;
    if (P <= 64) {
        if (tid < 32) {
            for (int size = 2; size <= P; size <<= 1)
                for (int stride = size >> 1; stride > 0; stride >>= 1) {
                    for (int i = tid; i < P / 2; i += 32) {
                        const int lo = 2 * i - (i & (stride - 1));
                        const int hi = lo + stride;
                        const bool up = (lo & size) == 0;
                        const unsigned long long a = keys[lo], b = keys[hi];
                        if ((a > b) == up) { keys[lo] = b; keys[hi] = a; }
                    }
                    __syncwarp();
                }
        }
        __syncthreads();
        return;
    }
    for (int size = 2; size <= P; size <<= 1)
        for (int stride = size >> 1; stride > 0; stride >>= 1) {
            for (int i = tid; i < P / 2; i += (int)blockDim.x) {
                const int lo = 2 * i - (i & (stride - 1));  // index with the `stride` bit clear
                const int hi = lo + stride;
                const bool up = (lo & size) == 0;
                const unsigned long long a = keys[lo], b = keys[hi];
                if ((a > b) == up) { keys[lo] = b; keys[hi] = a; }
            }
            __syncthreads();
        }
}

// Work layout of both kernels: a SUPER-CHUNK is 16 blockDim.x consecutive tiles (16384 for 1024 threads); thread t
// owns the kCandPerThread = 16 consecutive tiles [16 t, 16 t + 16) of it, so index order == (thread, j) order and one
// block scan per super-chunk orders everything.  Matrices of up to one super-chunk are read from memory once.

// values [n_maps][n]; indices [n_maps][capacity] (ascending tile index, first `capacity` only);
// counts [n_maps] = number of tiles below the threshold (may exceed capacity).
__global__ void __launch_bounds__(kCandThreads)
below_kernel(const float* __restrict__ values, int n, float threshold, int* __restrict__ indices, int capacity,
             int* __restrict__ counts) {
    __shared__ int warp_tot[kCandThreads / 32];
    pdl_prologue();
    const float* v = values + (size_t)blockIdx.x * n;
    int* out = indices + (size_t)blockIdx.x * capacity;
    const int kCandChunk = (int)blockDim.x * kCandPerThread;
    int base = 0;
    for (int c0 = 0; c0 < n; c0 += kCandChunk) {
        const int i0 = c0 + threadIdx.x * kCandPerThread;
        uint32_t flags = 0;
        float f[kCandPerThread];
        load_run16(v, i0, n, __int_as_float(0x7f800000), f);             // +Inf is never below a threshold
#pragma unroll
        for (int j = 0; j < kCandPerThread; ++j)
            if (f[j] < threshold) flags |= 1u << j;
        int total;
        int pos = base + block_exclusive_scan(__popc(flags), warp_tot, total);
        for (uint32_t f = flags; f; f &= f - 1) {
            if (pos < capacity) out[pos] = i0 + (__ffs(f) - 1);
            ++pos;
        }
        base += total;
    }
    if (threadIdx.x == 0) counts[blockIdx.x] = base;
}

// values [n_maps][n]; indices [n_maps][k], vals [n_maps][k] (nullable).  Entries beyond
// min(k, n) are filled with index -1 and value +Inf.  k <= kMaxBottomK.
__global__ void __launch_bounds__(kCandThreads)
bottom_k_kernel(const float* __restrict__ values, int n, int k, int* __restrict__ indices, float* __restrict__ vals,
                float threshold, int* __restrict__ below_idx, int capacity, int* __restrict__ below_counts) {
    __shared__ int hist[256];
    __shared__ int warp_tot[kCandThreads / 32];
    __shared__ uint32_t s_prefix, s_and[kCandThreads / 32], s_or[kCandThreads / 32];
    __shared__ int s_rank;
    __shared__ unsigned long long s_tau;
    __shared__ unsigned long long keys[kMaxBottomK];
    pdl_prologue();
    const float* v = values + (size_t)blockIdx.x * n;
    const int kk = k < n ? k : n;                           // entries that exist
    const int tid = threadIdx.x;
    const int kCandChunk = (int)blockDim.x * kCandPerThread;
    const bool resident = n <= kCandChunk;                  // the whole matrix sits in registers: read once
    uint32_t u[kCandPerThread];                             // order keys of this thread's tiles of a super-chunk
    uint32_t below_flags = 0;                               // resident matrices with below_counts: tiles < threshold
    auto load_keys = [&](int c0) {
        const int i0 = c0 + tid * kCandPerThread;
        float f[kCandPerThread];
        load_run16(v, i0, n, __int_as_float(0x7fc00000), f);             // NaN: order key 0xffffffff, never below
#pragma unroll
        for (int j = 0; j < kCandPerThread; ++j) {
            u[j] = order_key(f[j]);
            if (below_counts && f[j] < threshold) below_flags |= 1u << j;
        }
    };
    if (resident) load_keys(0);

    // ---- the threshold list of the same matrix (iqa_series_find: one launch, one read of the matrix), as below_kernel ----
    if (below_counts && resident) {
        int total;
        int pos = block_exclusive_scan(__popc(below_flags), warp_tot, total);
        int* out = below_idx + (size_t)blockIdx.x * capacity;
        for (uint32_t fl = below_flags; fl; fl &= fl - 1) {
            if (pos < capacity) out[pos] = tid * kCandPerThread + (__ffs(fl) - 1);
            ++pos;
        }
        if (tid == 0) below_counts[blockIdx.x] = total;
    }

    // ---- small k (<= 32) of a resident matrix: no radix passes.  A threshold tau with at least kk tiles <= tau is the
    //      kk-th smallest of >= kk GROUP minima: the minima of the warps' 512-tile runs when at least kk warps hold
    //      tiles (one shuffle reduction per warp, one rank count in warp 0), else the minima of the threads' 16-tile
    //      runs (every warp sorts its 32 thread minima, a tree of bitonic merges keeps the 32 smallest of the CTA:
    //      exact, and then all tiles <= tau belong to kk threads: at most 16 kk <= 512 of them).  The tiles <= tau are
    //      gathered (any order: the (key, index) pairs are unique) and sorted.  Warp minima bound nothing from above:
    //      should more than kMaxBottomK tiles pass (spatially sorted matrices), the radix select below takes over. ----
    if (resident && kk <= 32) {
        const int lane = tid & 31, w = tid >> 5, nw = (int)(blockDim.x >> 5);
        const int i0 = tid * kCandPerThread;
        unsigned long long m = ~0ull;                       // threads past the matrix hold no tile
        {
            uint32_t best = 0xffffffffu; int bj = -1;       // first minimum of the run: lowest index among equals
#pragma unroll
            for (int j = 0; j < kCandPerThread; ++j)
                if (i0 + j < n && (bj < 0 || u[j] < best)) { best = u[j]; bj = j; }
            if (bj >= 0) m = key64(best, i0 + bj);
        }
        const int data_warps = (n + 32 * kCandPerThread - 1) / (32 * kCandPerThread);
        if (tid == 0) { s_rank = 0; s_tau = ~0ull; }
        if (data_warps >= kk) {
            unsigned long long x = m;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) x = umin64(x, __shfl_xor_sync(0xffffffffu, x, o));
            if (lane == 0) keys[w] = x;
            __syncthreads();
            if (w == 0) {
                x = lane < nw ? keys[lane] : ~0ull;
                int r = 0;                                  // keys smaller than this lane's (real keys are unique)
#pragma unroll
                for (int l = 0; l < 32; ++l) r += __shfl_sync(0xffffffffu, x, l) < x ? 1 : 0;
                if (r == kk - 1 && x != ~0ull) s_tau = x;
            }
        } else {
            unsigned long long x = warp_sort32(m, lane);
            for (int r = 1; r < nw; r <<= 1) {              // nw is a power of two
                if ((w & (2 * r - 1)) == r) keys[w * 32 + lane] = x;
                __syncthreads();
                if ((w & (2 * r - 1)) == 0) x = warp_merge_low32(x, keys[(w + r) * 32 + 31 - lane], lane);
            }
            if (w == 0) {
                const unsigned long long t = __shfl_sync(0xffffffffu, x, kk - 1);
                if (lane == 0) s_tau = t;                   // ~0ull when fewer than kk threads hold tiles: every tile passes
            }
        }
        __syncthreads();                                    // s_tau is set; the lists in keys[] have been read
        const unsigned long long tau = s_tau;
        const uint32_t tau_hi = (uint32_t)(tau >> 32), tau_lo = (uint32_t)tau;
        uint32_t sel = 0;
#pragma unroll
        for (int j = 0; j < kCandPerThread; ++j)
            if (i0 + j < n && (u[j] < tau_hi || (u[j] == tau_hi && (uint32_t)(i0 + j) <= tau_lo))) sel |= 1u << j;
        if (sel) {
            int pos = atomicAdd(&s_rank, __popc(sel));
#pragma unroll
            for (int j = 0; j < kCandPerThread; ++j)
                if (sel & (1u << j)) {
                    if (pos < kMaxBottomK) keys[pos] = key64(u[j], i0 + j);
                    ++pos;
                }
        }
        __syncthreads();
        const int total = s_rank;                           // >= kk
        if (total <= kMaxBottomK) {
            int* out_i = indices + (size_t)blockIdx.x * k;
            float* out_v = vals ? vals + (size_t)blockIdx.x * k : nullptr;
            for (int i = kk + tid; i < k; i += (int)blockDim.x) {
                out_i[i] = -1;
                if (out_v) out_v[i] = __int_as_float(0x7f800000);
            }
            if (total <= 32) {                              // one key per lane of warp 0: its rank is its place
                if (w == 0) {
                    const unsigned long long x = lane < total ? keys[lane] : ~0ull;
                    int r = 0;
#pragma unroll
                    for (int l = 0; l < 32; ++l) r += __shfl_sync(0xffffffffu, x, l) < x ? 1 : 0;
                    if (lane < total && r < kk) {
                        const int idx = (int)(uint32_t)x;
                        out_i[r] = idx;
                        if (out_v) out_v[r] = v[idx];
                    }
                }
                return;
            }
            int P = 64;
            while (P < total) P <<= 1;
            for (int i = total + tid; i < P; i += (int)blockDim.x) keys[i] = ~0ull;
            __syncthreads();
            sort_keys_shared(keys, P);
            for (int i = tid; i < kk; i += (int)blockDim.x) {
                const int idx = (int)(uint32_t)keys[i];
                out_i[i] = idx;
                if (out_v) out_v[i] = v[idx];
            }
            return;
        }
        __syncthreads();                                    // (uniform) too many tiles passed: radix select
    }

    // ---- the bits all keys share: similarity values cluster (augLISI ~ 0.99x), so their leading bits are equal;
    //      a digit on which every key agrees would send all the atomics of a pass to ONE histogram bucket ----
    uint32_t k_and = 0xffffffffu, k_or = 0u;
    for (int c0 = 0; c0 < n; c0 += kCandChunk) {
        if (!resident) load_keys(c0);
        const int i0 = c0 + tid * kCandPerThread;
#pragma unroll
        for (int j = 0; j < kCandPerThread; ++j)
            if (i0 + j < n) { k_and &= u[j]; k_or |= u[j]; }
    }
    k_and = __reduce_and_sync(0xffffffffu, k_and);
    k_or = __reduce_or_sync(0xffffffffu, k_or);
    if ((tid & 31) == 0) { s_and[tid >> 5] = k_and; s_or[tid >> 5] = k_or; }
    __syncthreads();
    for (int i = 0; i < (int)(blockDim.x >> 5); ++i) { k_and &= s_and[i]; k_or |= s_or[i]; }
    const uint32_t diff = k_and ^ k_or;                     // bits on which the keys differ
    const int hi = 31 - __clz(diff | 1u);                   // highest such bit (0 when all keys are equal)

    // ---- radix select below the common prefix: the kk-th smallest order key (rank counts from 1) ----
    uint32_t mask = hi >= 31 ? 0u : ~((2u << hi) - 1u);     // bits above `hi` are settled
    uint32_t prefix = k_and & mask;
    int rank = kk;
    for (int shift = hi > 7 ? hi - 7 : 0; kk > 0; shift = shift > 8 ? shift - 8 : 0) {
        for (int i = tid; i < 256; i += (int)blockDim.x) hist[i] = 0;
        __syncthreads();
        for (int c0 = 0; c0 < n; c0 += kCandChunk) {
            if (!resident) load_keys(c0);
            const int i0 = c0 + tid * kCandPerThread;
#pragma unroll
            for (int j = 0; j < kCandPerThread; ++j)
                if (i0 + j < n && (u[j] & mask) == prefix) atomicAdd(&hist[(u[j] >> shift) & 255u], 1);
        }
        __syncthreads();
        if (tid < 32) {                                     // warp 0 finds the bucket that holds the rank-th key
            int c[8], sum = 0;
#pragma unroll
            for (int j = 0; j < 8; ++j) { c[j] = hist[tid * 8 + j]; sum += c[j]; }
            int inc = sum;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, inc, o);
                if (tid >= o) inc += t;
            }
            int cum = inc - sum;                            // keys in the buckets before this lane's eight
            if (cum < rank && rank <= inc) {                // exactly one lane (the histogram holds >= rank keys)
                int b = 0;
                for (; b < 7; ++b) {
                    if (cum + c[b] >= rank) break;
                    cum += c[b];
                }
                s_prefix = prefix | ((uint32_t)(tid * 8 + b) << shift);   // digits may overlap settled bits: same bits
                s_rank = rank - cum;
            }
        }
        __syncthreads();
        prefix = s_prefix;
        rank = s_rank;
        mask |= 255u << shift;
        if (shift == 0) break;
    }
    const uint32_t pivot = prefix;                          // key of the kk-th smallest value
    const int take_eq = rank;                               // how many tiles equal to it belong to the answer

    // ---- ordered compaction of the selected (key, index) pairs into shared memory ----
    int base = 0, eq_seen = 0;
    for (int c0 = 0; c0 < n && kk > 0; c0 += kCandChunk) {
        if (!resident) load_keys(c0);
        const int i0 = c0 + tid * kCandPerThread;
        uint32_t eq = 0, less = 0;
#pragma unroll
        for (int j = 0; j < kCandPerThread; ++j)
            if (i0 + j < n) {
                if (u[j] == pivot) eq |= 1u << j;
                if (u[j] < pivot) less |= 1u << j;
            }
        int tot_e;
        int erank = eq_seen + block_exclusive_scan(__popc(eq), warp_tot, tot_e);
        uint32_t sel = less;                                // plus the first take_eq equals, in index order
        for (uint32_t f = eq; f && erank < take_eq; f &= f - 1, ++erank) sel |= f & (0u - f);
        int tot_s;
        int pos = base + block_exclusive_scan(__popc(sel), warp_tot, tot_s);
#pragma unroll
        for (int j = 0; j < kCandPerThread; ++j)
            if (sel & (1u << j)) keys[pos++] = ((unsigned long long)u[j] << 32) | (uint32_t)(i0 + j);
        base += tot_s;
        eq_seen += tot_e;
    }
    // base == kk here.  Pad to a power of two and sort ascending by (key, index).
    int P = 1;
    while (P < kk) P <<= 1;
    for (int i = kk + tid; i < P; i += (int)blockDim.x) keys[i] = ~0ull;
    __syncthreads();
    for (int size = 2; size <= P; size <<= 1)
        for (int stride = size >> 1; stride > 0; stride >>= 1) {
            for (int i = tid; i < P / 2; i += (int)blockDim.x) {
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
    for (int i = tid; i < k; i += (int)blockDim.x) {
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

// -----------------------------------------------------------------------------
// bottom-k of a LARGE matrix (16384 < n <= 8 x 16384 tiles: N = 16384 at N_T = 64, N = 2048 at N_T = 8): one
// thread-block CLUSTER of C = ceil(n / 16384) CTAs per matrix instead of one CTA looping over super-chunks and
// re-reading them in every radix pass.  CTA r keeps tiles [16384 r, 16384 (r+1)) in registers; the per-CTA
// AND / OR words, histograms and selection counts are read across the cluster through distributed shared memory
// (every CTA sums the C histograms itself and reaches the same bucket, so nothing is broadcast); the selected
// (key, index) pairs are written straight into CTA 0's shared memory at their global position, and CTA 0 sorts
// and stores them.  Same selection, same order, same output as bottom_k_kernel.
// -----------------------------------------------------------------------------
constexpr int kCandMaxCluster = 8;

inline int cand_cluster_size(int n) {                       // 0: use the single-CTA kernel
    const int chunk = kCandThreads * kCandPerThread;
    if (n <= chunk || n > kCandMaxCluster * chunk) return 0;
    return (n + chunk - 1) / chunk;
}

__global__ void __launch_bounds__(kCandThreads)
bottom_k_cluster_kernel(const float* __restrict__ values, int n, int k, int* __restrict__ indices,
                        float* __restrict__ vals) {
    namespace cg = cooperative_groups;
    __shared__ int hist[256];
    __shared__ int warp_tot[kCandThreads / 32];
    __shared__ uint32_t s_prefix, s_and[kCandThreads / 32], s_or[kCandThreads / 32];
    __shared__ int s_rank;
    __shared__ uint32_t cta_and, cta_or;                    // this CTA's words, read by the others
    __shared__ int cta_tot_e, cta_tot_s;
    __shared__ unsigned long long keys[kMaxBottomK];        // used in CTA 0 only
    cg::cluster_group cluster = cg::this_cluster();
    pdl_prologue();
    const int C = (int)cluster.num_blocks(), r = (int)cluster.block_rank();
    const size_t map = blockIdx.x / C;
    const float* v = values + map * (size_t)n;
    const int kk = k < n ? k : n;
    const int tid = threadIdx.x;
    const int i0 = (r * kCandThreads + tid) * kCandPerThread;               // first tile of this thread
    uint32_t u[kCandPerThread];
    {
        float f[kCandPerThread];
        load_run16(v, i0, n, __int_as_float(0x7fc00000), f);
#pragma unroll
        for (int j = 0; j < kCandPerThread; ++j) u[j] = order_key(f[j]);
    }

    // ---- bits all keys of the matrix share ----
    uint32_t k_and = 0xffffffffu, k_or = 0u;
#pragma unroll
    for (int j = 0; j < kCandPerThread; ++j)
        if (i0 + j < n) { k_and &= u[j]; k_or |= u[j]; }
    k_and = __reduce_and_sync(0xffffffffu, k_and);
    k_or = __reduce_or_sync(0xffffffffu, k_or);
    if ((tid & 31) == 0) { s_and[tid >> 5] = k_and; s_or[tid >> 5] = k_or; }
    __syncthreads();
    if (tid == 0) {
        uint32_t a = 0xffffffffu, o = 0u;
        for (int i = 0; i < kCandThreads / 32; ++i) { a &= s_and[i]; o |= s_or[i]; }
        cta_and = a; cta_or = o;
    }
    cluster.sync();
    k_and = 0xffffffffu; k_or = 0u;
    for (int q = 0; q < C; ++q) { k_and &= *cluster.map_shared_rank(&cta_and, q); k_or |= *cluster.map_shared_rank(&cta_or, q); }
    const uint32_t diff = k_and ^ k_or;
    const int hi = 31 - __clz(diff | 1u);

    // ---- radix select below the common prefix; every CTA sums the C histograms and finds the same bucket ----
    uint32_t mask = hi >= 31 ? 0u : ~((2u << hi) - 1u);
    uint32_t prefix = k_and & mask;
    int rank = kk;
    for (int shift = hi > 7 ? hi - 7 : 0; kk > 0; shift = shift > 8 ? shift - 8 : 0) {
        if (tid < 256) hist[tid] = 0;
        __syncthreads();
#pragma unroll
        for (int j = 0; j < kCandPerThread; ++j)
            if (i0 + j < n && (u[j] & mask) == prefix) atomicAdd(&hist[(u[j] >> shift) & 255u], 1);
        cluster.sync();                                     // every CTA's histogram is complete
        if (tid < 32) {
            int c[8], sum = 0;
#pragma unroll
            for (int j = 0; j < 8; ++j) c[j] = 0;
            for (int q = 0; q < C; ++q) {
                const int* h = cluster.map_shared_rank(hist, q);
#pragma unroll
                for (int j = 0; j < 8; ++j) c[j] += h[tid * 8 + j];
            }
#pragma unroll
            for (int j = 0; j < 8; ++j) sum += c[j];
            int inc = sum;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, inc, o);
                if (tid >= o) inc += t;
            }
            int cum = inc - sum;
            if (cum < rank && rank <= inc) {
                int b = 0;
                for (; b < 7; ++b) {
                    if (cum + c[b] >= rank) break;
                    cum += c[b];
                }
                s_prefix = prefix | ((uint32_t)(tid * 8 + b) << shift);
                s_rank = rank - cum;
            }
        }
        cluster.sync();                                     // all histograms have been read: they may be cleared
        prefix = s_prefix;
        rank = s_rank;
        mask |= 255u << shift;
        if (shift == 0) break;
    }
    const uint32_t pivot = prefix;
    const int take_eq = rank;

    // ---- ordered compaction across the cluster into CTA 0's shared memory ----
    uint32_t eq = 0, less = 0;
#pragma unroll
    for (int j = 0; j < kCandPerThread; ++j)
        if (i0 + j < n) {
            if (u[j] == pivot) eq |= 1u << j;
            if (u[j] < pivot) less |= 1u << j;
        }
    int tot_e;
    int erank = block_exclusive_scan(__popc(eq), warp_tot, tot_e);
    if (tid == 0) cta_tot_e = tot_e;
    cluster.sync();
    for (int q = 0; q < r; ++q) erank += *cluster.map_shared_rank(&cta_tot_e, q);       // equals in the CTAs before this one
    uint32_t sel = less;
    for (uint32_t f = eq; f && erank < take_eq; f &= f - 1, ++erank) sel |= f & (0u - f);
    int tot_s;
    int pos = block_exclusive_scan(__popc(sel), warp_tot, tot_s);
    if (tid == 0) cta_tot_s = tot_s;
    cluster.sync();
    for (int q = 0; q < r; ++q) pos += *cluster.map_shared_rank(&cta_tot_s, q);
    unsigned long long* keys0 = cluster.map_shared_rank(keys, 0);
#pragma unroll
    for (int j = 0; j < kCandPerThread; ++j)
        if (kk > 0 && (sel & (1u << j))) keys0[pos++] = ((unsigned long long)u[j] << 32) | (uint32_t)(i0 + j);
    cluster.sync();                                         // CTA 0 holds all kk pairs; the other CTAs are done
    if (r != 0) return;

    int P = 1;
    while (P < kk) P <<= 1;
    for (int i = kk + tid; i < P; i += kCandThreads) keys[i] = ~0ull;
    __syncthreads();
    for (int size = 2; size <= P; size <<= 1)
        for (int stride = size >> 1; stride > 0; stride >>= 1) {
            for (int i = tid; i < P / 2; i += kCandThreads) {
                const int lo = 2 * i - (i & (stride - 1));
                const int hi2 = lo + stride;
                const bool up = (lo & size) == 0;
                const unsigned long long a = keys[lo], b = keys[hi2];
                if ((a > b) == up) { keys[lo] = b; keys[hi2] = a; }
            }
            __syncthreads();
        }
    int* out_i = indices + map * (size_t)k;
    float* out_v = vals ? vals + map * (size_t)k : nullptr;
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

// Threshold list of a large matrix with the same cluster layout: CTA r flags its 16384 tiles, the counts of the
// CTAs before it (distributed shared memory) give its offset in the ascending list.
__global__ void __launch_bounds__(kCandThreads)
below_cluster_kernel(const float* __restrict__ values, int n, float threshold, int* __restrict__ indices, int capacity,
                     int* __restrict__ counts) {
    namespace cg = cooperative_groups;
    __shared__ int warp_tot[kCandThreads / 32];
    __shared__ int cta_total;
    cg::cluster_group cluster = cg::this_cluster();
    pdl_prologue();
    const int C = (int)cluster.num_blocks(), r = (int)cluster.block_rank();
    const size_t map = blockIdx.x / C;
    const float* v = values + map * (size_t)n;
    int* out = indices + map * (size_t)capacity;
    const int i0 = (r * kCandThreads + (int)threadIdx.x) * kCandPerThread;
    uint32_t flags = 0;
    float f[kCandPerThread];
    load_run16(v, i0, n, __int_as_float(0x7f800000), f);
#pragma unroll
    for (int j = 0; j < kCandPerThread; ++j)
        if (f[j] < threshold) flags |= 1u << j;
    int total;
    int pos = block_exclusive_scan(__popc(flags), warp_tot, total);
    if (threadIdx.x == 0) cta_total = total;
    cluster.sync();
    int before = 0, all = 0;
    for (int q = 0; q < C; ++q) {
        const int t = *cluster.map_shared_rank(&cta_total, q);
        if (q < r) before += t;
        all += t;
    }
    pos += before;
    for (uint32_t f = flags; f; f &= f - 1) {
        if (pos < capacity) out[pos] = i0 + (__ffs(f) - 1);
        ++pos;
    }
    if (r == 0 && threadIdx.x == 0) counts[map] = all;
    cluster.sync();                                         // nobody exits while its total may still be read
}

}  // namespace iqa
