// =============================================================================
// iqa_aggregate.cuh -- S5: tile -> whole-image aggregation, Eqs. 3-4, and the
// g x g tile merge the paper mentions at PAPER.md:66.  Inputs are the four per-tile fp32
// arrays (<= a few MiB); all sums are taken in double, in a fixed order.
//
//   Eq. 3  LISI    = sum_t lisi_t * (max(X_t, Y_t) + C2) / (max(SX, SY) + C2)
//   Eq. 4  augLISI = (sum_t auglisi_t * (X_t + Y_t + C) - (n - 1) C) / (SX + SY + C)
//   with SX = sum_t X_t, SY = sum_t Y_t and n the number of merged tiles.
// =============================================================================
#pragma once
#include <cuda_runtime.h>

#include "iqa_kernels.cuh"

namespace iqa {

constexpr int kAggThreads = 1024;

struct Agg4 { double n3, n4, sx, sy; };

__device__ __forceinline__ void agg_add(Agg4& a, float lisi, float aug, float X, float Y,
                                        double C2, double C) {
    const double xd = (double)X, yd = (double)Y;
    a.n3 += (double)lisi * (fmax(xd, yd) + C2);     // Eq. 3 numerator term
    a.n4 += (double)aug * (xd + yd + C);            // Eq. 4 numerator term
    a.sx += xd;
    a.sy += yd;
}

__device__ __forceinline__ Agg4 agg_warp_sum(Agg4 a) {
    for (int o = 16; o > 0; o >>= 1) {
        a.n3 += __shfl_xor_sync(0xffffffffu, a.n3, o);
        a.n4 += __shfl_xor_sync(0xffffffffu, a.n4, o);
        a.sx += __shfl_xor_sync(0xffffffffu, a.sx, o);
        a.sy += __shfl_xor_sync(0xffffffffu, a.sy, o);
    }
    return a;
}

__device__ __forceinline__ void agg_finish(const Agg4& a, double n, double C2, double C,
                                           float* lisi_out, float* aug_out) {
    *lisi_out = (float)(a.n3 / (fmax(a.sx, a.sy) + C2));                 // Eq. 3
    *aug_out = (float)((a.n4 - (n - 1.0) * C) / (a.sx + a.sy + C));      // Eq. 4
}

// One CTA of 1024 threads per image pair (blockIdx.x = pair of the batch; arrays are
// [n_pairs][n]): thread-strided partial sums, warp butterfly, then warp order.
__global__ void __launch_bounds__(kAggThreads)
aggregate_kernel(const float* __restrict__ lisi, const float* __restrict__ aug,
                 const float* __restrict__ X, const float* __restrict__ Y, int n,
                 float C2f, float Cf, float* __restrict__ out2) {
    __shared__ Agg4 part[kAggThreads / 32];
    pdl_prologue();
    const size_t base = (size_t)blockIdx.x * (size_t)n;
    lisi += base; aug += base; X += base; Y += base; out2 += 2 * (size_t)blockIdx.x;
    const double C2 = (double)C2f, C = (double)Cf;
    Agg4 a = {0.0, 0.0, 0.0, 0.0};
    for (int t = threadIdx.x; t < n; t += kAggThreads)
        agg_add(a, lisi[t], aug[t], X[t], Y[t], C2, C);
    a = agg_warp_sum(a);
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = a;
    __syncthreads();
    if (threadIdx.x < 32) {
        Agg4 b = part[threadIdx.x];          // kAggThreads / 32 == 32 entries
        b = agg_warp_sum(b);
        if (threadIdx.x == 0) agg_finish(b, (double)n, C2, C, out2, out2 + 1);
    }
}

// P:66 merge: one warp per output tile; lanes stride over the g*g input tiles (row-major
// inside the block), then a warp butterfly.  Output tile (oy, ox) merges input tiles
// (oy*g .. oy*g+g-1, ox*g .. ox*g+g-1) of the nt x nt matrix.
__global__ void __launch_bounds__(256)
merge_kernel(const float* __restrict__ lisi, const float* __restrict__ aug,
             const float* __restrict__ X, const float* __restrict__ Y, int nt, int g,
             float C2f, float Cf,
             float* __restrict__ lisi_o, float* __restrict__ aug_o,
             float* __restrict__ X_o, float* __restrict__ Y_o) {
    pdl_prologue();
    const int nto = nt / g;
    const long long o = (long long)blockIdx.x * 8 + (threadIdx.x >> 5);
    if (o >= (long long)nto * nto) return;
    const int lane = threadIdx.x & 31;
    const int oy = (int)(o / nto), ox = (int)(o % nto);
    const double C2 = (double)C2f, C = (double)Cf;
    Agg4 a = {0.0, 0.0, 0.0, 0.0};
    const int gg = g * g;
    for (int k = lane; k < gg; k += 32) {
        const size_t t = (size_t)(oy * g + k / g) * nt + (size_t)(ox * g + k % g);
        agg_add(a, lisi[t], aug[t], X[t], Y[t], C2, C);
    }
    a = agg_warp_sum(a);
    if (lane == 0) {
        agg_finish(a, (double)gg, C2, C, lisi_o + o, aug_o + o);
        X_o[o] = (float)a.sx;
        Y_o[o] = (float)a.sy;
    }
}

}  // namespace iqa
