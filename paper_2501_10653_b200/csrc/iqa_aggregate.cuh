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
#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "iqa_kernels.cuh"

namespace iqa {

constexpr int kAggThreads = 256;
constexpr int kAggCluster = 8;      // CTAs per image pair for large tile counts (portable cluster size)
constexpr int kAggClusterMinTiles = 8192;   // below this one CTA is faster (measured: the cluster barriers cost ~0.5 us)

// Cluster size used for n tiles: a function of n only, so the order of additions stays fixed.
inline int agg_cluster_size(long long n) { return n >= kAggClusterMinTiles ? kAggCluster : 1; }

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

// One thread-block CLUSTER of agg_cluster_size(n) CTAs per image pair (arrays are [n_pairs][n]; cluster
// c = pair c).  A pair's arrays are at most a few MiB out of L2, so the loop is bound by load
// latency and by the fp32 -> fp64 conversions of one SM: the cluster spreads a pair over
// kAggCluster SMs, every thread takes 128-bit loads when the arrays allow it and issues
// kAggUnroll of them before the first double is added.  CTA r of the cluster owns the contiguous
// element range [r * per, (r + 1) * per); its partial (thread-strided, warp butterfly, warp
// order) goes to its own shared memory, and after a cluster barrier CTA 0 adds the kAggCluster
// partials in rank order through distributed shared memory and applies Eqs. 3-4.  The order
// of every addition is fixed by (n, thread, rank): results are bit-reproducible.
constexpr int kAggUnroll = 4;

__global__ void __launch_bounds__(kAggThreads)
aggregate_kernel(const float* __restrict__ lisi, const float* __restrict__ aug,
                 const float* __restrict__ X, const float* __restrict__ Y, int n,
                 float C2f, float Cf, float* __restrict__ out2, double* __restrict__ sums4) {
    namespace cg = cooperative_groups;
    __shared__ Agg4 part[kAggThreads / 32];
    __shared__ Agg4 cta_part;
    cg::cluster_group cluster = cg::this_cluster();
    pdl_prologue();
    const int rank = (int)cluster.block_rank();
    const int csize = (int)cluster.num_blocks();              // launch attribute: agg_cluster_size(n)
    const size_t pair = blockIdx.x / csize;
    const size_t base = pair * (size_t)n;
    lisi += base; aug += base; X += base; Y += base;
    const double C2 = (double)C2f, C = (double)Cf;
    Agg4 a = {0.0, 0.0, 0.0, 0.0};
    // this CTA's element range; a multiple of 4 long so the 128-bit groups never straddle ranks
    const int per = ((n + 4 * csize - 1) / (4 * csize)) * 4;
    const int e0 = min(n, rank * per), e1 = min(n, e0 + per);
    const bool vec = ((((uintptr_t)lisi | (uintptr_t)aug | (uintptr_t)X | (uintptr_t)Y) & 15u) == 0);
    const int g0 = e0 >> 2;                                   // first float4 group of the range
    const int g1 = vec ? (e1 >> 2) : g0;                      // one past the last whole group
    const float4* l4 = reinterpret_cast<const float4*>(lisi);
    const float4* a4 = reinterpret_cast<const float4*>(aug);
    const float4* x4 = reinterpret_cast<const float4*>(X);
    const float4* y4 = reinterpret_cast<const float4*>(Y);
    for (int i0 = g0 + threadIdx.x; i0 < g1; i0 += kAggThreads * kAggUnroll) {
        float4 vl[kAggUnroll], va[kAggUnroll], vx[kAggUnroll], vy[kAggUnroll];
#pragma unroll
        for (int u = 0; u < kAggUnroll; ++u) {
            const int i = i0 + u * kAggThreads;
            if (i < g1) { vl[u] = __ldg(l4 + i); va[u] = __ldg(a4 + i); vx[u] = __ldg(x4 + i); vy[u] = __ldg(y4 + i); }
        }
#pragma unroll
        for (int u = 0; u < kAggUnroll; ++u) {
            if (i0 + u * kAggThreads < g1) {
                agg_add(a, vl[u].x, va[u].x, vx[u].x, vy[u].x, C2, C);
                agg_add(a, vl[u].y, va[u].y, vx[u].y, vy[u].y, C2, C);
                agg_add(a, vl[u].z, va[u].z, vx[u].z, vy[u].z, C2, C);
                agg_add(a, vl[u].w, va[u].w, vx[u].w, vy[u].w, C2, C);
            }
        }
    }
    for (int t = (vec ? 4 * g1 : e0) + threadIdx.x; t < e1; t += kAggThreads)     // scalar rest of the range
        agg_add(a, lisi[t], aug[t], X[t], Y[t], C2, C);
    a = agg_warp_sum(a);
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = a;
    __syncthreads();
    if (threadIdx.x < 32) {
        Agg4 b = {0.0, 0.0, 0.0, 0.0};
        if (threadIdx.x < kAggThreads / 32) b = part[threadIdx.x];
        b = agg_warp_sum(b);
        if (threadIdx.x == 0) cta_part = b;
    }
    cluster.sync();                                           // every CTA's partial is in its shared memory
    if (rank == 0 && threadIdx.x == 0) {
        Agg4 s = cta_part;
        for (int r = 1; r < csize; ++r) {
            const Agg4* q = cluster.map_shared_rank(&cta_part, r);
            s.n3 += q->n3; s.n4 += q->n4; s.sx += q->sx; s.sy += q->sy;
        }
        if (out2) agg_finish(s, (double)n, C2, C, out2 + 2 * pair, out2 + 2 * pair + 1);
        if (sums4) {                                          // raw sums of Eqs. 3-4 (a band of a sharded image)
            double* q4 = sums4 + 4 * pair;
            q4[0] = s.n3; q4[1] = s.n4; q4[2] = s.sx; q4[3] = s.sy;
        }
    }
    cluster.sync();                                           // nobody exits while CTA 0 reads its shared memory
}

// Eqs. 3-4 from the (all-reduced) sums of all bands: sums4 = {sum lisi_t (max(X_t,Y_t)+C2),
// sum auglisi_t (X_t+Y_t+C), sum X_t, sum Y_t} over the n tiles of the whole image.
__global__ void aggregate_finish_kernel(const double* __restrict__ sums4, double n, float C2f, float Cf,
                                        float* __restrict__ out2) {
    pdl_prologue();
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        const Agg4 s = {sums4[0], sums4[1], sums4[2], sums4[3]};
        agg_finish(s, n, (double)C2f, (double)Cf, out2, out2 + 1);
    }
}

// P:66 merge: one warp per output tile; lanes stride over the g*g input tiles (row-major
// inside the block), then a warp butterfly.  Output tile (oy, ox) merges input tiles
// (oy*g .. oy*g+g-1, ox*g .. ox*g+g-1) of the nt x nt matrix.
__global__ void __launch_bounds__(256)
merge_kernel(const float* __restrict__ lisi, const float* __restrict__ aug,
             const float* __restrict__ X, const float* __restrict__ Y, int nt, int g, int n_maps,
             float C2f, float Cf,
             float* __restrict__ lisi_o, float* __restrict__ aug_o,
             float* __restrict__ X_o, float* __restrict__ Y_o) {
    pdl_prologue();
    const int nto = nt / g;
    const long long per_map = (long long)nto * nto;
    const long long og = (long long)blockIdx.x * 8 + (threadIdx.x >> 5);      // output tile over all maps
    if (og >= per_map * n_maps) return;
    const long long map = og / per_map, o = og % per_map;
    const size_t in0 = (size_t)map * nt * nt;
    const int lane = threadIdx.x & 31;
    const int oy = (int)(o / nto), ox = (int)(o % nto);
    const double C2 = (double)C2f, C = (double)Cf;
    Agg4 a = {0.0, 0.0, 0.0, 0.0};
    const int gg = g * g;
    for (int k = lane; k < gg; k += 32) {
        const size_t t = in0 + (size_t)(oy * g + k / g) * nt + (size_t)(ox * g + k % g);
        agg_add(a, lisi[t], aug[t], X[t], Y[t], C2, C);
    }
    a = agg_warp_sum(a);
    if (lane == 0) {
        agg_finish(a, (double)gg, C2, C, lisi_o + og, aug_o + og);
        X_o[og] = (float)a.sx;
        Y_o[og] = (float)a.sy;
    }
}

// ---- P:66, every level in one launch -------------------------------------------------------------------------------
// Level j >= 1 of the pyramid over an nty x ntx tile matrix merges blocks of 2^j x 2^j base tiles (tile size 2^j N_T):
// ceil(nty / 2^j) x ceil(ntx / 2^j) output tiles; a block over the right / bottom border holds only the base tiles that
// exist, and Eq. 4's n is that count.  EVERY output tile is summed directly from the BASE arrays in double
// (never from the re-rounded level below), so level j is the tile matrix of size 2^j N_T up to one fp32 rounding.
// One launch: a unit (map, level, block) is taken by a warp (blocks of up to kPyrWarpTiles base tiles, 8 units per CTA)
// or by a whole CTA (larger blocks); lanes / threads stride over the block's tiles, then butterflies, fixed order.
constexpr int kPyrMaxLevels = 21;
constexpr int kPyrWarpTiles = 1024;
struct PyramidLevel { int shift, nby, nbx, cta_mode; long long out_off; unsigned first_cta; };
struct PyramidParams {
    PyramidLevel lv[kPyrMaxLevels];
    int n_levels, nty, ntx, n_maps;
    long long out_per_map;                  // output tiles of all levels of one map
};

__global__ void __launch_bounds__(256)
pyramid_kernel(const float* __restrict__ lisi, const float* __restrict__ aug,
               const float* __restrict__ X, const float* __restrict__ Y, const __grid_constant__ PyramidParams p,
               float C2f, float Cf, float* __restrict__ lisi_o, float* __restrict__ aug_o,
               float* __restrict__ X_o, float* __restrict__ Y_o) {
    __shared__ Agg4 part[8];
    pdl_prologue();
    int l = 0;
    while (l + 1 < p.n_levels && blockIdx.x >= p.lv[l + 1].first_cta) ++l;
    const PyramidLevel& L = p.lv[l];
    const long long per_map = (long long)L.nby * L.nbx;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const long long unit = L.cta_mode ? (long long)(blockIdx.x - L.first_cta)
                                      : (long long)(blockIdx.x - L.first_cta) * 8 + w;
    if (unit >= per_map * p.n_maps) return;                  // (whole warps / CTAs: no barrier is skipped by part of one)
    const long long map = unit / per_map, o = unit - map * per_map;
    const int oy = (int)(o / L.nbx), ox = (int)(o - (long long)oy * L.nbx);
    const int r0 = oy << L.shift, c0 = ox << L.shift;
    const int rows = min(p.nty - r0, 1 << L.shift), cols = min(p.ntx - c0, 1 << L.shift);
    const int nb = rows * cols;                               // base tiles actually merged: Eq. 4's n
    const size_t in0 = (size_t)map * p.nty * p.ntx + (size_t)r0 * p.ntx + c0;
    const double C2 = (double)C2f, C = (double)Cf;
    Agg4 a = {0.0, 0.0, 0.0, 0.0};
    const int t0 = L.cta_mode ? (int)threadIdx.x : lane, dt = L.cta_mode ? 256 : 32;
    int r = t0 / cols, c = t0 - r * cols;                     // tile k = r * cols + c of the block
    const int dr = dt / cols, dc = dt - dr * cols;
    for (int k = t0; k < nb; k += dt) {
        const size_t t = in0 + (size_t)r * p.ntx + c;
        agg_add(a, lisi[t], aug[t], X[t], Y[t], C2, C);
        r += dr; c += dc;
        if (c >= cols) { c -= cols; ++r; }
    }
    a = agg_warp_sum(a);
    if (L.cta_mode) {
        if (lane == 0) part[w] = a;
        __syncthreads();
        if (threadIdx.x >= 32) return;
        Agg4 b = {0.0, 0.0, 0.0, 0.0};
        if (lane < 8) b = part[lane];
        a = agg_warp_sum(b);
    }
    if (lane == 0) {
        const size_t og = (size_t)map * p.out_per_map + (size_t)L.out_off + (size_t)o;
        agg_finish(a, (double)nb, C2, C, lisi_o + og, aug_o + og);
        X_o[og] = (float)a.sx;
        Y_o[og] = (float)a.sy;
    }
}

}  // namespace iqa
