// =============================================================================
// iqa_kernels.cuh -- sm_100a kernels for tile-wise LISI / augLISI (arxiv 2501.10653).
//
// Hot path ("P:NN" = PAPER.md line NN):
//   S1 load + clamp   S2 per-pixel terms (Eqs. 1-2)   S3 per-tile sums
//   S4 per-tile finalise     S5 Eqs. 3-4 aggregation and g x g merge
//
// The paper's H100 design is one thread block per tile with a shared-memory tree.
// Here the CTA -> pixel mapping does NOT depend on the tile size: a CTA of 8 warps owns a
// fixed "unit" of 128 columns x (8*RW) rows; warp w owns RW consecutive rows of it and
// lane l the four columns 4l..4l+3 (one 128-bit load per row and image, 512 contiguous
// bytes per warp and row).  A unit therefore holds several whole tiles (N_T < 64), exactly
// two (N_T = 64, RW = 8) or a piece of one (larger N_T); the tile size only decides how
// far the reduction goes:
//   lane   4 columns x RW rows in 16 independent fp32 accumulators (chain length RW)
//   warp   segmented xor-shuffle over the min(32, N_T/4) lanes that share a tile row
//   CTA    shared-memory combine of the warps that share a tile, fixed order
//   grid   (split tiles only) per-piece partials -> workspace -> finalise kernel, fixed order
// No floating-point atomics anywhere, so results are bit-reproducible.
// =============================================================================
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace iqa {

constexpr int kWarpsPerCta = 8;
constexpr int kCtaThreads = kWarpsPerCta * 32;
constexpr int kUnitCols = 128;          // 32 lanes x 4 columns

enum : int { kModeLisi = 1, kModeAug = 2, kModeFused = 3 };

struct TileParams {
    const float* __restrict__ x;
    const float* __restrict__ y;
    int N;               // image side
    int log2_nt;         // log2(N_T)           (strip kernels: N_T is a power of two >= 8)
    int nt;              // tiles per side, N / N_T
    int units_x;         // ceil(N / 128)
    float C1, C2, C, D;
    float* lisi;         // [n] or nullptr (mode without LISI)
    float* auglisi;      // [n] or nullptr
    float* sum_x;        // [n] or nullptr
    float* sum_y;        // [n] or nullptr
    float* lisi_num;     // [n] or nullptr: raw L_t
    float* aug_num;      // [n] or nullptr: raw A_t
    float4* ws;          // split tiles: [n][pieces] partial (L, A, X, Y)
    int pieces_x;        // pieces per tile across (max(1, N_T/128))
    int pieces_y;        // pieces per tile down   (max(1, N_T/(8*RW)))
};

// 128-bit streaming load: read-only path, no L1 allocation (every pixel is read once).
__device__ __forceinline__ float4 ldg_stream(const float* p) {
    float4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0, %1, %2, %3}, [%4];"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}

__device__ __forceinline__ float rcp_approx(float v) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(v));
    return r;
}

// S1 + S2 for one pixel pair: clamp, then the Eq. 1 and Eq. 2 terms.
//   s = |x + y| = x + y after the clamp;  d = |x - y|
//   L += s / (d + C1)   (MUFU.RCP: <= 1 ulp, far inside the 1e-5 budget)
//   A += s * d ;  X += x ;  Y += y
template <int MODE>
__device__ __forceinline__ void pixel_terms(float xv, float yv, float C1,
                                            float& aL, float& aA, float& aX, float& aY) {
    const float xc = fmaxf(xv, 0.0f);          // NaN -> 0, negatives -> 0
    const float yc = fmaxf(yv, 0.0f);
    const float s = xc + yc;
    const float d = fabsf(xc - yc);
    if (MODE & kModeLisi) aL = fmaf(s, rcp_approx(d + C1), aL);
    if (MODE & kModeAug) aA = fmaf(s, d, aA);
    aX += xc;
    aY += yc;
}

// S4: Eq. 1 / Eq. 2 from the four sums of one tile, true fp32 division.
__device__ __forceinline__ void finalise_tile(const TileParams& p, int t, float4 v /*L,A,X,Y*/) {
    if (p.lisi) p.lisi[t] = p.D * v.x / (fmaxf(v.z, v.w) + p.C2);        // Eq. 1
    if (p.auglisi) p.auglisi[t] = 1.0f - v.y / (v.z + v.w + p.C);          // Eq. 2
    if (p.sum_x) p.sum_x[t] = v.z;
    if (p.sum_y) p.sum_y[t] = v.w;
    if (p.lisi_num) p.lisi_num[t] = v.x;
    if (p.aug_num) p.aug_num[t] = v.y;
}

// -----------------------------------------------------------------------------
// Strip kernel.  grid = units_x * ceil(N / (8*RW)) CTAs of 256 threads, x-major so that
// consecutive CTAs read horizontally adjacent 512-byte segments (whole image rows are in
// flight together).  Requires: N_T a power of two >= max(8, RW), N % N_T == 0, x and y
// 16-byte aligned (N % 4 == 0 follows).  Ragged right/bottom edges (N % 128, N % (8*RW))
// are handled by idle lanes / warps: they contribute exact zeros.
// MIN_CTAS is the register budget handed to ptxas (65536 / (256 * MIN_CTAS) registers per
// thread): with the default "maximise occupancy" heuristic ptxas sinks each load next to its
// use and keeps only 2-4 of them in flight; with MIN_CTAS = 2 it hoists all 2*RW loads of a
// lane above the arithmetic (checked in SASS), which is what keeps HBM busy.
// -----------------------------------------------------------------------------
template <int MODE, int RW, int MIN_CTAS = 2>
__global__ void __launch_bounds__(kCtaThreads, MIN_CTAS)
strip_kernel(const TileParams p) {
    constexpr int RB = kWarpsPerCta * RW;      // rows per unit
    __shared__ float4 part[kWarpsPerCta][16];  // per warp: <= 16 tile segments (N_T = 8)

    const int lane = threadIdx.x & 31;
    const int w = threadIdx.x >> 5;
    const int ux = blockIdx.x % p.units_x;
    const int uy = blockIdx.x / p.units_x;
    const int N = p.N;
    const int col = ux * kUnitCols + lane * 4;
    const int row0 = uy * RB + w * RW;

    float aL[4] = {0.f, 0.f, 0.f, 0.f}, aA[4] = {0.f, 0.f, 0.f, 0.f};
    float aX[4] = {0.f, 0.f, 0.f, 0.f}, aY[4] = {0.f, 0.f, 0.f, 0.f};

    if (row0 < N) {                            // warp-uniform: the whole warp is inside or outside
        const bool in_cols = col < N;          // ragged right edge: idle lanes contribute exact zeros
        const size_t off = (size_t)row0 * (size_t)N + (size_t)(in_cols ? col : 0);
        const float* px = p.x + off;
        const float* py = p.y + off;
        const float C1 = p.C1;
#pragma unroll
        for (int i = 0; i < RW; i += 4) {
            float4 vx[4], vy[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                vx[k] = vy[k] = make_float4(0.f, 0.f, 0.f, 0.f);
                if (in_cols) {
                    vx[k] = ldg_stream(px + (size_t)(i + k) * (size_t)N);
                    vy[k] = ldg_stream(py + (size_t)(i + k) * (size_t)N);
                }
            }
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                pixel_terms<MODE>(vx[k].x, vy[k].x, C1, aL[0], aA[0], aX[0], aY[0]);
                pixel_terms<MODE>(vx[k].y, vy[k].y, C1, aL[1], aA[1], aX[1], aY[1]);
                pixel_terms<MODE>(vx[k].z, vy[k].z, C1, aL[2], aA[2], aX[2], aY[2]);
                pixel_terms<MODE>(vx[k].w, vy[k].w, C1, aL[3], aA[3], aX[3], aY[3]);
            }
        }
    }

    // lane: 4 columns -> 1
    float4 v;
    v.x = (aL[0] + aL[1]) + (aL[2] + aL[3]);
    v.y = (aA[0] + aA[1]) + (aA[2] + aA[3]);
    v.z = (aX[0] + aX[1]) + (aX[2] + aX[3]);
    v.w = (aY[0] + aY[1]) + (aY[2] + aY[3]);

    // warp: segmented butterfly over the g lanes that share a tile row
    const int log2_nt = p.log2_nt;
    const int log2_g = min(log2_nt - 2, 5);                 // g = min(32, N_T / 4)
    for (int o = (1 << log2_g) >> 1; o > 0; o >>= 1) {
        if (MODE & kModeLisi) v.x += __shfl_xor_sync(0xffffffffu, v.x, o);
        if (MODE & kModeAug) v.y += __shfl_xor_sync(0xffffffffu, v.y, o);
        v.z += __shfl_xor_sync(0xffffffffu, v.z, o);
        v.w += __shfl_xor_sync(0xffffffffu, v.w, o);
    }
    if ((lane & ((1 << log2_g) - 1)) == 0) part[w][lane >> log2_g] = v;
    __syncthreads();

    // CTA: combine the warps that share a tile (fixed order), one thread per tile of the unit
    const int log2_tpw = 5 - log2_g;                        // tile segments per warp row: 128/N_T or 1
    const int N_T = 1 << log2_nt;
    const int wpt = (N_T >= RB) ? kWarpsPerCta : (N_T / RW);   // warps per tile (down)
    const int n_ty = kWarpsPerCta / wpt;                    // tile rows in the unit
    const int t = threadIdx.x;
    if (t < (n_ty << log2_tpw)) {
        const int jy = t >> log2_tpw;
        const int jx = t & ((1 << log2_tpw) - 1);
        const int c0 = ux * kUnitCols + (jx << log2_nt);    // jx == 0 when N_T >= 128
        const int r0 = uy * RB + jy * wpt * RW;
        if (c0 < N && r0 < N) {
            float4 s = part[jy * wpt][jx];
            for (int k = 1; k < wpt; ++k) {
                const float4 q = part[jy * wpt + k][jx];
                s.x += q.x; s.y += q.y; s.z += q.z; s.w += q.w;
            }
            const int tile = (r0 >> log2_nt) * p.nt + (c0 >> log2_nt);
            if (p.ws == nullptr) {
                finalise_tile(p, tile, s);
            } else {                                        // split tile: piece -> workspace
                const int pxi = ux & (p.pieces_x - 1);
                const int pyi = uy & (p.pieces_y - 1);
                p.ws[((size_t)tile * p.pieces_y + pyi) * p.pieces_x + pxi] = s;
            }
        }
    }
}

// -----------------------------------------------------------------------------
// Generic kernel: any N_T dividing N, any 4-byte aligned pointers (the strip kernel needs a
// power-of-two N_T >= 8 and 16-byte alignment).  One CTA per (tile, piece), a piece being up
// to kGenericRows rows of the tile; scalar coalesced loads, thread-strided partial sums,
// warp butterfly, warp order.  pieces == 1: the CTA finalises its tile; otherwise the
// partial goes to the workspace and finalise_kernel finishes.
// -----------------------------------------------------------------------------
constexpr int kGenericRows = 64;

struct GenericParams {
    TileParams tp;
    int N_T;
    int pieces;               // ceil(N_T / kGenericRows)
};

template <int MODE>
__global__ void __launch_bounds__(kCtaThreads)
generic_kernel(const GenericParams g) {
    __shared__ float4 part[kWarpsPerCta];
    const TileParams& p = g.tp;
    const int N_T = g.N_T;
    const long long b = blockIdx.x;
    const int piece = (int)(b % g.pieces);
    const int tile = (int)(b / g.pieces);
    const int ty = tile / p.nt, tx = tile % p.nt;
    const int r_begin = piece * kGenericRows;
    const int r_end = min(N_T, r_begin + kGenericRows);
    const long long npix = (long long)(r_end - r_begin) * N_T;
    const size_t base = ((size_t)ty * N_T + r_begin) * (size_t)p.N + (size_t)tx * N_T;

    float aL = 0.f, aA = 0.f, aX = 0.f, aY = 0.f;
    for (long long k = threadIdx.x; k < npix; k += kCtaThreads) {
        const int r = (int)(k / N_T), c = (int)(k % N_T);
        const size_t off = base + (size_t)r * (size_t)p.N + (size_t)c;
        pixel_terms<MODE>(__ldg(p.x + off), __ldg(p.y + off), p.C1, aL, aA, aX, aY);
    }
    float4 v = make_float4(aL, aA, aX, aY);
    for (int o = 16; o > 0; o >>= 1) {
        v.x += __shfl_xor_sync(0xffffffffu, v.x, o);
        v.y += __shfl_xor_sync(0xffffffffu, v.y, o);
        v.z += __shfl_xor_sync(0xffffffffu, v.z, o);
        v.w += __shfl_xor_sync(0xffffffffu, v.w, o);
    }
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        float4 s = part[0];
        for (int k = 1; k < kWarpsPerCta; ++k) {
            s.x += part[k].x; s.y += part[k].y; s.z += part[k].z; s.w += part[k].w;
        }
        if (p.ws == nullptr) finalise_tile(p, tile, s);
        else p.ws[(size_t)tile * g.pieces + piece] = s;
    }
}

// -----------------------------------------------------------------------------
// Finalise kernel (split tiles): one CTA per tile sums the tile's pieces in a fixed order
// (thread-strided, then warp butterfly, then warp order) and applies Eqs. 1-2.
// -----------------------------------------------------------------------------
__global__ void __launch_bounds__(kCtaThreads)
finalise_kernel(const TileParams p, int pieces) {
    __shared__ float4 part[kWarpsPerCta];
    const int tile = blockIdx.x;
    const float4* src = p.ws + (size_t)tile * pieces;
    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int k = threadIdx.x; k < pieces; k += kCtaThreads) {
        const float4 q = src[k];
        v.x += q.x; v.y += q.y; v.z += q.z; v.w += q.w;
    }
    for (int o = 16; o > 0; o >>= 1) {
        v.x += __shfl_xor_sync(0xffffffffu, v.x, o);
        v.y += __shfl_xor_sync(0xffffffffu, v.y, o);
        v.z += __shfl_xor_sync(0xffffffffu, v.z, o);
        v.w += __shfl_xor_sync(0xffffffffu, v.w, o);
    }
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        float4 s = part[0];
        for (int k = 1; k < kWarpsPerCta; ++k) {
            s.x += part[k].x; s.y += part[k].y; s.z += part[k].z; s.w += part[k].w;
        }
        finalise_tile(p, tile, s);
    }
}

// Few pieces per tile (the common split case: 2..32): one thread per tile, sequential order.
__global__ void __launch_bounds__(kCtaThreads)
finalise_small_kernel(const TileParams p, int pieces, int n_tiles) {
    const int tile = blockIdx.x * kCtaThreads + threadIdx.x;
    if (tile >= n_tiles) return;
    const float4* src = p.ws + (size_t)tile * pieces;
    float4 s = src[0];
    for (int k = 1; k < pieces; ++k) {
        const float4 q = src[k];
        s.x += q.x; s.y += q.y; s.z += q.z; s.w += q.w;
    }
    finalise_tile(p, tile, s);
}

}  // namespace iqa
