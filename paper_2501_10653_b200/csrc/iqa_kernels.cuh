// =============================================================================
// iqa_kernels.cuh -- shared device pieces of the tile-wise LISI / augLISI kernels
// (arxiv 2501.10653; "P:NN" = PAPER.md line NN):
//   pixel_terms      S1 clamp + S2 per-pixel terms of Eqs. 1-2
//   finalise_tile    S4: Eq. 1 / Eq. 2 from the four sums of one tile
//   generic_kernel   any N_T dividing N, any 4-byte aligned pointers (slow path, still CUDA)
//   finalise_*       second pass for tiles that were split over several CTAs (workspace)
// The fast paths are iqa_tma.cuh (fp32, power-of-two N_T >= 8) and iqa_any.cuh (any N_T >= 4, any pixel type).
// Every kernel starts with pdl_prologue(): when launched with the programmatic-stream-
// serialisation attribute its CTAs may become resident while the previous kernel of the
// stream drains; griddepcontrol.wait then blocks until that kernel has completed and its
// writes are visible, so nothing is read or written early.
// No floating-point atomics anywhere, so results are bit-reproducible.
// =============================================================================
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace iqa {

constexpr int kWarpsPerCta = 8;
constexpr int kCtaThreads = kWarpsPerCta * 32;
constexpr int kUnitCols = 128;          // 32 lanes x 4 columns

enum : int { kModeLisi = 1, kModeAug = 2, kModeFused = 3 };

struct TileParams {
    const float* __restrict__ x;   // typed entry point: pixels of another type behind the same pointer
    const float* __restrict__ y;
    int N;               // image width W (= side N of the square API)
    int H;               // image height
    long long pitch_x, pitch_y;   // elements between rows of x / y (N when contiguous)
    int nt;              // tiles per row: ceil(W / N_T)
    float C1, C2, C, D;
    float* lisi;         // [n] or nullptr (mode without LISI)
    float* auglisi;      // [n] or nullptr
    float* sum_x;        // [n] or nullptr
    float* sum_y;        // [n] or nullptr
    float* lisi_num;     // [n] or nullptr: raw L_t
    float* aug_num;      // [n] or nullptr: raw A_t
    float4* ws;          // split tiles: [n][pieces] partial (L, A, X, Y)
};

// Programmatic dependent launch (sm_90+): wait for the previous kernel of the stream (no-op
// when launched without the attribute), then let the next one start its prologue.
__device__ __forceinline__ void pdl_prologue() {
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}

__device__ __forceinline__ float rcp_approx(float v) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(v));
    return r;
}

// Position of one persistent CTA in its item sequence b, b+G, b+2G, ... kept as (pair, uy, ux) and advanced
// by the decoded stride (no integer division in the loop).  Items are numbered pair-major, then row-major.
struct ItemCursor {
    int pair, uy, ux;
    __device__ __forceinline__ void advance(const ItemCursor& d, int units_x, int units_y) {
        ux += d.ux;
        const int cx = ux >= units_x;
        ux -= cx ? units_x : 0;
        uy += d.uy + cx;
        const int cy = uy >= units_y;
        uy -= cy ? units_y : 0;
        pair += d.pair + cy;
    }
};
__device__ __forceinline__ ItemCursor decode_item(int q, int units_x, int units_y) {
    ItemCursor c;
    const int t = q / units_x;
    c.ux = q - t * units_x;
    c.pair = t / units_y;
    c.uy = t - c.pair * units_y;
    return c;
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

// S1 + S2 for one pixel pair of ANY supported pixel type T (the generic kernels).
// Types whose values are exact in fp32 (float, half, int16, uint8) are converted and go through
// pixel_terms.  double and int32 are clamped, added and SUBTRACTED in fp64 and only then rounded: the
// Eq. 1 term (x+y)/(|x-y|+C1) is ill-conditioned in the inputs once |x-y| is of the order of C1, so
// rounding x and y to fp32 first would be wrong by percents (tests/test_oracle_2d_pins.py T2).
template <typename T> struct PixelExactInFloat { static constexpr bool value = true; };
template <> struct PixelExactInFloat<double> { static constexpr bool value = false; };
template <> struct PixelExactInFloat<int> { static constexpr bool value = false; };

// One pixel of type T already in a register -> the terms.  (Loads are issued by the caller, several at a time.)
template <int MODE, typename T>
__device__ __forceinline__ void pixel_terms_val(T xr, T yr, float C1, float& aL, float& aA, float& aX, float& aY) {
    if constexpr (PixelExactInFloat<T>::value) {
        pixel_terms<MODE>((float)xr, (float)yr, C1, aL, aA, aX, aY);
    } else {
        const double xv = (double)xr, yv = (double)yr;
        const double xc = xv > 0.0 ? xv : 0.0;      // P:27; NaN -> 0
        const double yc = yv > 0.0 ? yv : 0.0;
        const float s = (float)(xc + yc);
        const float d = (float)fabs(xc - yc);
        if (MODE & kModeLisi) aL = fmaf(s, rcp_approx(d + C1), aL);
        if (MODE & kModeAug) aA = fmaf(s, d, aA);
        aX += (float)xc;
        aY += (float)yc;
    }
}
template <int MODE, typename T>
__device__ __forceinline__ void pixel_terms_any(const T* __restrict__ x, const T* __restrict__ y, size_t ox, size_t oy,
                                                float C1, float& aL, float& aA, float& aX, float& aY) {
    pixel_terms_val<MODE, T>(x[ox], y[oy], C1, aL, aA, aX, aY);
}

// S4: Eq. 1 / Eq. 2 from the four sums of one tile, true fp32 division.
// Per-tile results are stored with an L2 evict-last policy: they are a few MiB, they are read again right away
// (finalise / aggregate / merge / candidate kernels), and keeping them in L2 keeps their write-back out of the
// DRAM read stream of the images.
// (plain stores, an evict-first policy and st.global.cs were measured against this: profiles/r02_store_variants.md)
__device__ __forceinline__ uint64_t policy_evict_last() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void store_result(float* dst, float v, uint64_t pol) {
    asm volatile("st.global.L2::cache_hint.f32 [%0], %1, %2;" ::"l"(dst), "f"(v), "l"(pol) : "memory");
}

template <class Params>
__device__ __forceinline__ void finalise_tile(const Params& p, size_t t, float4 v /*L,A,X,Y*/, uint64_t pol) {
    if (p.lisi) store_result(p.lisi + t, p.D * v.x / (fmaxf(v.z, v.w) + p.C2), pol);        // Eq. 1
    if (p.auglisi) store_result(p.auglisi + t, 1.0f - v.y / (v.z + v.w + p.C), pol);          // Eq. 2
    if (p.sum_x) store_result(p.sum_x + t, v.z, pol);
    if (p.sum_y) store_result(p.sum_y + t, v.w, pol);
    if (p.lisi_num) store_result(p.lisi_num + t, v.x, pol);
    if (p.aug_num) store_result(p.aug_num + t, v.y, pol);
}
template <class Params>
__device__ __forceinline__ void finalise_tile(const Params& p, size_t t, float4 v) {
    finalise_tile(p, t, v, policy_evict_last());
}

// -----------------------------------------------------------------------------
// Generic kernel: any N_T, any H x W with ANY row pitch (edge tiles), any element-aligned pointers -- what is
// left when no tensor map can describe the image (row pitch not a multiple of 16 bytes) or N_T < 4.  One CTA per (tile, piece), a piece being up
// to kGenericRows rows of the tile; scalar coalesced loads, thread-strided partial sums,
// warp butterfly, warp order.  pieces == 1: the CTA finalises its tile; otherwise the
// partial goes to the workspace and finalise_kernel finishes.
// -----------------------------------------------------------------------------
constexpr int kGenericRows = 64;
constexpr int kGenericInFlight = 4;      // generic_kernel: rows whose loads a thread issues before it computes
constexpr int kWarpInFlight = 8;         // generic_warp_kernel: pixel pairs a lane loads before it computes

struct GenericParams {
    TileParams tp;
    int N_T;
    int pieces;               // ceil(N_T / kGenericRows) pieces of ceil(N_T / pieces) rows
};

template <int MODE, typename T = float>
__global__ void __launch_bounds__(kCtaThreads)
generic_kernel(const GenericParams g) {
    __shared__ float4 part[kWarpsPerCta];
    pdl_prologue();
    const TileParams& p = g.tp;
    const int N_T = g.N_T;
    const long long b = blockIdx.x;
    const int piece = (int)(b % g.pieces);
    const int tile = (int)(b / g.pieces);
    const int ty = tile / p.nt, tx = tile % p.nt;
    const int rows_t = min(N_T, p.H - ty * N_T);             // edge tiles hold only the pixels that exist
    const int cols_t = min(N_T, p.N - tx * N_T);
    const int rpp = (N_T + g.pieces - 1) / g.pieces;          // rows per piece: ceil(N_T / 64) pieces of equal height
    const int r_begin = piece * rpp;
    const int r_end = min(rows_t, r_begin + rpp);
    const long long npix = r_end > r_begin ? (long long)(r_end - r_begin) * cols_t : 0;
    const size_t row0 = (size_t)ty * N_T + r_begin, col0 = (size_t)tx * N_T;

    float aL = 0.f, aA = 0.f, aX = 0.f, aY = 0.f;
    // warp w takes rows w, w + 8, ...; lanes stride over the columns (coalesced, no division per pixel).  The loads
    // of kGenericInFlight rows of both images are issued before the first term is computed: a lone scalar load per
    // thread would leave the kernel waiting on the latency of each one.
    (void)npix;
    const int lane = (int)(threadIdx.x & 31), w = (int)(threadIdx.x >> 5);
    const int nrows = r_end - r_begin;
    const size_t sx = (size_t)kWarpsPerCta * (size_t)p.pitch_x, sy = (size_t)kWarpsPerCta * (size_t)p.pitch_y;
    const T* xrow = reinterpret_cast<const T*>(p.x) + (row0 + w) * (size_t)p.pitch_x + col0;     // row w of the piece
    const T* yrow = reinterpret_cast<const T*>(p.y) + (row0 + w) * (size_t)p.pitch_y + col0;
    for (int r = w; r < nrows; r += kWarpsPerCta * kGenericInFlight, xrow += kGenericInFlight * sx, yrow += kGenericInFlight * sy) {
        const int nr = min(kGenericInFlight, (nrows - r + kWarpsPerCta - 1) / kWarpsPerCta);   // rows r, r + 8, ... of this round
        for (int c = lane; c < cols_t; c += 32) {
            T vx[kGenericInFlight], vy[kGenericInFlight];
#pragma unroll
            for (int u = 0; u < kGenericInFlight; ++u)
                if (u < nr) { vx[u] = xrow[u * sx + c]; vy[u] = yrow[u * sy + c]; }
#pragma unroll
            for (int u = 0; u < kGenericInFlight; ++u)
                if (u < nr) pixel_terms_val<MODE, T>(vx[u], vy[u], p.C1, aL, aA, aX, aY);
        }
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

// Small tiles (N_T * N_T <= kWarpTilePixels): one WARP per tile, eight tiles per CTA -- a CTA per
// 64-pixel tile would be all launch overhead.  Lanes stride over the tile's pixels, warp butterfly,
// lane 0 applies Eqs. 1-2.  Same sums, same edge-tile rule as generic_kernel.
constexpr int kWarpTilePixels = 2048;

template <int MODE, typename T = float>
__global__ void __launch_bounds__(kCtaThreads)
generic_warp_kernel(const GenericParams g, long long n_tiles) {
    pdl_prologue();
    const TileParams& p = g.tp;
    const int N_T = g.N_T;
    const long long tile = (long long)blockIdx.x * kWarpsPerCta + (threadIdx.x >> 5);
    if (tile >= n_tiles) return;
    const int lane = threadIdx.x & 31;
    const int ty = (int)(tile / p.nt), tx = (int)(tile % p.nt);
    const int rows_t = min(N_T, p.H - ty * N_T);
    const int cols_t = min(N_T, p.N - tx * N_T);
    const int npix = rows_t * cols_t;
    const size_t row0 = (size_t)ty * N_T, col0 = (size_t)tx * N_T;
    float aL = 0.f, aA = 0.f, aX = 0.f, aY = 0.f;
    // lanes stride over the tile's pixels in row-major order; (row, column) advance by additions, and the loads of
    // kWarpInFlight pixels of both images are issued before the first term is computed
    const T* xp = reinterpret_cast<const T*>(p.x);
    const T* yp = reinterpret_cast<const T*>(p.y);
    int r = lane / cols_t, c = lane - r * cols_t;
    const int dr = 32 / cols_t, dc = 32 - dr * cols_t;
    for (int k0 = lane; k0 < npix; k0 += 32 * kWarpInFlight) {
        T vx[kWarpInFlight], vy[kWarpInFlight];
#pragma unroll
        for (int u = 0; u < kWarpInFlight; ++u) {
            if (k0 + 32 * u < npix) {
                vx[u] = xp[(row0 + r) * (size_t)p.pitch_x + col0 + c];
                vy[u] = yp[(row0 + r) * (size_t)p.pitch_y + col0 + c];
                r += dr; c += dc;
                if (c >= cols_t) { c -= cols_t; ++r; }
            }
        }
#pragma unroll
        for (int u = 0; u < kWarpInFlight; ++u)
            if (k0 + 32 * u < npix) pixel_terms_val<MODE, T>(vx[u], vy[u], p.C1, aL, aA, aX, aY);
    }
    float4 v = make_float4(aL, aA, aX, aY);
    for (int o = 16; o > 0; o >>= 1) {
        v.x += __shfl_xor_sync(0xffffffffu, v.x, o);
        v.y += __shfl_xor_sync(0xffffffffu, v.y, o);
        v.z += __shfl_xor_sync(0xffffffffu, v.z, o);
        v.w += __shfl_xor_sync(0xffffffffu, v.w, o);
    }
    if (lane == 0) finalise_tile(p, (size_t)tile, v);
}

// -----------------------------------------------------------------------------
// Finalise kernel (split tiles): one CTA per tile sums the tile's pieces in a fixed order
// (thread-strided, then warp butterfly, then warp order) and applies Eqs. 1-2.
// -----------------------------------------------------------------------------
__global__ void __launch_bounds__(kCtaThreads)
finalise_kernel(const TileParams p, int pieces) {
    __shared__ float4 part[kWarpsPerCta];
    pdl_prologue();
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
    pdl_prologue();
    const int tile = blockIdx.x * kCtaThreads + threadIdx.x;     // host guarantees n_tiles < 2^31
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
