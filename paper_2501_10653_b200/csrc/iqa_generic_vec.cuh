// =============================================================================
// iqa_generic_vec.cuh -- the generic kernels with 128-bit loads: images no tensor map can describe
// (a row pitch that is not a multiple of 16 bytes -- a contiguous 8190-pixel-wide fp32 plane, say -- or N_T < 4), as
// long as x and y have the SAME alignment row by row: equal offsets of the bases inside their 16-byte lines and
// equal row pitches modulo 16 bytes.  (Otherwise: the scalar kernels of iqa_kernels.cuh.)
// S1-S4 of SURVEY.md 8(a): clamp, Eq. 1 / Eq. 2 terms, per-tile sums, Eqs. 1-2.
//
// Row r of a tile starts a(r) elements past a 16-byte boundary, and a(r) changes from row to row when the pitch is
// odd.  A SLOT is one or two 16-byte-aligned groups (kSlotE elements: 4 fp32 / int32, 4 fp64, 16 fp16 / int16, 32 uint8) of
// one tile row; a row of cols_t pixels needs at most qmax = ceil((16 / sizeof(T) - 1 + cols_t) / kSlotE) slots.  The lanes of a warp (one
// warp per tile piece) stride over the rows x qmax slots of their piece, so every lane is
// busy whatever the tile width; each thread issues the loads of kVecInFlight slots of both images before the first
// term is computed.  Elements of a slot outside the tile's columns are zeroed in the raw words (a (0, 0) pixel pair
// adds nothing to any of the four sums) and the slot goes through Pixel4<T>::terms -- the packed arithmetic of the TMA
// kernels.  A 16-byte group that holds at least one pixel of the tile lies inside the 16-byte line of that pixel, hence
// inside the allocation; groups without one are not loaded.
// Same pieces, workspace and second pass as generic_kernel.
// =============================================================================
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "iqa_any.cuh"
#include "iqa_kernels.cuh"

namespace iqa {

constexpr int kVecInFlight = 4;      // slots (32 bytes of each image, 64 for fp64) a thread loads before it computes

template <typename T> struct VecGeom {
    static constexpr int kES = (int)sizeof(T);
    static constexpr int kAL = 16 / kES;                  // elements per 16 bytes
    // elements per slot: one 16-byte group (4-byte pixels), two groups for fp64 (4 pixels) and for 1- and 2-byte pixels
    // (32 / 16 pixels: the slot's addressing and masks are paid per slot -- int16 N_T = 200 4.2 -> 4.6 TB/s)
    static constexpr int kSlotE = kES == 4 ? kAL : 2 * kAL;
    static constexpr int kVecs = kSlotE / kAL;            // 16-byte loads per slot and image
    // slots a thread loads before it computes: 4 (fp32 / int32), 2 for the two-group slots (measured; three lose on narrow
    // tiles).  A software pipeline (next round's loads in flight while this round is computed) needs more than the 80
    // registers that three CTAs per SM leave and was slower in every variant.
    static constexpr int kInFlight = kVecs == 2 ? 2 : kVecInFlight;
};

// Zero the elements of one 16-byte group whose tile column c_first + e is outside [0, cols_t).
template <typename T>
__device__ __forceinline__ void mask_group(uint4& a, uint4& b, int c_first, int cols_t) {
    constexpr int ES = (int)sizeof(T), AL = 16 / ES;
    if constexpr (ES >= 4) {                              // whole words: one predicate per element
        uint32_t* wa = reinterpret_cast<uint32_t*>(&a);
        uint32_t* wb = reinterpret_cast<uint32_t*>(&b);
#pragma unroll
        for (int e = 0; e < AL; ++e) {
            const bool ok = (unsigned)(c_first + e) < (unsigned)cols_t;
#pragma unroll
            for (int w = e * (ES / 4); w < (e + 1) * (ES / 4); ++w) { wa[w] = ok ? wa[w] : 0u; wb[w] = ok ? wb[w] : 0u; }
        }
    } else {                                              // the valid elements are a byte range [lo, hi) of the 16
        const int lo = max(0, -c_first) * (8 * ES), hi = min(AL, cols_t - c_first) * (8 * ES);     // in bits
        uint32_t* wa = reinterpret_cast<uint32_t*>(&a);
        uint32_t* wb = reinterpret_cast<uint32_t*>(&b);
#pragma unroll
        for (int w = 0; w < 4; ++w) {
            // low t bits set, t clamped to [0, 32]: the clamping funnel shift of (0 : 0xffffffff) by t
            const uint32_t mu = __funnelshift_lc(0xffffffffu, 0u, (uint32_t)max(0, hi - 32 * w));
            const uint32_t ml = __funnelshift_lc(0xffffffffu, 0u, (uint32_t)max(0, lo - 32 * w));
            const uint32_t m = mu & ~ml;
            wa[w] &= m;
            wb[w] &= m;
        }
    }
}

// The four sums (L, A, X, Y) of this thread's slots of rows [row0, row0 + nrows) x columns [col0, col0 + cols_t).
template <int MODE, typename T>
__device__ __forceinline__ float4 vec_tile_sums(const T* __restrict__ x, const T* __restrict__ y, long long pitch_x,
                                                long long pitch_y, size_t row0, int nrows, size_t col0, int cols_t,
                                                float C1, int tid, int group) {
    using G = VecGeom<T>;
    Acc16 acc;
    acc.clear();
    if (nrows <= 0 || cols_t <= 0) return acc_cols(acc);
    const int qmax = (G::kAL - 1 + cols_t + G::kSlotE - 1) / G::kSlotE;
    const int n_slots = nrows * qmax;
    // byte addresses of pixel (row0 + r, col0) of x and y, kept for the thread's current row r and advanced by additions;
    // the slot's 16-byte groups start at (address & ~15) + q * slot bytes, a(r) = (address & 15) / sizeof(T) elements
    // before the row's first pixel (the same for x and y: host)
    const long long pbx = pitch_x * G::kES, pby = pitch_y * G::kES;
    int r = tid / qmax, q = tid - r * qmax;                          // slot k = r * qmax + q, advanced by additions
    const int dr = group / qmax, dq = group - dr * qmax;
    uintptr_t tx = (uintptr_t)(x + row0 * (size_t)pitch_x + col0) + (uintptr_t)((long long)r * pbx);
    uintptr_t ty = (uintptr_t)(y + row0 * (size_t)pitch_y + col0) + (uintptr_t)((long long)r * pby);
    const long long sx = (long long)dr * pbx, sy = (long long)dr * pby;
    const uint4 zero = make_uint4(0u, 0u, 0u, 0u);
    constexpr int U = G::kInFlight, V = G::kVecs;
    // one round = U slots of this thread: issue their loads (advancing the thread's (row, slot) position) ...
    auto load_round = [&](int k0, uint4 (&vx)[U][V], uint4 (&vy)[U][V], int (&cl)[U]) {
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const bool live = k0 + u * group < n_slots;
            const int a = (int)(tx & 15u) / G::kES;
            const int c_lo = q * G::kSlotE - a;                       // tile column of the slot's first element
            cl[u] = live ? c_lo : cols_t;                             // dead slots: every element masked
            const uint4* px = reinterpret_cast<const uint4*>((tx & ~(uintptr_t)15u) + (uintptr_t)(q * (G::kSlotE * G::kES)));
            const uint4* py = reinterpret_cast<const uint4*>((ty & ~(uintptr_t)15u) + (uintptr_t)(q * (G::kSlotE * G::kES)));
#pragma unroll
            for (int v = 0; v < V; ++v) {
                const int cf = c_lo + v * G::kAL;
                const bool any = live && cf < cols_t && cf + G::kAL > 0;
                vx[u][v] = any ? __ldg(px + v) : zero;
                vy[u][v] = any ? __ldg(py + v) : zero;
            }
            q += dq; tx += sx; ty += sy;
            if (q >= qmax) { q -= qmax; tx += pbx; ty += pby; }
        }
    };
    // ... and, a round later, mask them and add their terms
    auto compute_round = [&](uint4 (&vx)[U][V], uint4 (&vy)[U][V], const int (&cl)[U]) {
#pragma unroll
        for (int u = 0; u < U; ++u) {
#pragma unroll
            for (int v = 0; v < V; ++v) mask_group<T>(vx[u][v], vy[u][v], cl[u] + v * G::kAL, cols_t);
            const uint32_t* wx = reinterpret_cast<const uint32_t*>(&vx[u][0]);
            const uint32_t* wy = reinterpret_cast<const uint32_t*>(&vy[u][0]);
            constexpr int kW = Pixel4<T>::kWords;
#pragma unroll
            for (int c = 0; c < G::kSlotE / 4; ++c) Pixel4<T>::template terms<MODE>(wx + c * kW, wy + c * kW, C1, acc);
        }
    };
    for (int k0 = tid; k0 < n_slots; k0 += group * U) {
        uint4 vx[U][V], vy[U][V];
        int cl[U];
        load_round(k0, vx, vy, cl);
        compute_round(vx, vy, cl);
    }
    return acc_cols(acc);
}

__device__ __forceinline__ float4 warp_sum4(float4 v) {
    for (int o = 16; o > 0; o >>= 1) {
        v.x += __shfl_xor_sync(0xffffffffu, v.x, o);
        v.y += __shfl_xor_sync(0xffffffffu, v.y, o);
        v.z += __shfl_xor_sync(0xffffffffu, v.z, o);
        v.w += __shfl_xor_sync(0xffffffffu, v.w, o);
    }
    return v;
}

// The pairs of one launch: image pointers in the kernel parameters (a batch of independent pairs, or the comparisons of
// a time series, which share images).
constexpr int kVecMaxPairs = 32;
struct VecBatch {
    const void* x[kVecMaxPairs];
    const void* y[kVecMaxPairs];
    int n_pairs;
    int pair_minor;      // unit order: 0 = pair-major; 1 = the pairs of one tile piece next to each other (series: an image
                         // shared by two comparisons comes from DRAM once and from L2 afterwards, as in any_kernel)
};

// One WARP per (pair, tile, piece of ceil(N_T / pieces) rows), eight units per CTA: the units are independent streams
// (no CTA barrier, no serial tail per tile), so the loads of up to 24 warps per SM overlap.  (A CTA per tile -- the
// mapping of the scalar generic_kernel -- was measured at 3.7 TB/s here: a 64 x 64 tile is 32 KiB, and a CTA that
// loads, reduces and exits leaves the SM waiting on one DRAM latency per tile.)  pieces == 1: the warp finalises its
// tile; otherwise the partial goes to the workspace [pair][tile][piece] and finalise_*_kernel finishes.
// g.tp.x / g.tp.y are unused (the images are b.x / b.y); the output arrays and the workspace start at pair 0 of the launch.
template <int MODE, typename T>
__global__ void __launch_bounds__(kCtaThreads, 3)
generic_vec_kernel(const GenericParams g, const __grid_constant__ VecBatch b, long long units_per_pair) {
    pdl_prologue();
    const TileParams& p = g.tp;
    const int N_T = g.N_T;
    const long long unit = (long long)blockIdx.x * kWarpsPerCta + (threadIdx.x >> 5);
    if (unit >= units_per_pair * b.n_pairs) return;
    const int lane = threadIdx.x & 31;
    int pair;
    long long v_unit;                                        // (tile, piece) inside the pair
    if (b.pair_minor) { v_unit = unit / b.n_pairs; pair = (int)(unit - v_unit * b.n_pairs); }
    else { pair = (int)(unit / units_per_pair); v_unit = unit - pair * units_per_pair; }
    const long long tile = v_unit / g.pieces;
    const int piece = (int)(v_unit - tile * g.pieces);
    const int ty = (int)(tile / p.nt), tx = (int)(tile % p.nt);
    const int rows_t = min(N_T, p.H - ty * N_T);             // edge tiles hold only the pixels that exist
    const int cols_t = min(N_T, p.N - tx * N_T);
    const int rpp = (N_T + g.pieces - 1) / g.pieces;          // rows per piece: ceil(N_T / 64) pieces of equal height
    const int r_begin = piece * rpp;
    const int r_end = min(rows_t, r_begin + rpp);
    float4 v = vec_tile_sums<MODE, T>(reinterpret_cast<const T*>(b.x[pair]), reinterpret_cast<const T*>(b.y[pair]), p.pitch_x,
                                      p.pitch_y, (size_t)ty * N_T + r_begin, r_end - r_begin, (size_t)tx * N_T, cols_t,
                                      p.C1, lane, 32);
    v = warp_sum4(v);
    if (lane == 0) {
        const size_t t = (size_t)pair * (size_t)(units_per_pair / g.pieces) + (size_t)tile;
        if (p.ws == nullptr) finalise_tile(p, t, v);
        else p.ws[t * g.pieces + piece] = v;
    }
}

}  // namespace iqa
