// =============================================================================
// iqa_any.cuh -- the TMA-fed persistent kernel for everything the power-of-two kernel of
// iqa_tma.cuh does not take ("allowing input of FITS images"):
//   * any tile side N_T >= 4 (48, 100, 50, 7 ...), tiles larger than an item are split,
//   * pixels of type fp32, fp64, fp16, int16, int32, uint8 (FITS BITPIX -32, -64, 16, 32, 8),
//   * image bases aligned to the element size only, as long as x and y sit at the SAME offset inside
//     their 16-byte line (two windows cut at the same column out of aligned images): the tensor maps
//     start at the 16-byte boundary below the bases,
//   * H x W images with row pitches and edge tiles (zero-filled by the TMA unit).
// S1-S4 of SURVEY.md 8(a): clamp, Eq. 1 / Eq. 2 terms, per-tile sums, Eqs. 1-2.
//
// Same roles as tma_kernel: eight consumer warps, one producer lane issuing cp.async.bulk.tensor.2d
// into a ring of box slots (full / empty mbarriers), one finaliser warp.  What differs is that the
// geometry is a RUN-TIME description computed on the host (any_geometry() in iqa_tiles.cu):
//   item     kx x ky whole tiles (N_T <= 128), or one piece pw x ph of a split tile (N_T > 128);
//            columns c0 .. c0 + cv, rows r0 .. r0 + rv of the image; items are numbered pair-major,
//            then row-major; CTA b takes items b, b + G, ...
//   box      box_w columns x b rows of the element type (<= 128 columns; b <= 256), about 16-20 KiB; an
//            item is ceil(rv / b) boxes per image; a ragged last box starts EARLIER (it overlaps the
//            previous one) and the rows already counted are skipped, so nothing outside the item's rows
//            is ever fetched.  The TMA unit needs the global address of a box row to be 16-byte aligned
//            (measured: anything else traps), so a box starts at the 16-byte boundary at or below the
//            item's first pixel and the item's columns sit s = 0 .. 16/sizeof(T) - 1 columns into it
//   lane     lane l owns BOX columns 4l .. 4l+3 for every pixel type (LDS.128 / .64 / .32 / 2 x .128
//            for 4- / 2- / 1- / 8-byte pixels): 16 accumulators, the packed-pair arithmetic of
//            pixel_terms2, no mask and no shift in the pixel loop -- the offset s only enters when the
//            lane's four column sums are assigned to tiles at the end of the item;
//            fp64 and int32 form x + y and |x - y| exactly before rounding to fp32.
//            When N_T is a multiple of 8 and the bases are 16-byte aligned, a lane owns EIGHT columns
//            (8l .. 8l+7, all in one tile) and folds columns j and j + 4 into the same accumulator:
//            boxes of up to 256 columns, twice the pixels per item for the same per-item bookkeeping
//   warp     warp w owns rows [w rpw, (w+1) rpw) of a box (ky == 1), or rows of tile row w / wpt
//            (ky > 1: several tile rows per box, wpt = 8 / ky warps each)
//   reduce   per item: every lane folds its 4 columns into the partial of the tile its FIRST column
//            lies in; columns that belong to the next tile (N_T % 4 != 0) travel one lane up by a
//            shuffle; part[buf][warp][lane] -> the finaliser warp sums the (warp, lane) entries of
//            each tile in a fixed order (groups of 32 / pow2(tiles) lanes per tile, then a butterfly)
//            and applies Eq. 1 / Eq. 2, or writes the piece's sums to the workspace.
// No floating-point atomics: results are bit-reproducible and do not depend on the grid size.
// =============================================================================
#pragma once
#include <cuda.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "iqa_kernels.cuh"
#include "iqa_tma.cuh"

namespace iqa {

constexpr int kAnyMaxImages = 64;      // tensor maps per launch: 32 pairs
constexpr int kAnyPartBufs = 4;
constexpr int kAnyMaxSlots = 8;

struct AnyParams {
    CUtensorMap maps[kAnyMaxImages];   // images 2p (x) and 2p + 1 (y) of pair p; box box_w x box_rows, OOB -> 0
    int shift;             // elements between the 16-byte aligned tensor bases and pixel (0, 0): the same for all images
    int pad_mask;          // 16 / sizeof(T) - 1: box columns start at multiples of 16 bytes
    int const_s;           // the items' column offset s is the same for every item (s = shift)
    int n_pairs;
    int pair_minor;        // item order: 0 = pair-major (batches), 1 = the pairs of one item location next to each other (series)
    int W, H, N_T;
    int ntx, nty, n_tiles;
    int kx, ky;            // whole tiles per item across / down (1, 1 when tiles are split)
    int px, py;            // pieces per tile across / down (1, 1 unless split)
    int pw, ph;            // item extent: columns (pw + s <= box_w <= 32 lanes x 4 or 8 columns), rows
    int units_x, units_y;  // items across / down
    int box_rows;          // b
    int row_bytes;         // bytes between two box rows in shared memory (box_w * sizeof(T), multiple of 16)
    int slot_bytes;        // ring slot stride (multiple of 128)
    int n_slots;           // even, 4 .. kAnyMaxSlots
    int rpw, wpt;          // rows per warp inside a box (or inside a tile when ky > 1); warps per tile row
    int fin_gsz;           // finaliser lanes per tile: max(1, 32 / pow2ceil(kx * ky))
    int cpl_log2;          // log2 of the columns a lane owns: 2 (four) or 3 (eight: N_T % 8 == 0, every base 16-byte aligned)
    int boxes_per_item;    // ceil(ph / box_rows)
    unsigned nt_magic;     // floor(2^32 / N_T) + 1: n / N_T == umulhi(n, nt_magic) for the small n used here
    float C1, C2, C, D;
    float *lisi, *auglisi, *sum_x, *sum_y, *lisi_num, *aug_num;   // [n_pairs * n_tiles] or nullptr
    float4* ws;            // split tiles: [pair][tile][py][px] partial (L, A, X, Y)
};

inline size_t any_smem_bytes(int n_slots, int slot_bytes) {
    return 1024 /* alignment slack */ + (size_t)n_slots * slot_bytes +
           (size_t)kAnyPartBufs * kWarpsPerCta * 32 * sizeof(float4) + (2 * kAnyMaxSlots + 2 * kAnyPartBufs) * sizeof(uint64_t);
}

// Image region of item (ux, uy).
struct AnyItem {
    int c0, r0;      // first column / row in the image
    int cv, rv;      // valid columns / rows (the box may hold more columns: they belong to the neighbour)
    int tx0, ty0;    // tile of the item's top-left corner
    int ix, iy;      // piece index inside the tile (split tiles)
    int bc0;         // first TENSOR column of the item's boxes (a multiple of 16 bytes)
    int s;           // box column of the item's first column: c0 + shift - bc0
};
__device__ __forceinline__ AnyItem any_item(const AnyParams& p, int ux, int uy) {
    AnyItem it;
    const int gx = p.px == 1 ? ux : ux / p.px, gy = p.py == 1 ? uy : uy / p.py;
    it.ix = ux - gx * p.px;
    it.iy = uy - gy * p.py;
    it.tx0 = gx * p.kx;
    it.ty0 = gy * p.ky;
    const int GW = p.kx * p.N_T, GH = p.ky * p.N_T;
    it.c0 = gx * GW + it.ix * p.pw;
    it.cv = min(p.pw, GW - it.ix * p.pw);
    it.r0 = gy * GH + it.iy * p.ph;
    it.rv = min(p.ph, GH - it.iy * p.ph);
    it.bc0 = (it.c0 + p.shift) & ~p.pad_mask;
    it.s = (it.c0 + p.shift) & p.pad_mask;
    return it;
}
// Box s of an item with rv valid rows: the box starts o rows below the item's first row and its rows
// [lo, hi) are the ones not yet counted (a ragged last box overlaps its predecessor).
struct AnyBox { int o, lo, hi; };
__device__ __forceinline__ AnyBox any_box(int s, int b, int rv) {
    AnyBox x;
    const int done = s * b;
    x.o = min(done, max(0, rv - b));
    x.lo = done - x.o;
    x.hi = min(b, rv - x.o);
    return x;
}

// ---- 4 pixels of type T at p (shared memory) -> S1 + S2 into this lane's accumulators ---------------------------
// Types whose values are exact in fp32 are converted and follow pixel_terms2 (the arithmetic of the fp32
// kernel); fp64 and int32 are clamped, added and subtracted exactly first (R19:
// the Eq. 1 term is ill-conditioned in x - y once |x - y| is of the order of C1).
template <int MODE>
__device__ __forceinline__ void terms_wide2(float s0, float s1, float d0, float d1, float x0, float x1, float y0,
                                            float y1, float C1, uint64_t& aL, float& aA0, float& aA1, uint64_t& aX,
                                            uint64_t& aY) {
    if (MODE & kModeLisi) aL = fma2(pack2(s0, s1), pack2(rcp_approx(d0 + C1), rcp_approx(d1 + C1)), aL);
    if (MODE & kModeAug) { aA0 = fmaf(s0, d0, aA0); aA1 = fmaf(s1, d1, aA1); }
    aX = add2(aX, pack2(x0, x1));
    aY = add2(aY, pack2(y0, y1));
}

// Pixel4<T>: four horizontally adjacent pixels of type T.  terms() takes them as the kWords 32-bit words they occupy
// (registers: the generic kernels load them from global memory), row() reads them from shared memory.
template <typename T> struct Pixel4;

template <> struct Pixel4<float> {
    static constexpr int kBytes = 16, kWords = 4;
    template <int MODE>
    static __device__ __forceinline__ void terms(const uint32_t* x, const uint32_t* y, float C1, Acc16& a) {
        pixel_terms2<MODE>(__uint_as_float(x[0]), __uint_as_float(x[1]), __uint_as_float(y[0]), __uint_as_float(y[1]), C1,
                           a.L[0], a.A[0], a.A[1], a.X[0], a.Y[0]);
        pixel_terms2<MODE>(__uint_as_float(x[2]), __uint_as_float(x[3]), __uint_as_float(y[2]), __uint_as_float(y[3]), C1,
                           a.L[1], a.A[2], a.A[3], a.X[1], a.Y[1]);
    }
    template <int MODE>
    static __device__ __forceinline__ void row(const unsigned char* xs, const unsigned char* ys, float C1, Acc16& a) {
        const uint4 vx = *reinterpret_cast<const uint4*>(xs);
        const uint4 vy = *reinterpret_cast<const uint4*>(ys);
        const uint32_t wx[4] = {vx.x, vx.y, vx.z, vx.w}, wy[4] = {vy.x, vy.y, vy.z, vy.w};
        terms<MODE>(wx, wy, C1, a);
    }
};

template <> struct Pixel4<__half> {
    static constexpr int kBytes = 8, kWords = 2;
    template <int MODE>
    static __device__ __forceinline__ void terms(const uint32_t* x, const uint32_t* y, float C1, Acc16& a) {
        // the clamp on two pixels at once in fp16 (max(NaN, 0) = 0, as in fp32), then the exact conversion
        const __half2 zero = __float2half2_rn(0.0f);
        const float2 x01 = __half22float2(__hmax2(*reinterpret_cast<const __half2*>(&x[0]), zero));
        const float2 x23 = __half22float2(__hmax2(*reinterpret_cast<const __half2*>(&x[1]), zero));
        const float2 y01 = __half22float2(__hmax2(*reinterpret_cast<const __half2*>(&y[0]), zero));
        const float2 y23 = __half22float2(__hmax2(*reinterpret_cast<const __half2*>(&y[1]), zero));
        pixel_terms2<MODE, false>(x01.x, x01.y, y01.x, y01.y, C1, a.L[0], a.A[0], a.A[1], a.X[0], a.Y[0]);
        pixel_terms2<MODE, false>(x23.x, x23.y, y23.x, y23.y, C1, a.L[1], a.A[2], a.A[3], a.X[1], a.Y[1]);
    }
    template <int MODE>
    static __device__ __forceinline__ void row(const unsigned char* xs, const unsigned char* ys, float C1, Acc16& a) {
        const uint2 qx = *reinterpret_cast<const uint2*>(xs);
        const uint2 qy = *reinterpret_cast<const uint2*>(ys);
        const uint32_t wx[2] = {qx.x, qx.y}, wy[2] = {qy.x, qy.y};
        terms<MODE>(wx, wy, C1, a);
    }
};

// int16 -> fp32 without the conversion unit: the clamp on both halves at once leaves u in [0, 32767];
// the float with bits 0x4B000000 | u is exactly 2^23 + u, and subtracting 2^23 leaves u.
__device__ __forceinline__ void s16x2_to_float(uint32_t w, float& lo, float& hi) {
    const uint32_t u = __vimax_s16x2_relu(w, w);               // max(v, 0) on both halves: VIMNMX.S16x2.RELU
    const uint64_t m = pack2(8388608.0f, 8388608.0f);
    const uint64_t f = sub2(pack2(__uint_as_float(__byte_perm(u, 0x4B000000u, 0x7610)),
                                  __uint_as_float(__byte_perm(u, 0x4B000000u, 0x7632))), m);
    unpack2(f, lo, hi);
}
template <> struct Pixel4<short> {
    static constexpr int kBytes = 8, kWords = 2;
    template <int MODE>
    static __device__ __forceinline__ void terms(const uint32_t* x, const uint32_t* y, float C1, Acc16& a) {
        float x0, x1, x2, x3, y0, y1, y2, y3;
        s16x2_to_float(x[0], x0, x1); s16x2_to_float(x[1], x2, x3);
        s16x2_to_float(y[0], y0, y1); s16x2_to_float(y[1], y2, y3);
        pixel_terms2<MODE, false>(x0, x1, y0, y1, C1, a.L[0], a.A[0], a.A[1], a.X[0], a.Y[0]);
        pixel_terms2<MODE, false>(x2, x3, y2, y3, C1, a.L[1], a.A[2], a.A[3], a.X[1], a.Y[1]);
    }
    template <int MODE>
    static __device__ __forceinline__ void row(const unsigned char* xs, const unsigned char* ys, float C1, Acc16& a) {
        const uint2 qx = *reinterpret_cast<const uint2*>(xs);
        const uint2 qy = *reinterpret_cast<const uint2*>(ys);
        const uint32_t wx[2] = {qx.x, qx.y}, wy[2] = {qy.x, qy.y};
        terms<MODE>(wx, wy, C1, a);
    }
};

// uint8 -> fp32 the same way: bits 0x4B000000 | v are exactly 2^23 + v.
__device__ __forceinline__ void u8x4_to_float(uint32_t w, float& f0, float& f1, float& f2, float& f3) {
    const uint64_t m = pack2(8388608.0f, 8388608.0f);
    unpack2(sub2(pack2(__uint_as_float(__byte_perm(w, 0x4B000000u, 0x7650)),
                       __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7651))), m), f0, f1);
    unpack2(sub2(pack2(__uint_as_float(__byte_perm(w, 0x4B000000u, 0x7652)),
                       __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7653))), m), f2, f3);
}
template <> struct Pixel4<unsigned char> {
    static constexpr int kBytes = 4, kWords = 1;
    template <int MODE>
    static __device__ __forceinline__ void terms(const uint32_t* x, const uint32_t* y, float C1, Acc16& a) {
        float x0, x1, x2, x3, y0, y1, y2, y3;
        u8x4_to_float(x[0], x0, x1, x2, x3);
        u8x4_to_float(y[0], y0, y1, y2, y3);
        pixel_terms2<MODE, false>(x0, x1, y0, y1, C1, a.L[0], a.A[0], a.A[1], a.X[0], a.Y[0]);      // unsigned: nothing to clamp
        pixel_terms2<MODE, false>(x2, x3, y2, y3, C1, a.L[1], a.A[2], a.A[3], a.X[1], a.Y[1]);
    }
    template <int MODE>
    static __device__ __forceinline__ void row(const unsigned char* xs, const unsigned char* ys, float C1, Acc16& a) {
        const uint32_t qx = *reinterpret_cast<const uint32_t*>(xs);
        const uint32_t qy = *reinterpret_cast<const uint32_t*>(ys);
        terms<MODE>(&qx, &qy, C1, a);
    }
};

template <> struct Pixel4<double> {
    static constexpr int kBytes = 32, kWords = 8;
    static __device__ __forceinline__ void one(double xv, double yv, float& s, float& d, float& xc, float& yc) {
        const double xd = xv > 0.0 ? xv : 0.0;      // P:27; NaN -> 0
        const double yd = yv > 0.0 ? yv : 0.0;
        s = (float)(xd + yd);
        d = (float)fabs(xd - yd);
        xc = (float)xd;
        yc = (float)yd;
    }
    template <int MODE>
    static __device__ __forceinline__ void terms(const uint32_t* x, const uint32_t* y, float C1, Acc16& a) {
        float s0, s1, d0, d1, cx0, cx1, cy0, cy1;
        one(__hiloint2double((int)x[1], (int)x[0]), __hiloint2double((int)y[1], (int)y[0]), s0, d0, cx0, cy0);
        one(__hiloint2double((int)x[3], (int)x[2]), __hiloint2double((int)y[3], (int)y[2]), s1, d1, cx1, cy1);
        terms_wide2<MODE>(s0, s1, d0, d1, cx0, cx1, cy0, cy1, C1, a.L[0], a.A[0], a.A[1], a.X[0], a.Y[0]);
        one(__hiloint2double((int)x[5], (int)x[4]), __hiloint2double((int)y[5], (int)y[4]), s0, d0, cx0, cy0);
        one(__hiloint2double((int)x[7], (int)x[6]), __hiloint2double((int)y[7], (int)y[6]), s1, d1, cx1, cy1);
        terms_wide2<MODE>(s0, s1, d0, d1, cx0, cx1, cy0, cy1, C1, a.L[1], a.A[2], a.A[3], a.X[1], a.Y[1]);
    }
    template <int MODE>
    static __device__ __forceinline__ void row(const unsigned char* xs, const unsigned char* ys, float C1, Acc16& a) {
        const uint4 xa = *reinterpret_cast<const uint4*>(xs), xb = *reinterpret_cast<const uint4*>(xs + 16);
        const uint4 ya = *reinterpret_cast<const uint4*>(ys), yb = *reinterpret_cast<const uint4*>(ys + 16);
        const uint32_t wx[8] = {xa.x, xa.y, xa.z, xa.w, xb.x, xb.y, xb.z, xb.w};
        const uint32_t wy[8] = {ya.x, ya.y, ya.z, ya.w, yb.x, yb.y, yb.z, yb.w};
        terms<MODE>(wx, wy, C1, a);
    }
};

template <> struct Pixel4<int> {
    static constexpr int kBytes = 16, kWords = 4;
    // after the clamp x, y are in [0, 2^31): x + y and |x - y| are exact as unsigned 32-bit integers, and one
    // integer -> fp32 conversion rounds exactly like the fp64 route of the oracle's definition
    static __device__ __forceinline__ void one(int xv, int yv, float& s, float& d, float& xc, float& yc) {
        const uint32_t xu = (uint32_t)max(xv, 0), yu = (uint32_t)max(yv, 0);
        s = __uint2float_rn(xu + yu);
        d = __uint2float_rn(xu > yu ? xu - yu : yu - xu);
        xc = __uint2float_rn(xu);
        yc = __uint2float_rn(yu);
    }
    template <int MODE>
    static __device__ __forceinline__ void terms(const uint32_t* x, const uint32_t* y, float C1, Acc16& a) {
        float s0, s1, d0, d1, cx0, cx1, cy0, cy1;
        one((int)x[0], (int)y[0], s0, d0, cx0, cy0); one((int)x[1], (int)y[1], s1, d1, cx1, cy1);
        terms_wide2<MODE>(s0, s1, d0, d1, cx0, cx1, cy0, cy1, C1, a.L[0], a.A[0], a.A[1], a.X[0], a.Y[0]);
        one((int)x[2], (int)y[2], s0, d0, cx0, cy0); one((int)x[3], (int)y[3], s1, d1, cx1, cy1);
        terms_wide2<MODE>(s0, s1, d0, d1, cx0, cx1, cy0, cy1, C1, a.L[1], a.A[2], a.A[3], a.X[1], a.Y[1]);
    }
    template <int MODE>
    static __device__ __forceinline__ void row(const unsigned char* xs, const unsigned char* ys, float C1, Acc16& a) {
        const uint4 vx = *reinterpret_cast<const uint4*>(xs);
        const uint4 vy = *reinterpret_cast<const uint4*>(ys);
        const uint32_t wx[4] = {vx.x, vx.y, vx.z, vx.w}, wy[4] = {vy.x, vy.y, vy.z, vy.w};
        terms<MODE>(wx, wy, C1, a);
    }
};

// Sum of the columns j of this lane with lo <= j < hi (0 <= lo, hi <= 4), fixed order (c0 + c1) + (c2 + c3).
__device__ __forceinline__ float col_sum(float c0, float c1, float c2, float c3, int lo, int hi) {
    const float v0 = (lo <= 0 && 0 < hi) ? c0 : 0.0f, v1 = (lo <= 1 && 1 < hi) ? c1 : 0.0f;
    const float v2 = (lo <= 2 && 2 < hi) ? c2 : 0.0f, v3 = (lo <= 3 && 3 < hi) ? c3 : 0.0f;
    return (v0 + v1) + (v2 + v3);
}
__device__ __forceinline__ float4 acc_cols(const Acc16& a, int lo, int hi) {
    float l0, l1, l2, l3, x0, x1, x2, x3, y0, y1, y2, y3;
    unpack2(a.L[0], l0, l1); unpack2(a.L[1], l2, l3);
    unpack2(a.X[0], x0, x1); unpack2(a.X[1], x2, x3);
    unpack2(a.Y[0], y0, y1); unpack2(a.Y[1], y2, y3);
    return make_float4(col_sum(l0, l1, l2, l3, lo, hi), col_sum(a.A[0], a.A[1], a.A[2], a.A[3], lo, hi),
                       col_sum(x0, x1, x2, x3, lo, hi), col_sum(y0, y1, y2, y3, lo, hi));
}

// All four columns: (c0 + c1) + (c2 + c3), the order of col_sum.
__device__ __forceinline__ float4 acc_cols(const Acc16& a) {
    float l0, l1, l2, l3, x0, x1, x2, x3, y0, y1, y2, y3;
    unpack2(a.L[0], l0, l1); unpack2(a.L[1], l2, l3);
    unpack2(a.X[0], x0, x1); unpack2(a.X[1], x2, x3);
    unpack2(a.Y[0], y0, y1); unpack2(a.Y[1], y2, y3);
    return make_float4((l0 + l1) + (l2 + l3), (a.A[0] + a.A[1]) + (a.A[2] + a.A[3]), (x0 + x1) + (x2 + x3),
                       (y0 + y1) + (y2 + y3));
}

// Position of a persistent CTA in its item sequence b, b + G, ...: three digits advanced by the decoded stride.
//   pair-major (batches of independent pairs)  item = (pair, uy, ux), ux fastest
//   pair-minor (the comparisons of a series)   item = (uy, ux, pair), pair fastest: the K comparisons of one item
//     location run on neighbouring CTAs at the same time, so an image that two comparisons share -- I_k+1 is the y of
//     comparison k and the x of comparison k+1, I_0 the x of every comparison in reference mode -- comes from DRAM once
//     and from L2 afterwards
struct AnyCursor {
    int d0, d1, d2;
    __device__ __forceinline__ void advance(const AnyCursor& s, int r0, int r1) {
        d0 += s.d0;
        const int c0 = d0 >= r0;
        d0 -= c0 ? r0 : 0;
        d1 += s.d1 + c0;
        const int c1 = d1 >= r1;
        d1 -= c1 ? r1 : 0;
        d2 += s.d2 + c1;
    }
};
__device__ __forceinline__ AnyCursor any_decode(int q, int r0, int r1) {
    AnyCursor c;
    const int t = q / r0;
    c.d0 = q - t * r0;
    c.d2 = t / r1;
    c.d1 = t - c.d2 * r1;
    return c;
}

template <int MODE, typename T>
__global__ void __launch_bounds__(kTmaThreads, 2)
any_kernel(const __grid_constant__ AnyParams p) {
    extern __shared__ unsigned char smem_dyn[];
    unsigned char* base = smem_dyn + ((1024u - (smem_addr(smem_dyn) & 1023u)) & 1023u);
    const int n_slots = p.n_slots;
    const uint32_t slot_bytes = (uint32_t)p.slot_bytes;
    const size_t part_off = (size_t)n_slots * slot_bytes;
    float4 (*part)[kWarpsPerCta][32] = reinterpret_cast<float4 (*)[kWarpsPerCta][32]>(base + part_off);
    const uint32_t boxes_u32 = smem_addr(base);
    const uint32_t full_u32 = smem_addr(base + part_off + kAnyPartBufs * kWarpsPerCta * 32 * sizeof(float4));
    const uint32_t empty_u32 = full_u32 + 8u * kAnyMaxSlots;
    const uint32_t pfull_u32 = empty_u32 + 8u * kAnyMaxSlots;
    const uint32_t pempty_u32 = pfull_u32 + 8u * kAnyPartBufs;

    if (threadIdx.x == 0) {
        for (int i = 0; i < n_slots; ++i) {
            mbar_init(full_u32 + 8u * i, 1u);
            mbar_init(empty_u32 + 8u * i, (uint32_t)kWarpsPerCta);
        }
        for (int i = 0; i < kAnyPartBufs; ++i) {
            mbar_init(pfull_u32 + 8u * i, (uint32_t)kWarpsPerCta);
            mbar_init(pempty_u32 + 8u * i, 1u);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();
    pdl_prologue();

    const int lane = threadIdx.x & 31;
    const int w = threadIdx.x >> 5;
    const int units_x = p.units_x, units_y = p.units_y;
    const int b = p.box_rows;
    const bool pm = p.pair_minor != 0;
    const int r0 = pm ? p.n_pairs : units_x, r1 = pm ? units_x : units_y, r2 = pm ? units_y : p.n_pairs;
    const AnyCursor stride = any_decode((int)gridDim.x, r0, r1);
#define IQA_ANY_PAIR(c) (pm ? (c).d0 : (c).d2)
#define IQA_ANY_UX(c) (pm ? (c).d1 : (c).d0)
#define IQA_ANY_UY(c) (pm ? (c).d2 : (c).d1)

    if (w == kWarpsPerCta) {
        // ================= producer: one elected lane issues every TMA load =================
        if (lane != 0) return;
        const uint32_t box_bytes = (uint32_t)(b * p.row_bytes);
        RingPos r{0, 0, n_slots, 0u};
        for (AnyCursor c = any_decode((int)blockIdx.x, r0, r1); c.d2 < r2; c.advance(stride, r0, r1)) {
            const AnyItem it = any_item(p, IQA_ANY_UX(c), IQA_ANY_UY(c));
            const int n_boxes = it.rv == p.ph ? p.boxes_per_item : (it.rv + b - 1) / b;
            for (int s = 0; s < n_boxes; ++s) {
                const AnyBox bx = any_box(s, b, it.rv);
                for (int j = 0; j < 2; ++j) {
                    const int img = 2 * IQA_ANY_PAIR(c) + j;
                    mbar_wait(empty_u32 + 8u * r.slot, r.phase ^ 1u);
                    mbar_expect_tx(full_u32 + 8u * r.slot, box_bytes);
                    tma_load_box(boxes_u32 + (uint32_t)r.slot * slot_bytes, p.maps + img, it.bc0, it.r0 + bx.o,
                                 full_u32 + 8u * r.slot);
                    r.advance();
                }
            }
        }
        return;
    }

    const bool split = p.px * p.py > 1;

    if (w == kWarpsPerCta + 1) {
        // ================= finaliser: (warp, lane) partials -> tiles -> Eqs. 1-2 (or pieces -> workspace) ========
        int buf = 0;
        uint32_t phase = 0u;
        const int n_it = p.kx * p.ky;                 // tiles per item (1 when split)
        const int gsz = p.fin_gsz;                    // lanes per tile
        const int groups = 32 / gsz;
        const int m = lane & (gsz - 1);
        const int nw = p.ky > 1 ? p.wpt : kWarpsPerCta;        // warps that share a tile: a power of two
        const int log2_nw = 31 - __clz(nw);
        const uint64_t pol = policy_evict_last();
        const int t_lane = lane / gsz;                // this lane's tile of the first round (the only one when gsz > 1)
        const int jy_lane = t_lane / p.kx, jx_lane = t_lane - jy_lane * p.kx;
        for (AnyCursor c = any_decode((int)blockIdx.x, r0, r1); c.d2 < r2; c.advance(stride, r0, r1)) {
            const AnyItem it = any_item(p, IQA_ANY_UX(c), IQA_ANY_UY(c));
            mbar_wait(pfull_u32 + 8u * buf, phase);
            for (int t0 = 0; t0 < n_it; t0 += groups) {
                const int t = t0 + t_lane;
                const bool active = t < n_it;
                int jy = jy_lane, jx = jx_lane;
                if (t0 > 0) { jy = t / p.kx; jx = t - jy * p.kx; }
                if (!active) jy = jx = 0;
                // lanes whose FIRST valid column lies in tile column jx (the columns a lane holds of the next tile
                // were moved one lane up by the consumers); the item's column c is box column c + s
                const int cl = p.cpl_log2, cr = (1 << cl) - 1;         // a lane owns 4 or 8 box columns
                const int la = (split || jx == 0) ? it.s >> cl : (jx * p.N_T + it.s + cr) >> cl;
                const int lb = split ? (it.cv + it.s + cr) >> cl : ((jx + 1) * p.N_T + it.s + cr) >> cl;
                const int w0 = p.ky > 1 ? jy * p.wpt : 0;
                float4 s = make_float4(0.f, 0.f, 0.f, 0.f);
                if (active) {
                    // the tile's entries are part[buf][w0 .. w0 + nw)[la .. lb): the gsz lanes of the tile's group
                    // split them without a division (nw and gsz are powers of two), each in a fixed order
                    if (gsz >= nw) {                 // gsz / nw lanes per warp row
                        const float4* row = part[buf][w0 + (m & (nw - 1))];
                        for (int l = la + (m >> log2_nw); l < lb; l += gsz >> log2_nw) {
                            const float4 u = row[l];
                            s.x += u.x; s.y += u.y; s.z += u.z; s.w += u.w;
                        }
                    } else {                         // several warp rows per lane
                        for (int ew = m; ew < nw; ew += gsz)
                            for (int l = la; l < lb; ++l) {
                                const float4 u = part[buf][w0 + ew][l];
                                s.x += u.x; s.y += u.y; s.z += u.z; s.w += u.w;
                            }
                    }
                }
                for (int o = gsz >> 1; o > 0; o >>= 1) {
                    s.x += __shfl_xor_sync(0xffffffffu, s.x, o);
                    s.y += __shfl_xor_sync(0xffffffffu, s.y, o);
                    s.z += __shfl_xor_sync(0xffffffffu, s.z, o);
                    s.w += __shfl_xor_sync(0xffffffffu, s.w, o);
                }
                const int tx = it.tx0 + jx, ty = it.ty0 + jy;
                if (active && m == 0 && (split || (tx < p.ntx && ty < p.nty))) {
                    const size_t tile = (size_t)IQA_ANY_PAIR(c) * p.n_tiles + (size_t)ty * p.ntx + tx;
                    if (!split) finalise_tile(p, tile, s, pol);
                    else p.ws[(tile * p.py + it.iy) * p.px + it.ix] = s;
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(pempty_u32 + 8u * buf);
            if (++buf == kAnyPartBufs) { buf = 0; phase ^= 1u; }
        }
        return;
    }

    // ================= consumer warps =================
    const float C1 = p.C1;
    const int row_bytes = p.row_bytes;
    // this warp's rows inside a box
    int row_lo, row_hi;
    if (p.ky > 1) {
        const int jy = w / p.wpt, q = w - jy * p.wpt;
        row_lo = jy * p.N_T + q * p.rpw;
        row_hi = min(row_lo + p.rpw, (jy + 1) * p.N_T);
    } else {
        row_lo = w * p.rpw;
        row_hi = min(b, row_lo + p.rpw);
    }
    // Whole tiles per item (N_T <= 112): every item has pw columns and ph rows; when the column offset s is the same
    // for all of them as well (`fixed`), nothing about an item has to be computed in this loop.
    const bool fixed = !split && p.const_s;
    // this lane's box columns 4 lane .. 4 lane + 3 are the item's columns 4 lane - s ..: [j_lo, j_end) of them lie
    // inside the item, and from j_cb on they belong to the tile after the one of the first (whole tiles only)
    const bool straddle = !split && (((p.N_T & 3) != 0) || !p.const_s || (p.shift & 3) != 0);
    int j_lo = 0, j_cb = 4, j_end = 4;
    auto lane_columns = [&](int s, int cv) {
        const int c = 4 * lane - s;                            // item column of j = 0
        j_lo = max(0, min(4, -c));
        j_end = max(0, min(4, cv - c));
        // tile of the first valid column: (c + j_lo) / N_T by multiplication (columns < 256, exact)
        const int t = (int)__umulhi((unsigned)max(c + j_lo, 0), p.nt_magic);
        j_cb = split ? 4 : max(0, min(4, (t + 1) * p.N_T - c));
    };
    if (fixed) lane_columns(p.shift, p.pw);
    // every lane holds either four columns of ONE tile or none of the item: nothing to mask (lanes outside the item
    // are never read by the finaliser)
    const bool wide = p.cpl_log2 == 3;                         // eight columns per lane (host: fixed, N_T % 8 == 0, s == 0)
    const bool whole_lanes = wide || (fixed && (p.N_T & 3) == 0 && (p.shift & 3) == 0);
    // lanes past the box re-read its last chunk (their columns are masked at the end / never read by the finaliser)
    const int lane_bytes = Pixel4<T>::kBytes << (p.cpl_log2 - 2);
    const unsigned char* my_base = base + min(lane * lane_bytes, row_bytes - lane_bytes);
    const int boxes_full = p.boxes_per_item;                   // boxes of an item with all ph rows
    int buf = 0;
    uint32_t part_phase = 0u;
    RingPos cy{0, 0, n_slots, 0u};
    Acc16 acc;
    for (AnyCursor c = any_decode((int)blockIdx.x, r0, r1); c.d2 < r2; c.advance(stride, r0, r1)) {
        int rv = p.ph;
        if (!fixed) {
            const AnyItem it = any_item(p, IQA_ANY_UX(c), IQA_ANY_UY(c));
            rv = it.rv;
            lane_columns(it.s, it.cv);
        }
        const int n_boxes = rv == p.ph ? boxes_full : (rv + b - 1) / b;
        acc.clear();
        for (int s = 0; s < n_boxes; ++s) {
            const AnyBox bx = any_box(s, b, rv);
            const int xs = cy.slot; const uint32_t xp = cy.phase; cy.advance();
            const int ys = cy.slot; const uint32_t yp = cy.phase; cy.advance();
            mbar_wait(full_u32 + 8u * xs, xp);
            mbar_wait(full_u32 + 8u * ys, yp);
            const int ra = max(row_lo, bx.lo);
            int nr = min(row_hi, bx.hi) - ra;
            const unsigned char* xr = my_base + (size_t)xs * slot_bytes + (size_t)ra * row_bytes;
            const unsigned char* yr = my_base + (size_t)ys * slot_bytes + (size_t)ra * row_bytes;
            if (!wide) {
#pragma unroll 1
                for (; nr >= 4; nr -= 4) {
#pragma unroll
                    for (int k = 0; k < 4; ++k) Pixel4<T>::template row<MODE>(xr + k * row_bytes, yr + k * row_bytes, C1, acc);
                    xr += 4 * row_bytes;
                    yr += 4 * row_bytes;
                }
                if (nr >= 2) {
                    Pixel4<T>::template row<MODE>(xr, yr, C1, acc);
                    Pixel4<T>::template row<MODE>(xr + row_bytes, yr + row_bytes, C1, acc);
                    xr += 2 * row_bytes;
                    yr += 2 * row_bytes;
                    nr -= 2;
                }
                if (nr >= 1) Pixel4<T>::template row<MODE>(xr, yr, C1, acc);
            } else {                                               // columns j and j + 4 of the lane share accumulator j
                constexpr int kHalf = Pixel4<T>::kBytes;
#pragma unroll 1
                for (; nr >= 4; nr -= 4) {                         // four rows at a time: uint8 +3.5 %, int16 +1.7 %
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        Pixel4<T>::template row<MODE>(xr + k * row_bytes, yr + k * row_bytes, C1, acc);
                        Pixel4<T>::template row<MODE>(xr + k * row_bytes + kHalf, yr + k * row_bytes + kHalf, C1, acc);
                    }
                    xr += 4 * row_bytes;
                    yr += 4 * row_bytes;
                }
#pragma unroll 1
                for (; nr >= 2; nr -= 2) {
                    Pixel4<T>::template row<MODE>(xr, yr, C1, acc);
                    Pixel4<T>::template row<MODE>(xr + kHalf, yr + kHalf, C1, acc);
                    Pixel4<T>::template row<MODE>(xr + row_bytes, yr + row_bytes, C1, acc);
                    Pixel4<T>::template row<MODE>(xr + row_bytes + kHalf, yr + row_bytes + kHalf, C1, acc);
                    xr += 2 * row_bytes;
                    yr += 2 * row_bytes;
                }
                if (nr >= 1) {
                    Pixel4<T>::template row<MODE>(xr, yr, C1, acc);
                    Pixel4<T>::template row<MODE>(xr + kHalf, yr + kHalf, C1, acc);
                }
            }
            __syncwarp();
            if (lane == 0) { mbar_arrive(empty_u32 + 8u * xs); mbar_arrive(empty_u32 + 8u * ys); }
        }
        // lane -> (warp, lane) partial of the tile of its first valid column
        float4 v = whole_lanes ? acc_cols(acc) : acc_cols(acc, j_lo, min(j_cb, j_end));
        if (straddle) {
            const float4 h = acc_cols(acc, max(j_cb, j_lo), j_end);    // columns of the NEXT tile: one lane up
            const float hx = __shfl_up_sync(0xffffffffu, h.x, 1), hy = __shfl_up_sync(0xffffffffu, h.y, 1);
            const float hz = __shfl_up_sync(0xffffffffu, h.z, 1), hw = __shfl_up_sync(0xffffffffu, h.w, 1);
            if (lane > 0) { v.x += hx; v.y += hy; v.z += hz; v.w += hw; }
        }
        mbar_wait(pempty_u32 + 8u * buf, part_phase ^ 1u);     // part[buf] of kAnyPartBufs items ago has been read
        part[buf][w][lane] = v;
        __syncwarp();
        if (lane == 0) mbar_arrive(pfull_u32 + 8u * buf);
        if (++buf == kAnyPartBufs) { buf = 0; part_phase ^= 1u; }
    }
}

#undef IQA_ANY_PAIR
#undef IQA_ANY_UX
#undef IQA_ANY_UY

}  // namespace iqa
