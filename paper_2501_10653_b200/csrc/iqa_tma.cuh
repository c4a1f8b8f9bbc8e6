// =============================================================================
// iqa_tma.cuh -- the TMA-fed persistent sm_100a kernel for tile-wise LISI / augLISI over
// image PAIRS and over TIME SERIES (S1-S4 of SURVEY.md 8(a); Eqs. 1-2; clamp
// PAPER.md:27; series: SURVEY.md 8(f)-2).
//
// Data movement is done by the Tensor Memory Accelerator: one elected thread of a producer
// warp issues cp.async.bulk.tensor.2d (SASS UTMALDG) for BOXES of 128 columns x 8 RPW rows
// (RPW = 4: 32 rows, 16 KiB) straight into shared memory; completion is signalled on an mbarrier per box
// ("full"), the eight consumer warps give a box back through a second mbarrier ("empty").
// Against a per-thread cp.async ring (the first version of this kernel, round 1)
// this removes every address computation and 8 LDGSTS per thread and stage from the instruction
// stream (that kernel spent ~19.5 instructions per pixel pair, ~10.5 of them arithmetic), which is what
// the time-series modes need: they halve the HBM bytes per comparison, so the instruction
// issue rate, not HBM, would otherwise bound them.  Rows / columns outside the image are
// zero-filled by the TMA unit, and zeros add exact zeros to all four sums.
//
// The per-pixel arithmetic uses the packed fp32 pair instructions of sm_100
// (add/sub/fma.rn.f32x2 -> FADD2 / FFMA2): the same roundings as the scalar form, half the
// issue slots for s = x + y, d = x - y, L += s * r, X += x, Y += y.
//
// Work decomposition
//   group     a set of M images compared with one another: M = 2 for an image pair
//             (x, y); a time series of M snapshots gives K = M - 1 comparisons
//               kPairs        (x, y) = (I_0, I_1)
//               kReference    (x, y) = (I_0, I_k+1)    k = 0 .. M-2
//               kConsecutive  (x, y) = (I_k, I_k+1)
//   item      128 columns x R rows of a group (R = S box heights; 32-row boxes: S = 1 for N_T <= 32, else 2); items
//             are numbered group-major, then row-major over the image; CTA b takes items b,
//             b+G, b+2G, ... (persistent grid).  For an item ALL comparisons of the group are
//             computed before the next item, so in the series modes the x box of a comparison
//             is still in shared memory: every image is read from HBM once per group, i.e.
//             4 (K+1)/K bytes per pixel and comparison instead of 8.
//   box order kPairs: stage-major  x(s0) y(s0) x(s1) y(s1)      -- ring of kNumBoxes boxes
//             kConsecutive: image-major I_0(s0..) I_1(s0..) ... -- ring; box q is the y of one
//                           comparison and, S boxes later, the x of the next
//             kReference: I_0's S boxes live in S dedicated slots for the whole item, the
//                           snapshots stream through a ring of kNumBoxes - S boxes
//   consume   warp w owns rows RPW w .. RPW w + RPW - 1 of a box, lane l the columns 4l..4l+3: conflict-free
//             LDS.128, 16 fp32 accumulators per lane
//   reduce    per item and comparison: lane -> warp (segmented reduce-scatter butterfly) ->
//             part[buf][warp][segment] in shared memory, handed through an mbarrier to a tenth
//             FINALISER warp, which combines the warps of a tile in warp order and applies Eq. 1 /
//             Eq. 2 (or writes the piece's partial sums to the workspace: tiles larger than an
//             item).  The consumer warps never meet at a CTA barrier.
// No floating-point atomics: results are bit-reproducible and do not depend on the grid size.
// =============================================================================
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "iqa_kernels.cuh"

namespace iqa {

constexpr int kMaxImages = 128;                // tensor maps per launch (kernel parameter space: 16 KiB of the 32 KiB limit)
// Box geometry and ring size are template parameters of the kernel:
//   RPW  rows per consumer warp and box (box = 8 RPW rows x 128 columns: 16 KiB for RPW = 4)
//   NB   box slots per CTA (NB boxes of shared memory; 2 CTAs per SM)
constexpr int kTmaThreads = kCtaThreads + 64;  // + the producer warp + the finaliser warp
constexpr int kPartBufs = 4;                   // per-warp partial sums in flight between consumers and finaliser

enum : int { kPairs = 0, kReference = 1, kConsecutive = 2 };

struct TmaParams {
    CUtensorMap maps[kMaxImages];   // image i of group g is maps[g * M + i]; box 128 x 8 RPW, OOB -> 0
    int n_groups;
    int M;               // images per group (2 for pairs)
    int W, H;            // image width and height in pixels (the square API passes N, N)
    int log2_nt;         // log2(N_T), N_T a power of two >= 8
    int ntx;             // tiles per row: ceil(W / N_T)
    int n_tiles;         // ntx * ceil(H / N_T)
    int units_x;         // items across: ceil(W / 128), or the full tile grid when tiles are split
    int units_y;         // items down:   ceil(H / R),   or the full tile grid when tiles are split
    int S;               // boxes (stages) per item and image: R = S * box rows
    float C1, C2, C, D;
    float* lisi;         // [n_groups * (M-1) * n_tiles] or nullptr; comparison c = g (M-1) + k
    float* auglisi;
    float* sum_x;
    float* sum_y;
    float* lisi_num;
    float* aug_num;
    float4* ws;          // split tiles: [comparison][tile][pieces_y][pieces_x] partial (L, A, X, Y)
    int pieces_x, pieces_y;
};

constexpr size_t tma_smem_bytes(int NB, int RPW) {
    return 1024 /* alignment slack */ + (size_t)NB * (kWarpsPerCta * RPW * kUnitCols * 4) +
           kPartBufs * kWarpsPerCta * 16 * sizeof(float4) + (2 * NB + 2 * kPartBufs) * sizeof(uint64_t);
}

// ---- mbarrier / TMA primitives (PTX ISA: mbarrier, cp.async.bulk.tensor) --------------------
__device__ __forceinline__ uint32_t smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar), "r"(parity), "r"(0x989680u) /* suspend-time hint: sleep in hardware, not in a spin */
        : "memory");
}
// One box (128 columns x 8 RPW rows, fixed by the tensor map) of the image described by `map`, top-left (col, row), -> dst.
__device__ __forceinline__ void tma_load_box(uint32_t dst, const CUtensorMap* map, int col, int row, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
        ::"r"(dst), "l"(map), "r"(col), "r"(row), "r"(bar) : "memory");
}

// ---- packed fp32 pairs ---------------------------------------------------------------------
__device__ __forceinline__ uint64_t pack2(float lo, float hi) {
    uint64_t r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(uint64_t v, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ uint64_t add2(uint64_t a, uint64_t b) {
    uint64_t r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ uint64_t sub2(uint64_t a, uint64_t b) {
    uint64_t r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ uint64_t fma2(uint64_t a, uint64_t b, uint64_t c) {
    uint64_t r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}

// 16 accumulators of one lane: columns (0,1) and (2,3) packed for L, X, Y; A scalar (its
// multiplicand |d| needs the absolute-value operand modifier, which the packed form lacks).
struct Acc16 {
    uint64_t L[2], X[2], Y[2];
    float A[4];
    __device__ __forceinline__ void clear() {
        L[0] = L[1] = X[0] = X[1] = Y[0] = Y[1] = 0ull;
        A[0] = A[1] = A[2] = A[3] = 0.f;
    }
};

// S1 + S2 for two horizontally adjacent pixel pairs: clamp, then the Eq. 1 / Eq. 2 terms
// with the roundings of pixel_terms() (iqa_kernels.cuh).
// CLAMP = false: the caller has clamped already (or the pixel type has no negative values).
template <int MODE, bool CLAMP = true>
__device__ __forceinline__ void pixel_terms2(float x0, float x1, float y0, float y1, float C1,
                                             uint64_t& aL, float& aA0, float& aA1, uint64_t& aX, uint64_t& aY) {
    const uint64_t xc = CLAMP ? pack2(fmaxf(x0, 0.0f), fmaxf(x1, 0.0f)) : pack2(x0, x1);     // NaN -> 0, negatives -> 0
    const uint64_t yc = CLAMP ? pack2(fmaxf(y0, 0.0f), fmaxf(y1, 0.0f)) : pack2(y0, y1);
    const uint64_t s = add2(xc, yc);            // |x + y| = x + y after the clamp
    const uint64_t d = sub2(xc, yc);
    float d0, d1;
    unpack2(d, d0, d1);
    if (MODE & kModeLisi) {
        const float r0 = rcp_approx(fabsf(d0) + C1);
        const float r1 = rcp_approx(fabsf(d1) + C1);
        aL = fma2(s, pack2(r0, r1), aL);
    }
    if (MODE & kModeAug) {
        float s0, s1;
        unpack2(s, s0, s1);
        aA0 = fmaf(s0, fabsf(d0), aA0);
        aA1 = fmaf(s1, fabsf(d1), aA1);
    }
    aX = add2(aX, xc);
    aY = add2(aY, yc);
}

// One box pair (x box, y box) -> this thread's RPW rows x 4 columns into the accumulators.
template <int MODE, int kRowsPerWarp>
__device__ __forceinline__ void consume_boxes(const float* xs, const float* ys, float C1, Acc16& a) {
    float4 vx[kRowsPerWarp], vy[kRowsPerWarp];
#pragma unroll
    for (int k = 0; k < kRowsPerWarp; ++k) {
        vx[k] = *reinterpret_cast<const float4*>(xs + k * kUnitCols);
        vy[k] = *reinterpret_cast<const float4*>(ys + k * kUnitCols);
    }
#pragma unroll
    for (int k = 0; k < kRowsPerWarp; ++k) {
        pixel_terms2<MODE>(vx[k].x, vx[k].y, vy[k].x, vy[k].y, C1, a.L[0], a.A[0], a.A[1], a.X[0], a.Y[0]);
        pixel_terms2<MODE>(vx[k].z, vx[k].w, vy[k].z, vy[k].w, C1, a.L[1], a.A[2], a.A[3], a.X[1], a.Y[1]);
    }
}

// Position in a ring of box slots [first, first + n): slot index and the parity of the phase
// the CONSUMER waits for on the slot's full barrier (the producer waits for parity ^ 1 on empty).
struct RingPos {
    int slot, first, n;
    uint32_t phase;
    __device__ __forceinline__ void advance() {
        if (++slot == first + n) { slot = first; phase ^= 1u; }
    }
};

// Consumer side of the per-item reduction: lane (4 columns -> 1) -> warp.  The g = min(32, N_T/4)
// lanes of a tile row are combined with a reduce-scatter butterfly: at the first two levels every
// lane gives away half of what it holds (4 -> 2 -> 1 values), so a segment of 16 lanes costs 5
// shuffles + 5 adds instead of the 16 + 16 of an all-reduce.  Afterwards lane (seg << log2_g) + c'
// holds component c of segment seg (c' = bit-reversed c: L at +0, X at +1, A at +2, Y at +3; for
// g = 2: lane +0 holds (L, A), lane +1 holds (X, Y)) and stores it into part[w][seg].
__device__ __forceinline__ void warp_partials(const Acc16& a, float4* part_w /* part[w] */, int log2_g, int lane) {
    float lo, hi;
    unpack2(add2(a.L[0], a.L[1]), lo, hi); const float vL = lo + hi;          // (c0 + c2) + (c1 + c3)
    const float vA = (a.A[0] + a.A[2]) + (a.A[1] + a.A[3]);
    unpack2(add2(a.X[0], a.X[1]), lo, hi); const float vX = lo + hi;
    unpack2(add2(a.Y[0], a.Y[1]), lo, hi); const float vY = lo + hi;
    const bool b0 = lane & 1, b1 = lane & 2;
    // level 1 (xor 1): even lanes keep (L, A), odd lanes keep (X, Y)
    float k0 = b0 ? vX : vL, k1 = b0 ? vY : vA;
    k0 += __shfl_xor_sync(0xffffffffu, b0 ? vL : vX, 1);
    k1 += __shfl_xor_sync(0xffffffffu, b0 ? vA : vY, 1);
    float* dst = reinterpret_cast<float*>(part_w + (lane >> log2_g));
    if (log2_g == 1) {                                     // N_T = 8: two lanes per segment
        *reinterpret_cast<float2*>(dst + (b0 ? 2 : 0)) = make_float2(k0, k1);   // (L, A) or (X, Y)
        return;
    }
    // level 2 (xor 2): lanes with bit 1 clear keep the first value, the others the second
    float k = b1 ? k1 : k0;
    k += __shfl_xor_sync(0xffffffffu, b1 ? k0 : k1, 2);
    for (int o = 4; o < (1 << log2_g); o <<= 1) k += __shfl_xor_sync(0xffffffffu, k, o);
    if ((lane & ((1 << log2_g) - 1)) < 4) dst[(b0 ? 2 : 0) + (b1 ? 1 : 0)] = k;   // float4 order (L, A, X, Y)
}

// Finaliser side: combine the warps of every tile of the item in warp order, then Eq. 1 / Eq. 2
// (or the piece's partial sums to the workspace).  Executed by one warp; lanes take tiles.
template <int kRowsPerWarp>
__device__ __forceinline__ void finalise_item(const TmaParams& p, const float4 (*part)[16], int cmp, int uy, int ux,
                                              int lane) {
    constexpr int kBoxRows = kWarpsPerCta * kRowsPerWarp;
    const int log2_nt = p.log2_nt;
    const int log2_g = min(log2_nt - 2, 5);                       // g = min(32, N_T / 4) lanes per tile row
    const int log2_tpw = 5 - log2_g;                              // tile segments per warp row
    const int wpt = min(kWarpsPerCta, (1 << log2_nt) / kRowsPerWarp);   // warps per tile row-band of a box
    const int n_ty = kWarpsPerCta / wpt;                          // tile rows per item (> 1 only when N_T < box rows)
    const int R = p.S * kBoxRows;
    for (int t = lane; t < (n_ty << log2_tpw); t += 32) {
        const int jy = t >> log2_tpw;
        const int jx = t & ((1 << log2_tpw) - 1);
        const int c0 = ux * kUnitCols + (jx << log2_nt);          // jx == 0 when N_T >= 128
        const int r0 = uy * R + (jy << log2_nt);                  // jy == 0 unless N_T < box rows
        // split tiles: the items cover the whole tile grid and EVERY piece is written (a piece outside the
        // image is all zeros); otherwise tiles that start outside the image do not exist
        if (p.ws != nullptr || (c0 < p.W && r0 < p.H)) {
            float4 s = part[jy * wpt][jx];
            for (int k = 1; k < wpt; ++k) {
                const float4 u = part[jy * wpt + k][jx];
                s.x += u.x; s.y += u.y; s.z += u.z; s.w += u.w;
            }
            const size_t tile = (size_t)cmp * p.n_tiles + (size_t)(r0 >> log2_nt) * p.ntx + (c0 >> log2_nt);
            if (p.ws == nullptr) {
                finalise_tile(p, tile, s);                        // S4: Eq. 1 / Eq. 2
            } else {                                              // split tile: piece -> workspace
                const int pxi = ux & (p.pieces_x - 1);
                const int pyi = uy & (p.pieces_y - 1);
                p.ws[(tile * p.pieces_y + pyi) * p.pieces_x + pxi] = s;
            }
        }
    }
}

template <int MODE, int SERIES, int kNumBoxes, int kRowsPerWarp>
__global__ void __launch_bounds__(kTmaThreads, 2)
tma_kernel(const __grid_constant__ TmaParams p) {
    constexpr int kBoxRows = kWarpsPerCta * kRowsPerWarp;
    constexpr int kBoxFloats = kBoxRows * kUnitCols;
    constexpr uint32_t kBoxBytes = kBoxFloats * 4u;
    extern __shared__ unsigned char smem_dyn[];
    // 1 KiB-aligned start of the boxes (pointer arithmetic on smem_dyn keeps the shared address space)
    unsigned char* base = smem_dyn + ((1024u - (smem_addr(smem_dyn) & 1023u)) & 1023u);
    float* boxes = reinterpret_cast<float*>(base);
    constexpr size_t kPartOff = (size_t)kNumBoxes * kBoxBytes;
    constexpr size_t kBarOff = kPartOff + kPartBufs * kWarpsPerCta * 16 * sizeof(float4);
    float4 (*part)[kWarpsPerCta][16] = reinterpret_cast<float4 (*)[kWarpsPerCta][16]>(base + kPartOff);
    const uint32_t boxes_u32 = smem_addr(boxes);
    const uint32_t full_u32 = smem_addr(base + kBarOff);          // full[slot]  at full_u32  + 8 slot
    const uint32_t empty_u32 = full_u32 + 8u * kNumBoxes;         // empty[slot] at empty_u32 + 8 slot
    const uint32_t pfull_u32 = empty_u32 + 8u * kNumBoxes;        // part_full[buf]: 8 consumer warps -> finaliser
    const uint32_t pempty_u32 = pfull_u32 + 8u * kPartBufs;       // part_empty[buf]: finaliser -> consumers

    if (threadIdx.x == 0) {
        for (int i = 0; i < kNumBoxes; ++i) {
            mbar_init(full_u32 + 8u * i, 1u);                     // the producer's expect_tx arrival
            mbar_init(empty_u32 + 8u * i, (uint32_t)kWarpsPerCta); // one arrival per consumer warp
        }
        for (int i = 0; i < kPartBufs; ++i) {
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
    const int S = p.S, M = p.M;
    const int units_x = p.units_x, units_y = p.units_y;
    const int R = S * kBoxRows;
    const ItemCursor stride = decode_item((int)gridDim.x, units_x, units_y);
    const int ring_first = SERIES == kReference ? S : 0;          // kReference: slots [0, S) hold I_0's boxes

    if (w == kWarpsPerCta) {
        // ================= producer warp: one elected lane issues every TMA load =================
        if (lane != 0) return;
        RingPos r{ring_first, ring_first, kNumBoxes - ring_first, 0u};
        uint32_t ref_phase = 0u;
        auto fill = [&](int slot, uint32_t phase, const CUtensorMap* map, int col, int row) {
            mbar_wait(empty_u32 + 8u * slot, phase ^ 1u);         // the slot's previous box has been consumed
            mbar_expect_tx(full_u32 + 8u * slot, kBoxBytes);
            tma_load_box(boxes_u32 + (uint32_t)slot * kBoxBytes, map, col, row, full_u32 + 8u * slot);
        };
        for (ItemCursor c = decode_item((int)blockIdx.x, units_x, units_y); c.pair < p.n_groups;
             c.advance(stride, units_x, units_y)) {
            const CUtensorMap* maps = p.maps + c.pair * M;
            const int col = c.ux * kUnitCols, row = c.uy * R;
            if (SERIES == kPairs) {
                for (int s = 0; s < S; ++s)
                    for (int j = 0; j < 2; ++j) { fill(r.slot, r.phase, maps + j, col, row + s * kBoxRows); r.advance(); }
            } else {
                if (SERIES == kReference) {
                    for (int s = 0; s < S; ++s) fill(s, ref_phase, maps, col, row + s * kBoxRows);
                    ref_phase ^= 1u;
                }
                for (int j = SERIES == kReference ? 1 : 0; j < M; ++j)
                    for (int s = 0; s < S; ++s) { fill(r.slot, r.phase, maps + j, col, row + s * kBoxRows); r.advance(); }
            }
        }
        return;
    }

    if (w == kWarpsPerCta + 1) {
        // ================= finaliser warp: per item and comparison, warps -> tiles -> Eqs. 1-2 =================
        int buf = 0;
        uint32_t phase = 0u;
        for (ItemCursor c = decode_item((int)blockIdx.x, units_x, units_y); c.pair < p.n_groups;
             c.advance(stride, units_x, units_y)) {
            for (int j = 1; j < M; ++j) {
                mbar_wait(pfull_u32 + 8u * buf, phase);           // the eight warps' partial sums are in part[buf]
                finalise_item<kRowsPerWarp>(p, part[buf], c.pair * (M - 1) + (j - 1), c.uy, c.ux, lane);
                __syncwarp();
                if (lane == 0) mbar_arrive(pempty_u32 + 8u * buf);
                if (++buf == kPartBufs) { buf = 0; phase ^= 1u; }
            }
        }
        return;
    }

    // ================= consumer warps =================
    const float C1 = p.C1;
    const int log2_g = min(p.log2_nt - 2, 5);
    const int my_off = (w * kRowsPerWarp) * kUnitCols + lane * 4;   // this thread's RPW x 4 patch inside a box
    const float* my_boxes = boxes + my_off;
    auto wait_full = [&](int slot, uint32_t phase) { mbar_wait(full_u32 + 8u * slot, phase); };
    auto release = [&](int slot) {                                  // after __syncwarp(): every lane has read the box
        if (lane == 0) mbar_arrive(empty_u32 + 8u * slot);
    };
    int buf = 0;
    uint32_t part_phase = 0u;
    auto hand_over = [&](const Acc16& acc) {                        // this warp's partial sums -> finaliser warp
        mbar_wait(pempty_u32 + 8u * buf, part_phase ^ 1u);          // part[buf] of kPartBufs reductions ago has been read
        warp_partials(acc, part[buf][w], log2_g, lane);
        __syncwarp();
        if (lane == 0) mbar_arrive(pfull_u32 + 8u * buf);
        if (++buf == kPartBufs) { buf = 0; part_phase ^= 1u; }
    };
    RingPos cy{ring_first, ring_first, kNumBoxes - ring_first, 0u};
    RingPos cx = cy;                                                // kConsecutive: trails cy by S boxes
    if (SERIES == kConsecutive)
        for (int s = 0; s < S; ++s) cy.advance();
    uint32_t ref_phase = 0u;
    Acc16 acc;
    for (ItemCursor c = decode_item((int)blockIdx.x, units_x, units_y); c.pair < p.n_groups;
         c.advance(stride, units_x, units_y)) {
        if (SERIES == kPairs) {
            acc.clear();
            for (int s = 0; s < S; ++s) {
                const int xs = cy.slot; const uint32_t xp = cy.phase; cy.advance();
                const int ys = cy.slot; const uint32_t yp = cy.phase; cy.advance();
                wait_full(xs, xp);
                wait_full(ys, yp);
                consume_boxes<MODE, kRowsPerWarp>(my_boxes + xs * kBoxFloats, my_boxes + ys * kBoxFloats, C1, acc);
                __syncwarp();
                release(xs);
                release(ys);
            }
            hand_over(acc);
        } else {
            for (int j = 1; j < M; ++j) {
                acc.clear();
                for (int s = 0; s < S; ++s) {
                    const int xs = SERIES == kReference ? s : cx.slot;
                    if (j == 1) wait_full(xs, SERIES == kReference ? ref_phase : cx.phase);
                    wait_full(cy.slot, cy.phase);
                    consume_boxes<MODE, kRowsPerWarp>(my_boxes + xs * kBoxFloats, my_boxes + cy.slot * kBoxFloats, C1, acc);
                    __syncwarp();
                    if (SERIES == kReference) {
                        release(cy.slot);
                        if (j == M - 1) release(s);                 // I_0's box: free for the next item
                    } else {
                        release(cx.slot);                           // the x box; the y box is the next x
                        if (j == M - 1) release(cy.slot);
                        cx.advance();
                    }
                    cy.advance();
                }
                hand_over(acc);
            }
            if (SERIES == kReference) ref_phase ^= 1u;
            if (SERIES == kConsecutive)
                for (int s = 0; s < S; ++s) {
                    cx.advance();           // skip the last image's boxes (already released)
                    cy.advance();           // the next item's I_0 boxes are its first x boxes
                }
        }
    }
}

}  // namespace iqa
