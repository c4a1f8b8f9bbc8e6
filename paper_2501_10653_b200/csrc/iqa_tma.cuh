// =============================================================================
// iqa_tma.cuh -- the TMA-fed persistent sm_100a kernel for tile-wise LISI / augLISI over
// image PAIRS and over TIME SERIES (S1-S4 of SURVEY.md 8(a); Eqs. 1-2; clamp
// PAPER.md:27; series: SURVEY.md 8(f)-2).
//
// Data movement is done by the Tensor Memory Accelerator: one elected thread of a producer
// warp issues cp.async.bulk.tensor.2d (SASS UTMALDG) for BOXES of 128 columns x 32 rows
// (16 KiB) straight into shared memory; completion is signalled on an mbarrier per box
// ("full"), the eight consumer warps give a box back through a second mbarrier ("empty").
// Against the per-thread cp.async ring of iqa_stream.cuh this removes every address
// computation and 8 LDGSTS per thread and stage from the instruction stream (the cp.async
// kernel spends ~19.5 instructions per pixel pair, ~10.5 of them arithmetic), which is what
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
//   item      128 columns x R rows of a group (R = 32 S; S = 1 for N_T <= 32, else 2); items
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
//   consume   warp w owns rows 4w..4w+3 of a box, lane l the columns 4l..4l+3: conflict-free
//             LDS.128, 16 fp32 accumulators per lane
//   reduce    per item and comparison exactly as iqa_stream.cuh: lane -> segmented warp
//             butterfly -> shared-memory combine of the warps of a tile (fixed order) -> Eq. 1 /
//             Eq. 2, or the piece's partial sums to the workspace (tiles larger than an item)
// No floating-point atomics: results are bit-reproducible and do not depend on the grid size.
// =============================================================================
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "iqa_kernels.cuh"
#include "iqa_stream.cuh"     // ItemCursor, decode_item

namespace iqa {

constexpr int kMaxImages = 64;                 // tensor maps per launch (kernel parameter space: 8 KiB)
constexpr int kBoxRows = 32;                   // 8 consumer warps x 4 rows
constexpr int kRowsPerWarp = kBoxRows / kWarpsPerCta;
constexpr int kBoxFloats = kBoxRows * kUnitCols;
constexpr uint32_t kBoxBytes = kBoxFloats * 4u;
constexpr int kNumBoxes = 6;                   // 96 KiB of boxes per CTA, 2 CTAs per SM
constexpr int kTmaThreads = kCtaThreads + 32;  // + the producer warp
constexpr int kConsumerBarrier = 1;            // named barrier of the 256 consumer threads

enum : int { kPairs = 0, kReference = 1, kConsecutive = 2 };

struct TmaParams {
    CUtensorMap maps[kMaxImages];   // image i of group g is maps[g * M + i]; box 128 x 32, OOB -> 0
    int n_groups;
    int M;               // images per group (2 for pairs)
    int N;               // image side
    int log2_nt;         // log2(N_T), N_T a power of two >= 8
    int nt;              // tiles per side
    int n_tiles;         // nt * nt
    int units_x;         // items across: ceil(N / 128)
    int units_y;         // items down:   ceil(N / R)
    int S;               // boxes (stages) per item and image: R = 32 S
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

constexpr size_t tma_smem_bytes() {
    return 1024 /* alignment slack */ + (size_t)kNumBoxes * kBoxBytes + 2 * kWarpsPerCta * 16 * sizeof(float4) +
           2 * kNumBoxes * sizeof(uint64_t);
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
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
// One box: 128 columns x 32 rows of the image described by `map`, top-left (col, row), -> dst.
__device__ __forceinline__ void tma_load_box(uint32_t dst, const CUtensorMap* map, int col, int row, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
        ::"r"(dst), "l"(map), "r"(col), "r"(row), "r"(bar) : "memory");
}
__device__ __forceinline__ void consumer_barrier() {
    asm volatile("bar.sync %0, %1;" ::"n"(kConsumerBarrier), "n"(kCtaThreads) : "memory");
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
template <int MODE>
__device__ __forceinline__ void pixel_terms2(float x0, float x1, float y0, float y1, float C1,
                                             uint64_t& aL, float& aA0, float& aA1, uint64_t& aX, uint64_t& aY) {
    const uint64_t xc = pack2(fmaxf(x0, 0.0f), fmaxf(x1, 0.0f));     // NaN -> 0, negatives -> 0
    const uint64_t yc = pack2(fmaxf(y0, 0.0f), fmaxf(y1, 0.0f));
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

// One box pair (x box, y box) -> this thread's 4 rows x 4 columns into the accumulators.
template <int MODE>
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

// Per item and comparison: lane -> warp (segmented butterfly) -> CTA (shared memory, warp
// order) -> Eq. 1 / Eq. 2 or the workspace.  Called by the 256 consumer threads.
template <int MODE>
__device__ __forceinline__ void reduce_item(const TmaParams& p, const Acc16& a, float4 (*part)[16],
                                            int cmp, int uy, int ux, int lane, int w) {
    const int log2_nt = p.log2_nt;
    const int log2_g = min(log2_nt - 2, 5);                       // g = min(32, N_T / 4) lanes per tile row
    const int log2_tpw = 5 - log2_g;                              // tile segments per warp row
    const int wpt = min(kWarpsPerCta, (1 << log2_nt) / kRowsPerWarp);   // warps per tile row-band of a box
    const int n_ty = kWarpsPerCta / wpt;                          // tile rows per item (> 1 only when N_T < 32)
    const int R = p.S * kBoxRows;
    // lane: 4 columns -> 1   ((c0 + c2) + (c1 + c3))
    float4 v;
    float lo, hi;
    unpack2(add2(a.L[0], a.L[1]), lo, hi); v.x = lo + hi;
    v.y = (a.A[0] + a.A[2]) + (a.A[1] + a.A[3]);
    unpack2(add2(a.X[0], a.X[1]), lo, hi); v.z = lo + hi;
    unpack2(add2(a.Y[0], a.Y[1]), lo, hi); v.w = lo + hi;
    // warp: segmented butterfly over the g lanes that share a tile row
    for (int o = (1 << log2_g) >> 1; o > 0; o >>= 1) {
        if (MODE & kModeLisi) v.x += __shfl_xor_sync(0xffffffffu, v.x, o);
        if (MODE & kModeAug) v.y += __shfl_xor_sync(0xffffffffu, v.y, o);
        v.z += __shfl_xor_sync(0xffffffffu, v.z, o);
        v.w += __shfl_xor_sync(0xffffffffu, v.w, o);
    }
    if ((lane & ((1 << log2_g) - 1)) == 0) part[w][lane >> log2_g] = v;
    consumer_barrier();      // part[] of this buffer complete; the other buffer is rewritten only after the next barrier

    const int t = threadIdx.x;
    if (t < (n_ty << log2_tpw)) {
        const int jy = t >> log2_tpw;
        const int jx = t & ((1 << log2_tpw) - 1);
        const int c0 = ux * kUnitCols + (jx << log2_nt);          // jx == 0 when N_T >= 128
        const int r0 = uy * R + (jy << log2_nt);                  // jy == 0 unless N_T < 32
        if (c0 < p.N && r0 < p.N) {
            float4 s = part[jy * wpt][jx];
            for (int k = 1; k < wpt; ++k) {
                const float4 u = part[jy * wpt + k][jx];
                s.x += u.x; s.y += u.y; s.z += u.z; s.w += u.w;
            }
            const size_t tile = (size_t)cmp * p.n_tiles + (size_t)(r0 >> log2_nt) * p.nt + (c0 >> log2_nt);
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

template <int MODE, int SERIES>
__global__ void __launch_bounds__(kTmaThreads, 2)
tma_kernel(const __grid_constant__ TmaParams p) {
    extern __shared__ unsigned char smem_dyn[];
    // 1 KiB-aligned start of the boxes (pointer arithmetic on smem_dyn keeps the shared address space)
    unsigned char* base = smem_dyn + ((1024u - (smem_addr(smem_dyn) & 1023u)) & 1023u);
    float* boxes = reinterpret_cast<float*>(base);
    float4 (*part)[kWarpsPerCta][16] =
        reinterpret_cast<float4 (*)[kWarpsPerCta][16]>(base + (size_t)kNumBoxes * kBoxBytes);
    uint64_t* bars = reinterpret_cast<uint64_t*>(base + (size_t)kNumBoxes * kBoxBytes + 2 * kWarpsPerCta * 16 * sizeof(float4));
    const uint32_t boxes_u32 = smem_addr(boxes);
    const uint32_t full_u32 = smem_addr(bars);                    // full[slot]  at full_u32  + 8 slot
    const uint32_t empty_u32 = full_u32 + 8u * kNumBoxes;         // empty[slot] at empty_u32 + 8 slot

    if (threadIdx.x == 0) {
        for (int i = 0; i < kNumBoxes; ++i) {
            mbar_init(full_u32 + 8u * i, 1u);                     // the producer's expect_tx arrival
            mbar_init(empty_u32 + 8u * i, (uint32_t)kWarpsPerCta); // one arrival per consumer warp
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

    // ================= consumer warps =================
    const float C1 = p.C1;
    const int my_off = (w * kRowsPerWarp) * kUnitCols + lane * 4;   // this thread's 4 x 4 patch inside a box
    const float* my_boxes = boxes + my_off;
    auto wait_full = [&](int slot, uint32_t phase) { mbar_wait(full_u32 + 8u * slot, phase); };
    auto release = [&](int slot) {                                  // after __syncwarp(): every lane has read the box
        if (lane == 0) mbar_arrive(empty_u32 + 8u * slot);
    };
    RingPos cy{ring_first, ring_first, kNumBoxes - ring_first, 0u};
    RingPos cx = cy;                                                // kConsecutive: trails cy by S boxes
    if (SERIES == kConsecutive)
        for (int s = 0; s < S; ++s) cy.advance();
    uint32_t ref_phase = 0u;
    int buf = 0;
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
                consume_boxes<MODE>(my_boxes + xs * kBoxFloats, my_boxes + ys * kBoxFloats, C1, acc);
                __syncwarp();
                release(xs);
                release(ys);
            }
            reduce_item<MODE>(p, acc, part[buf], c.pair, c.uy, c.ux, lane, w);
            buf ^= 1;
        } else {
            for (int j = 1; j < M; ++j) {
                acc.clear();
                for (int s = 0; s < S; ++s) {
                    const int xs = SERIES == kReference ? s : cx.slot;
                    if (j == 1) wait_full(xs, SERIES == kReference ? ref_phase : cx.phase);
                    wait_full(cy.slot, cy.phase);
                    consume_boxes<MODE>(my_boxes + xs * kBoxFloats, my_boxes + cy.slot * kBoxFloats, C1, acc);
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
                reduce_item<MODE>(p, acc, part[buf], c.pair * (M - 1) + (j - 1), c.uy, c.ux, lane, w);
                buf ^= 1;
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
