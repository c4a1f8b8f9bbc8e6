// =============================================================================
// iqa_stream.cuh -- the persistent, cp.async-pipelined sm_100a kernel for tile-wise LISI /
// augLISI over a BATCH of image pairs (S1-S4 of SURVEY.md 8(a); Eqs. 1-2, PAPER.md:15-21;
// clamp PAPER.md:27).
//
// Why not the paper's design (one thread block per tile, shared-memory tree):
// a 64 x 64 tile is 32 KiB of input, far too little for a CTA to keep HBM3e busy, and the
// load -> reduce -> exit shape leaves the memory system idle during every CTA's ramp and
// tail.  Here the CTAs are persistent (grid = resident CTAs of the chip) and every thread
// runs a private ring of DEPTH shared-memory stages filled by 128-bit asynchronous copies
// (cp.async.cg global -> shared, L1 bypassed, L2 evict-first; SASS LDGSTS.E.BYPASS.128),
// so the loads of the next DEPTH-1 stages are in flight while the current one is reduced.
// A thread only ever reads the bytes it copied itself: cp.async.wait_group is the only
// synchronisation of the pipeline (no mbarrier, no producer warp, no CTA barrier).
//
//   item     128 columns x R rows of one pair (R = item_rows, a multiple of the stage height
//            8*K chosen on the host from N_T); items are numbered pair-major, then row-major
//            over the image (horizontally adjacent items run at the same time); CTA b takes
//            items b, b+G, b+2G, ...
//   stage    8*K rows of the item; warp w owns rows wK..wK+K-1 of the stage, lane l the
//            columns 4l..4l+3: K 16-byte copies per image and thread, 512 contiguous bytes
//            per warp and row; rows / columns outside the image are zero-filled by the copy
//            (src-size 0), so ragged edges add exact zeros
//   consume  conflict-free LDS.128, 16 fp32 accumulators per lane (chain length R/8)
//   reduce   at the end of the item, exactly as the strip kernel: lane -> segmented warp
//            butterfly over the min(32, N_T/4) lanes of a tile row -> shared-memory combine
//            of the warps of a tile (fixed order) -> Eq. 1 / Eq. 2, or (tiles larger than an
//            item) the piece's partial sums to the workspace for the finalise kernel
// No floating-point atomics: results are bit-reproducible and do not depend on the grid size.
// =============================================================================
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "iqa_kernels.cuh"

namespace iqa {

constexpr int kMaxBatch = 32;                 // pairs per launch (the pointer table lives in the kernel parameters)

struct BatchParams {
    const float* x[kMaxBatch];
    const float* y[kMaxBatch];
    int n_pairs;
    int N;               // image side
    int log2_nt;         // log2(N_T), N_T a power of two >= 8
    int nt;              // tiles per side
    int n_tiles;         // nt * nt
    int units_x;         // items across: ceil(N / 128)
    int units_y;         // items down:   ceil(N / item_rows)
    int item_rows;       // R: multiple of the stage height; a tile of side <= 64 sits inside one item
    int n_items;         // n_pairs * units_x * units_y
    float C1, C2, C, D;
    float* lisi;         // [n_pairs * n_tiles] or nullptr
    float* auglisi;
    float* sum_x;
    float* sum_y;
    float* lisi_num;
    float* aug_num;
    float4* ws;          // split tiles: [n_pairs * n_tiles][pieces_y][pieces_x] partial (L, A, X, Y)
    int pieces_x, pieces_y;
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ uint64_t policy_evict_first() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
// 16-byte asynchronous copy global -> shared, L1 bypassed (.cg), L2 evict-first (every pixel is
// read once).  src_bytes = 16 copies, src_bytes = 0 writes 16 zero bytes and reads nothing.
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, uint32_t src_bytes, uint64_t pol) {
#ifdef IQA_CP_ASYNC_L2_HINT
    asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2, %3;"
                 ::"r"(dst), "l"(src), "r"(src_bytes), "l"(pol) : "memory");
#else
    (void)pol;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
#endif
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int PENDING>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(PENDING) : "memory"); }

// Dynamic shared memory: [DEPTH][2 images][8*K rows][128] floats, then part[2][8][16] float4.
template <int K, int DEPTH>
constexpr size_t stream_smem_bytes() {
    return (size_t)DEPTH * 2 * (kWarpsPerCta * K) * kUnitCols * sizeof(float) + 2 * kWarpsPerCta * 16 * sizeof(float4);
}

// Position of one CTA in its item sequence b, b+G, b+2G, ... kept as (pair, uy, ux) and advanced
// by the decoded stride (no integer division in the loop).
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

template <int MODE, int K, int DEPTH, int MIN_CTAS>
__global__ void __launch_bounds__(kCtaThreads, MIN_CTAS)
stream_kernel(const __grid_constant__ BatchParams p) {
    constexpr int RS = kWarpsPerCta * K;                    // rows per stage
    constexpr int kImgFloats = RS * kUnitCols;              // one image block of a stage
    constexpr int kStageFloats = 2 * kImgFloats;
    constexpr uint32_t kStageBytes = kStageFloats * 4u;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* ring = reinterpret_cast<float*>(smem_raw);
    float4 (*part)[kWarpsPerCta][16] =
        reinterpret_cast<float4 (*)[kWarpsPerCta][16]>(smem_raw + (size_t)DEPTH * kStageBytes);

    pdl_prologue();
    const int lane = threadIdx.x & 31;
    const int w = threadIdx.x >> 5;
    const int N = p.N;
    const int R = p.item_rows;
    const int stages_per_item = R / RS;
    const int units_x = p.units_x, units_y = p.units_y;
    const uint64_t pol = policy_evict_first();
    // this thread's slot inside a stage (the same for the copy and for the read)
    const int my_off = (w * K) * kUnitCols + lane * 4;
    const uint32_t ring_u32 = smem_u32(ring) + (uint32_t)my_off * 4u;
    const ItemCursor stride = decode_item((int)gridDim.x, units_x, units_y);
    const size_t stage_step = (size_t)RS * (size_t)N;      // elements between two stages of an item

    // ---- issue side: runs DEPTH-1 stages ahead of the consume side ---------------------------
    ItemCursor a = decode_item((int)blockIdx.x, units_x, units_y);
    int a_s = 0;                    // stage inside the item
    uint32_t a_dst = ring_u32;      // shared address of this thread's slot in the stage being filled
    int a_slot = 0;
    const float* ax = nullptr;      // this thread's first pixel of the stage, in x and in y
    const float* ay = nullptr;
    bool a_inside = false;          // item entirely inside the image: no predicates, no zero fill
    auto issue = [&]() {
        if (a.pair < p.n_pairs) {
            if (a_s == 0) {         // new item: base pointers and the inside test
                const int col = a.ux * kUnitCols + lane * 4;
                const int row = a.uy * R + w * K;
                a_inside = (a.ux + 1) * kUnitCols <= N && (a.uy + 1) * R <= N;       // CTA-uniform
                const size_t off = a_inside ? (size_t)row * (size_t)N + (size_t)col : 0;
                ax = p.x[a.pair] + off;
                ay = p.y[a.pair] + off;
            }
            if (a_inside) {
#pragma unroll
                for (int k = 0; k < K; ++k) {
                    cp_async16(a_dst + k * (kUnitCols * 4u), ax + (size_t)k * (size_t)N, 16u, pol);
                    cp_async16(a_dst + (kImgFloats + k * kUnitCols) * 4u, ay + (size_t)k * (size_t)N, 16u, pol);
                }
                ax += stage_step;
                ay += stage_step;
            } else {                // ragged right / bottom edge: rows and columns outside are zero-filled
                const int col = a.ux * kUnitCols + lane * 4;
                const int row = a.uy * R + a_s * RS + w * K;
#pragma unroll
                for (int k = 0; k < K; ++k) {
                    const bool ok = col < N && row + k < N;
                    const size_t off = ok ? (size_t)(row + k) * (size_t)N + (size_t)col : 0;
                    cp_async16(a_dst + k * (kUnitCols * 4u), ax + off, ok ? 16u : 0u, pol);
                    cp_async16(a_dst + (kImgFloats + k * kUnitCols) * 4u, ay + off, ok ? 16u : 0u, pol);
                }
            }
            if (++a_s == stages_per_item) {
                a_s = 0;
                a.advance(stride, units_x, units_y);
            }
            if (++a_slot == DEPTH) { a_slot = 0; a_dst = ring_u32; } else { a_dst += kStageBytes; }
        }
        cp_async_commit();                                  // always: keeps the group count uniform
    };
#pragma unroll
    for (int i = 0; i < DEPTH - 1; ++i) issue();

    // ---- consume side -------------------------------------------------------------------
    const float C1 = p.C1;
    const int log2_nt = p.log2_nt;
    const int log2_g = min(log2_nt - 2, 5);                       // g = min(32, N_T / 4) lanes per tile row
    const int log2_tpw = 5 - log2_g;                              // tile segments per warp row
    const int wpt = min(kWarpsPerCta, (1 << log2_nt) / K);        // warps per tile row of the item
    const int n_ty = kWarpsPerCta / wpt;                          // tile rows per item (> 1 only when N_T < 8*K)
    const float* c_src = ring + my_off;                           // this thread's slot in the stage being consumed
    int c_slot = 0;
    int buf = 0;
    for (ItemCursor c = decode_item((int)blockIdx.x, units_x, units_y); c.pair < p.n_pairs;
         c.advance(stride, units_x, units_y), buf ^= 1) {
        float aL[4] = {0.f, 0.f, 0.f, 0.f}, aA[4] = {0.f, 0.f, 0.f, 0.f};
        float aX[4] = {0.f, 0.f, 0.f, 0.f}, aY[4] = {0.f, 0.f, 0.f, 0.f};
        for (int s = 0; s < stages_per_item; ++s) {
            issue();                                              // stage (now + DEPTH - 1)
            cp_async_wait<DEPTH - 1>();                           // the oldest stage of this thread has landed
            float4 vx[K], vy[K];
#pragma unroll
            for (int k = 0; k < K; ++k) {
                vx[k] = *reinterpret_cast<const float4*>(c_src + k * kUnitCols);
                vy[k] = *reinterpret_cast<const float4*>(c_src + kImgFloats + k * kUnitCols);
            }
#pragma unroll
            for (int k = 0; k < K; ++k) {
                pixel_terms<MODE>(vx[k].x, vy[k].x, C1, aL[0], aA[0], aX[0], aY[0]);
                pixel_terms<MODE>(vx[k].y, vy[k].y, C1, aL[1], aA[1], aX[1], aY[1]);
                pixel_terms<MODE>(vx[k].z, vy[k].z, C1, aL[2], aA[2], aX[2], aY[2]);
                pixel_terms<MODE>(vx[k].w, vy[k].w, C1, aL[3], aA[3], aX[3], aY[3]);
            }
            if (++c_slot == DEPTH) { c_slot = 0; c_src = ring + my_off; } else { c_src += kStageFloats; }
        }

        const int pair = c.pair, uy = c.uy, ux = c.ux;
        // lane: 4 columns -> 1
        float4 v;
        v.x = (aL[0] + aL[1]) + (aL[2] + aL[3]);
        v.y = (aA[0] + aA[1]) + (aA[2] + aA[3]);
        v.z = (aX[0] + aX[1]) + (aX[2] + aX[3]);
        v.w = (aY[0] + aY[1]) + (aY[2] + aY[3]);
        // warp: segmented butterfly over the g lanes that share a tile row
        for (int o = (1 << log2_g) >> 1; o > 0; o >>= 1) {
            if (MODE & kModeLisi) v.x += __shfl_xor_sync(0xffffffffu, v.x, o);
            if (MODE & kModeAug) v.y += __shfl_xor_sync(0xffffffffu, v.y, o);
            v.z += __shfl_xor_sync(0xffffffffu, v.z, o);
            v.w += __shfl_xor_sync(0xffffffffu, v.w, o);
        }
        if ((lane & ((1 << log2_g) - 1)) == 0) part[buf][w][lane >> log2_g] = v;
        __syncthreads();     // part[buf] complete; part[buf ^ 1] is rewritten only after the next barrier

        // CTA: combine the warps that share a tile (fixed order), one thread per tile of the item
        const int t = threadIdx.x;
        if (t < (n_ty << log2_tpw)) {
            const int jy = t >> log2_tpw;
            const int jx = t & ((1 << log2_tpw) - 1);
            const int c0 = ux * kUnitCols + (jx << log2_nt);      // jx == 0 when N_T >= 128
            const int r0 = uy * R + (jy << log2_nt);              // jy == 0 unless N_T < 8*K
            if (c0 < N && r0 < N) {
                float4 s = part[buf][jy * wpt][jx];
                for (int k = 1; k < wpt; ++k) {
                    const float4 u = part[buf][jy * wpt + k][jx];
                    s.x += u.x; s.y += u.y; s.z += u.z; s.w += u.w;
                }
                const size_t tile = (size_t)pair * p.n_tiles + (size_t)(r0 >> log2_nt) * p.nt + (c0 >> log2_nt);
                if (p.ws == nullptr) {
                    finalise_tile(p, tile, s);                    // S4: Eq. 1 / Eq. 2
                } else {                                          // split tile: piece -> workspace
                    const int pxi = ux & (p.pieces_x - 1);
                    const int pyi = uy & (p.pieces_y - 1);
                    p.ws[(tile * p.pieces_y + pyi) * p.pieces_x + pxi] = s;
                }
            }
        }
    }
    cp_async_wait<0>();
}

}  // namespace iqa
