// =============================================================================
// iqa_tiles.cu -- the C ABI of include/iqa_tiles.h: argument validation, the choice of kernel and
// mapping, tensor-map encoding, and the launches.  No torch types, no allocation of device memory; the
// only things kept between calls are a per-device cache of launch geometry (SM count, CTAs per SM) and
// the test / tuning knobs of iqa_debug_knob.
// Order of every entry point: validate -> plan -> encode EVERY tensor map of the call on the host ->
// launch.  Nothing is enqueued unless all of the first three succeeded.
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -shared -Xcompiler -fPIC
// =============================================================================
#include "../../include/iqa_tiles.h"

#include <atomic>
#include <cfloat>
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <type_traits>
#include <utility>
#include <vector>

#include "iqa_aggregate.cuh"
#include "iqa_any.cuh"
#include "iqa_candidates.cuh"
#include "iqa_generic_vec.cuh"
#include "iqa_kernels.cuh"
#include "iqa_tma.cuh"

namespace {

using namespace iqa;

constexpr int kMaxN = 1 << 20;   // 2^40 pixels; keeps every grid and tile index inside int
constexpr int kMaxDevices = 64;

bool is_pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }
int ilog2(int v) { int l = 0; while ((1 << l) < v) ++l; return l; }
int ceil_div(int a, int b) { return (a + b - 1) / b; }
int round_up(int a, int b) { return ceil_div(a, b) * b; }
bool pos_finite(float v) { return std::isfinite(v) && v > 0.0f; }
// C1 feeds rcp.approx.ftz (|x - y| + C1 with x == y): a subnormal C1 would be flushed to zero there
bool pos_normal(float v) { return std::isfinite(v) && v >= FLT_MIN; }

// ---- test / tuning knobs (iqa_debug_knob): plain atomics, set by iqa_debug_knob only --------------------------------
// The shipping library does NOT read the environment: a stray IQA_FORCE_GENERIC=1 in a user's shell must not cost
// 40 % of the bandwidth silently.  A build with -DIQA_TESTING takes the initial values from the environment
// variables of the same names (read once), which is handy under ncu.
//   IQA_FORCE_GENERIC    1: every call takes the generic kernels
//   IQA_FORCE_ANY        1: fp32 power-of-two shapes take the general TMA kernel (iqa_any.cuh) instead of tma_kernel
//   IQA_TMA_CONFIG       0..4: ring / box configuration of tma_kernel (-1: default)
//   IQA_TMA_MAX_CTAS     cap of the persistent grid (0: none)
//   IQA_NO_PDL           1: launch without programmatic dependent launch
//   IQA_CAND_NO_CLUSTER  1: candidate kernels never use the cluster twins
//   IQA_ANY_NO_WIDE      1: any_kernel never lets a lane own eight columns
//   IQA_GENERIC_NO_VEC   1: the generic path always takes the scalar-load kernels
//   IQA_SERIES_PAIR_MAJOR 1: any_kernel runs the comparisons of a series in pair-major item order (no L2 sharing)
//   IQA_PLAN_LARGE_JOB   1: every call is planned as if it had enough work to fill the GPU (no small-job rule in make_plan)
enum Knob { kKnobForceGeneric, kKnobForceAny, kKnobTmaConfig, kKnobTmaMaxCtas, kKnobNoPdl, kKnobCandNoCluster, kKnobNoWide,
            kKnobGenericNoVec, kKnobSeriesPairMajor, kKnobPlanLargeJob, kNumKnobs };
const char* const kKnobNames[kNumKnobs] = {"IQA_FORCE_GENERIC", "IQA_FORCE_ANY", "IQA_TMA_CONFIG", "IQA_TMA_MAX_CTAS",
                                           "IQA_NO_PDL", "IQA_CAND_NO_CLUSTER", "IQA_ANY_NO_WIDE", "IQA_GENERIC_NO_VEC",
                                           "IQA_SERIES_PAIR_MAJOR", "IQA_PLAN_LARGE_JOB"};
const int kKnobDefaults[kNumKnobs] = {0, 0, -1, 0, 0, 0, 0, 0, 0, 0};
struct Knobs {
    std::atomic<int> v[kNumKnobs];
    Knobs() {
        for (int i = 0; i < kNumKnobs; ++i) {
#ifdef IQA_TESTING
            const char* s = std::getenv(kKnobNames[i]);
            v[i].store((s && *s) ? std::atoi(s) : kKnobDefaults[i], std::memory_order_relaxed);
#else
            v[i].store(kKnobDefaults[i], std::memory_order_relaxed);
#endif
        }
    }
};
Knobs& knobs() { static Knobs k; return k; }
int knob(Knob k) { return knobs().v[k].load(std::memory_order_relaxed); }

// ---- pixel types -----------------------------------------------------------------------------------------
int esize_of(int ptype) {
    switch (ptype) {
        case IQA_PIXEL_F32: case IQA_PIXEL_I32: return 4;
        case IQA_PIXEL_F64: return 8;
        case IQA_PIXEL_F16: case IQA_PIXEL_I16: return 2;
        case IQA_PIXEL_U8: return 1;
        default: return 0;
    }
}
CUtensorMapDataType tma_type_of(int ptype) {
    switch (ptype) {
        case IQA_PIXEL_F64: return CU_TENSOR_MAP_DATA_TYPE_FLOAT64;
        case IQA_PIXEL_F16: return CU_TENSOR_MAP_DATA_TYPE_FLOAT16;
        case IQA_PIXEL_I16: return CU_TENSOR_MAP_DATA_TYPE_UINT16;     // bits only; the kernel reinterprets
        case IQA_PIXEL_I32: return CU_TENSOR_MAP_DATA_TYPE_INT32;
        case IQA_PIXEL_U8: return CU_TENSOR_MAP_DATA_TYPE_UINT8;
        default: return CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
    }
}

// ---- tma_kernel configurations: {box slots per CTA, rows per warp and box} ------------------------------------
// Measured on B200 (profiles/r01g_tma_configs.md): pairs are HBM-bound and want FEW bytes in flight (config 1: two
// 16 KiB boxes in flight per CTA while two are consumed; six boxes lose 3-6 % to DRAM locality); the series modes
// keep S + 1 boxes alive and want the deeper ring of config 0.
struct TmaConfig { int boxes, rpw; };
constexpr int kNumTmaConfigs = 5;
constexpr TmaConfig kTmaConfigs[kNumTmaConfigs] = {{6, 4}, {4, 4}, {8, 2}, {6, 2}, {4, 2}};

using TmaFn = void (*)(const TmaParams);
template <int MODE, int SERIES>
TmaFn tma_fn_cfg(int cfg) {
    switch (cfg) {
        case 1: return tma_kernel<MODE, SERIES, 4, 4>;
        case 2: return tma_kernel<MODE, SERIES, 8, 2>;
        case 3: return tma_kernel<MODE, SERIES, 6, 2>;
        case 4: return tma_kernel<MODE, SERIES, 4, 2>;
        default: return tma_kernel<MODE, SERIES, 6, 4>;
    }
}
// The standalone LISI / augLISI entry points only exist for pairs; the series modes are fused.
TmaFn tma_fn(int mode, int series, int cfg) {
    if (series == kPairs) {
        switch (mode) {
            case kModeLisi: return tma_fn_cfg<kModeLisi, kPairs>(cfg);
            case kModeAug: return tma_fn_cfg<kModeAug, kPairs>(cfg);
            default: return tma_fn_cfg<kModeFused, kPairs>(cfg);
        }
    }
    if (mode != kModeFused) return nullptr;
    return series == kReference ? tma_fn_cfg<kModeFused, kReference>(cfg) : tma_fn_cfg<kModeFused, kConsecutive>(cfg);
}
size_t tma_smem(int cfg) { return tma_smem_bytes(kTmaConfigs[cfg].boxes, kTmaConfigs[cfg].rpw); }

// any_kernel instantiations: the three modes for fp32 (paper-named entry points with odd N_T), fused for the rest.
using AnyFn = void (*)(const AnyParams);
constexpr int kNumAnyFns = 8;
AnyFn any_fn_at(int i) {
    switch (i) {
        case 0: return any_kernel<kModeLisi, float>;
        case 1: return any_kernel<kModeAug, float>;
        case 2: return any_kernel<kModeFused, float>;
        case 3: return any_kernel<kModeFused, double>;
        case 4: return any_kernel<kModeFused, __half>;
        case 5: return any_kernel<kModeFused, short>;
        case 6: return any_kernel<kModeFused, int>;
        default: return any_kernel<kModeFused, unsigned char>;
    }
}
int any_fn_index(int mode, int ptype) {
    switch (ptype) {
        case IQA_PIXEL_F32: return mode == kModeLisi ? 0 : mode == kModeAug ? 1 : 2;
        case IQA_PIXEL_F64: return 3;
        case IQA_PIXEL_F16: return 4;
        case IQA_PIXEL_I16: return 5;
        case IQA_PIXEL_I32: return 6;
        default: return 7;
    }
}
constexpr int kAnyBoxBudget = 20480;    // bytes of one box
constexpr int kAnyRingBudget = 81920;   // bytes of the ring of boxes of one CTA (2 CTAs per SM)
constexpr size_t kAnyMaxSmem = 1024 + kAnyRingBudget + 128 * kAnyMaxSlots + kAnyPartBufs * kWarpsPerCta * 32 * 16 + 256;

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda).
using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                   const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                   CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled_fn() {
    static const EncodeTiledFn fn = [] {
        void* f = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess ||
            q != cudaDriverEntryPointSuccess)
            f = nullptr;
        return (EncodeTiledFn)f;
    }();
    return fn;
}

// Tensor map of one H x W row-major image of `ptype` pixels with a row pitch (in elements): boxes of box_w columns x
// box_rows rows, no swizzle (a box lands as [box_rows][box_w] elements), out-of-bounds elements read as zero.
// The image base only needs the alignment of its element type: the tensor starts at the 16-byte boundary below it and
// is (base & 15) / sizeof(pixel) elements wider on the left; any_kernel works in tensor columns and masks those
// elements (they lie in the same 16-byte line as pixel (0, 0), hence inside the allocation).  The row pitch must be
// a multiple of 16 bytes.
bool encode_image_map(CUtensorMap* map, const void* img, int ptype, int H, int W, long long pitch,
                      int box_w, int box_rows) {
    const EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) return false;
    const int es = esize_of(ptype);
    const uintptr_t addr = (uintptr_t)img;
    const unsigned sh = (unsigned)((addr & 15u) / (unsigned)es);
    const cuuint64_t dims[2] = {(cuuint64_t)W + sh, (cuuint64_t)H};
    const cuuint64_t strides[1] = {(cuuint64_t)pitch * (cuuint64_t)es};
    const cuuint32_t box[2] = {(cuuint32_t)box_w, (cuuint32_t)box_rows};
    const cuuint32_t estr[2] = {1u, 1u};
    return enc(map, tma_type_of(ptype), 2u, (void*)(addr & ~(uintptr_t)15u), dims, strides, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// Per-device launch geometry, filled on first use under a mutex (`ready` is the lock-free fast path afterwards).
// any_occ: resident CTAs per SM of any_kernel instantiation i at a given dynamic shared-memory size -- asked of the
// runtime once per (device, instantiation, size) instead of on every call (the single-pair path is host-latency bound).
constexpr int kAnyOccSlots = 4;
struct AnyOcc { std::atomic<size_t> smem{0}; std::atomic<int> occ{0}; };
struct Geometry {
    std::atomic<int> ready{0};
    int sms;
    int tma_ctas[kNumTmaConfigs];
    AnyOcc any_occ[kNumAnyFns][kAnyOccSlots];
};
Geometry g_geo[kMaxDevices];
std::mutex g_geo_mutex;

const Geometry* geometry() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return nullptr;
    Geometry& g = g_geo[dev];
    if (g.ready.load(std::memory_order_acquire)) return &g;
    std::lock_guard<std::mutex> lock(g_geo_mutex);
    if (g.ready.load(std::memory_order_acquire)) return &g;
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) return nullptr;
    for (int c = 0; c < kNumTmaConfigs; ++c) {
        g.tma_ctas[c] = 0;
        for (int m = 1; m <= 3; ++m)
            for (int ser = 0; ser < 3; ++ser) {
                TmaFn fn = tma_fn(m, ser, c);
                if (!fn) continue;
                if (cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tma_smem(c)) != cudaSuccess) return nullptr;
                int occ = 0;
                if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, kTmaThreads, tma_smem(c)) != cudaSuccess || occ <= 0) return nullptr;
                occ = occ < 2 ? occ : 2;
                g.tma_ctas[c] = g.tma_ctas[c] == 0 || occ < g.tma_ctas[c] ? occ : g.tma_ctas[c];
            }
    }
    for (int i = 0; i < kNumAnyFns; ++i)
        if (cudaFuncSetAttribute(any_fn_at(i), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kAnyMaxSmem) != cudaSuccess)
            return nullptr;
    g.sms = sms;
    g.ready.store(1, std::memory_order_release);
    return &g;
}

// Resident CTAs per SM of any_kernel instantiation `fi` with `smem` bytes of dynamic shared memory on the current
// device (0: unknown).  A handful of sizes occur per instantiation (one per ring geometry); they are kept in a small
// table that threads fill under the mutex; a full table just asks the runtime again.
int any_occupancy(int fi, size_t smem) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return 0;
    AnyOcc* slots = g_geo[dev].any_occ[fi];
    for (int i = 0; i < kAnyOccSlots; ++i) {
        const int occ = slots[i].occ.load(std::memory_order_acquire);
        if (occ == 0) break;
        if (slots[i].smem.load(std::memory_order_relaxed) == smem) return occ;
    }
    int occ = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, any_fn_at(fi), kTmaThreads, smem) != cudaSuccess || occ <= 0)
        return 0;
    std::lock_guard<std::mutex> lock(g_geo_mutex);
    for (int i = 0; i < kAnyOccSlots; ++i)
        if (slots[i].occ.load(std::memory_order_relaxed) == 0) {
            slots[i].smem.store(smem, std::memory_order_relaxed);
            slots[i].occ.store(occ, std::memory_order_release);
            break;
        }
    return occ;
}

// Launch with the programmatic-stream-serialisation attribute (PDL): the kernel may become
// resident while the previous kernel of the stream drains; every kernel of this library
// starts with griddepcontrol.wait, so nothing is read or written before that kernel is done.
template <typename... KArgs, typename... Args>
cudaError_t launch_cluster(void (*kernel)(KArgs...), unsigned grid, unsigned block, size_t smem, cudaStream_t st,
                           unsigned cluster, Args&&... args) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(block);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[2];
    unsigned na = 0;
    if (!knob(kKnobNoPdl)) {
        attr[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[na].val.programmaticStreamSerializationAllowed = 1;
        ++na;
    }
    if (cluster > 0) {                        // thread-block cluster of `cluster` CTAs along x
        attr[na].id = cudaLaunchAttributeClusterDimension;
        attr[na].val.clusterDim.x = cluster;
        attr[na].val.clusterDim.y = 1;
        attr[na].val.clusterDim.z = 1;
        ++na;
    }
    cfg.attrs = attr;
    cfg.numAttrs = na;
    return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}
template <typename... KArgs, typename... Args>
cudaError_t launch(void (*kernel)(KArgs...), unsigned grid, unsigned block, size_t smem, cudaStream_t st,
                   Args&&... args) {
    return launch_cluster(kernel, grid, block, smem, st, 0u, std::forward<Args>(args)...);
}

int status_of_shape(int N, int N_T) {
    if (N <= 0 || N_T <= 0 || N > kMaxN || N_T > N || N % N_T != 0) return IQA_ERR_SHAPE;
    const long long nt = N / N_T;
    if (nt * nt > 0x7fffffffLL) return IQA_ERR_SHAPE;
    return IQA_OK;
}

// Geometry of the images of one call: the x images share pitch_x, the y images pitch_y (elements).
struct Geom { int H, W; long long pitch_x, pitch_y; int ptype; };
Geom square_geom(int N) { return Geom{N, N, (long long)N, (long long)N, IQA_PIXEL_F32}; }

// ---- run-time geometry of any_kernel (iqa_any.cuh) ------------------------------------------------------------
struct AnyGeom {
    int kx, ky, px, py, pw, ph, box_w, box_rows, row_bytes, slot_bytes, n_slots, rpw, wpt, fin_gsz, units_x, units_y;
    int const_s;       // every item sits at the same column offset inside its box
    int cpl_log2;      // columns per lane: 2 -> four, 3 -> eight
};
constexpr int kAnySplitAbove = 112;   // tiles wider than this are split (128 lanes-columns minus the widest 16-byte pad)
// Pieces per split tile (N_T > kAnySplitAbove): pw x 64 pixels each, pw a multiple of 16 columns; the same for every
// pixel type and alignment, so that the workspace size is a function of N_T alone.
void any_pieces(int N_T, int* pw, int* px, int* py) {
    const int px0 = ceil_div(N_T, kAnySplitAbove);
    *pw = round_up(ceil_div(N_T, px0), 16);
    *px = ceil_div(N_T, *pw);
    *py = ceil_div(N_T, 64);
}
// shift: elements between the 16-byte boundary below the image bases and pixel (0, 0) (the same for every image).
AnyGeom any_geometry(int esize, int N_T, int H, int W, int shift) {
    AnyGeom g{};
    const int pad = 16 / esize;                       // elements per 16 bytes: a TMA box starts at a multiple of it
    const int wpad = pad < 4 ? 4 : pad;               // box widths are whole lanes (4 columns) as well
    const int ntx = ceil_div(W, N_T), nty = ceil_div(H, N_T);
    g.cpl_log2 = 2;
    if (N_T <= kAnySplitAbove) {                      // whole tiles inside one item: kx across, ky down
        // kx_a: items that start on 16-byte boundaries (s = 0 everywhere); kx_s: items at any column, which costs
        // pad - 1 columns of the box
        int kx_a = 0;
        if (shift == 0)
            for (int k = kUnitCols / N_T; k >= 1; --k)
                if ((k * N_T) % pad == 0) { kx_a = k; break; }
        int kx_s = (kUnitCols - pad + 1) / N_T;
        if (kx_a > ntx) kx_a = ntx;
        if (kx_s > ntx) kx_s = ntx;
        // kx_w: eight columns per lane (boxes of up to 256 columns): every lane inside one tile, items on 16-byte
        // boundaries.  Twice the pixels per item, and tile sides such as 48 fill 30 of 32 lanes instead of 24.
        int kx_w = 0;
        if (shift == 0 && N_T % 8 == 0 && esize <= 4 && !knob(kKnobNoWide))     // (fp64: 64 bytes per lane and row: slower)
            for (int k = 2 * kUnitCols / N_T; k >= 1; --k)
                if ((k * N_T) % pad == 0) { kx_w = k; break; }
        if (kx_w > ntx) kx_w = ntx;
        if (kx_w > 0 && kx_w * N_T > kUnitCols) {
            g.kx = kx_w;
            g.const_s = 1;
            g.cpl_log2 = 3;
            g.box_w = g.kx * N_T;
        } else if (kx_a > 0 && kx_a * 8 >= kx_s * 7) {
            g.kx = kx_a;
            g.const_s = 1;
            g.box_w = round_up(g.kx * N_T, wpad);
        } else {
            g.kx = kx_s;
            g.const_s = (g.kx * N_T) % pad == 0 || g.kx >= ntx;      // one item column: c0 = 0 everywhere
            g.box_w = round_up(g.kx * N_T + pad - 1, wpad);
        }
        g.pw = g.kx * N_T;
        g.row_bytes = g.box_w * esize;
        int rows_fit = kAnyBoxBudget / g.row_bytes;
        if (rows_fit > 256) rows_fit = 256;
        g.ky = 1;
        if (N_T <= rows_fit) {                        // several tile rows per box, 8 / ky warps each
            while (g.ky < kWarpsPerCta && 2 * g.ky * N_T <= rows_fit && g.ky < nty) g.ky *= 2;
            g.box_rows = g.ky * N_T;
            g.wpt = kWarpsPerCta / g.ky;
            g.rpw = ceil_div(N_T, g.wpt);
        } else {                                      // the tile's rows in S boxes
            const int S = ceil_div(N_T, rows_fit);
            g.box_rows = ceil_div(N_T, S);
            g.wpt = kWarpsPerCta;
            g.rpw = ceil_div(g.box_rows, kWarpsPerCta);
        }
        g.ph = g.ky * N_T;
        g.px = g.py = 1;
    } else {                                          // split tiles: pieces of pw x 64 pixels
        any_pieces(N_T, &g.pw, &g.px, &g.py);
        g.kx = g.ky = 1;
        g.const_s = N_T % pad == 0;                   // pw is a multiple of 16 columns
        g.box_w = g.const_s && shift == 0 ? g.pw : round_up(g.pw + pad - 1, wpad);
        g.row_bytes = g.box_w * esize;
        g.box_rows = 64;
        while (g.box_rows * g.row_bytes > kAnyBoxBudget) g.box_rows /= 2;
        g.ph = 64;
        g.wpt = kWarpsPerCta;
        g.rpw = ceil_div(g.box_rows, kWarpsPerCta);
    }
    g.slot_bytes = round_up(g.box_rows * g.row_bytes, 128);
    g.n_slots = (kAnyRingBudget / g.slot_bytes) & ~1;
    if (g.n_slots < 4) g.n_slots = 4;
    if (g.n_slots > kAnyMaxSlots) g.n_slots = kAnyMaxSlots;
    int p2 = 1;
    while (p2 < g.kx * g.ky) p2 <<= 1;
    g.fin_gsz = p2 >= 32 ? 1 : 32 / p2;
    g.units_x = ceil_div(ntx, g.kx) * g.px;
    g.units_y = ceil_div(nty, g.ky) * g.py;
    return g;
}

// How a call is mapped onto kernels.  DESIGN.md "Kernels".
enum PlanKind { kPlanGeneric = 0, kPlanTma = 2, kPlanAny = 3 };
struct Plan {
    PlanKind kind;     // generic kernels / tma_kernel (fp32, power-of-two N_T) / any_kernel
    int tma_cfg;       // tma: index into kTmaConfigs
    int item_rows;     // tma: R
    int pieces_x, pieces_y, pieces;   // pieces per tile; pieces == 1 -> finished inside one CTA
    AnyGeom any;
};

constexpr int kSplitItemRows = 64;   // tma_kernel, tiles of side >= 128: items of 128 x 64, pieces to the workspace

void generic_plan(Plan& pl, int N_T) {
    pl.kind = kPlanGeneric;
    pl.pieces_x = 1;
    pl.pieces_y = ceil_div(N_T, kGenericRows);
    pl.pieces = pl.pieces_y;
}

// Alignment of the images of a call: `lo16` = the offset of every base inside its 16-byte line when all images
// share it (-1 when they differ: no common column grid for the TMA boxes).
struct Align { int lo16; };
Align align_of(const void* const* a, int na, const void* const* b, int nb) {
    const int lo = (int)((uintptr_t)a[0] & 15u);
    for (int i = 0; i < na; ++i)
        if ((int)((uintptr_t)a[i] & 15u) != lo) return Align{-1};
    for (int i = 0; i < nb; ++i)
        if ((int)((uintptr_t)b[i] & 15u) != lo) return Align{-1};
    return Align{lo};
}

// The 128-bit generic kernel runs one WARP per piece of a tile (<= 64 rows) and keeps a few 16-byte loads per lane in
// flight: it only beats any_kernel's idle lanes when there are enough pieces to give every SM several warps.  Below that
// (one or two pairs of a 1024^2 / 2048^2 image with tiles of 113 .. 400 columns) any_kernel, whose TMA ring keeps tens of
// KiB in flight per SM whatever the item count, is up to 3x faster.  Measured crossovers (pieces of the whole call per
// SM; sweeps at N = 1024 / 2048 with 2, 4 and 32 pairs): ~4.5 for 4-byte pixels, ~12 for fp64, ~4 for 1- and 2-byte pixels.
// Without a device (a CPU-only box asking iqa_query_plan) the rule is off.
bool small_job(const Geom& g, int N_T, int es, long long n_cmp) {
    if (knob(kKnobPlanLargeJob)) return false;
    const Geometry* geo = geometry();
    if (!geo) return false;
    const long long units = (long long)ceil_div(g.W, N_T) * ceil_div(g.H, N_T) * ceil_div(N_T, kGenericRows) * n_cmp;
    const long long per_sm_x2 = es == 8 ? 24 : es == 4 ? 9 : 8;          // twice the crossover
    return 2 * units < per_sm_x2 * geo->sms;
}

// A tensor map can describe the images when every row pitch is a multiple of 16 bytes; the boxes of x and y share
// their column grid when all bases have the same offset inside a 16-byte line (al.lo16 >= 0).
// series: the call is a time series (tma_kernel's series ring; any_kernel's pair-minor order); n_cmp: its comparisons.
Plan make_plan(const Geom& g, int N_T, Align al, bool series, int n_cmp) {
    Plan pl{};
    generic_plan(pl, N_T);
    const int es = esize_of(g.ptype);
    const bool tma_able = (g.pitch_x * es) % 16 == 0 && (g.pitch_y * es) % 16 == 0 && al.lo16 >= 0;
    if (!tma_able || N_T < 4 || knob(kKnobForceGeneric)) return pl;
    if (g.ptype == IQA_PIXEL_F32 && is_pow2(N_T) && N_T >= 8 && al.lo16 == 0 && !knob(kKnobForceAny)) {
        pl.kind = kPlanTma;
        const int dflt = series ? 0 : 1;
        const int c = knob(kKnobTmaConfig);
        pl.tma_cfg = c >= 0 && c < kNumTmaConfigs ? c : dflt;
        // the series modes keep S + 1 boxes alive (S = 64 / box rows for N_T >= 64): small rings fall back
        if (series && kTmaConfigs[pl.tma_cfg].boxes < 64 / (kWarpsPerCta * kTmaConfigs[pl.tma_cfg].rpw) + 2) pl.tma_cfg = 0;
        const int rs = kWarpsPerCta * kTmaConfigs[pl.tma_cfg].rpw;       // box height
        if (N_T <= 64) {
            pl.item_rows = N_T > rs ? N_T : rs;                  // whole tiles inside one item
            pl.pieces_x = pl.pieces_y = 1;
        } else {
            pl.item_rows = kSplitItemRows;
            pl.pieces_x = N_T / kUnitCols;
            pl.pieces_y = N_T / kSplitItemRows;
        }
        pl.pieces = pl.pieces_x * pl.pieces_y;
        return pl;
    }
    pl.kind = kPlanAny;
    pl.any = any_geometry(es, N_T, g.H, g.W, al.lo16 / es);
    // any_kernel binds lanes to box columns, and an item is whole tiles or ONE piece of a tile: a 64-column tile behind a
    // shifted base fills 17 of 32 lanes, a 130-column tile two pieces of 20 lanes.  The warp-per-piece kernel with 128-bit
    // loads (iqa_generic_vec.cuh: every lane busy whatever the width; x and y are aligned alike here) is faster there.
    // Thresholds measured at N = 8192: whole tiles at <= 0.56 lane fill; split tiles below 0.8 (4- and
    // 8-byte pixels) / always (1- and 2-byte pixels: split pieces run four columns per lane).
    if ((long long)N_T * N_T > kWarpTilePixels && !knob(kKnobForceAny)) {
        const AnyGeom& a = pl.any;
        const bool split = a.px * a.py > 1;
        const double fill = split ? (double)N_T / (128.0 * a.px) : (double)(a.kx * N_T) / (32.0 * (1 << a.cpl_log2));
        // (the comparisons of a series share images through L2 in any_kernel's pair-minor order, worth 1.2-1.35x for 4- and
        //  8-byte pixels: the generic kernel, which runs them pair by pair, has to win by more)
        const double whole = es == 1 ? 0.5 : 0.56;       // whole tiles: N_T = 64 behind a shift, N_T = 65 .. 71 (uint8: 64 only)
        const bool sharing = series && n_cmp > 1;        // a series of two images is one pair: nothing to share
        const double limit = es <= 2 ? (split ? 2.0 : whole)
                           : sharing ? (split ? 0.5 : -1.0)
                                     : (!split ? whole : 0.8);
        const bool narrow_image = !split && a.kx >= ceil_div(g.W, N_T);       // the image, not the mapping, limits the fill
        if (!narrow_image && (split ? fill < limit : fill <= limit) && !small_job(g, N_T, es, n_cmp)) {
            generic_plan(pl, N_T);
            return pl;
        }
    }
    pl.pieces_x = pl.any.px;
    pl.pieces_y = pl.any.py;
    pl.pieces = pl.pieces_x * pl.pieces_y;
    return pl;
}

// Pieces per tile in the worst case over the mappings a call may take (tma, any or generic).
size_t max_pieces(int N_T) {
    if (N_T <= 64) return 1;                                      // every path finishes tiles inside one CTA
    size_t pieces = (size_t)ceil_div(N_T, kGenericRows);
    if (N_T > kAnySplitAbove) {
        int pw, px, py;
        any_pieces(N_T, &pw, &px, &py);
        if ((size_t)px * py > pieces) pieces = (size_t)px * py;
    }
    if (is_pow2(N_T)) {
        const size_t s = (size_t)(N_T / kUnitCols) * (size_t)(N_T / kSplitItemRows);
        if (s > pieces) pieces = s;
    }
    return pieces;
}

size_t workspace_bytes_for(int n_pairs, int N, int N_T) {
    const size_t pieces = max_pieces(N_T);
    if (pieces <= 1) return 0;
    const size_t n = (size_t)(N / N_T) * (size_t)(N / N_T);
    return (size_t)n_pairs * n * pieces * sizeof(float4);
}

struct Outputs {
    float *lisi, *auglisi, *sum_x, *sum_y, *lisi_num, *aug_num;   // [n_comparisons * n] each (or nullptr)
    Outputs offset(size_t k) const {
        auto o = [k](float* p) { return p ? p + k : nullptr; };
        return {o(lisi), o(auglisi), o(sum_x), o(sum_y), o(lisi_num), o(aug_num)};
    }
    Outputs for_mode(int mode) const {
        return {(mode & kModeLisi) ? lisi : nullptr, (mode & kModeAug) ? auglisi : nullptr, sum_x, sum_y,
                (mode & kModeLisi) ? lisi_num : nullptr, (mode & kModeAug) ? aug_num : nullptr};
    }
};

struct Consts { float C1, C2, C, D; };

// ---- tma_kernel: encode, then launch --------------------------------------------------------------------------
struct TmaLaunch { TmaParams p; TmaFn fn; unsigned grid; size_t smem; };

// n_groups groups of M images (imgs[g * M + i], HOST array of device pointers); `out` and `ws` point at the first
// comparison of the first group.  n_groups * M may exceed kMaxImages (several launches); M itself may not.  Image i of
// a group has pitch_y when (i & 1) else pitch_x (pairs: x, y; series: both pitches are equal).
// Appends the prepared launches; false when a tensor map could not be encoded (nothing was launched).
bool prepare_tma(std::vector<TmaLaunch>& q, int mode, int series, const void* const* imgs, int n_groups, int M,
                 const Geom& g, int N_T, const Consts& k, const Outputs& out, float4* ws, const Plan& pl) {
    const Geometry* geo = geometry();
    TmaFn fn = tma_fn(mode, series, pl.tma_cfg);
    const int box_rows = kWarpsPerCta * kTmaConfigs[pl.tma_cfg].rpw;
    if (!geo || !fn || geo->tma_ctas[pl.tma_cfg] <= 0 || M < 2 || M > kMaxImages) return false;
    const int H = g.H, W = g.W;
    const int ntx = ceil_div(W, N_T), nty = ceil_div(H, N_T);
    const long long n = (long long)ntx * nty;
    // split tiles: the items cover the whole tile grid, so that every piece of an edge tile is written
    // (boxes entirely outside the image are zero-filled by the TMA unit without touching memory)
    const int units_x = pl.pieces > 1 ? ntx * pl.pieces_x : ceil_div(W, kUnitCols);
    const int units_y = pl.pieces > 1 ? nty * pl.pieces_y : ceil_div(H, pl.item_rows);
    const long long items_per_group = (long long)units_x * units_y;
    const int groups_per_launch = kMaxImages / M;
    if (items_per_group * groups_per_launch > 0x7fffffffLL) return false;
    for (int first = 0; first < n_groups; first += groups_per_launch) {
        const int ng = n_groups - first < groups_per_launch ? n_groups - first : groups_per_launch;
        q.emplace_back();
        TmaLaunch& L = q.back();
        TmaParams& p = L.p;
        std::memset(&p, 0, sizeof(p));
        for (int i = 0; i < ng * M; ++i)
            if (!encode_image_map(&p.maps[i], imgs[(size_t)first * M + i], IQA_PIXEL_F32, H, W,
                                  (i & 1) ? g.pitch_y : g.pitch_x, kUnitCols, box_rows))
                return false;
        p.n_groups = ng; p.M = M; p.W = W; p.H = H; p.log2_nt = ilog2(N_T); p.ntx = ntx; p.n_tiles = (int)n;
        p.units_x = units_x; p.units_y = units_y; p.S = pl.item_rows / box_rows;
        p.C1 = k.C1; p.C2 = k.C2; p.C = k.C; p.D = k.D;
        const size_t cmp0 = (size_t)first * (size_t)(M - 1);
        const Outputs o = out.offset(cmp0 * (size_t)n);
        p.lisi = o.lisi; p.auglisi = o.auglisi; p.sum_x = o.sum_x; p.sum_y = o.sum_y;
        p.lisi_num = o.lisi_num; p.aug_num = o.aug_num;
        p.ws = (ws && pl.pieces > 1) ? ws + cmp0 * (size_t)n * pl.pieces : nullptr;
        p.pieces_x = pl.pieces_x; p.pieces_y = pl.pieces_y;
        const long long n_items = items_per_group * ng;
        long long resident = (long long)geo->sms * geo->tma_ctas[pl.tma_cfg];
        const int max_ctas = knob(kKnobTmaMaxCtas);
        if (max_ctas > 0 && max_ctas < resident) resident = max_ctas;
        L.fn = fn;
        L.grid = (unsigned)(n_items < resident ? n_items : resident);
        L.smem = tma_smem(pl.tma_cfg);
    }
    return true;
}
int fire(const std::vector<TmaLaunch>& q, cudaStream_t st) {
    for (const TmaLaunch& L : q)
        if (launch(L.fn, L.grid, kTmaThreads, L.smem, st, L.p) != cudaSuccess) return IQA_ERR_CUDA;
    return IQA_OK;
}

// ---- any_kernel: encode, then launch ---------------------------------------------------------------------------
struct AnyLaunch { AnyParams p; AnyFn fn; unsigned grid; size_t smem; };

// pair_minor: the pairs are the comparisons of a time series (they share images): item order of AnyCursor.
bool prepare_any(std::vector<AnyLaunch>& q, int mode, const void* const* xs, const void* const* ys, int n_pairs,
                 const Geom& g, int N_T, const Consts& k, const Outputs& out, float4* ws, const Plan& pl, bool pair_minor) {
    const Geometry* geo = geometry();
    if (!geo) return false;
    const AnyGeom& a = pl.any;
    AnyFn fn = any_fn_at(any_fn_index(mode, g.ptype));
    const size_t smem = any_smem_bytes(a.n_slots, a.slot_bytes);
    if (smem > kAnyMaxSmem) return false;
    int occ = any_occupancy(any_fn_index(mode, g.ptype), smem);
    if (occ <= 0) return false;
    if (occ > 2) occ = 2;
    const int ntx = ceil_div(g.W, N_T), nty = ceil_div(g.H, N_T);
    const long long n = (long long)ntx * nty;
    const long long items_per_pair = (long long)a.units_x * a.units_y;
    const int pairs_per_launch = kAnyMaxImages / 2;
    if (items_per_pair * pairs_per_launch > 0x7fffffffLL) return false;
    for (int first = 0; first < n_pairs; first += pairs_per_launch) {
        const int np = n_pairs - first < pairs_per_launch ? n_pairs - first : pairs_per_launch;
        q.emplace_back();
        AnyLaunch& L = q.back();
        AnyParams& p = L.p;
        std::memset(&p, 0, sizeof(p));
        for (int i = 0; i < np; ++i) {
            if (!encode_image_map(&p.maps[2 * i], xs[first + i], g.ptype, g.H, g.W, g.pitch_x, a.box_w, a.box_rows) ||
                !encode_image_map(&p.maps[2 * i + 1], ys[first + i], g.ptype, g.H, g.W, g.pitch_y, a.box_w, a.box_rows))
                return false;
        }
        p.shift = (int)(((uintptr_t)xs[0] & 15u) / (unsigned)esize_of(g.ptype));
        p.pad_mask = 16 / esize_of(g.ptype) - 1;
        p.const_s = a.const_s;
        p.pair_minor = pair_minor && np > 1 && !knob(kKnobSeriesPairMajor) ? 1 : 0;
        p.n_pairs = np; p.W = g.W; p.H = g.H; p.N_T = N_T; p.ntx = ntx; p.nty = nty; p.n_tiles = (int)n;
        p.kx = a.kx; p.ky = a.ky; p.px = a.px; p.py = a.py; p.pw = a.pw; p.ph = a.ph;
        p.units_x = a.units_x; p.units_y = a.units_y; p.box_rows = a.box_rows; p.row_bytes = a.row_bytes;
        p.slot_bytes = a.slot_bytes; p.n_slots = a.n_slots; p.rpw = a.rpw; p.wpt = a.wpt; p.fin_gsz = a.fin_gsz;
        p.cpl_log2 = a.cpl_log2;
        p.boxes_per_item = ceil_div(a.ph, a.box_rows);
        p.nt_magic = (unsigned)(0x100000000ull / (unsigned)N_T) + 1u;
        p.C1 = k.C1; p.C2 = k.C2; p.C = k.C; p.D = k.D;
        const Outputs o = out.offset((size_t)first * (size_t)n);
        p.lisi = o.lisi; p.auglisi = o.auglisi; p.sum_x = o.sum_x; p.sum_y = o.sum_y;
        p.lisi_num = o.lisi_num; p.aug_num = o.aug_num;
        p.ws = (ws && pl.pieces > 1) ? ws + (size_t)first * (size_t)n * pl.pieces : nullptr;
        const long long n_items = items_per_pair * np;
        long long resident = (long long)geo->sms * occ;
        const int max_ctas = knob(kKnobTmaMaxCtas);
        if (max_ctas > 0 && max_ctas < resident) resident = max_ctas;
        L.fn = fn;
        L.grid = (unsigned)(n_items < resident ? n_items : resident);
        L.smem = smem;
    }
    return true;
}
int fire(const std::vector<AnyLaunch>& q, cudaStream_t st) {
    for (const AnyLaunch& L : q)
        if (launch(L.fn, L.grid, kTmaThreads, L.smem, st, L.p) != cudaSuccess) return IQA_ERR_CUDA;
    return IQA_OK;
}

// ---- generic kernels (pair by pair) ---------------------------------------------------------------------------
// The scalar-load generic kernels, one pair per launch.
template <int MODE, typename T>
cudaError_t launch_generic_one(const GenericParams& g, long long n, int N_T, int pieces, cudaStream_t st) {
    if ((long long)N_T * N_T <= kWarpTilePixels)          // small tiles: one warp per tile (pieces == 1 here)
        return launch(generic_warp_kernel<MODE, T>, (unsigned)((n + kWarpsPerCta - 1) / kWarpsPerCta), kCtaThreads, 0, st, g, n);
    return launch(generic_kernel<MODE, T>, (unsigned)(n * pieces), kCtaThreads, 0, st, g);
}
// The warp-per-piece kernel with 128-bit loads (iqa_generic_vec.cuh): up to kVecMaxPairs pairs per launch.
template <int MODE, typename T>
cudaError_t launch_generic_vec(const GenericParams& g, const VecBatch& b, long long n, int pieces, cudaStream_t st) {
    const long long upp = n * pieces, units = upp * b.n_pairs;
    return launch(generic_vec_kernel<MODE, T>, (unsigned)((units + kWarpsPerCta - 1) / kWarpsPerCta), kCtaThreads, 0, st, g, b,
                  upp);
}
template <typename F32, typename Other>
cudaError_t by_pixel_type(int ptype, int mode, F32&& f32, Other&& other) {
    switch (ptype) {
        case IQA_PIXEL_F64: return other((double*)nullptr);
        case IQA_PIXEL_F16: return other((__half*)nullptr);
        case IQA_PIXEL_I16: return other((short*)nullptr);
        case IQA_PIXEL_I32: return other((int*)nullptr);
        case IQA_PIXEL_U8: return other((unsigned char*)nullptr);
        default: return f32(mode);
    }
}

// series_order: the pairs are the comparisons of a time series (pair-minor unit order in the 128-bit kernel).
int launch_generic(int mode, const void* const* xs, const void* const* ys, int n_pairs, const Geom& g2, int N_T,
                   const Consts& k, const Outputs& out, float4* ws, const Plan& pl, cudaStream_t st, bool series_order) {
    const int nt = ceil_div(g2.W, N_T);
    const long long n = (long long)nt * ceil_div(g2.H, N_T);
    if (n * pl.pieces > 0x7fffffffLL) return IQA_ERR_SHAPE;
    const int es = esize_of(g2.ptype);
    // x and y aligned alike row by row (every pair): the kernel with 128-bit loads, kVecMaxPairs pairs per launch
    bool vec = !knob(kKnobGenericNoVec) && (((g2.pitch_x - g2.pitch_y) * es) & 15) == 0;
    for (int i = 0; i < n_pairs && vec; ++i) vec = (((uintptr_t)xs[i] ^ (uintptr_t)ys[i]) & 15u) == 0;
    const int per_launch = vec ? kVecMaxPairs : 1;
    if (n * pl.pieces * per_launch > 0x7fffffffLL) return IQA_ERR_SHAPE;
    for (int i = 0; i < n_pairs; i += per_launch) {
        const int np = n_pairs - i < per_launch ? n_pairs - i : per_launch;
        GenericParams g{};
        TileParams& p = g.tp;
        p.x = (const float*)xs[i]; p.y = (const float*)ys[i]; p.N = g2.W; p.H = g2.H; p.nt = nt;
        p.pitch_x = g2.pitch_x; p.pitch_y = g2.pitch_y;
        p.C1 = k.C1; p.C2 = k.C2; p.C = k.C; p.D = k.D;
        const Outputs o = out.offset((size_t)i * (size_t)n);
        p.lisi = o.lisi; p.auglisi = o.auglisi; p.sum_x = o.sum_x; p.sum_y = o.sum_y;
        p.lisi_num = o.lisi_num; p.aug_num = o.aug_num;
        p.ws = (ws && pl.pieces > 1) ? ws + (size_t)i * (size_t)n * pl.pieces : nullptr;
        g.N_T = N_T; g.pieces = pl.pieces;
        cudaError_t e;
        if (vec) {
            VecBatch b{};
            for (int j = 0; j < np; ++j) { b.x[j] = xs[i + j]; b.y[j] = ys[i + j]; }
            b.n_pairs = np;
            b.pair_minor = series_order && np > 1 && !knob(kKnobSeriesPairMajor) ? 1 : 0;
            e = by_pixel_type(g2.ptype, mode,
                [&](int m) { return m == kModeLisi  ? launch_generic_vec<kModeLisi, float>(g, b, n, pl.pieces, st)
                                    : m == kModeAug ? launch_generic_vec<kModeAug, float>(g, b, n, pl.pieces, st)
                                                    : launch_generic_vec<kModeFused, float>(g, b, n, pl.pieces, st); },
                [&](auto* t) { using T = std::remove_pointer_t<decltype(t)>;
                               return launch_generic_vec<kModeFused, T>(g, b, n, pl.pieces, st); });
        } else {
            e = by_pixel_type(g2.ptype, mode,
                [&](int m) { return m == kModeLisi  ? launch_generic_one<kModeLisi, float>(g, n, N_T, pl.pieces, st)
                                    : m == kModeAug ? launch_generic_one<kModeAug, float>(g, n, N_T, pl.pieces, st)
                                                    : launch_generic_one<kModeFused, float>(g, n, N_T, pl.pieces, st); },
                [&](auto* t) { using T = std::remove_pointer_t<decltype(t)>;
                               return launch_generic_one<kModeFused, T>(g, n, N_T, pl.pieces, st); });
        }
        if (e != cudaSuccess) return IQA_ERR_CUDA;
    }
    return IQA_OK;
}

// Which second pass a split-tile call takes: a function of (pieces, tiles per comparison) only, so that a batch and
// the same pairs one by one sum the pieces in the same order.
bool finalise_is_small(int pieces, long long n) { return pieces <= 32 && n >= 64; }

// S1-S4 for n_pairs pairs (xs[i], ys[i]) with the plan's kernel; `out` / `ws` point at pair 0.  The plan is
// downgraded to the generic kernels (before anything is launched) when a tensor map cannot be encoded.
int launch_pairs(int mode, const void* const* xs, const void* const* ys, int n_pairs, const Geom& g, int N_T,
                 const Consts& k, const Outputs& out, float4* ws, Plan& pl, cudaStream_t st, bool series_order = false) {
    if (pl.kind == kPlanTma) {
        std::vector<TmaLaunch> q;
        q.reserve((size_t)ceil_div(n_pairs, kMaxImages / 2));
        std::vector<const void*> imgs((size_t)2 * n_pairs);
        for (int i = 0; i < n_pairs; ++i) { imgs[2 * (size_t)i] = xs[i]; imgs[2 * (size_t)i + 1] = ys[i]; }
        if (prepare_tma(q, mode, kPairs, imgs.data(), n_pairs, 2, g, N_T, k, out, ws, pl)) return fire(q, st);
        generic_plan(pl, N_T);
    } else if (pl.kind == kPlanAny) {
        std::vector<AnyLaunch> q;
        q.reserve((size_t)ceil_div(n_pairs, kAnyMaxImages / 2));
        if (prepare_any(q, mode, xs, ys, n_pairs, g, N_T, k, out, ws, pl, series_order)) return fire(q, st);
        generic_plan(pl, N_T);
    }
    return launch_generic(mode, xs, ys, n_pairs, g, N_T, k, out, ws, pl, st, series_order);
}

// After S1-S4 of n_cmp comparisons: the second pass of split tiles, then Eqs. 3-4 per comparison.
int finish_comparisons(const Outputs& out, float* out2, int n_cmp, long long n, const Consts& k, float4* ws,
                       const Plan& pl, cudaStream_t st) {
    if (pl.pieces > 1) {                       // second pass over all tiles of the batch, fixed order
        TileParams p{};
        p.C1 = k.C1; p.C2 = k.C2; p.C = k.C; p.D = k.D;
        p.lisi = out.lisi; p.auglisi = out.auglisi; p.sum_x = out.sum_x; p.sum_y = out.sum_y;
        p.lisi_num = out.lisi_num; p.aug_num = out.aug_num;
        p.ws = ws;
        const int total = (int)(n * n_cmp);
        cudaError_t e;
        if (finalise_is_small(pl.pieces, n))
            e = launch(finalise_small_kernel, (unsigned)((total + kCtaThreads - 1) / kCtaThreads), kCtaThreads, 0, st,
                       p, pl.pieces, total);
        else
            e = launch(finalise_kernel, (unsigned)total, kCtaThreads, 0, st, p, pl.pieces);
        if (e != cudaSuccess) return IQA_ERR_CUDA;
    }
    if (out2) {                                // Eqs. 3-4 per comparison
        const unsigned cs = (unsigned)agg_cluster_size(n);
        if (launch_cluster(aggregate_kernel, (unsigned)n_cmp * cs, kAggThreads, 0, st, cs,
                   (const float*)out.lisi, (const float*)out.auglisi, (const float*)out.sum_x,
                   (const float*)out.sum_y, (int)n, k.C2, k.C, out2, (double*)nullptr) != cudaSuccess)
            return IQA_ERR_CUDA;
    }
    return cudaGetLastError() == cudaSuccess ? IQA_OK : IQA_ERR_CUDA;
}

// Shape of the images of a call: status and tile count.  `square`: the paper-named entry points keep the paper's
// requirement N % N_T == 0.
int status_of_geometry(const Geom& g, int N_T, bool square, long long* n_tiles) {
    if (square) {
        if (const int s = status_of_shape(g.W, N_T)) return s;
        *n_tiles = (long long)(g.W / N_T) * (g.W / N_T);
        return IQA_OK;
    }
    if (esize_of(g.ptype) == 0) return IQA_ERR_SHAPE;
    if (g.H <= 0 || g.W <= 0 || N_T <= 0 || g.H > kMaxN || g.W > kMaxN || g.pitch_x < g.W || g.pitch_y < g.W)
        return IQA_ERR_SHAPE;
    *n_tiles = (long long)ceil_div(g.W, N_T) * ceil_div(g.H, N_T);
    return *n_tiles > 0x7fffffffLL ? IQA_ERR_SHAPE : IQA_OK;
}

int validate_common(int mode, int n_cmp, const Geom& g, int N_T, bool square, float C1, float C2, float C, float D,
                    const Outputs& out, const float* out2) {
    if (n_cmp <= 0) return IQA_ERR_SHAPE;
    if ((mode & kModeLisi) && !out.lisi) return IQA_ERR_NULL;
    if ((mode & kModeAug) && !out.auglisi) return IQA_ERR_NULL;
    if (mode == kModeFused && (!out.sum_x || !out.sum_y)) return IQA_ERR_NULL;
    long long n = 0;
    if (const int s = status_of_geometry(g, N_T, square, &n)) return s;
    if (n * n_cmp > 0x7fffffffLL) return IQA_ERR_SHAPE;
    if ((mode & kModeLisi) && (!pos_normal(C1) || !pos_finite(C2) || !std::isfinite(D))) return IQA_ERR_PARAM;
    if ((mode & kModeAug) && !pos_finite(C)) return IQA_ERR_PARAM;
    if (out2 && (!pos_finite(C2) || !pos_finite(C))) return IQA_ERR_PARAM;
    return IQA_OK;
}

size_t pieces_bytes(long long n_cmp, long long n, int N_T) {
    const size_t mp = max_pieces(N_T);
    return mp > 1 ? (size_t)n_cmp * (size_t)n * mp * sizeof(float4) : 0;
}

// Shared body of every *_tiles / *_batch entry point: validation, then the launches.
// xs, ys: HOST arrays of n_pairs device pointers.  out2 (nullable): Eqs. 3-4 per pair.
int run_batch(int mode, const void* const* xs, const void* const* ys, int n_pairs, const Geom& g, int N_T, bool square,
              float C1, float C2, float C, float D, Outputs out, float* out2,
              void* workspace, size_t workspace_bytes, void* stream) {
    if (!xs || !ys) return IQA_ERR_NULL;
    if (n_pairs <= 0) return IQA_ERR_SHAPE;
    for (int i = 0; i < n_pairs; ++i)
        if (!xs[i] || !ys[i]) return IQA_ERR_NULL;
    if (const int s = validate_common(mode, n_pairs, g, N_T, square, C1, C2, C, D, out, out2)) return s;
    long long n = 0;
    status_of_geometry(g, N_T, square, &n);
    uintptr_t bits = 0;
    for (int i = 0; i < n_pairs; ++i) bits |= (uintptr_t)xs[i] | (uintptr_t)ys[i];
    if (bits & (uintptr_t)(esize_of(g.ptype) - 1)) return IQA_ERR_ALIGN;
    const size_t need = pieces_bytes(n_pairs, n, N_T);
    if (need > 0 && (!workspace || workspace_bytes < need)) return IQA_ERR_WORKSPACE;
    if (need > 0 && ((uintptr_t)workspace & 15u)) return IQA_ERR_ALIGN;

    cudaStream_t st = (cudaStream_t)stream;
    float4* ws = need > 0 ? (float4*)workspace : nullptr;
    out = out.for_mode(mode);
    const Consts k{C1, C2, C, D};
    // One plan per RUN of consecutive pairs of the same alignment class (the offset of x and y inside their 16-byte
    // lines, -1 when the two differ), each run planned exactly like a call of its own: one pair behind a shifted base
    // does not drag the aligned pairs of its batch onto the generic kernels, and every pair is summed in the order the
    // single-pair call would use.  A uniform batch -- the usual case -- is one run.
    const size_t ws_per_pair = (size_t)n * max_pieces(N_T);          // float4 slots; >= n * pieces of any plan
    // (a mixed batch must not fail half way: the one shape check a later run could still trip over is made up front)
    if (align_of(xs, n_pairs, ys, n_pairs).lo16 < 0 && (long long)ws_per_pair * kVecMaxPairs > 0x7fffffffLL)
        return IQA_ERR_SHAPE;
    for (int first = 0; first < n_pairs;) {
        const Align al = align_of(xs + first, 1, ys + first, 1);
        int np = 1;
        while (first + np < n_pairs && align_of(xs + first + np, 1, ys + first + np, 1).lo16 == al.lo16) ++np;
        Plan pl = make_plan(g, N_T, al, false, n_pairs);          // (the job's size is the call's, not the run's)
        const Outputs o = out.offset((size_t)first * (size_t)n);
        float4* w = ws ? ws + (size_t)first * ws_per_pair : nullptr;
        if (const int rc = launch_pairs(mode, xs + first, ys + first, np, g, N_T, k, o, w, pl, st)) return rc;
        if (const int rc = finish_comparisons(o, out2 ? out2 + 2 * (size_t)first : nullptr, np, n, k, w, pl, st)) return rc;
        first += np;
    }
    return IQA_OK;
}

// Time series: imgs = HOST array of n_images device pointers; K = n_images - 1
// comparisons, (I_0, I_k+1) or (I_k, I_k+1).  fp32 images with a power-of-two N_T take tma_kernel, which
// keeps the x box of every comparison in shared memory (each image is read from HBM once);
// everything else runs the K pair computations with the kernels of the pair entry points in series order
// (any_kernel / the 128-bit generic kernel: one launch per 32 comparisons, pair-minor, shared images from L2).
int run_series(const void* const* imgs, int n_images, int series, const Geom& g, int N_T, bool square,
               float C1, float C2, float C, float D, Outputs out, float* out2,
               void* workspace, size_t workspace_bytes, void* stream) {
    if (!imgs) return IQA_ERR_NULL;
    if (n_images < 2 || (series != kReference && series != kConsecutive)) return IQA_ERR_SHAPE;
    for (int i = 0; i < n_images; ++i)
        if (!imgs[i]) return IQA_ERR_NULL;
    const int K = n_images - 1;
    if (const int s = validate_common(kModeFused, K, g, N_T, square, C1, C2, C, D, out, out2)) return s;
    long long n = 0;
    status_of_geometry(g, N_T, square, &n);
    uintptr_t bits = 0;
    for (int i = 0; i < n_images; ++i) bits |= (uintptr_t)imgs[i];
    if (bits & (uintptr_t)(esize_of(g.ptype) - 1)) return IQA_ERR_ALIGN;
    const size_t need = pieces_bytes(K, n, N_T);
    if (need > 0 && (!workspace || workspace_bytes < need)) return IQA_ERR_WORKSPACE;
    if (need > 0 && ((uintptr_t)workspace & 15u)) return IQA_ERR_ALIGN;

    Plan pl = make_plan(g, N_T, align_of(imgs, n_images, imgs, 0), true, K);
    cudaStream_t st = (cudaStream_t)stream;
    float4* ws = need > 0 ? (float4*)workspace : nullptr;
    const Consts k{C1, C2, C, D};
    if (pl.kind == kPlanTma) {
        // chunks of at most kMaxImages images; consecutive chunks share one image
        std::vector<TmaLaunch> q;
        q.reserve((size_t)ceil_div(K, kMaxImages - 1));
        const void* chunk[kMaxImages];
        bool ok = true;
        for (int first = 0; first < K && ok; first += kMaxImages - 1) {       // first = first comparison of the chunk
            const int kc = K - first < kMaxImages - 1 ? K - first : kMaxImages - 1;
            chunk[0] = series == kReference ? imgs[0] : imgs[first];
            for (int i = 0; i < kc; ++i) chunk[1 + i] = imgs[first + 1 + i];
            ok = prepare_tma(q, kModeFused, series, chunk, 1, kc + 1, g, N_T, k, out.offset((size_t)first * (size_t)n),
                             ws ? ws + (size_t)first * (size_t)n * pl.pieces : nullptr, pl);
        }
        if (ok) {
            if (const int rc = fire(q, st)) return rc;
            return finish_comparisons(out, out2, K, n, k, ws, pl, st);
        }
        generic_plan(pl, N_T);
    }
    // pair by pair; a plan downgraded by one chunk stays downgraded for the rest (one finalise pass fits all)
    std::vector<const void*> xs((size_t)K), ys((size_t)K);
    for (int i = 0; i < K; ++i) {
        xs[i] = series == kReference ? imgs[0] : imgs[i];
        ys[i] = imgs[i + 1];
    }
    if (const int rc = launch_pairs(kModeFused, xs.data(), ys.data(), K, g, N_T, k, out, ws, pl, st, true)) return rc;
    return finish_comparisons(out, out2, K, n, k, ws, pl, st);
}

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

}  // namespace

// ---- built-in workspace of iqa_fused_tiles_static ------------------------------------------------------------
// For callers that cannot allocate device memory (include/iqa_tiles.h explains who): the partial sums of split
// tiles land here instead of in a caller-supplied workspace.  The array is part of the library's device image, so
// every GPU that loads this library holds these IQA_STATIC_WORKSPACE_BYTES until the process exits.  One array per
// device, shared by every call on that device and never cleared (nothing in it has to start at zero: the second pass
// reads only slots the first pass of the same call wrote); calls that overlap on the GPU race on it.
static __device__ __align__(256) unsigned char g_static_workspace[IQA_STATIC_WORKSPACE_BYTES];

namespace {

// In host code `g_static_workspace` is only the host-side handle of the symbol: handing it to a kernel would pass a
// host address.  Its device address differs from GPU to GPU and comes from cudaGetSymbolAddress, asked once per
// device with that device current and then kept.  Allocates nothing.
int static_workspace(void** ws) {
    static std::mutex mu;
    static void* addr[kMaxDevices] = {};
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return IQA_ERR_CUDA;
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[dev]) {
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, g_static_workspace) != cudaSuccess || !p) return IQA_ERR_CUDA;
        addr[dev] = p;
    }
    *ws = addr[dev];
    return IQA_OK;
}

}  // namespace

extern "C" {

const char* iqa_status_string(int status) {
    switch (status) {
        case IQA_OK: return "ok";
        case IQA_ERR_NULL: return "required pointer is NULL";
        case IQA_ERR_SHAPE: return "bad shape: need 0 < N_T <= N <= 2^20, N % N_T == 0, n_pairs >= 1, tile count < 2^31, a known pixel type";
        case IQA_ERR_PARAM: return "bad constant: C1 must be a normal float > 0, C2 and C finite and > 0, D finite";
        case IQA_ERR_ALIGN: return "pointer alignment: images to their element size, workspace 16-byte";
        case IQA_ERR_WORKSPACE: return "workspace missing or smaller than iqa_workspace_bytes / iqa_batch_workspace_bytes";
        case IQA_ERR_CUDA: return "CUDA launch or copy failed";
        case IQA_ERR_STATIC_LIMIT: return "iqa_fused_tiles_static: this shape needs more than IQA_STATIC_WORKSPACE_BYTES of workspace; call iqa_fused_tiles with a workspace of your own";
        default: return "unknown status";
    }
}

const char* iqa_version(void) { return "0.8.0"; }

int iqa_debug_knob(const char* name, int value) {
    if (!name) return -1;
    for (int i = 0; i < kNumKnobs; ++i)
        if (std::strcmp(name, kKnobNames[i]) == 0) return knobs().v[i].exchange(value, std::memory_order_relaxed);
    return -1;
}

size_t iqa_workspace_bytes(int N, int N_T) {
    if (status_of_shape(N, N_T) != IQA_OK) return 0;
    return workspace_bytes_for(1, N, N_T);
}

size_t iqa_batch_workspace_bytes(int n_pairs, int N, int N_T) {
    if (n_pairs <= 0 || status_of_shape(N, N_T) != IQA_OK) return 0;
    return workspace_bytes_for(n_pairs, N, N_T);
}

int iqa_lisi_tiles(const float* x, const float* y, int N, int N_T,
                   float C1, float C2, float D, float* lisi,
                   void* workspace, size_t workspace_bytes, void* stream) {
    const Outputs o{lisi, nullptr, nullptr, nullptr, nullptr, nullptr};
    const void* xs[1] = {x};
    const void* ys[1] = {y};
    return run_batch(kModeLisi, xs, ys, 1, square_geom(N), N_T, true, C1, C2, 1.0f, D, o, nullptr, workspace,
                     workspace_bytes, stream);
}

int iqa_auglisi_tiles(const float* x, const float* y, int N, int N_T, float C,
                      float* auglisi, void* workspace, size_t workspace_bytes, void* stream) {
    const Outputs o{nullptr, auglisi, nullptr, nullptr, nullptr, nullptr};
    const void* xs[1] = {x};
    const void* ys[1] = {y};
    return run_batch(kModeAug, xs, ys, 1, square_geom(N), N_T, true, 1.0f, 1.0f, C, 0.0f, o, nullptr, workspace,
                     workspace_bytes, stream);
}

int iqa_fused_tiles(const float* x, const float* y, int N, int N_T,
                    float C1, float C2, float C, float D,
                    float* lisi, float* auglisi, float* sum_x, float* sum_y,
                    float* lisi_num, float* auglisi_num,
                    void* workspace, size_t workspace_bytes, void* stream) {
    const Outputs o{lisi, auglisi, sum_x, sum_y, lisi_num, auglisi_num};
    const void* xs[1] = {x};
    const void* ys[1] = {y};
    return run_batch(kModeFused, xs, ys, 1, square_geom(N), N_T, true, C1, C2, C, D, o, nullptr, workspace,
                     workspace_bytes, stream);
}

// iqa_fused_tiles without a workspace argument and without any allocation: split-tile partial sums go to
// g_static_workspace (above).  Everything is validated, and a shape beyond the array refused, BEFORE the first CUDA call;
// the first call on a device that needs the array looks its address up (do that outside stream capture).
int iqa_fused_tiles_static(const float* x, const float* y, int N, int N_T,
                           float C1, float C2, float C, float D,
                           float* lisi, float* auglisi, float* sum_x, float* sum_y,
                           float* lisi_num, float* auglisi_num, void* stream) {
    const Outputs o{lisi, auglisi, sum_x, sum_y, lisi_num, auglisi_num};
    if (!x || !y) return IQA_ERR_NULL;
    if (const int s = validate_common(kModeFused, 1, square_geom(N), N_T, true, C1, C2, C, D, o, nullptr)) return s;
    if (((uintptr_t)x | (uintptr_t)y) & 3u) return IQA_ERR_ALIGN;
    const size_t need = workspace_bytes_for(1, N, N_T);
    if (need > (size_t)IQA_STATIC_WORKSPACE_BYTES) return IQA_ERR_STATIC_LIMIT;
    void* ws = nullptr;
    if (need > 0)
        if (const int s = static_workspace(&ws)) return s;
    const void* xs[1] = {x};
    const void* ys[1] = {y};
    return run_batch(kModeFused, xs, ys, 1, square_geom(N), N_T, true, C1, C2, C, D, o, nullptr, ws,
                     need > 0 ? (size_t)IQA_STATIC_WORKSPACE_BYTES : 0, stream);
}

int iqa_query_plan(const void* x, int pixel_type, int H, int W, long long pitch, int N_T, int series) {
    return iqa_query_plan_n(x, pixel_type, H, W, pitch, N_T, series, 0);
}

int iqa_query_plan_n(const void* x, int pixel_type, int H, int W, long long pitch, int N_T, int series, int n_cmp) {
    const int es = esize_of(pixel_type);
    if (!x || es == 0 || H <= 0 || W <= 0 || N_T <= 0 || n_cmp < 0 || pitch < W || ((uintptr_t)x & (uintptr_t)(es - 1))) return -1;
    const Geom g{H, W, pitch, pitch, pixel_type};
    const Plan pl = make_plan(g, N_T, align_of(&x, 1, &x, 0), series != 0, n_cmp > 0 ? n_cmp : 1 << 30);
    if (pl.kind == kPlanTma) return IQA_PLAN_TMA + pl.tma_cfg;
    // (a series runs any_kernel as one launch per 32 comparisons in pair-minor item order)
    return pl.kind == kPlanAny ? IQA_PLAN_TMA_ANY : IQA_PLAN_GENERIC;
}

size_t iqa_workspace_bytes_2d(int H, int W, int N_T) {
    if (H <= 0 || W <= 0 || N_T <= 0 || H > kMaxN || W > kMaxN) return 0;
    const size_t pieces = max_pieces(N_T);
    if (pieces <= 1) return 0;
    const size_t n = (size_t)ceil_div(H, N_T) * (size_t)ceil_div(W, N_T);
    return n * pieces * sizeof(float4);
}

int iqa_fused_tiles_2d_typed(const void* x, const void* y, int pixel_type,
                             int H, int W, long long pitch_x, long long pitch_y, int N_T,
                             float C1, float C2, float C, float D,
                             float* lisi, float* auglisi, float* sum_x, float* sum_y,
                             float* lisi_num, float* auglisi_num,
                             void* workspace, size_t workspace_bytes, void* stream) {
    const Outputs o{lisi, auglisi, sum_x, sum_y, lisi_num, auglisi_num};
    const Geom g{H, W, pitch_x, pitch_y, pixel_type};
    const void* xs[1] = {x};
    const void* ys[1] = {y};
    return run_batch(kModeFused, xs, ys, 1, g, N_T, false, C1, C2, C, D, o, nullptr, workspace, workspace_bytes, stream);
}

int iqa_fused_tiles_2d(const float* x, const float* y, int H, int W, long long pitch_x, long long pitch_y, int N_T,
                       float C1, float C2, float C, float D,
                       float* lisi, float* auglisi, float* sum_x, float* sum_y,
                       float* lisi_num, float* auglisi_num,
                       void* workspace, size_t workspace_bytes, void* stream) {
    return iqa_fused_tiles_2d_typed(x, y, IQA_PIXEL_F32, H, W, pitch_x, pitch_y, N_T, C1, C2, C, D, lisi, auglisi, sum_x,
                                    sum_y, lisi_num, auglisi_num, workspace, workspace_bytes, stream);
}

int iqa_fused_batch_2d_typed(const void* const* x_ptrs_host, const void* const* y_ptrs_host, int n_pairs, int pixel_type,
                             int H, int W, long long pitch, int N_T, float C1, float C2, float C, float D,
                             float* lisi, float* auglisi, float* sum_x, float* sum_y,
                             float* lisi_num, float* auglisi_num, float* out2,
                             void* workspace, size_t workspace_bytes, void* stream) {
    const Outputs o{lisi, auglisi, sum_x, sum_y, lisi_num, auglisi_num};
    const Geom g{H, W, pitch, pitch, pixel_type};
    return run_batch(kModeFused, x_ptrs_host, y_ptrs_host, n_pairs, g, N_T, false, C1, C2, C, D, o, out2,
                     workspace, workspace_bytes, stream);
}

int iqa_fused_batch_2d(const float* const* x_ptrs_host, const float* const* y_ptrs_host, int n_pairs,
                       int H, int W, long long pitch, int N_T, float C1, float C2, float C, float D,
                       float* lisi, float* auglisi, float* sum_x, float* sum_y,
                       float* lisi_num, float* auglisi_num, float* out2,
                       void* workspace, size_t workspace_bytes, void* stream) {
    return iqa_fused_batch_2d_typed((const void* const*)x_ptrs_host, (const void* const*)y_ptrs_host, n_pairs, IQA_PIXEL_F32,
                                    H, W, pitch, N_T, C1, C2, C, D, lisi, auglisi, sum_x, sum_y, lisi_num, auglisi_num,
                                    out2, workspace, workspace_bytes, stream);
}

int iqa_series_tiles_2d_typed(const void* const* img_ptrs_host, int n_images, int mode, int pixel_type,
                              int H, int W, long long pitch, int N_T, float C1, float C2, float C, float D,
                              float* lisi, float* auglisi, float* sum_x, float* sum_y,
                              float* lisi_num, float* auglisi_num, float* out2,
                              void* workspace, size_t workspace_bytes, void* stream) {
    const Outputs o{lisi, auglisi, sum_x, sum_y, lisi_num, auglisi_num};
    const int series = mode == IQA_SERIES_REFERENCE ? kReference : mode == IQA_SERIES_CONSECUTIVE ? kConsecutive : -1;
    const Geom g{H, W, pitch, pitch, pixel_type};
    return run_series(img_ptrs_host, n_images, series, g, N_T, false, C1, C2, C, D, o, out2,
                      workspace, workspace_bytes, stream);
}

int iqa_series_tiles_2d(const float* const* img_ptrs_host, int n_images, int mode,
                        int H, int W, long long pitch, int N_T, float C1, float C2, float C, float D,
                        float* lisi, float* auglisi, float* sum_x, float* sum_y,
                        float* lisi_num, float* auglisi_num, float* out2,
                        void* workspace, size_t workspace_bytes, void* stream) {
    return iqa_series_tiles_2d_typed((const void* const*)img_ptrs_host, n_images, mode, IQA_PIXEL_F32, H, W, pitch, N_T,
                                     C1, C2, C, D, lisi, auglisi, sum_x, sum_y, lisi_num, auglisi_num, out2,
                                     workspace, workspace_bytes, stream);
}

int iqa_fused_batch(const float* const* x_ptrs_host, const float* const* y_ptrs_host, int n_pairs,
                    int N, int N_T, float C1, float C2, float C, float D,
                    float* lisi, float* auglisi, float* sum_x, float* sum_y,
                    float* lisi_num, float* auglisi_num, float* out2,
                    void* workspace, size_t workspace_bytes, void* stream) {
    const Outputs o{lisi, auglisi, sum_x, sum_y, lisi_num, auglisi_num};
    return run_batch(kModeFused, (const void* const*)x_ptrs_host, (const void* const*)y_ptrs_host, n_pairs, square_geom(N),
                     N_T, true, C1, C2, C, D, o, out2, workspace, workspace_bytes, stream);
}

size_t iqa_series_workspace_bytes(int n_images, int N, int N_T) {
    if (n_images < 2 || status_of_shape(N, N_T) != IQA_OK) return 0;
    return workspace_bytes_for(n_images - 1, N, N_T);
}

int iqa_series_tiles(const float* const* img_ptrs_host, int n_images, int mode,
                     int N, int N_T, float C1, float C2, float C, float D,
                     float* lisi, float* auglisi, float* sum_x, float* sum_y,
                     float* lisi_num, float* auglisi_num, float* out2,
                     void* workspace, size_t workspace_bytes, void* stream) {
    const Outputs o{lisi, auglisi, sum_x, sum_y, lisi_num, auglisi_num};
    const int series = mode == IQA_SERIES_REFERENCE ? kReference : mode == IQA_SERIES_CONSECUTIVE ? kConsecutive : -1;
    return run_series((const void* const*)img_ptrs_host, n_images, series, square_geom(N), N_T, true, C1, C2, C, D, o, out2,
                      workspace, workspace_bytes, stream);
}

int iqa_aggregate(const float* lisi, const float* auglisi,
                  const float* sum_x, const float* sum_y, int n_tiles,
                  float C2, float C, float* out2, void* stream) {
    if (!lisi || !auglisi || !sum_x || !sum_y || !out2) return IQA_ERR_NULL;
    if (n_tiles <= 0) return IQA_ERR_SHAPE;
    if (!pos_finite(C2) || !pos_finite(C)) return IQA_ERR_PARAM;
    const unsigned cs = (unsigned)agg_cluster_size(n_tiles);
    if (launch_cluster(aggregate_kernel, cs, kAggThreads, 0, (cudaStream_t)stream, cs, lisi, auglisi, sum_x, sum_y,
               n_tiles, C2, C, out2, (double*)nullptr) != cudaSuccess)
        return IQA_ERR_CUDA;
    return cudaGetLastError() == cudaSuccess ? IQA_OK : IQA_ERR_CUDA;
}

int iqa_aggregate_partial(const float* lisi, const float* auglisi,
                          const float* sum_x, const float* sum_y, int n_tiles,
                          float C2, float C, double* sums4, void* stream) {
    if (!lisi || !auglisi || !sum_x || !sum_y || !sums4) return IQA_ERR_NULL;
    if (n_tiles <= 0) return IQA_ERR_SHAPE;
    if (!pos_finite(C2) || !pos_finite(C)) return IQA_ERR_PARAM;
    if ((uintptr_t)sums4 & 7u) return IQA_ERR_ALIGN;
    const unsigned cs = (unsigned)agg_cluster_size(n_tiles);
    if (launch_cluster(aggregate_kernel, cs, kAggThreads, 0, (cudaStream_t)stream, cs, lisi, auglisi, sum_x, sum_y,
               n_tiles, C2, C, (float*)nullptr, sums4) != cudaSuccess)
        return IQA_ERR_CUDA;
    return cudaGetLastError() == cudaSuccess ? IQA_OK : IQA_ERR_CUDA;
}

int iqa_aggregate_finish(const double* sums4, long long n_tiles_total, float C2, float C, float* out2, void* stream) {
    if (!sums4 || !out2) return IQA_ERR_NULL;
    if (n_tiles_total <= 0) return IQA_ERR_SHAPE;
    if (!pos_finite(C2) || !pos_finite(C)) return IQA_ERR_PARAM;
    if ((uintptr_t)sums4 & 7u) return IQA_ERR_ALIGN;
    if (launch(aggregate_finish_kernel, 1u, 32u, 0, (cudaStream_t)stream, sums4, (double)n_tiles_total, C2, C, out2) !=
        cudaSuccess)
        return IQA_ERR_CUDA;
    return cudaGetLastError() == cudaSuccess ? IQA_OK : IQA_ERR_CUDA;
}

int iqa_tiles_below(const float* values, int n_tiles, int n_maps, float threshold,
                    int* indices, int capacity, int* counts, void* stream) {
    if (!values || !counts || (capacity > 0 && !indices)) return IQA_ERR_NULL;
    if (n_tiles <= 0 || n_maps <= 0 || capacity < 0) return IQA_ERR_SHAPE;
    if (threshold != threshold) return IQA_ERR_PARAM;
    const int cs = knob(kKnobCandNoCluster) ? 0 : cand_cluster_size(n_tiles);
    const cudaError_t e = cs > 0
        ? launch_cluster(below_cluster_kernel, (unsigned)n_maps * (unsigned)cs, (unsigned)kCandThreads, 0,
                         (cudaStream_t)stream, (unsigned)cs, values, n_tiles, threshold, indices, capacity, counts)
        : launch(below_kernel, (unsigned)n_maps, (unsigned)cand_threads(n_tiles), 0, (cudaStream_t)stream, values,
                 n_tiles, threshold, indices, capacity, counts);
    if (e != cudaSuccess) return IQA_ERR_CUDA;
    return cudaGetLastError() == cudaSuccess ? IQA_OK : IQA_ERR_CUDA;
}

int iqa_tiles_bottom_k(const float* values, int n_tiles, int n_maps, int k,
                       int* indices, float* vals, void* stream) {
    if (!values || !indices) return IQA_ERR_NULL;
    if (n_tiles <= 0 || n_maps <= 0 || k <= 0 || k > kMaxBottomK) return IQA_ERR_SHAPE;
    const int cs = knob(kKnobCandNoCluster) ? 0 : cand_cluster_size(n_tiles);
    const cudaError_t e = cs > 0
        ? launch_cluster(bottom_k_cluster_kernel, (unsigned)n_maps * (unsigned)cs, (unsigned)kCandThreads, 0,
                         (cudaStream_t)stream, (unsigned)cs, values, n_tiles, k, indices, vals)
        : launch(bottom_k_kernel, (unsigned)n_maps, (unsigned)cand_threads(n_tiles), 0, (cudaStream_t)stream, values,
                 n_tiles, k, indices, vals, 0.0f, (int*)nullptr, 0, (int*)nullptr);
    if (e != cudaSuccess) return IQA_ERR_CUDA;
    return cudaGetLastError() == cudaSuccess ? IQA_OK : IQA_ERR_CUDA;
}

namespace {
int check_find_args(int index, int k, const int* bottom_idx, float threshold, const int* below_idx, int capacity,
                    const int* below_counts) {
    if (index != IQA_FIND_LISI && index != IQA_FIND_AUGLISI) return IQA_ERR_SHAPE;
    if (k < 0 || k > kMaxBottomK || capacity < 0) return IQA_ERR_SHAPE;
    if (k == 0 && !below_counts) return IQA_ERR_NULL;
    if (k > 0 && !bottom_idx) return IQA_ERR_NULL;
    if (below_counts && capacity > 0 && !below_idx) return IQA_ERR_NULL;
    if (below_counts && threshold != threshold) return IQA_ERR_PARAM;
    return IQA_OK;
}
// The candidate lists of K matrices of n tiles behind the series kernels of the same call.
int launch_find(const float* values, int n, int K, int k, int* bottom_idx, float* bottom_val, float threshold,
                int* below_idx, int capacity, int* below_counts, void* stream) {
    // both lists of a matrix that one CTA keeps in registers: ONE launch, the matrix is read once
    if (k > 0 && below_counts && n <= cand_threads(n) * kCandPerThread) {
        if (launch(bottom_k_kernel, (unsigned)K, (unsigned)cand_threads(n), 0, (cudaStream_t)stream, values, n, k,
                   bottom_idx, bottom_val, threshold, below_idx, capacity, below_counts) != cudaSuccess)
            return IQA_ERR_CUDA;
        return cudaGetLastError() == cudaSuccess ? IQA_OK : IQA_ERR_CUDA;
    }
    if (k > 0)
        if (const int rc = iqa_tiles_bottom_k(values, n, K, k, bottom_idx, bottom_val, stream)) return rc;
    if (below_counts)
        if (const int rc = iqa_tiles_below(values, n, K, threshold, below_idx, capacity, below_counts, stream)) return rc;
    return IQA_OK;
}
}  // namespace

int iqa_series_find(const float* const* img_ptrs_host, int n_images, int mode,
                    int N, int N_T, float C1, float C2, float C, float D,
                    float* lisi, float* auglisi, float* sum_x, float* sum_y,
                    float* lisi_num, float* auglisi_num, float* out2,
                    void* workspace, size_t workspace_bytes,
                    int index, int k, int* bottom_idx, float* bottom_val,
                    float threshold, int* below_idx, int capacity, int* below_counts, void* stream) {
    // every argument of the candidate step is checked before the series is enqueued
    if (const int rc = check_find_args(index, k, bottom_idx, threshold, below_idx, capacity, below_counts)) return rc;
    if (const int rc = iqa_series_tiles(img_ptrs_host, n_images, mode, N, N_T, C1, C2, C, D, lisi, auglisi, sum_x, sum_y,
                                        lisi_num, auglisi_num, out2, workspace, workspace_bytes, stream))
        return rc;
    return launch_find(index == IQA_FIND_LISI ? lisi : auglisi, (N / N_T) * (N / N_T), n_images - 1, k, bottom_idx,
                       bottom_val, threshold, below_idx, capacity, below_counts, stream);
}

int iqa_series_find_2d_typed(const void* const* img_ptrs_host, int n_images, int mode, int pixel_type,
                             int H, int W, long long pitch, int N_T, float C1, float C2, float C, float D,
                             float* lisi, float* auglisi, float* sum_x, float* sum_y,
                             float* lisi_num, float* auglisi_num, float* out2,
                             void* workspace, size_t workspace_bytes,
                             int index, int k, int* bottom_idx, float* bottom_val,
                             float threshold, int* below_idx, int capacity, int* below_counts, void* stream) {
    if (const int rc = check_find_args(index, k, bottom_idx, threshold, below_idx, capacity, below_counts)) return rc;
    if (const int rc = iqa_series_tiles_2d_typed(img_ptrs_host, n_images, mode, pixel_type, H, W, pitch, N_T, C1, C2, C, D,
                                                 lisi, auglisi, sum_x, sum_y, lisi_num, auglisi_num, out2, workspace,
                                                 workspace_bytes, stream))
        return rc;
    return launch_find(index == IQA_FIND_LISI ? lisi : auglisi, ceil_div(H, N_T) * ceil_div(W, N_T), n_images - 1, k,
                       bottom_idx, bottom_val, threshold, below_idx, capacity, below_counts, stream);
}

int iqa_merge_tiles_batch(const float* lisi, const float* auglisi,
                          const float* sum_x, const float* sum_y, int nt, int g, int n_maps,
                          float C2, float C,
                          float* lisi_out, float* auglisi_out,
                          float* sum_x_out, float* sum_y_out, void* stream) {
    if (!lisi || !auglisi || !sum_x || !sum_y || !lisi_out || !auglisi_out || !sum_x_out || !sum_y_out)
        return IQA_ERR_NULL;
    if (nt <= 0 || g <= 0 || g > nt || nt % g != 0 || n_maps <= 0 || (long long)nt * nt * n_maps > 0x7fffffffLL)
        return IQA_ERR_SHAPE;
    if (!pos_finite(C2) || !pos_finite(C)) return IQA_ERR_PARAM;
    const long long n_out = (long long)(nt / g) * (nt / g) * n_maps;
    const unsigned grid = (unsigned)((n_out + 7) / 8);
    if (launch(merge_kernel, grid, 256u, 0, (cudaStream_t)stream, lisi, auglisi, sum_x, sum_y, nt, g, n_maps, C2, C,
               lisi_out, auglisi_out, sum_x_out, sum_y_out) != cudaSuccess)
        return IQA_ERR_CUDA;
    return cudaGetLastError() == cudaSuccess ? IQA_OK : IQA_ERR_CUDA;
}

int iqa_pyramid_levels(int nty, int ntx) {
    if (nty <= 0 || ntx <= 0) return 0;
    int L = 0;
    while ((1 << L) < (nty > ntx ? nty : ntx)) ++L;
    return L;
}

size_t iqa_pyramid_tiles(int nty, int ntx) {
    const int L = iqa_pyramid_levels(nty, ntx);
    size_t total = 0;
    for (int j = 1; j <= L; ++j) total += (size_t)ceil_div(nty, 1 << j) * (size_t)ceil_div(ntx, 1 << j);
    return total;
}

int iqa_pyramid(const float* lisi, const float* auglisi, const float* sum_x, const float* sum_y,
                int nty, int ntx, int n_maps, float C2, float C,
                float* lisi_out, float* auglisi_out, float* sum_x_out, float* sum_y_out, void* stream) {
    if (!lisi || !auglisi || !sum_x || !sum_y) return IQA_ERR_NULL;
    if (nty <= 0 || ntx <= 0 || n_maps <= 0 || (long long)nty * ntx * n_maps > 0x7fffffffLL) return IQA_ERR_SHAPE;
    if (!pos_finite(C2) || !pos_finite(C)) return IQA_ERR_PARAM;
    const int L = iqa_pyramid_levels(nty, ntx);
    if (L == 0) return IQA_OK;                                // a 1 x 1 matrix is its own top: no level to emit
    if (!lisi_out || !auglisi_out || !sum_x_out || !sum_y_out) return IQA_ERR_NULL;
    if (L > kPyrMaxLevels) return IQA_ERR_SHAPE;
    PyramidParams p{};
    p.n_levels = L; p.nty = nty; p.ntx = ntx; p.n_maps = n_maps;
    long long off = 0, cta = 0;
    for (int j = 1; j <= L; ++j) {
        PyramidLevel& lv = p.lv[j - 1];
        lv.shift = j;
        lv.nby = ceil_div(nty, 1 << j);
        lv.nbx = ceil_div(ntx, 1 << j);
        const long long side = 1LL << j;
        lv.cta_mode = side * side > kPyrWarpTiles;
        lv.out_off = off;
        lv.first_cta = (unsigned)cta;
        const long long units = (long long)lv.nby * lv.nbx * n_maps;
        off += (long long)lv.nby * lv.nbx;
        cta += lv.cta_mode ? units : (units + 7) / 8;
    }
    p.out_per_map = off;
    if (cta > 0x7fffffffLL) return IQA_ERR_SHAPE;
    if (launch(pyramid_kernel, (unsigned)cta, 256u, 0, (cudaStream_t)stream, lisi, auglisi, sum_x, sum_y, p, C2, C,
               lisi_out, auglisi_out, sum_x_out, sum_y_out) != cudaSuccess)
        return IQA_ERR_CUDA;
    return cudaGetLastError() == cudaSuccess ? IQA_OK : IQA_ERR_CUDA;
}

int iqa_merge_tiles(const float* lisi, const float* auglisi,
                    const float* sum_x, const float* sum_y, int nt, int g,
                    float C2, float C,
                    float* lisi_out, float* auglisi_out,
                    float* sum_x_out, float* sum_y_out, void* stream) {
    return iqa_merge_tiles_batch(lisi, auglisi, sum_x, sum_y, nt, g, 1, C2, C, lisi_out, auglisi_out, sum_x_out,
                                 sum_y_out, stream);
}

size_t iqa_host_scratch_bytes(int N, int N_T) { return iqa_host_scratch_bytes_typed(N, N_T, IQA_PIXEL_F32); }

size_t iqa_host_scratch_bytes_typed(int N, int N_T, int pixel_type) {
    if (status_of_shape(N, N_T) != IQA_OK || esize_of(pixel_type) == 0) return 0;
    const size_t img = align_up((size_t)N * (size_t)N * (size_t)esize_of(pixel_type), 256);
    const size_t n = (size_t)(N / N_T) * (size_t)(N / N_T);
    const size_t per_tile = align_up(n * sizeof(float), 256);
    return 2 * img + 4 * per_tile + 256 + align_up(workspace_bytes_for(1, N, N_T), 256);
}

namespace {
int fused_host_impl(const void* x_host, const void* y_host, int ptype, int N, int N_T,
                    float C1, float C2, float C, float D,
                    float* lisi_host, float* auglisi_host,
                    float* sum_x_host, float* sum_y_host, float* out2_host,
                    void* dev_scratch, size_t dev_scratch_bytes, void* stream, bool synchronise) {
    if (!x_host || !y_host || !dev_scratch) return IQA_ERR_NULL;
    if (esize_of(ptype) == 0) return IQA_ERR_SHAPE;
    if (const int s = status_of_shape(N, N_T)) return s;
    if (!pos_normal(C1) || !pos_finite(C2) || !pos_finite(C) || !std::isfinite(D)) return IQA_ERR_PARAM;
    if (dev_scratch_bytes < iqa_host_scratch_bytes_typed(N, N_T, ptype)) return IQA_ERR_WORKSPACE;
    if ((uintptr_t)dev_scratch & 255u) return IQA_ERR_ALIGN;

    cudaStream_t st = (cudaStream_t)stream;
    const size_t img_bytes = (size_t)N * (size_t)N * (size_t)esize_of(ptype);
    const size_t img = align_up(img_bytes, 256);
    const size_t n = (size_t)(N / N_T) * (size_t)(N / N_T);
    const size_t per_tile = align_up(n * sizeof(float), 256);
    char* base = (char*)dev_scratch;
    void* xd = base;
    void* yd = base + img;
    float* d_lisi = (float*)(base + 2 * img);
    float* d_aug = (float*)(base + 2 * img + per_tile);
    float* d_sx = (float*)(base + 2 * img + 2 * per_tile);
    float* d_sy = (float*)(base + 2 * img + 3 * per_tile);
    float* d_out2 = (float*)(base + 2 * img + 4 * per_tile);
    void* ws = base + 2 * img + 4 * per_tile + 256;
    const size_t ws_bytes = workspace_bytes_for(1, N, N_T);

    if (cudaMemcpyAsync(xd, x_host, img_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) return IQA_ERR_CUDA;
    if (cudaMemcpyAsync(yd, y_host, img_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) return IQA_ERR_CUDA;
    // (the uploaded pixels are computed on as they are: no conversion pass, 2 sizeof(pixel) bytes per pixel pair over PCIe)
    const void* xs[1] = {xd};
    const void* ys[1] = {yd};
    const Outputs o{d_lisi, d_aug, d_sx, d_sy, nullptr, nullptr};
    Geom g = square_geom(N);
    g.ptype = ptype;
    const int rc = run_batch(kModeFused, xs, ys, 1, g, N_T, true, C1, C2, C, D, o, d_out2, ws_bytes ? ws : nullptr, ws_bytes,
                             stream);
    if (rc != IQA_OK) return rc;
    const size_t nb = n * sizeof(float);
    cudaError_t e = cudaSuccess;
    if (lisi_host && e == cudaSuccess) e = cudaMemcpyAsync(lisi_host, d_lisi, nb, cudaMemcpyDeviceToHost, st);
    if (auglisi_host && e == cudaSuccess) e = cudaMemcpyAsync(auglisi_host, d_aug, nb, cudaMemcpyDeviceToHost, st);
    if (sum_x_host && e == cudaSuccess) e = cudaMemcpyAsync(sum_x_host, d_sx, nb, cudaMemcpyDeviceToHost, st);
    if (sum_y_host && e == cudaSuccess) e = cudaMemcpyAsync(sum_y_host, d_sy, nb, cudaMemcpyDeviceToHost, st);
    if (out2_host && e == cudaSuccess) e = cudaMemcpyAsync(out2_host, d_out2, 2 * sizeof(float), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && synchronise) e = cudaStreamSynchronize(st);
    return e == cudaSuccess ? IQA_OK : IQA_ERR_CUDA;
}
}  // namespace

int iqa_fused_host(const float* x_host, const float* y_host, int N, int N_T,
                   float C1, float C2, float C, float D,
                   float* lisi_host, float* auglisi_host,
                   float* sum_x_host, float* sum_y_host, float* out2_host,
                   void* dev_scratch, size_t dev_scratch_bytes, void* stream) {
    return fused_host_impl(x_host, y_host, IQA_PIXEL_F32, N, N_T, C1, C2, C, D, lisi_host, auglisi_host, sum_x_host,
                           sum_y_host, out2_host, dev_scratch, dev_scratch_bytes, stream, true);
}

int iqa_fused_host_async(const float* x_host, const float* y_host, int N, int N_T,
                         float C1, float C2, float C, float D,
                         float* lisi_host, float* auglisi_host,
                         float* sum_x_host, float* sum_y_host, float* out2_host,
                         void* dev_scratch, size_t dev_scratch_bytes, void* stream) {
    return fused_host_impl(x_host, y_host, IQA_PIXEL_F32, N, N_T, C1, C2, C, D, lisi_host, auglisi_host, sum_x_host,
                           sum_y_host, out2_host, dev_scratch, dev_scratch_bytes, stream, false);
}

int iqa_fused_host_typed(const void* x_host, const void* y_host, int pixel_type, int N, int N_T,
                         float C1, float C2, float C, float D,
                         float* lisi_host, float* auglisi_host,
                         float* sum_x_host, float* sum_y_host, float* out2_host,
                         void* dev_scratch, size_t dev_scratch_bytes, void* stream) {
    return fused_host_impl(x_host, y_host, pixel_type, N, N_T, C1, C2, C, D, lisi_host, auglisi_host, sum_x_host,
                           sum_y_host, out2_host, dev_scratch, dev_scratch_bytes, stream, true);
}

int iqa_fused_host_typed_async(const void* x_host, const void* y_host, int pixel_type, int N, int N_T,
                               float C1, float C2, float C, float D,
                               float* lisi_host, float* auglisi_host,
                               float* sum_x_host, float* sum_y_host, float* out2_host,
                               void* dev_scratch, size_t dev_scratch_bytes, void* stream) {
    return fused_host_impl(x_host, y_host, pixel_type, N, N_T, C1, C2, C, D, lisi_host, auglisi_host, sum_x_host,
                           sum_y_host, out2_host, dev_scratch, dev_scratch_bytes, stream, false);
}

}  // extern "C"
