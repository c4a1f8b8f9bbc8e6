// =============================================================================
// iqa_tiles.cu -- the C ABI of include/iqa_tiles.h: argument validation, the N_T-dependent
// choice of mapping, and the launches.  No torch types, no allocation; the only thing kept
// between calls is a per-device cache of launch geometry (SM count, CTAs per SM).
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -shared -Xcompiler -fPIC
// =============================================================================
#include "../../include/iqa_tiles.h"

#include <atomic>
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <utility>

#include "iqa_aggregate.cuh"
#include "iqa_candidates.cuh"
#include "iqa_kernels.cuh"
#include "iqa_stream.cuh"
#include "iqa_tma.cuh"

namespace {

using namespace iqa;

constexpr int kMaxN = 1 << 20;   // 2^40 pixels; keeps every grid and tile index inside int
constexpr int kMaxDevices = 64;

bool is_pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }
int ilog2(int v) { int l = 0; while ((1 << l) < v) ++l; return l; }
bool pos_finite(float v) { return std::isfinite(v) && v > 0.0f; }

int env_int(const char* name, int dflt) {
    const char* s = std::getenv(name);
    return (s && *s) ? std::atoi(s) : dflt;
}

// ---- stream-kernel variants (rows per warp and stage K, ring depth, CTAs per SM) -----------
// Measured on B200 (profiles/r01*_variants.md): 48-64 KiB of copies in
// flight per SM is the sweet spot; deeper rings or more CTAs lose DRAM locality (down to
// 6.1-6.4 TB/s), fewer warps lose latency hiding.  Variants 0 and 1 are within 1 % of each other.
//   variant 0  K=4, depth 2, 2 CTAs/SM  (stage = 32 rows, 68 KiB smem/CTA, 64 KiB in flight per SM)  default
//   variant 1  K=2, depth 2, 3 CTAs/SM  (stage = 16 rows, 36 KiB smem/CTA, 48 KiB in flight per SM)
//   variant 2  K=8, depth 2, 1 CTA/SM   (stage = 64 rows, 132 KiB smem/CTA)  mapping-independence tests only
// The default path is the TMA-fed kernel of iqa_tma.cuh (kTmaConfigs below); the cp.async variants stay as the
// fallback when a tensor map cannot be encoded and for the mapping-independence tests.
// IQA_FORCE_VARIANT=v selects one of them (debug / tuning knob); all kernels agree to ~1e-7 relative.
constexpr int kNumVariants = 3;
struct VariantInfo { int K, depth, min_ctas; };
constexpr VariantInfo kVariants[kNumVariants] = {{4, 2, 2}, {2, 2, 3}, {8, 2, 1}};

using StreamFn = void (*)(const BatchParams);

template <int MODE>
StreamFn stream_fn(int variant) {
    switch (variant) {
        case 1: return stream_kernel<MODE, 2, 2, 3>;
        case 2: return stream_kernel<MODE, 8, 2, 1>;
        default: return stream_kernel<MODE, 4, 2, 2>;
    }
}
StreamFn stream_fn(int mode, int variant) {
    switch (mode) {
        case kModeLisi: return stream_fn<kModeLisi>(variant);
        case kModeAug: return stream_fn<kModeAug>(variant);
        default: return stream_fn<kModeFused>(variant);
    }
}
size_t stream_smem(int variant) {
    switch (variant) {
        case 1: return stream_smem_bytes<2, 2>();
        case 2: return stream_smem_bytes<8, 2>();
        default: return stream_smem_bytes<4, 2>();
    }
}

using TmaFn = void (*)(const TmaParams);

// TMA kernel configurations: {box slots per CTA, rows per warp and box}.  Measured on B200
// (profiles/r01g_tma_configs.md): pairs are HBM-bound and want FEW bytes in flight (config 1: two
// 16 KiB boxes in flight per CTA while two are consumed; six boxes lose 3-6 % to DRAM locality, as
// the cp.async variants did); the series modes keep S + 1 boxes alive and want the deeper ring of
// config 0.  IQA_TMA_CONFIG=c forces one (tuning knob).
struct TmaConfig { int boxes, rpw; };
constexpr int kNumTmaConfigs = 5;
constexpr TmaConfig kTmaConfigs[kNumTmaConfigs] = {{6, 4}, {4, 4}, {8, 2}, {6, 2}, {4, 2}};

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

// Tensor map of one H x W fp32 row-major image with a row pitch (in elements): boxes of 128 columns x box_rows rows, no swizzle (a box
// lands as [box_rows][128] floats), out-of-bounds elements read as zero.  Needs a 16-byte aligned base
// and pitch % 4 == 0 (row pitch a multiple of 16 bytes); W itself is free.
bool encode_image_map(CUtensorMap* map, const float* img, int H, int W, long long pitch, int box_rows) {
    const EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) return false;
    const cuuint64_t dims[2] = {(cuuint64_t)W, (cuuint64_t)H};
    const cuuint64_t strides[1] = {(cuuint64_t)pitch * sizeof(float)};
    const cuuint32_t box[2] = {(cuuint32_t)kUnitCols, (cuuint32_t)box_rows};
    const cuuint32_t estr[2] = {1u, 1u};
    return enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2u, const_cast<float*>(img), dims, strides, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// Per-device launch geometry, filled on first use (benign race: every thread computes the same values).
struct Geometry { std::atomic<int> ready{0}; int sms; int ctas[3][kNumVariants]; int tma_ctas[kNumTmaConfigs]; };
Geometry g_geo[kMaxDevices];

const Geometry* geometry() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return nullptr;
    Geometry& g = g_geo[dev];
    if (g.ready.load(std::memory_order_acquire)) return &g;
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) return nullptr;
    for (int m = 0; m < 3; ++m)
        for (int v = 0; v < kNumVariants; ++v) {
            StreamFn fn = stream_fn(m + 1, v);
            const size_t smem = stream_smem(v);
            if (cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return nullptr;
            int occ = 0;
            if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, kCtaThreads, smem) != cudaSuccess || occ <= 0) return nullptr;
            g.ctas[m][v] = occ < kVariants[v].min_ctas ? occ : kVariants[v].min_ctas;
        }
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
    g.sms = sms;
    g.ready.store(1, std::memory_order_release);
    return &g;
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
    static const bool no_pdl = env_int("IQA_NO_PDL", 0) != 0;
    if (!no_pdl) {
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

// How (N, N_T) is mapped onto CTAs.  DESIGN.md "Mapping".
enum PlanKind { kPlanGeneric = 0, kPlanStream = 1, kPlanTma = 2 };
struct Plan {
    PlanKind kind;     // generic kernel / cp.async stream kernel / TMA kernel
    int variant;       // stream: index into kVariants
    int tma_cfg;       // tma: index into kTmaConfigs
    int item_rows;     // stream, tma: R
    int pieces_x, pieces_y, pieces;   // pieces per tile; pieces == 1 -> finished inside one CTA
};

constexpr int kSplitItemRows = 64;   // tiles of side >= 128: items of 128 x 64, pieces to the workspace

// General image geometry of the 2-D entry point (pairs only): x has pitch_x, y has pitch_y.
struct Geom2D { int H, W; long long pitch_x, pitch_y; };

// first_image: one image of the call (the TMA path is taken only when its tensor map encodes).
Plan make_plan(int N, int N_T, bool aligned16, const float* first_image, bool series, const Geom2D* g2 = nullptr) {
    Plan pl{};
    const bool fast = is_pow2(N_T) && N_T >= 8 && aligned16 && !env_int("IQA_FORCE_GENERIC", 0);
    pl.kind = fast ? kPlanTma : kPlanGeneric;
    if (fast) {
        const int forced = env_int("IQA_FORCE_VARIANT", -1);     // debug knob (tests: mapping independence)
        if (forced >= 0 && forced < kNumVariants && !g2) { pl.kind = kPlanStream; pl.variant = forced; }
        if (pl.kind == kPlanTma) {
            const int dflt = series ? 0 : 1;
            const int c = env_int("IQA_TMA_CONFIG", dflt);
            pl.tma_cfg = c >= 0 && c < kNumTmaConfigs ? c : dflt;
            // the series modes keep S + 1 boxes alive (S = 64 / box rows for N_T >= 64): small rings fall back
            if (series && kTmaConfigs[pl.tma_cfg].boxes < 64 / (kWarpsPerCta * kTmaConfigs[pl.tma_cfg].rpw) + 2) pl.tma_cfg = 0;
            CUtensorMap probe;
            const bool ok = g2 ? encode_image_map(&probe, first_image, g2->H, g2->W, g2->pitch_x, kWarpsPerCta * kTmaConfigs[pl.tma_cfg].rpw)
                               : encode_image_map(&probe, first_image, N, N, N, kWarpsPerCta * kTmaConfigs[pl.tma_cfg].rpw);
            if (!ok) { pl.kind = g2 ? kPlanGeneric : kPlanStream; pl.variant = 0; }
        }
        const int rs = pl.kind == kPlanTma ? kWarpsPerCta * kTmaConfigs[pl.tma_cfg].rpw
                                           : kWarpsPerCta * kVariants[pl.variant].K;   // stage height
        if (N_T <= 64) {
            pl.item_rows = N_T > rs ? N_T : rs;                  // whole tiles inside one item
            pl.pieces_x = pl.pieces_y = 1;
        } else {
            pl.item_rows = kSplitItemRows;
            pl.pieces_x = N_T / kUnitCols;
            pl.pieces_y = N_T / kSplitItemRows;
        }
    }
    if (pl.kind == kPlanGeneric) {
        pl.pieces_x = 1;
        pl.pieces_y = (N_T + kGenericRows - 1) / kGenericRows;
    }
    pl.pieces = pl.pieces_x * pl.pieces_y;
    return pl;
}

// Pieces per tile in the worst case over the mappings a call may take (tma, stream or generic).
size_t max_pieces(int N_T) {
    if (N_T <= 64) return 1;                                      // every path finishes tiles inside one CTA
    size_t pieces = (size_t)(N_T + kGenericRows - 1) / kGenericRows;
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

// The TMA kernel over n_groups groups of M images (imgs[g * M + i], HOST array of device pointers);
// `out` and `ws` point at the first comparison of the first group.  n_groups * M may exceed
// kMaxImages (several launches); M itself may not.
int launch_tma(int mode, int series, const float* const* imgs, int n_groups, int M, int N, int N_T, const Consts& k,
               const Outputs& out, float4* ws, const Plan& pl, cudaStream_t st, const Geom2D* g2 = nullptr) {
    const Geometry* geo = geometry();
    TmaFn fn = tma_fn(mode, series, pl.tma_cfg);
    const int box_rows = kWarpsPerCta * kTmaConfigs[pl.tma_cfg].rpw;
    if (!geo || !fn || geo->tma_ctas[pl.tma_cfg] <= 0 || M < 2 || M > kMaxImages) return IQA_ERR_CUDA;
    const int H = g2 ? g2->H : N, W = g2 ? g2->W : N;
    const int ntx = (W + N_T - 1) / N_T, nty = (H + N_T - 1) / N_T;
    const long long n = (long long)ntx * nty;
    // split tiles: the items cover the whole tile grid, so that every piece of an edge tile is written
    // (boxes entirely outside the image are zero-filled by the TMA unit without touching memory)
    const int units_x = pl.pieces > 1 ? ntx * pl.pieces_x : (W + kUnitCols - 1) / kUnitCols;
    const int units_y = pl.pieces > 1 ? nty * pl.pieces_y : (H + pl.item_rows - 1) / pl.item_rows;
    const long long items_per_group = (long long)units_x * units_y;
    const int groups_per_launch = kMaxImages / M;
    if (items_per_group * groups_per_launch > 0x7fffffffLL) return IQA_ERR_SHAPE;
    for (int first = 0; first < n_groups; first += groups_per_launch) {
        const int ng = n_groups - first < groups_per_launch ? n_groups - first : groups_per_launch;
        TmaParams p{};
        for (int i = 0; i < ng * M; ++i)
            if (!encode_image_map(&p.maps[i], imgs[(size_t)first * M + i], H, W,
                                  g2 ? ((i & 1) ? g2->pitch_y : g2->pitch_x) : (long long)N, box_rows))
                return IQA_ERR_CUDA;
        p.n_groups = ng; p.M = M; p.W = W; p.H = H; p.log2_nt = ilog2(N_T); p.ntx = ntx; p.n_tiles = (int)n;
        p.units_x = units_x; p.units_y = units_y; p.S = pl.item_rows / box_rows;
        p.C1 = k.C1; p.C2 = k.C2; p.C = k.C; p.D = k.D;
        const size_t cmp0 = (size_t)first * (size_t)(M - 1);
        const Outputs o = out.offset(cmp0 * (size_t)n);
        p.lisi = o.lisi; p.auglisi = o.auglisi; p.sum_x = o.sum_x; p.sum_y = o.sum_y;
        p.lisi_num = o.lisi_num; p.aug_num = o.aug_num;
        p.ws = ws ? ws + cmp0 * (size_t)n * pl.pieces : nullptr;
        p.pieces_x = pl.pieces_x; p.pieces_y = pl.pieces_y;
        const long long n_items = items_per_group * ng;
        long long resident = (long long)geo->sms * geo->tma_ctas[pl.tma_cfg];
        static const int max_ctas = env_int("IQA_TMA_MAX_CTAS", 0);     // tuning knob
        if (max_ctas > 0 && max_ctas < resident) resident = max_ctas;
        const unsigned grid = (unsigned)(n_items < resident ? n_items : resident);
        if (launch(fn, grid, kTmaThreads, tma_smem(pl.tma_cfg), st, p) != cudaSuccess) return IQA_ERR_CUDA;
    }
    return IQA_OK;
}

// S1-S4 for n_pairs pairs (xs[i], ys[i]) with the plan's kernel; `out` / `ws` point at pair 0.
int launch_pairs(int mode, const float* const* xs, const float* const* ys, int n_pairs, int N, int N_T,
                 const Consts& k, const Outputs& out, float4* ws, const Plan& pl, cudaStream_t st,
                 const Geom2D* g2 = nullptr) {
    const int H = g2 ? g2->H : N, W = g2 ? g2->W : N;
    const int nt = (W + N_T - 1) / N_T;                       // tiles per row
    const long long n = (long long)nt * ((H + N_T - 1) / N_T);
    if (pl.kind == kPlanTma) {
        const float* imgs[kMaxImages];
        for (int first = 0; first < n_pairs; first += kMaxImages / 2) {
            const int np = n_pairs - first < kMaxImages / 2 ? n_pairs - first : kMaxImages / 2;
            for (int i = 0; i < np; ++i) { imgs[2 * i] = xs[first + i]; imgs[2 * i + 1] = ys[first + i]; }
            const int rc = launch_tma(mode, kPairs, imgs, np, 2, N, N_T, k, out.offset((size_t)first * (size_t)n),
                                      ws ? ws + (size_t)first * (size_t)n * pl.pieces : nullptr, pl, st, g2);
            if (rc != IQA_OK) return rc;
        }
    } else if (pl.kind == kPlanStream) {
        const Geometry* geo = geometry();
        if (!geo) return IQA_ERR_CUDA;
        const int units_x = (N + kUnitCols - 1) / kUnitCols;
        const int units_y = (N + pl.item_rows - 1) / pl.item_rows;
        const long long items_per_pair = (long long)units_x * units_y;
        if (items_per_pair * kMaxBatch > 0x7fffffffLL) return IQA_ERR_SHAPE;
        StreamFn fn = stream_fn(mode, pl.variant);
        for (int first = 0; first < n_pairs; first += kMaxBatch) {
            const int np = n_pairs - first < kMaxBatch ? n_pairs - first : kMaxBatch;
            BatchParams p{};
            for (int i = 0; i < np; ++i) { p.x[i] = xs[first + i]; p.y[i] = ys[first + i]; }
            p.n_pairs = np; p.N = N; p.log2_nt = ilog2(N_T); p.nt = nt; p.n_tiles = (int)n;
            p.units_x = units_x; p.units_y = units_y; p.item_rows = pl.item_rows;
            p.n_items = (int)(items_per_pair * np);
            p.C1 = k.C1; p.C2 = k.C2; p.C = k.C; p.D = k.D;
            const Outputs o = out.offset((size_t)first * (size_t)n);
            p.lisi = o.lisi; p.auglisi = o.auglisi; p.sum_x = o.sum_x; p.sum_y = o.sum_y;
            p.lisi_num = o.lisi_num; p.aug_num = o.aug_num;
            p.ws = ws ? ws + (size_t)first * (size_t)n * pl.pieces : nullptr;
            p.pieces_x = pl.pieces_x; p.pieces_y = pl.pieces_y;
            const long long resident = (long long)geo->sms * geo->ctas[mode - 1][pl.variant];
            const unsigned grid = (unsigned)(p.n_items < resident ? p.n_items : resident);
            if (launch(fn, grid, kCtaThreads, stream_smem(pl.variant), st, p) != cudaSuccess) return IQA_ERR_CUDA;
        }
    } else {
        const long long grid = n * pl.pieces;
        if (grid > 0x7fffffffLL) return IQA_ERR_SHAPE;
        for (int i = 0; i < n_pairs; ++i) {
            GenericParams g{};
            TileParams& p = g.tp;
            p.x = xs[i]; p.y = ys[i]; p.N = W; p.H = H; p.nt = nt;
            p.pitch_x = g2 ? g2->pitch_x : (long long)N; p.pitch_y = g2 ? g2->pitch_y : (long long)N;
            p.C1 = k.C1; p.C2 = k.C2; p.C = k.C; p.D = k.D;
            const Outputs o = out.offset((size_t)i * (size_t)n);
            p.lisi = o.lisi; p.auglisi = o.auglisi; p.sum_x = o.sum_x; p.sum_y = o.sum_y;
            p.lisi_num = o.lisi_num; p.aug_num = o.aug_num;
            p.ws = ws ? ws + (size_t)i * (size_t)n * pl.pieces : nullptr;
            g.N_T = N_T; g.pieces = pl.pieces;
            cudaError_t e;
            if ((long long)N_T * N_T <= kWarpTilePixels) {        // small tiles: one warp per tile (pieces == 1 here)
                const unsigned wgrid = (unsigned)((n + kWarpsPerCta - 1) / kWarpsPerCta);
                switch (mode) {
                    case kModeLisi: e = launch(generic_warp_kernel<kModeLisi>, wgrid, kCtaThreads, 0, st, g, n); break;
                    case kModeAug: e = launch(generic_warp_kernel<kModeAug>, wgrid, kCtaThreads, 0, st, g, n); break;
                    default: e = launch(generic_warp_kernel<kModeFused>, wgrid, kCtaThreads, 0, st, g, n); break;
                }
            } else {
                switch (mode) {
                    case kModeLisi: e = launch(generic_kernel<kModeLisi>, (unsigned)grid, kCtaThreads, 0, st, g); break;
                    case kModeAug: e = launch(generic_kernel<kModeAug>, (unsigned)grid, kCtaThreads, 0, st, g); break;
                    default: e = launch(generic_kernel<kModeFused>, (unsigned)grid, kCtaThreads, 0, st, g); break;
                }
            }
            if (e != cudaSuccess) return IQA_ERR_CUDA;
        }
    }
    return IQA_OK;
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
        if (pl.pieces <= 32 && total >= 64)
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

// Validation shared by the batch and the series entry points (everything but the image lists).
// Shape of a general image (g2) or of the paper's square N x N image: status and tile count.
int status_of_geometry(int N, int N_T, const Geom2D* g2, long long* n_tiles) {
    if (!g2) {
        if (const int s = status_of_shape(N, N_T)) return s;
        *n_tiles = (long long)(N / N_T) * (N / N_T);
        return IQA_OK;
    }
    if (g2->H <= 0 || g2->W <= 0 || N_T <= 0 || g2->H > kMaxN || g2->W > kMaxN || g2->pitch_x < g2->W ||
        g2->pitch_y < g2->W)
        return IQA_ERR_SHAPE;
    *n_tiles = (long long)((g2->W + N_T - 1) / N_T) * ((g2->H + N_T - 1) / N_T);
    return *n_tiles > 0x7fffffffLL ? IQA_ERR_SHAPE : IQA_OK;
}

int validate_common(int mode, int n_cmp, int N, int N_T, float C1, float C2, float C, float D, const Outputs& out,
                    const float* out2, const Geom2D* g2 = nullptr) {
    if (n_cmp <= 0) return IQA_ERR_SHAPE;
    if ((mode & kModeLisi) && !out.lisi) return IQA_ERR_NULL;
    if ((mode & kModeAug) && !out.auglisi) return IQA_ERR_NULL;
    if (mode == kModeFused && (!out.sum_x || !out.sum_y)) return IQA_ERR_NULL;
    long long n = 0;
    if (const int s = status_of_geometry(N, N_T, g2, &n)) return s;
    if (n * n_cmp > 0x7fffffffLL) return IQA_ERR_SHAPE;
    if ((mode & kModeLisi) && (!pos_finite(C1) || !pos_finite(C2) || !std::isfinite(D))) return IQA_ERR_PARAM;
    if ((mode & kModeAug) && !pos_finite(C)) return IQA_ERR_PARAM;
    if (out2 && (!pos_finite(C2) || !pos_finite(C))) return IQA_ERR_PARAM;
    return IQA_OK;
}

// Shared body of every *_tiles / *_batch entry point: validation, then the launches.
// xs, ys: HOST arrays of n_pairs device pointers.  out2 (nullable): Eqs. 3-4 per pair.
int run_batch(int mode, const float* const* xs, const float* const* ys, int n_pairs, int N, int N_T,
              float C1, float C2, float C, float D, Outputs out, float* out2,
              void* workspace, size_t workspace_bytes, void* stream, const Geom2D* g2 = nullptr) {
    if (!xs || !ys) return IQA_ERR_NULL;
    if (n_pairs <= 0) return IQA_ERR_SHAPE;
    for (int i = 0; i < n_pairs; ++i)
        if (!xs[i] || !ys[i]) return IQA_ERR_NULL;
    if (const int s = validate_common(mode, n_pairs, N, N_T, C1, C2, C, D, out, out2, g2)) return s;
    long long n = 0;
    status_of_geometry(N, N_T, g2, &n);
    uintptr_t bits = 0;
    for (int i = 0; i < n_pairs; ++i) bits |= (uintptr_t)xs[i] | (uintptr_t)ys[i];
    if (bits & 3u) return IQA_ERR_ALIGN;
    const size_t need = (size_t)n_pairs * (size_t)n * (max_pieces(N_T) > 1 ? max_pieces(N_T) : 0) * sizeof(float4);
    if (need > 0 && (!workspace || workspace_bytes < need)) return IQA_ERR_WORKSPACE;
    if (need > 0 && ((uintptr_t)workspace & 15u)) return IQA_ERR_ALIGN;

    const bool aligned16 = ((bits & 15u) == 0) && (g2 ? (g2->pitch_x % 4 == 0 && g2->pitch_y % 4 == 0) : (N % 4 == 0));
    const Plan pl = make_plan(g2 ? g2->W : N, N_T, aligned16, xs[0], false, g2);
    cudaStream_t st = (cudaStream_t)stream;
    float4* ws = pl.pieces > 1 ? (float4*)workspace : nullptr;
    out = out.for_mode(mode);
    const Consts k{C1, C2, C, D};
    if (const int rc = launch_pairs(mode, xs, ys, n_pairs, g2 ? g2->W : N, N_T, k, out, ws, pl, st, g2)) return rc;
    return finish_comparisons(out, out2, n_pairs, n, k, ws, pl, st);
}

// Time series: imgs = HOST array of n_images device pointers; K = n_images - 1
// comparisons, (I_0, I_k+1) or (I_k, I_k+1).  Aligned power-of-two shapes take the TMA kernel, which
// keeps the x box of every comparison in shared memory (each image is read from HBM once);
// everything else is computed pair by pair with the kernels of the pair entry points.
int run_series(const float* const* imgs, int n_images, int series, int N, int N_T,
               float C1, float C2, float C, float D, Outputs out, float* out2,
               void* workspace, size_t workspace_bytes, void* stream, const Geom2D* g2 = nullptr) {
    if (!imgs) return IQA_ERR_NULL;
    if (n_images < 2 || (series != kReference && series != kConsecutive)) return IQA_ERR_SHAPE;
    for (int i = 0; i < n_images; ++i)
        if (!imgs[i]) return IQA_ERR_NULL;
    const int K = n_images - 1;
    if (const int s = validate_common(kModeFused, K, N, N_T, C1, C2, C, D, out, out2, g2)) return s;
    long long n = 0;
    status_of_geometry(N, N_T, g2, &n);
    uintptr_t bits = 0;
    for (int i = 0; i < n_images; ++i) bits |= (uintptr_t)imgs[i];
    if (bits & 3u) return IQA_ERR_ALIGN;
    const size_t need = (size_t)K * (size_t)n * (max_pieces(N_T) > 1 ? max_pieces(N_T) : 0) * sizeof(float4);
    if (need > 0 && (!workspace || workspace_bytes < need)) return IQA_ERR_WORKSPACE;
    if (need > 0 && ((uintptr_t)workspace & 15u)) return IQA_ERR_ALIGN;

    const bool aligned16 = ((bits & 15u) == 0) && (g2 ? g2->pitch_x % 4 == 0 : N % 4 == 0);
    if (g2) N = g2->W;
    const Plan pl = make_plan(N, N_T, aligned16, imgs[0], true, g2);
    cudaStream_t st = (cudaStream_t)stream;
    float4* ws = pl.pieces > 1 ? (float4*)workspace : nullptr;
    const Consts k{C1, C2, C, D};
    if (pl.kind == kPlanTma) {
        // chunks of at most kMaxImages images; consecutive chunks share one image
        const float* chunk[kMaxImages];
        for (int first = 0; first < K; first += kMaxImages - 1) {       // first = first comparison of the chunk
            const int kc = K - first < kMaxImages - 1 ? K - first : kMaxImages - 1;
            chunk[0] = series == kReference ? imgs[0] : imgs[first];
            for (int i = 0; i < kc; ++i) chunk[1 + i] = imgs[first + 1 + i];
            const int rc = launch_tma(kModeFused, series, chunk, 1, kc + 1, N, N_T, k, out.offset((size_t)first * (size_t)n),
                                      ws ? ws + (size_t)first * (size_t)n * pl.pieces : nullptr, pl, st, g2);
            if (rc != IQA_OK) return rc;
        }
    } else {
        const float* xs[kMaxBatch];
        const float* ys[kMaxBatch];
        for (int first = 0; first < K; first += kMaxBatch) {
            const int kc = K - first < kMaxBatch ? K - first : kMaxBatch;
            for (int i = 0; i < kc; ++i) {
                xs[i] = series == kReference ? imgs[0] : imgs[first + i];
                ys[i] = imgs[first + i + 1];
            }
            const int rc = launch_pairs(kModeFused, xs, ys, kc, N, N_T, k, out.offset((size_t)first * (size_t)n),
                                        ws ? ws + (size_t)first * (size_t)n * pl.pieces : nullptr, pl, st, g2);
            if (rc != IQA_OK) return rc;
        }
    }
    return finish_comparisons(out, out2, K, n, k, ws, pl, st);
}

// Generic kernels on pixels of type T (iqa_fused_tiles_2d_typed).
template <typename T>
int launch_typed(const void* x, const void* y, const Geom2D& g2, int N_T, const Consts& k, const Outputs& out, float4* ws,
                 const Plan& pl, cudaStream_t st) {
    const int nt = (g2.W + N_T - 1) / N_T;
    const long long n = (long long)nt * ((g2.H + N_T - 1) / N_T);
    GenericParams g{};
    TileParams& p = g.tp;
    p.x = (const float*)x; p.y = (const float*)y; p.N = g2.W; p.H = g2.H; p.nt = nt;
    p.pitch_x = g2.pitch_x; p.pitch_y = g2.pitch_y;
    p.C1 = k.C1; p.C2 = k.C2; p.C = k.C; p.D = k.D;
    p.lisi = out.lisi; p.auglisi = out.auglisi; p.sum_x = out.sum_x; p.sum_y = out.sum_y;
    p.lisi_num = out.lisi_num; p.aug_num = out.aug_num;
    p.ws = ws;
    g.N_T = N_T; g.pieces = pl.pieces;
    cudaError_t e;
    if ((long long)N_T * N_T <= kWarpTilePixels)
        e = launch(generic_warp_kernel<kModeFused, T>, (unsigned)((n + kWarpsPerCta - 1) / kWarpsPerCta), kCtaThreads, 0, st, g, n);
    else
        e = launch(generic_kernel<kModeFused, T>, (unsigned)(n * pl.pieces), kCtaThreads, 0, st, g);
    return e == cudaSuccess ? IQA_OK : IQA_ERR_CUDA;
}

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

}  // namespace

extern "C" {

const char* iqa_status_string(int status) {
    switch (status) {
        case IQA_OK: return "ok";
        case IQA_ERR_NULL: return "required pointer is NULL";
        case IQA_ERR_SHAPE: return "bad shape: need 0 < N_T <= N <= 2^20, N % N_T == 0, n_pairs >= 1, tile count < 2^31";
        case IQA_ERR_PARAM: return "bad constant: C1, C2, C must be finite and > 0, D finite";
        case IQA_ERR_ALIGN: return "pointer alignment: images 4-byte, workspace 16-byte";
        case IQA_ERR_WORKSPACE: return "workspace missing or smaller than iqa_workspace_bytes / iqa_batch_workspace_bytes";
        case IQA_ERR_CUDA: return "CUDA launch or copy failed";
        default: return "unknown status";
    }
}

const char* iqa_version(void) { return "0.4.0"; }

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
    return run_batch(kModeLisi, &x, &y, 1, N, N_T, C1, C2, 1.0f, D, o, nullptr, workspace, workspace_bytes, stream);
}

int iqa_auglisi_tiles(const float* x, const float* y, int N, int N_T, float C,
                      float* auglisi, void* workspace, size_t workspace_bytes, void* stream) {
    const Outputs o{nullptr, auglisi, nullptr, nullptr, nullptr, nullptr};
    return run_batch(kModeAug, &x, &y, 1, N, N_T, 1.0f, 1.0f, C, 0.0f, o, nullptr, workspace, workspace_bytes, stream);
}

int iqa_fused_tiles(const float* x, const float* y, int N, int N_T,
                    float C1, float C2, float C, float D,
                    float* lisi, float* auglisi, float* sum_x, float* sum_y,
                    float* lisi_num, float* auglisi_num,
                    void* workspace, size_t workspace_bytes, void* stream) {
    const Outputs o{lisi, auglisi, sum_x, sum_y, lisi_num, auglisi_num};
    return run_batch(kModeFused, &x, &y, 1, N, N_T, C1, C2, C, D, o, nullptr, workspace, workspace_bytes, stream);
}

int iqa_query_plan(const float* x, int H, int W, long long pitch, int N_T, int series) {
    if (!x || H <= 0 || W <= 0 || N_T <= 0 || pitch < W) return -1;
    const Geom2D g2{H, W, pitch, pitch};
    const bool aligned16 = (((uintptr_t)x & 15u) == 0) && (pitch % 4 == 0);
    const bool square = H == W && pitch == W && W % N_T == 0;      // what the paper-named entry points see
    const Plan pl = make_plan(W, N_T, aligned16, x, series != 0, square ? nullptr : &g2);
    return pl.kind == kPlanTma ? IQA_PLAN_TMA + pl.tma_cfg : pl.kind == kPlanStream ? IQA_PLAN_CP_ASYNC : IQA_PLAN_GENERIC;
}

size_t iqa_workspace_bytes_2d(int H, int W, int N_T) {
    if (H <= 0 || W <= 0 || N_T <= 0 || H > kMaxN || W > kMaxN) return 0;
    const size_t pieces = max_pieces(N_T);
    if (pieces <= 1) return 0;
    const size_t n = (size_t)((H + N_T - 1) / N_T) * (size_t)((W + N_T - 1) / N_T);
    return n * pieces * sizeof(float4);
}

int iqa_fused_tiles_2d(const float* x, const float* y, int H, int W, long long pitch_x, long long pitch_y, int N_T,
                       float C1, float C2, float C, float D,
                       float* lisi, float* auglisi, float* sum_x, float* sum_y,
                       float* lisi_num, float* auglisi_num,
                       void* workspace, size_t workspace_bytes, void* stream) {
    if (!x || !y || !lisi || !auglisi || !sum_x || !sum_y) return IQA_ERR_NULL;
    if (H <= 0 || W <= 0 || N_T <= 0 || H > kMaxN || W > kMaxN || pitch_x < W || pitch_y < W) return IQA_ERR_SHAPE;
    const long long ntx = (W + N_T - 1) / N_T, nty = (H + N_T - 1) / N_T;
    if (ntx * nty > 0x7fffffffLL) return IQA_ERR_SHAPE;
    if (!pos_finite(C1) || !pos_finite(C2) || !pos_finite(C) || !std::isfinite(D)) return IQA_ERR_PARAM;
    const uintptr_t bits = (uintptr_t)x | (uintptr_t)y;
    if (bits & 3u) return IQA_ERR_ALIGN;
    const size_t need = iqa_workspace_bytes_2d(H, W, N_T);
    if (need > 0 && (!workspace || workspace_bytes < need)) return IQA_ERR_WORKSPACE;
    if (need > 0 && ((uintptr_t)workspace & 15u)) return IQA_ERR_ALIGN;

    const Geom2D g2{H, W, pitch_x, pitch_y};
    const bool aligned16 = ((bits & 15u) == 0) && (pitch_x % 4 == 0) && (pitch_y % 4 == 0);
    const Plan pl = make_plan(W, N_T, aligned16, x, false, &g2);
    cudaStream_t st = (cudaStream_t)stream;
    float4* ws = pl.pieces > 1 ? (float4*)workspace : nullptr;
    const Outputs out{lisi, auglisi, sum_x, sum_y, lisi_num, auglisi_num};
    const Consts k{C1, C2, C, D};
    if (const int rc = launch_pairs(kModeFused, &x, &y, 1, W, N_T, k, out, ws, pl, st, &g2)) return rc;
    return finish_comparisons(out, nullptr, 1, ntx * nty, k, ws, pl, st);
}

int iqa_fused_tiles_2d_typed(const void* x, const void* y, int pixel_type,
                             int H, int W, long long pitch_x, long long pitch_y, int N_T,
                             float C1, float C2, float C, float D,
                             float* lisi, float* auglisi, float* sum_x, float* sum_y,
                             float* lisi_num, float* auglisi_num,
                             void* workspace, size_t workspace_bytes, void* stream) {
    if (pixel_type == IQA_PIXEL_F32)
        return iqa_fused_tiles_2d((const float*)x, (const float*)y, H, W, pitch_x, pitch_y, N_T, C1, C2, C, D, lisi, auglisi,
                                  sum_x, sum_y, lisi_num, auglisi_num, workspace, workspace_bytes, stream);
    if (!x || !y || !lisi || !auglisi || !sum_x || !sum_y) return IQA_ERR_NULL;
    size_t esize = 0;
    switch (pixel_type) {
        case IQA_PIXEL_F64: esize = 8; break;
        case IQA_PIXEL_F16: case IQA_PIXEL_I16: esize = 2; break;
        case IQA_PIXEL_I32: esize = 4; break;
        case IQA_PIXEL_U8: esize = 1; break;
        default: return IQA_ERR_SHAPE;
    }
    if (H <= 0 || W <= 0 || N_T <= 0 || H > kMaxN || W > kMaxN || pitch_x < W || pitch_y < W) return IQA_ERR_SHAPE;
    const long long n = (long long)((W + N_T - 1) / N_T) * ((H + N_T - 1) / N_T);
    if (n * (long long)((N_T + kGenericRows - 1) / kGenericRows) > 0x7fffffffLL) return IQA_ERR_SHAPE;
    if (!pos_finite(C1) || !pos_finite(C2) || !pos_finite(C) || !std::isfinite(D)) return IQA_ERR_PARAM;
    if ((((uintptr_t)x | (uintptr_t)y) & (esize - 1)) != 0) return IQA_ERR_ALIGN;
    const size_t need = iqa_workspace_bytes_2d(H, W, N_T);
    if (need > 0 && (!workspace || workspace_bytes < need)) return IQA_ERR_WORKSPACE;
    if (need > 0 && ((uintptr_t)workspace & 15u)) return IQA_ERR_ALIGN;

    const Geom2D g2{H, W, pitch_x, pitch_y};
    Plan pl{};
    pl.kind = kPlanGeneric;
    pl.pieces_x = 1;
    pl.pieces_y = (N_T + kGenericRows - 1) / kGenericRows;
    pl.pieces = pl.pieces_y;
    cudaStream_t st = (cudaStream_t)stream;
    float4* ws = pl.pieces > 1 ? (float4*)workspace : nullptr;
    const Outputs out{lisi, auglisi, sum_x, sum_y, lisi_num, auglisi_num};
    const Consts k{C1, C2, C, D};
    int rc;
    switch (pixel_type) {
        case IQA_PIXEL_F64: rc = launch_typed<double>(x, y, g2, N_T, k, out, ws, pl, st); break;
        case IQA_PIXEL_F16: rc = launch_typed<__half>(x, y, g2, N_T, k, out, ws, pl, st); break;
        case IQA_PIXEL_I16: rc = launch_typed<short>(x, y, g2, N_T, k, out, ws, pl, st); break;
        case IQA_PIXEL_I32: rc = launch_typed<int>(x, y, g2, N_T, k, out, ws, pl, st); break;
        default: rc = launch_typed<unsigned char>(x, y, g2, N_T, k, out, ws, pl, st); break;
    }
    if (rc != IQA_OK) return rc;
    return finish_comparisons(out, nullptr, 1, n, k, ws, pl, st);
}

int iqa_fused_batch_2d(const float* const* x_ptrs_host, const float* const* y_ptrs_host, int n_pairs,
                       int H, int W, long long pitch, int N_T, float C1, float C2, float C, float D,
                       float* lisi, float* auglisi, float* sum_x, float* sum_y,
                       float* lisi_num, float* auglisi_num, float* out2,
                       void* workspace, size_t workspace_bytes, void* stream) {
    const Outputs o{lisi, auglisi, sum_x, sum_y, lisi_num, auglisi_num};
    const Geom2D g2{H, W, pitch, pitch};
    return run_batch(kModeFused, x_ptrs_host, y_ptrs_host, n_pairs, W, N_T, C1, C2, C, D, o, out2,
                     workspace, workspace_bytes, stream, &g2);
}

int iqa_series_tiles_2d(const float* const* img_ptrs_host, int n_images, int mode,
                        int H, int W, long long pitch, int N_T, float C1, float C2, float C, float D,
                        float* lisi, float* auglisi, float* sum_x, float* sum_y,
                        float* lisi_num, float* auglisi_num, float* out2,
                        void* workspace, size_t workspace_bytes, void* stream) {
    const Outputs o{lisi, auglisi, sum_x, sum_y, lisi_num, auglisi_num};
    const int series = mode == IQA_SERIES_REFERENCE ? kReference : mode == IQA_SERIES_CONSECUTIVE ? kConsecutive : -1;
    const Geom2D g2{H, W, pitch, pitch};
    return run_series(img_ptrs_host, n_images, series, W, N_T, C1, C2, C, D, o, out2,
                      workspace, workspace_bytes, stream, &g2);
}

int iqa_fused_batch(const float* const* x_ptrs_host, const float* const* y_ptrs_host, int n_pairs,
                    int N, int N_T, float C1, float C2, float C, float D,
                    float* lisi, float* auglisi, float* sum_x, float* sum_y,
                    float* lisi_num, float* auglisi_num, float* out2,
                    void* workspace, size_t workspace_bytes, void* stream) {
    const Outputs o{lisi, auglisi, sum_x, sum_y, lisi_num, auglisi_num};
    return run_batch(kModeFused, x_ptrs_host, y_ptrs_host, n_pairs, N, N_T, C1, C2, C, D, o, out2,
                     workspace, workspace_bytes, stream);
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
    return run_series(img_ptrs_host, n_images, series, N, N_T, C1, C2, C, D, o, out2,
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
    const int cs = env_int("IQA_CAND_NO_CLUSTER", 0) ? 0 : cand_cluster_size(n_tiles);
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
    const int cs = env_int("IQA_CAND_NO_CLUSTER", 0) ? 0 : cand_cluster_size(n_tiles);
    const cudaError_t e = cs > 0
        ? launch_cluster(bottom_k_cluster_kernel, (unsigned)n_maps * (unsigned)cs, (unsigned)kCandThreads, 0,
                         (cudaStream_t)stream, (unsigned)cs, values, n_tiles, k, indices, vals)
        : launch(bottom_k_kernel, (unsigned)n_maps, (unsigned)cand_threads(n_tiles), 0, (cudaStream_t)stream, values,
                 n_tiles, k, indices, vals);
    if (e != cudaSuccess) return IQA_ERR_CUDA;
    return cudaGetLastError() == cudaSuccess ? IQA_OK : IQA_ERR_CUDA;
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

int iqa_merge_tiles(const float* lisi, const float* auglisi,
                    const float* sum_x, const float* sum_y, int nt, int g,
                    float C2, float C,
                    float* lisi_out, float* auglisi_out,
                    float* sum_x_out, float* sum_y_out, void* stream) {
    return iqa_merge_tiles_batch(lisi, auglisi, sum_x, sum_y, nt, g, 1, C2, C, lisi_out, auglisi_out, sum_x_out,
                                 sum_y_out, stream);
}

size_t iqa_host_scratch_bytes(int N, int N_T) {
    if (status_of_shape(N, N_T) != IQA_OK) return 0;
    const size_t img = align_up((size_t)N * (size_t)N * sizeof(float), 256);
    const size_t n = (size_t)(N / N_T) * (size_t)(N / N_T);
    const size_t per_tile = align_up(n * sizeof(float), 256);
    return 2 * img + 4 * per_tile + 256 + align_up(workspace_bytes_for(1, N, N_T), 256);
}

namespace {
int fused_host_impl(const float* x_host, const float* y_host, int N, int N_T,
                    float C1, float C2, float C, float D,
                    float* lisi_host, float* auglisi_host,
                    float* sum_x_host, float* sum_y_host, float* out2_host,
                    void* dev_scratch, size_t dev_scratch_bytes, void* stream, bool synchronise) {
    if (!x_host || !y_host || !dev_scratch) return IQA_ERR_NULL;
    if (const int s = status_of_shape(N, N_T)) return s;
    if (!pos_finite(C1) || !pos_finite(C2) || !pos_finite(C) || !std::isfinite(D)) return IQA_ERR_PARAM;
    if (dev_scratch_bytes < iqa_host_scratch_bytes(N, N_T)) return IQA_ERR_WORKSPACE;
    if ((uintptr_t)dev_scratch & 255u) return IQA_ERR_ALIGN;

    cudaStream_t st = (cudaStream_t)stream;
    const size_t img_bytes = (size_t)N * (size_t)N * sizeof(float);
    const size_t img = align_up(img_bytes, 256);
    const size_t n = (size_t)(N / N_T) * (size_t)(N / N_T);
    const size_t per_tile = align_up(n * sizeof(float), 256);
    char* base = (char*)dev_scratch;
    float* xd = (float*)base;
    float* yd = (float*)(base + img);
    float* d_lisi = (float*)(base + 2 * img);
    float* d_aug = (float*)(base + 2 * img + per_tile);
    float* d_sx = (float*)(base + 2 * img + 2 * per_tile);
    float* d_sy = (float*)(base + 2 * img + 3 * per_tile);
    float* d_out2 = (float*)(base + 2 * img + 4 * per_tile);
    void* ws = base + 2 * img + 4 * per_tile + 256;
    const size_t ws_bytes = workspace_bytes_for(1, N, N_T);

    if (cudaMemcpyAsync(xd, x_host, img_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) return IQA_ERR_CUDA;
    if (cudaMemcpyAsync(yd, y_host, img_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) return IQA_ERR_CUDA;
    const float* xs[1] = {xd};
    const float* ys[1] = {yd};
    const int rc = iqa_fused_batch(xs, ys, 1, N, N_T, C1, C2, C, D, d_lisi, d_aug, d_sx, d_sy, nullptr, nullptr,
                                   d_out2, ws_bytes ? ws : nullptr, ws_bytes, stream);
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
    return fused_host_impl(x_host, y_host, N, N_T, C1, C2, C, D, lisi_host, auglisi_host, sum_x_host, sum_y_host,
                           out2_host, dev_scratch, dev_scratch_bytes, stream, true);
}

int iqa_fused_host_async(const float* x_host, const float* y_host, int N, int N_T,
                         float C1, float C2, float C, float D,
                         float* lisi_host, float* auglisi_host,
                         float* sum_x_host, float* sum_y_host, float* out2_host,
                         void* dev_scratch, size_t dev_scratch_bytes, void* stream) {
    return fused_host_impl(x_host, y_host, N, N_T, C1, C2, C, D, lisi_host, auglisi_host, sum_x_host, sum_y_host,
                           out2_host, dev_scratch, dev_scratch_bytes, stream, false);
}

}  // extern "C"
