// =============================================================================
// iqa_tiles.cu -- the C ABI of include/iqa_tiles.h: argument validation, the N_T-dependent
// choice of mapping, and the launches.  No torch types, no allocation, no global state.
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -shared -Xcompiler -fPIC
// =============================================================================
#include "../../include/iqa_tiles.h"

#include <cmath>
#include <cstdint>
#include <cstdlib>

#include "iqa_aggregate.cuh"
#include "iqa_kernels.cuh"

namespace {

using namespace iqa;

constexpr int kMaxN = 1 << 20;   // 2^40 pixels; keeps every grid and tile index inside int

bool is_pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }
int ilog2(int v) { int l = 0; while ((1 << l) < v) ++l; return l; }
bool pos_finite(float v) { return std::isfinite(v) && v > 0.0f; }

int env_int(const char* name, int dflt) {
    const char* s = std::getenv(name);
    return (s && *s) ? std::atoi(s) : dflt;
}

// How (N, N_T) is mapped onto CTAs.  DESIGN.md "Mapping".
struct Plan {
    bool strip;        // vectorised strip kernel (else generic kernel)
    int rw;            // rows per warp (strip): 4, 8 or 16
    int pieces_x, pieces_y, pieces;   // pieces per tile; pieces == 1 -> finished in one CTA
    long long grid;    // CTAs of the first pass
};

int status_of_shape(int N, int N_T) {
    if (N <= 0 || N_T <= 0 || N > kMaxN || N_T > N || N % N_T != 0) return IQA_ERR_SHAPE;
    const long long nt = N / N_T;
    if (nt * nt > 0x7fffffffLL) return IQA_ERR_SHAPE;
    return IQA_OK;
}

// Rows per warp for the strip kernel.  A tile of side <= 64 must sit inside one unit
// (8*rw >= N_T) so that the common cases need no second pass; rw never exceeds N_T.
int choose_rw(int N, int N_T) {
    int rw = 8;
    const int forced = env_int("IQA_FORCE_RW", 0);          // debug knob (tests: mapping independence)
    if (forced == 4 || forced == 8 || forced == 16) rw = forced;
    if (rw > N_T) rw = N_T >= 8 ? 8 : 4;
    if (N_T <= 64 && 8 * rw < N_T) rw = N_T / 8;
    (void)N;
    return rw;
}

Plan make_plan(int N, int N_T, bool aligned16) {
    Plan pl{};
    const long long nt = N / N_T;
    pl.strip = is_pow2(N_T) && N_T >= 8 && aligned16 && !env_int("IQA_FORCE_GENERIC", 0);
    if (pl.strip) {
        pl.rw = choose_rw(N, N_T);
        const int rb = kWarpsPerCta * pl.rw;
        pl.pieces_x = N_T > kUnitCols ? N_T / kUnitCols : 1;
        pl.pieces_y = N_T > rb ? N_T / rb : 1;
        pl.pieces = pl.pieces_x * pl.pieces_y;
        const long long ux = (N + kUnitCols - 1) / kUnitCols, uy = (N + rb - 1) / rb;
        pl.grid = ux * uy;
    } else {
        pl.rw = 0;
        pl.pieces_x = 1;
        pl.pieces_y = (N_T + kGenericRows - 1) / kGenericRows;
        pl.pieces = pl.pieces_y;
        pl.grid = nt * nt * pl.pieces;
    }
    return pl;
}

size_t workspace_bytes_for(int N, int N_T) {
    if (N_T <= 64) return 0;                                  // every path finishes tiles in one CTA
    const size_t n = (size_t)(N / N_T) * (size_t)(N / N_T);
    size_t pieces = (size_t)(N_T + kGenericRows - 1) / kGenericRows;       // generic path
    if (is_pow2(N_T)) {                                       // strip path, worst case rw = 4
        const size_t px = N_T > kUnitCols ? N_T / kUnitCols : 1;
        const size_t py = N_T / 32;
        if (px * py > pieces) pieces = px * py;
    }
    return n * pieces * sizeof(float4);
}

template <int MODE>
void launch_strip(const TileParams& p, int rw, unsigned grid, cudaStream_t st) {
    switch (rw) {
        case 4: strip_kernel<MODE, 4><<<grid, kCtaThreads, 0, st>>>(p); break;
        case 16: strip_kernel<MODE, 16><<<grid, kCtaThreads, 0, st>>>(p); break;
        default: strip_kernel<MODE, 8><<<grid, kCtaThreads, 0, st>>>(p); break;
    }
}

void launch_generic(int mode, const GenericParams& g, unsigned grid, cudaStream_t st) {
    switch (mode) {
        case kModeLisi: generic_kernel<kModeLisi><<<grid, kCtaThreads, 0, st>>>(g); break;
        case kModeAug: generic_kernel<kModeAug><<<grid, kCtaThreads, 0, st>>>(g); break;
        default: generic_kernel<kModeFused><<<grid, kCtaThreads, 0, st>>>(g); break;
    }
}

// Shared body of the three *_tiles entry points.
int run_tiles(int mode, const float* x, const float* y, int N, int N_T,
              float C1, float C2, float C, float D,
              float* lisi, float* auglisi, float* sum_x, float* sum_y,
              float* lisi_num, float* aug_num,
              void* workspace, size_t workspace_bytes, void* stream) {
    if (!x || !y) return IQA_ERR_NULL;
    if ((mode & kModeLisi) && !lisi) return IQA_ERR_NULL;
    if ((mode & kModeAug) && !auglisi) return IQA_ERR_NULL;
    if (mode == kModeFused && (!sum_x || !sum_y)) return IQA_ERR_NULL;
    if (const int s = status_of_shape(N, N_T)) return s;
    if ((mode & kModeLisi) && (!pos_finite(C1) || !pos_finite(C2) || !std::isfinite(D)))
        return IQA_ERR_PARAM;
    if ((mode & kModeAug) && !pos_finite(C)) return IQA_ERR_PARAM;
    if (((uintptr_t)x | (uintptr_t)y) & 3u) return IQA_ERR_ALIGN;
    const size_t need = workspace_bytes_for(N, N_T);
    if (need > 0 && (!workspace || workspace_bytes < need)) return IQA_ERR_WORKSPACE;
    if (need > 0 && ((uintptr_t)workspace & 15u)) return IQA_ERR_ALIGN;

    const bool aligned16 = ((((uintptr_t)x | (uintptr_t)y) & 15u) == 0) && (N % 4 == 0);
    const Plan pl = make_plan(N, N_T, aligned16);
    if (pl.grid > 0x7fffffffLL) return IQA_ERR_SHAPE;
    cudaStream_t st = (cudaStream_t)stream;

    TileParams p{};
    p.x = x; p.y = y; p.N = N; p.nt = N / N_T;
    p.log2_nt = is_pow2(N_T) ? ilog2(N_T) : 0;
    p.units_x = (N + kUnitCols - 1) / kUnitCols;
    p.C1 = C1; p.C2 = C2; p.C = C; p.D = D;
    p.lisi = (mode & kModeLisi) ? lisi : nullptr;
    p.auglisi = (mode & kModeAug) ? auglisi : nullptr;
    p.sum_x = sum_x; p.sum_y = sum_y;
    p.lisi_num = (mode & kModeLisi) ? lisi_num : nullptr;
    p.aug_num = (mode & kModeAug) ? aug_num : nullptr;
    p.pieces_x = pl.pieces_x; p.pieces_y = pl.pieces_y;
    p.ws = pl.pieces > 1 ? (float4*)workspace : nullptr;

    if (pl.strip) {
        switch (mode) {
            case kModeLisi: launch_strip<kModeLisi>(p, pl.rw, (unsigned)pl.grid, st); break;
            case kModeAug: launch_strip<kModeAug>(p, pl.rw, (unsigned)pl.grid, st); break;
            default: launch_strip<kModeFused>(p, pl.rw, (unsigned)pl.grid, st); break;
        }
    } else {
        GenericParams g{};
        g.tp = p; g.N_T = N_T; g.pieces = pl.pieces;
        launch_generic(mode, g, (unsigned)pl.grid, st);
    }
    if (pl.pieces > 1) {
        const int n = p.nt * p.nt;
        if (pl.pieces <= 32 && n >= 64)
            finalise_small_kernel<<<(n + kCtaThreads - 1) / kCtaThreads, kCtaThreads, 0, st>>>(p, pl.pieces, n);
        else
            finalise_kernel<<<n, kCtaThreads, 0, st>>>(p, pl.pieces);
    }
    return cudaGetLastError() == cudaSuccess ? IQA_OK : IQA_ERR_CUDA;
}

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

}  // namespace

extern "C" {

const char* iqa_status_string(int status) {
    switch (status) {
        case IQA_OK: return "ok";
        case IQA_ERR_NULL: return "required pointer is NULL";
        case IQA_ERR_SHAPE: return "bad shape: need 0 < N_T <= N <= 2^20, N % N_T == 0, tile count < 2^31";
        case IQA_ERR_PARAM: return "bad constant: C1, C2, C must be finite and > 0, D finite";
        case IQA_ERR_ALIGN: return "pointer alignment: images 4-byte, workspace 16-byte";
        case IQA_ERR_WORKSPACE: return "workspace missing or smaller than iqa_workspace_bytes(N, N_T)";
        case IQA_ERR_CUDA: return "CUDA launch or copy failed";
        default: return "unknown status";
    }
}

const char* iqa_version(void) { return "0.1.0"; }

size_t iqa_workspace_bytes(int N, int N_T) {
    if (status_of_shape(N, N_T) != IQA_OK) return 0;
    return workspace_bytes_for(N, N_T);
}

int iqa_lisi_tiles(const float* x, const float* y, int N, int N_T,
                   float C1, float C2, float D, float* lisi,
                   void* workspace, size_t workspace_bytes, void* stream) {
    return run_tiles(kModeLisi, x, y, N, N_T, C1, C2, 1.0f, D, lisi, nullptr, nullptr, nullptr,
                     nullptr, nullptr, workspace, workspace_bytes, stream);
}

int iqa_auglisi_tiles(const float* x, const float* y, int N, int N_T, float C,
                      float* auglisi, void* workspace, size_t workspace_bytes, void* stream) {
    return run_tiles(kModeAug, x, y, N, N_T, 1.0f, 1.0f, C, 0.0f, nullptr, auglisi, nullptr, nullptr,
                     nullptr, nullptr, workspace, workspace_bytes, stream);
}

int iqa_fused_tiles(const float* x, const float* y, int N, int N_T,
                    float C1, float C2, float C, float D,
                    float* lisi, float* auglisi, float* sum_x, float* sum_y,
                    float* lisi_num, float* auglisi_num,
                    void* workspace, size_t workspace_bytes, void* stream) {
    return run_tiles(kModeFused, x, y, N, N_T, C1, C2, C, D, lisi, auglisi, sum_x, sum_y,
                     lisi_num, auglisi_num, workspace, workspace_bytes, stream);
}

int iqa_aggregate(const float* lisi, const float* auglisi,
                  const float* sum_x, const float* sum_y, int n_tiles,
                  float C2, float C, float* out2, void* stream) {
    if (!lisi || !auglisi || !sum_x || !sum_y || !out2) return IQA_ERR_NULL;
    if (n_tiles <= 0) return IQA_ERR_SHAPE;
    if (!pos_finite(C2) || !pos_finite(C)) return IQA_ERR_PARAM;
    aggregate_kernel<<<1, kAggThreads, 0, (cudaStream_t)stream>>>(lisi, auglisi, sum_x, sum_y,
                                                                  n_tiles, C2, C, out2);
    return cudaGetLastError() == cudaSuccess ? IQA_OK : IQA_ERR_CUDA;
}

int iqa_merge_tiles(const float* lisi, const float* auglisi,
                    const float* sum_x, const float* sum_y, int nt, int g,
                    float C2, float C,
                    float* lisi_out, float* auglisi_out,
                    float* sum_x_out, float* sum_y_out, void* stream) {
    if (!lisi || !auglisi || !sum_x || !sum_y || !lisi_out || !auglisi_out || !sum_x_out || !sum_y_out)
        return IQA_ERR_NULL;
    if (nt <= 0 || g <= 0 || g > nt || nt % g != 0 || (long long)nt * nt > 0x7fffffffLL)
        return IQA_ERR_SHAPE;
    if (!pos_finite(C2) || !pos_finite(C)) return IQA_ERR_PARAM;
    const long long n_out = (long long)(nt / g) * (nt / g);
    const unsigned grid = (unsigned)((n_out + 7) / 8);
    merge_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>(lisi, auglisi, sum_x, sum_y, nt, g, C2, C,
                                                         lisi_out, auglisi_out, sum_x_out, sum_y_out);
    return cudaGetLastError() == cudaSuccess ? IQA_OK : IQA_ERR_CUDA;
}

size_t iqa_host_scratch_bytes(int N, int N_T) {
    if (status_of_shape(N, N_T) != IQA_OK) return 0;
    const size_t img = align_up((size_t)N * (size_t)N * sizeof(float), 256);
    const size_t n = (size_t)(N / N_T) * (size_t)(N / N_T);
    const size_t per_tile = align_up(n * sizeof(float), 256);
    return 2 * img + 4 * per_tile + 256 + align_up(workspace_bytes_for(N, N_T), 256);
}

int iqa_fused_host(const float* x_host, const float* y_host, int N, int N_T,
                   float C1, float C2, float C, float D,
                   float* lisi_host, float* auglisi_host,
                   float* sum_x_host, float* sum_y_host, float* out2_host,
                   void* dev_scratch, size_t dev_scratch_bytes, void* stream) {
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
    const size_t ws_bytes = workspace_bytes_for(N, N_T);

    if (cudaMemcpyAsync(xd, x_host, img_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) return IQA_ERR_CUDA;
    if (cudaMemcpyAsync(yd, y_host, img_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) return IQA_ERR_CUDA;
    int rc = iqa_fused_tiles(xd, yd, N, N_T, C1, C2, C, D, d_lisi, d_aug, d_sx, d_sy, nullptr, nullptr,
                             ws_bytes ? ws : nullptr, ws_bytes, stream);
    if (rc != IQA_OK) return rc;
    rc = iqa_aggregate(d_lisi, d_aug, d_sx, d_sy, (int)n, C2, C, d_out2, stream);
    if (rc != IQA_OK) return rc;
    const size_t nb = n * sizeof(float);
    cudaError_t e = cudaSuccess;
    if (lisi_host && e == cudaSuccess) e = cudaMemcpyAsync(lisi_host, d_lisi, nb, cudaMemcpyDeviceToHost, st);
    if (auglisi_host && e == cudaSuccess) e = cudaMemcpyAsync(auglisi_host, d_aug, nb, cudaMemcpyDeviceToHost, st);
    if (sum_x_host && e == cudaSuccess) e = cudaMemcpyAsync(sum_x_host, d_sx, nb, cudaMemcpyDeviceToHost, st);
    if (sum_y_host && e == cudaSuccess) e = cudaMemcpyAsync(sum_y_host, d_sy, nb, cudaMemcpyDeviceToHost, st);
    if (out2_host && e == cudaSuccess) e = cudaMemcpyAsync(out2_host, d_out2, 2 * sizeof(float), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    return e == cudaSuccess ? IQA_OK : IQA_ERR_CUDA;
}

}  // extern "C"
