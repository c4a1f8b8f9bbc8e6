// =============================================================================
// iqa_oracle.cpp -- CPU ORACLE for tile-wise LISI / augLISI.  TEST INFRASTRUCTURE.
//
// This file is the plain definition of what the hot path computes, written out
// from the paper (arxiv 2501.10653; citations "P:NN" = line NN of PAPER.md):
//   * Eq. 1  LISI
//   * Eq. 2  augLISI
//   * clamp  "negative pixel values in the inputs are set to zeros"   P:27 (Sec. 2)
//   * tiling N x N image -> n = (N/N_T)^2 tiles of N_T x N_T
//   * Eq. 3  LISI aggregation over tiles
//   * Eq. 4  augLISI aggregation over tiles
//
// It is deliberately slow and obvious: one loop nest tiles -> rows -> pixels,
// every accumulation in double, no blocking, no fusion, no reordering.  The only
// parallelism is "#pragma omp parallel for" over tiles (tiles are independent,
// P:29), which does not change any arithmetic.
//
// It shares NO code with the CUDA path (paper_2501_10653_b200/csrc) and must
// never be imported, linked or executed by the product path.  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs use it.
//
// Parity pins (tests/test_oracle_pins.py): every function below is pinned by
// exact-rational brute force, a hand-derived worked example, closed forms and
// invariants -- nothing here is "parity unpinned".
//
// Readings of the paper where it is silent:
//   R1  D is a caller-supplied constant (the paper never defines it); callers use D = C1/2.
//   R2  the sums in Eqs. 1-2 run over the N_T x N_T pixels of the tile (Eq. 3 confirms).
//   R3  clamp is  v > 0 ? v : 0  (NaN -> 0, -0 -> +0, -Inf -> 0).
//   R5  the IQA matrix is row-major [ty][tx]; tile t = ty*(N/N_T)+tx.
//   R8  outputs are NOT clamped to [0,1] (augLISI can be negative).
//
// Build: g++ -O2 -std=c++17 -fopenmp -ffp-contract=off -shared -fPIC  (no -ffast-math)
// =============================================================================
#include <cmath>
#include <cstddef>
#include <cstdint>
#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {

// Number of threads the OpenMP runtime would use (reported by bench.py as "cores").
int iqa_oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

// Per-tile LISI (Eq. 1) and augLISI (Eq. 2) of two N x N row-major fp32 images.
//   x, y         [N*N]  input images, read only
//   N, N_T       image side and tile side; N % N_T must be 0
//   C1,C2,C,D    constants of Eqs. 1-2 (promoted from the caller's fp32 values)
//   lisi,auglisi [n]    per-tile index values, n = (N/N_T)^2, t = ty*(N/N_T)+tx
//   X, Y         [n]    per-tile sums of the clamped x and y   (denominators of Eqs. 1-2)
//   L, A         [n]    per-tile numerators: sum |x+y|/(|x-y|+C1) and sum |x+y||x-y|
//   threads      OpenMP threads (<=0: runtime default)
// Returns 0 on success, 1 on a bad argument.
int iqa_oracle_tiles(const float* x, const float* y, long N, long N_T,
                     double C1, double C2, double C, double D,
                     double* lisi, double* auglisi,
                     double* X, double* Y, double* L, double* A,
                     int threads) {
    if (!x || !y || !lisi || !auglisi || !X || !Y || !L || !A) return 1;
    if (N <= 0 || N_T <= 0 || N % N_T != 0) return 1;
    const long nt = N / N_T;          // tiles per side
    const long n = nt * nt;
#ifdef _OPENMP
    const int nthreads = threads > 0 ? threads : omp_get_max_threads();
#pragma omp parallel for schedule(static) num_threads(nthreads)
#else
    (void)threads;
#endif
    for (long t = 0; t < n; ++t) {
        const long ty = t / nt, tx = t % nt;
        double sumL = 0.0, sumA = 0.0, sumX = 0.0, sumY = 0.0;
        for (long r = 0; r < N_T; ++r) {
            const long row = ty * N_T + r;
            for (long c = 0; c < N_T; ++c) {
                const long k = row * N + (tx * N_T + c);
                // negative pixels are set to zero before anything else.
                const double xd = (x[k] > 0.0f) ? (double)x[k] : 0.0;
                const double yd = (y[k] > 0.0f) ? (double)y[k] : 0.0;
                const double s = std::fabs(xd + yd);     // |x_i + y_i|
                const double d = std::fabs(xd - yd);     // |x_i - y_i|
                sumL += s / (d + C1);                    // numerator of Eq. 1
                sumA += s * d;                           // numerator of Eq. 2
                sumX += xd;
                sumY += yd;
            }
        }
        const double mx = sumX > sumY ? sumX : sumY;
        lisi[t] = D * sumL / (mx + C2);                  // Eq. 1
        auglisi[t] = 1.0 - sumA / (sumX + sumY + C);     // Eq. 2
        X[t] = sumX; Y[t] = sumY; L[t] = sumL; A[t] = sumA;
    }
    return 0;
}

// The same per-tile Eq. 1 / Eq. 2 for a general H x W image with a row pitch (SURVEY.md 8(f)-4,
// DESIGN.md reading R18): the image is cut into cells of N_T x N_T starting at (0, 0); a cell that
// sticks out over the right / bottom border is an EDGE TILE and holds only the pixels that exist
// ("N" in Eqs. 1-2 is the pixel count of the region compared, reading R2).
//   x, y         row r, column c is x[r * pitch_x + c] / y[r * pitch_y + c]  (pitches in elements)
//   outputs      [nty * ntx] with nty = ceil(H / N_T), ntx = ceil(W / N_T), t = ty * ntx + tx
int iqa_oracle_tiles_2d(const float* x, const float* y, long H, long W, long pitch_x, long pitch_y, long N_T,
                        double C1, double C2, double C, double D,
                        double* lisi, double* auglisi, double* X, double* Y, double* L, double* A,
                        int threads) {
    if (!x || !y || !lisi || !auglisi || !X || !Y || !L || !A) return 1;
    if (H <= 0 || W <= 0 || N_T <= 0 || pitch_x < W || pitch_y < W) return 1;
    const long nty = (H + N_T - 1) / N_T, ntx = (W + N_T - 1) / N_T;
    const long n = nty * ntx;
#ifdef _OPENMP
    const int nthreads = threads > 0 ? threads : omp_get_max_threads();
#pragma omp parallel for schedule(static) num_threads(nthreads)
#else
    (void)threads;
#endif
    for (long t = 0; t < n; ++t) {
        const long ty = t / ntx, tx = t % ntx;
        const long r_end = (ty + 1) * N_T < H ? (ty + 1) * N_T : H;      // edge tiles stop at the border
        const long c_end = (tx + 1) * N_T < W ? (tx + 1) * N_T : W;
        double sumL = 0.0, sumA = 0.0, sumX = 0.0, sumY = 0.0;
        for (long r = ty * N_T; r < r_end; ++r) {
            for (long c = tx * N_T; c < c_end; ++c) {
                const float xv = x[r * pitch_x + c], yv = y[r * pitch_y + c];
                const double xd = (xv > 0.0f) ? (double)xv : 0.0;
                const double yd = (yv > 0.0f) ? (double)yv : 0.0;
                const double s = std::fabs(xd + yd);
                const double d = std::fabs(xd - yd);
                sumL += s / (d + C1);
                sumA += s * d;
                sumX += xd;
                sumY += yd;
            }
        }
        const double mx = sumX > sumY ? sumX : sumY;
        lisi[t] = D * sumL / (mx + C2);                  // Eq. 1
        auglisi[t] = 1.0 - sumA / (sumX + sumY + C);     // Eq. 2
        X[t] = sumX; Y[t] = sumY; L[t] = sumL; A[t] = sumA;
    }
    return 0;
}

// The same for pixels given as DOUBLES (FITS planes come as BITPIX -64, 16, 32, 8 ...;
// every such pixel value converts to double exactly, so the caller converts and this routine is the
// definition for all of them).  Identical loop nest; only the element type of x and y differs.
int iqa_oracle_tiles_2d_f64(const double* x, const double* y, long H, long W, long pitch_x, long pitch_y, long N_T,
                            double C1, double C2, double C, double D,
                            double* lisi, double* auglisi, double* X, double* Y, double* L, double* A,
                            int threads) {
    if (!x || !y || !lisi || !auglisi || !X || !Y || !L || !A) return 1;
    if (H <= 0 || W <= 0 || N_T <= 0 || pitch_x < W || pitch_y < W) return 1;
    const long nty = (H + N_T - 1) / N_T, ntx = (W + N_T - 1) / N_T;
    const long n = nty * ntx;
#ifdef _OPENMP
    const int nthreads = threads > 0 ? threads : omp_get_max_threads();
#pragma omp parallel for schedule(static) num_threads(nthreads)
#else
    (void)threads;
#endif
    for (long t = 0; t < n; ++t) {
        const long ty = t / ntx, tx = t % ntx;
        const long r_end = (ty + 1) * N_T < H ? (ty + 1) * N_T : H;
        const long c_end = (tx + 1) * N_T < W ? (tx + 1) * N_T : W;
        double sumL = 0.0, sumA = 0.0, sumX = 0.0, sumY = 0.0;
        for (long r = ty * N_T; r < r_end; ++r) {
            for (long c = tx * N_T; c < c_end; ++c) {
                const double xv = x[r * pitch_x + c], yv = y[r * pitch_y + c];
                const double xd = (xv > 0.0) ? xv : 0.0;                 // P:27 (NaN -> 0 as well)
                const double yd = (yv > 0.0) ? yv : 0.0;
                const double s = std::fabs(xd + yd);
                const double d = std::fabs(xd - yd);
                sumL += s / (d + C1);
                sumA += s * d;
                sumX += xd;
                sumY += yd;
            }
        }
        const double mx = sumX > sumY ? sumX : sumY;
        lisi[t] = D * sumL / (mx + C2);                  // Eq. 1
        auglisi[t] = 1.0 - sumA / (sumX + sumY + C);     // Eq. 2
        X[t] = sumX; Y[t] = sumY; L[t] = sumL; A[t] = sumA;
    }
    return 0;
}

// Tile -> whole-image aggregation, Eqs. 3-4, over n tiles (n >= 1).
//   out2[0] = LISI of the whole image, out2[1] = augLISI of the whole image.
// "Whole image" may be any set of tiles merged into a larger tile: the caller
// passes exactly the tiles to merge.
int iqa_oracle_aggregate(const double* lisi, const double* auglisi,
                         const double* X, const double* Y, long n,
                         double C2, double C, double* out2) {
    if (!lisi || !auglisi || !X || !Y || !out2 || n <= 0) return 1;
    double SX = 0.0, SY = 0.0;
    for (long t = 0; t < n; ++t) { SX += X[t]; SY += Y[t]; }
    double num3 = 0.0, num4 = 0.0;
    for (long t = 0; t < n; ++t) {
        const double mt = X[t] > Y[t] ? X[t] : Y[t];
        num3 += lisi[t] * (mt + C2);                     // Eq. 3 numerator
        num4 += auglisi[t] * (X[t] + Y[t] + C);          // Eq. 4 numerator (first part)
    }
    const double M = SX > SY ? SX : SY;
    out2[0] = num3 / (M + C2);                           // Eq. 3
    out2[1] = (num4 - (double)(n - 1) * C) / (SX + SY + C);   // Eq. 4
    return 0;
}

}  // extern "C"
