/* =============================================================================
 * iqa_tiles.h -- C ABI of libiqa_tiles.so: tile-wise LISI / augLISI on one B200.
 *
 * What the library computes (arxiv 2501.10653; "P:NN" = line NN of PAPER.md):
 *   clamp     negative pixels are set to zero before everything else        P:27  (Sec. 2)
 *   Eq. 1     lisi_t    = D * L_t / (max(X_t, Y_t) + C2),
 *             L_t = sum_k |x_k + y_k| / (|x_k - y_k| + C1)
 *   Eq. 2     auglisi_t = 1 - A_t / (X_t + Y_t + C),
 *             A_t = sum_k |x_k + y_k| * |x_k - y_k|
 *             X_t = sum_k x_k, Y_t = sum_k y_k over the N_T x N_T pixels of tile t
 *   tiling    N x N image -> n = (N/N_T)^2 tiles, one value per tile
 *             ("IQA matrix")
 *   Eq. 3/4   tile -> whole-image aggregation of the two matrices
 *   merge     the "entire image" of Eqs. 3-4 may be a larger tile formed by
 *             merging g x g smaller ones
 * and, built on the same kernels (each section below cites its passage):
 *   series    K comparisons of a time series, every snapshot read from HBM once
 *   finder    tiles below a threshold / the k lowest tiles of a matrix
 *   general   H x W images with a row pitch, edge tiles, other pixel types
 *   sharding  one pair over several GPUs by bands of tile rows
 *
 * Conventions (the paper states none; DESIGN.md "Boundary" and "Readings"):
 *   * Every pointer is a DEVICE pointer owned by the caller unless the argument name ends
 *     in `_host`.  The library allocates no device memory and keeps no state between calls
 *     (beyond a per-device cache of launch geometry: SM count, resident CTAs per SM).
 *   * `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Device
 *     entry points are ASYNCHRONOUS: they validate, enqueue and return; outputs are valid
 *     once the stream has reached that point.  x and y are never written.
 *   * Images are fp32, row-major, contiguous: pixel (r, c) is x[r*N + c].  Tile
 *     t = ty*(N/N_T) + tx covers rows ty*N_T.. and columns tx*N_T..; every per-tile array
 *     is indexed by t (a row-major (N/N_T) x (N/N_T) matrix with the image's orientation).
 *   * Clamp is v > 0 ? v : 0, so NaN, -0 and -Inf become +0 (FITS blank pixels read as
 *     empty sky).  +Inf pixels give unspecified output.  Outputs are NOT clamped to [0,1]
 *     (augLISI is negative when sum|x+y||x-y| exceeds sum x + sum y + C).
 *   * D is caller-supplied; the paper never defines it.  D = C1/2 makes LISI(x, x) -> 1.
 *   * Errors: a status code is returned, nothing is thrown or printed, and NOTHING is
 *     enqueued when the status is not IQA_OK (validation precedes the first launch).
 *       NULL required pointer ....................................... IQA_ERR_NULL
 *       N <= 0, N_T <= 0, N % N_T != 0, n_tiles <= 0,
 *       n_pairs <= 0, g bad, unknown pixel type ..................... IQA_ERR_SHAPE
 *       C2 or C not finite or <= 0, D not finite, C1 not a NORMAL
 *       positive float (C1 >= FLT_MIN: |x - y| + C1 feeds a
 *       flush-to-zero reciprocal) ................................... IQA_ERR_PARAM
 *       x or y not aligned to their element size (4 bytes for fp32) . IQA_ERR_ALIGN
 *       workspace NULL / too small when iqa_workspace_bytes() > 0 ... IQA_ERR_WORKSPACE
 *       CUDA launch / copy failure .................................. IQA_ERR_CUDA
 *     Every tensor map of a call is encoded on the host BEFORE its first launch (a map that cannot be
 *     encoded downgrades the whole call to the generic kernels), so validation, planning and encoding
 *     never leave work behind.  IQA_ERR_CUDA from a failing launch or copy is the one exception: earlier
 *     launches of the same call may already be enqueued and the outputs are then undefined.
 *   * Any N_T that divides N is accepted.  Images whose row pitch is a multiple of 16 bytes (N % 4 == 0
 *     for the square fp32 entry points) and whose bases sit at the same offset inside their 16-byte
 *     lines take a persistent TMA-fed kernel: tma_kernel for fp32 with a power-of-two N_T >= 8 and
 *     16-byte aligned bases, any_kernel for every other N_T >= 4, the other pixel types and shifted
 *     bases -- except the shapes that would leave most of any_kernel's lanes idle (split tiles of
 *     113 .. ~200 columns, a 64-column tile behind a shifted base), which, like every other pitch and
 *     N_T < 4, take the generic kernel (128-bit loads when x and y are aligned alike, scalar loads
 *     otherwise; still CUDA).  iqa_query_plan tells which.  Results are deterministic: fixed reduction
 *     order, no floating-point atomics; two calls on the same inputs are bit-identical.
 * ============================================================================= */
#ifndef IQA_TILES_H
#define IQA_TILES_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    IQA_OK = 0,
    IQA_ERR_NULL = 1,
    IQA_ERR_SHAPE = 2,
    IQA_ERR_PARAM = 3,
    IQA_ERR_ALIGN = 4,
    IQA_ERR_WORKSPACE = 5,
    IQA_ERR_CUDA = 6,
    IQA_ERR_STATIC_LIMIT = 7      /* iqa_fused_tiles_static only: the shape needs more than IQA_STATIC_WORKSPACE_BYTES */
} iqa_status;

/* Static, never-freed description of a status code ("unknown status" for other values). */
const char* iqa_status_string(int status);

/* Library version, "major.minor.patch". */
const char* iqa_version(void);

/* Bytes of device workspace the *_tiles entry points need for (N, N_T): 0 when every tile
 * is finished inside one CTA, else room for the per-piece partial sums of split tiles
 * (16 B per piece of 128 x 64 pixels).  Returns 0 for invalid shapes (the entry points report those). */
size_t iqa_workspace_bytes(int N, int N_T);

/* Eq. 1 per tile (clamp P:27).
 *   x, y      [N*N]  device, read-only
 *   lisi      [n]    device, written; n = (N/N_T)^2
 *   workspace        device scratch of >= iqa_workspace_bytes(N, N_T) bytes (may be NULL when 0),
 *                    contents undefined before and after */
int iqa_lisi_tiles(const float* x, const float* y, int N, int N_T,
                   float C1, float C2, float D,
                   float* lisi,
                   void* workspace, size_t workspace_bytes, void* stream);

/* Eq. 2 per tile (clamp P:27).  Arguments as above. */
int iqa_auglisi_tiles(const float* x, const float* y, int N, int N_T, float C,
                      float* auglisi,
                      void* workspace, size_t workspace_bytes, void* stream);

/* Eq. 1 and Eq. 2 per tile from ONE read of x and y, plus the per-tile sums Eqs. 3-4 need.
 *   lisi, auglisi        [n] each, required
 *   sum_x, sum_y         [n] each, required: X_t, Y_t (clamped sums)
 *   lisi_num, auglisi_num [n] each, MAY BE NULL: the raw numerators L_t and A_t */
int iqa_fused_tiles(const float* x, const float* y, int N, int N_T,
                    float C1, float C2, float C, float D,
                    float* lisi, float* auglisi,
                    float* sum_x, float* sum_y,
                    float* lisi_num, float* auglisi_num,
                    void* workspace, size_t workspace_bytes, void* stream);

/* ---- the same call for programs that may not allocate device memory ---------------------------
 * iqa_fused_tiles wants a workspace for tiles wider than 64 pixels, and somebody has to cudaMalloc it.
 * Some users of this library cannot: a plug-in inside a telescope pipeline or an inference server whose
 * host program hands out ALL device memory at start-up and gives a plug-in nothing but the pointers of its
 * input and output buffers; a per-snapshot loop that must never hit the device-wide synchronisation that
 * cudaMalloc / cudaFree imply; a binding from a language that has no CUDA allocator at hand.  For them
 * iqa_fused_tiles_static is iqa_fused_tiles with the workspace argument removed: the partial sums of split
 * tiles go to a fixed array of IQA_STATIC_WORKSPACE_BYTES that is part of the library image itself (a
 * file-scope __device__ array in iqa_tiles.cu).  Same kernels, same order of summation: the outputs are
 * bit-identical to iqa_fused_tiles on the same inputs.
 *
 *   cost      every GPU on which this process uses the library keeps those IQA_STATIC_WORKSPACE_BYTES (1 MiB)
 *             reserved from the moment the library's code is loaded onto it until the process ends, whether
 *             or not this entry point is ever called.
 *   limit     shapes with iqa_workspace_bytes(N, N_T) > IQA_STATIC_WORKSPACE_BYTES are refused with
 *             IQA_ERR_STATIC_LIMIT before anything is enqueued (1 MiB covers every BASELINE.json
 *             configuration up to N = 16384, N_T = 128; N = 32768, N_T = 128 would need 4 MiB: use
 *             iqa_fused_tiles with a workspace of your own there).  Shapes that need no workspace
 *             (N_T <= 64, ...) never touch the array.
 *   set-up    the FIRST call on each device that needs the array looks up its device address (one
 *             cudaGetSymbolAddress with that device current, cached per device afterwards; a failure is
 *             IQA_ERR_CUDA).  Make that first call during start-up, outside any stream capture.
 *   no allocation   the call itself never calls cudaMalloc, cudaFree, or a library routine that does.
 *   sharing   ALL calls on a device use the SAME array, and it keeps whatever the last call left in it.
 *             Nothing in it has to start at zero -- every slot the second pass reads was written by the
 *             first pass of the same call -- so no clearing is done or needed.  But two calls that may
 *             run on the GPU at the same time (different streams, or different host threads on
 *             different streams) RACE on it and both results are then garbage: keep the calls of one
 *             device on one stream, or order them with events.  Calls on different devices do not interact.
 * Arguments and every other error as iqa_fused_tiles (lisi_num, auglisi_num MAY BE NULL). */
#define IQA_STATIC_WORKSPACE_BYTES 1048576
int iqa_fused_tiles_static(const float* x, const float* y, int N, int N_T,
                           float C1, float C2, float C, float D,
                           float* lisi, float* auglisi,
                           float* sum_x, float* sum_y,
                           float* lisi_num, float* auglisi_num,
                           void* stream);

/* Diagnostic: which kernel a call on this image would take (host-side decision only, nothing is enqueued).
 *   x, pixel_type, H, W, pitch, N_T as for iqa_fused_tiles_2d_typed; series != 0: as for the time-series entry points.
 * Returns IQA_PLAN_GENERIC, IQA_PLAN_TMA_ANY (any_kernel: any N_T >= 4, any pixel type; the time-series entry points
 * run it as one launch per 32 comparisons in pair-minor order; `series` is answered for a series of three or more
 * images -- a two-image series is planned like the pair it is), or IQA_PLAN_TMA + c (tma_kernel, c = its ring / box
 * configuration, 0..4); -1 for bad arguments.  bench.py reports it, and the GPU tests assert that every BASELINE.json configuration takes tma_kernel
 * -- a silent fall-back would cost bandwidth, not parity. */
#define IQA_PLAN_GENERIC 0
#define IQA_PLAN_TMA_ANY 2
#define IQA_PLAN_TMA 16
int iqa_query_plan(const void* x, int pixel_type, int H, int W, long long pitch, int N_T, int series);

/* The same for a call of a given size.  One rule of the plan depends on how much work the call holds: the generic
 * kernel (one warp per piece of a tile) only beats any_kernel's idle lanes when the whole call has several pieces per
 * SM, so SMALL jobs -- one or two pairs of a 1024^2 or 2048^2 image with tiles of 113 .. 400 columns -- keep any_kernel
 * (up to 3x faster there).  iqa_query_plan answers for a job large enough to fill the GPU; iqa_query_plan_n answers for
 * n_cmp pairs (or comparisons of a series; 0 = large job) on the CURRENT device (without a device: the large-job answer). */
int iqa_query_plan_n(const void* x, int pixel_type, int H, int W, long long pitch, int N_T, int series, int n_cmp);

/* Test and tuning hook, NOT part of the stable ABI (names and meanings may change with any release): sets one of the
 * library's process-wide knobs and returns its previous value (-1: unknown name).  The library never reads the
 * environment; only a build with -DIQA_TESTING takes the knobs' initial values from the environment variables of
 * the same names:
 *   IQA_FORCE_GENERIC 1: generic kernels only        IQA_FORCE_ANY 1: any_kernel instead of tma_kernel
 *   IQA_TMA_CONFIG 0..4: tma_kernel ring / box configuration (-1: default)
 *   IQA_TMA_MAX_CTAS n: cap of the persistent grid (0: none)     IQA_NO_PDL 1: no programmatic dependent launch
 *   IQA_CAND_NO_CLUSTER 1: candidate kernels without thread-block clusters
 *   IQA_ANY_NO_WIDE 1: any_kernel lanes own four columns even when eight would fit
 *   IQA_PLAN_LARGE_JOB 1: plan every call as a large job (the small-job rule of iqa_query_plan_n off)
 * They select among kernels that all satisfy the same parity bar (tests/test_gpu_parity.py runs every one). */
int iqa_debug_knob(const char* name, int value);

/* ---- general images -------------------------------------------------------
 * The paper's images are square and N is a multiple of N_T.  This entry point drops
 * both: an H x W image with a row pitch (elements between rows; a sub-window of a larger array, a
 * padded FITS plane) is cut into cells of N_T x N_T starting at (0, 0); a cell that sticks out over
 * the right / bottom border is an EDGE TILE and holds only the pixels that exist ("N" in Eqs. 1-2
 * is the pixel count of the region compared).  That equals zero-padding both images to a multiple
 * of N_T, because after the clamp a zero pixel pair adds nothing to any of the four sums.
 *   x, y            pixel (r, c) is x[r * pitch_x + c] / y[r * pitch_y + c]; pitch >= W
 *   outputs         [nty * ntx], nty = ceil(H / N_T), ntx = ceil(W / N_T), t = ty * ntx + tx
 *   workspace       >= iqa_workspace_bytes_2d(H, W, N_T) bytes (may be NULL when 0)
 * Eqs. 3-4 over the result: iqa_aggregate with n_tiles = nty * ntx.  Pitches that are multiples of 4 take a
 * TMA-fed kernel (the TMA unit zero-fills what lies outside the image; the base needs 4-byte alignment only)
 * unless the shape would fill too few of that kernel's lanes (the lane-fill thresholds of the preamble: split tiles
 * of 113 .. ~200 columns, a 64-column tile behind a shifted base); those shapes, other pitches and N_T < 4 take the
 * generic kernel.  iqa_query_plan tells which. */
size_t iqa_workspace_bytes_2d(int H, int W, int N_T);
int iqa_fused_tiles_2d(const float* x, const float* y, int H, int W, long long pitch_x, long long pitch_y, int N_T,
                       float C1, float C2, float C, float D,
                       float* lisi, float* auglisi, float* sum_x, float* sum_y,
                       float* lisi_num, float* auglisi_num,
                       void* workspace, size_t workspace_bytes, void* stream);

/* Other pixel types (FITS BITPIX -64, 16, 32, 8; fp16 from a GPU imager): the same computation on an
 * H x W image of `pixel_type` pixels (pitches in ELEMENTS of that type; pointers aligned to the element
 * size).  Every such value is exact in double; types that are exact in fp32 (F16, I16, U8) are converted
 * and follow the fp32 arithmetic, F64 and I32 are clamped, added and subtracted in fp64 before rounding
 * (the Eq. 1 term is ill-conditioned in x - y).  Row pitches that are multiples of 16 BYTES and N_T >= 4 take the
 * TMA-fed any_kernel (tensor maps of the element type; algorithmic bytes 2 sizeof(pixel) per pixel pair); other
 * pitches take the generic kernels.  Unknown pixel_type: IQA_ERR_SHAPE. */
typedef enum {
    IQA_PIXEL_F32 = 0, IQA_PIXEL_F64 = 1, IQA_PIXEL_F16 = 2, IQA_PIXEL_I16 = 3, IQA_PIXEL_I32 = 4, IQA_PIXEL_U8 = 5
} iqa_pixel_type;
int iqa_fused_tiles_2d_typed(const void* x, const void* y, int pixel_type,
                             int H, int W, long long pitch_x, long long pitch_y, int N_T,
                             float C1, float C2, float C, float D,
                             float* lisi, float* auglisi, float* sum_x, float* sum_y,
                             float* lisi_num, float* auglisi_num,
                             void* workspace, size_t workspace_bytes, void* stream);

/* The batch and time-series entry points (below) for general images: all images of the call share
 * H, W and ONE row pitch.  Workspace: n_pairs (resp. n_images - 1) * iqa_workspace_bytes_2d(H, W, N_T).
 * Outputs as for the square entry points with n = ceil(H / N_T) * ceil(W / N_T) tiles per comparison. */
int iqa_fused_batch_2d(const float* const* x_ptrs_host, const float* const* y_ptrs_host, int n_pairs,
                       int H, int W, long long pitch, int N_T, float C1, float C2, float C, float D,
                       float* lisi, float* auglisi, float* sum_x, float* sum_y,
                       float* lisi_num, float* auglisi_num, float* out2,
                       void* workspace, size_t workspace_bytes, void* stream);
int iqa_series_tiles_2d(const float* const* img_ptrs_host, int n_images, int mode,
                        int H, int W, long long pitch, int N_T, float C1, float C2, float C, float D,
                        float* lisi, float* auglisi, float* sum_x, float* sum_y,
                        float* lisi_num, float* auglisi_num, float* out2,
                        void* workspace, size_t workspace_bytes, void* stream);

/* The same two entry points for images of `pixel_type` pixels (pitch in ELEMENTS of that type).  Batches run in
 * one any_kernel launch per 32 pairs.  A typed time series is ONE any_kernel launch per 32 comparisons in pair-minor
 * item order: the comparisons of one image location run on neighbouring CTAs, so each snapshot comes from HBM once
 * and its second reader finds it in L2 (only fp32 images with a power-of-two N_T have the kernel that keeps the
 * shared image in shared memory).  Shapes below the lane-fill thresholds, and pitches no tensor map can describe,
 * take the generic kernels instead; iqa_query_plan is the source of truth for which kernel a call takes. */
int iqa_fused_batch_2d_typed(const void* const* x_ptrs_host, const void* const* y_ptrs_host, int n_pairs, int pixel_type,
                             int H, int W, long long pitch, int N_T, float C1, float C2, float C, float D,
                             float* lisi, float* auglisi, float* sum_x, float* sum_y,
                             float* lisi_num, float* auglisi_num, float* out2,
                             void* workspace, size_t workspace_bytes, void* stream);
int iqa_series_tiles_2d_typed(const void* const* img_ptrs_host, int n_images, int mode, int pixel_type,
                              int H, int W, long long pitch, int N_T, float C1, float C2, float C, float D,
                              float* lisi, float* auglisi, float* sum_x, float* sum_y,
                              float* lisi_num, float* auglisi_num, float* out2,
                              void* workspace, size_t workspace_bytes, void* stream);

/* Bytes of device workspace iqa_fused_batch needs: n_pairs * iqa_workspace_bytes(N, N_T). */
size_t iqa_batch_workspace_bytes(int n_pairs, int N, int N_T);

/* The whole hot path over a BATCH of image pairs of one shape (e.g. the snapshots of a time
 * series, or the 16-pair throughput loop of BASELINE.json config [4]) in as few launches as
 * possible: one persistent kernel streams all pairs (Eqs. 1-2 per tile, clamp fused into the
 * load), then -- only for tiles larger than 64 -- one finalise pass, then, when out2 is given,
 * one launch applies Eqs. 3-4 to every pair.
 *   x_ptrs_host, y_ptrs_host  HOST arrays of n_pairs DEVICE pointers to [N*N] images; the
 *                        arrays are read during the call only (they may be freed on return)
 *   lisi, auglisi, sum_x, sum_y  [n_pairs * n] device, required; pair p occupies [p*n, (p+1)*n)
 *   lisi_num, auglisi_num        [n_pairs * n] device, MAY BE NULL
 *   out2                 [n_pairs * 2] device, MAY BE NULL: out2[2p] = LISI, out2[2p+1] = augLISI of pair p
 *   workspace            >= iqa_batch_workspace_bytes(n_pairs, N, N_T) bytes (may be NULL when 0)
 * n_pairs * n must stay below 2^31.  Results are bit-identical to n_pairs calls of
 * iqa_fused_tiles + iqa_aggregate whenever the batch and the single call take the same kernel (always for the
 * power-of-two tile sides of tma_kernel and for whole-tile any_kernel shapes; the one size-dependent rule, for split
 * tiles of 113 .. 400 columns on small images, is described at iqa_query_plan_n): the kernel is chosen per run of
 * consecutive pairs whose x and y
 * sit at the same offset inside their 16-byte lines, as it would be for each pair alone, so one
 * shifted pair costs the aligned pairs of its batch nothing (it only splits the batch into more launches). */
int iqa_fused_batch(const float* const* x_ptrs_host, const float* const* y_ptrs_host, int n_pairs,
                    int N, int N_T, float C1, float C2, float C, float D,
                    float* lisi, float* auglisi, float* sum_x, float* sum_y,
                    float* lisi_num, float* auglisi_num, float* out2,
                    void* workspace, size_t workspace_bytes, void* stream);

/* ---- time series ---------------------------------------------------------
 * "Transients typically exhibit on-and-off emission behaviour, causing intensity variations
 * between observations of the same section of the sky, while fixed sources remain unchanged"
 * (P:39); "the rest of the image remains largely stable with slight variations over time".
 * A series of n_images snapshots I_0 .. I_{n_images-1} of one field gives K = n_images - 1
 * comparisons, each of them exactly the pair computation above (clamp P:27, Eqs. 1-2 per tile,
 * Eqs. 3-4 for the whole image):
 *   IQA_SERIES_REFERENCE    comparison k is (x, y) = (I_0, I_{k+1})
 *   IQA_SERIES_CONSECUTIVE  comparison k is (x, y) = (I_k, I_{k+1})
 * For 16-byte aligned images and a power-of-two N_T >= 8 one persistent TMA-fed kernel keeps the
 * x block of every comparison in shared memory, so each image is read from HBM ONCE:
 * 4 (K+1)/K bytes per pixel and comparison instead of the 8 of K independent pair calls.  Other
 * tile sides and pixel types (the _typed entry points) run the K pair computations in ONE launch of
 * the general TMA kernel whose item order puts the comparisons of one image location on neighbouring
 * CTAs: every image still comes from HBM once, its second reader finds it in L2.  Row pitches no
 * tensor map can describe are computed pair by pair (same results, 8 bytes). */
#define IQA_SERIES_REFERENCE 0
#define IQA_SERIES_CONSECUTIVE 1

/* Bytes of device workspace iqa_series_tiles needs: (n_images - 1) * iqa_workspace_bytes(N, N_T). */
size_t iqa_series_workspace_bytes(int n_images, int N, int N_T);

/*   img_ptrs_host        HOST array of n_images DEVICE pointers to [N*N] images (read during the call only)
 *   mode                 IQA_SERIES_REFERENCE or IQA_SERIES_CONSECUTIVE (anything else: IQA_ERR_SHAPE)
 *   lisi, auglisi, sum_x, sum_y  [K * n] device, required; comparison k occupies [k*n, (k+1)*n);
 *                        sum_x holds the tile sums of the comparison's x image, sum_y of its y image
 *   lisi_num, auglisi_num        [K * n] device, MAY BE NULL
 *   out2                 [K * 2] device, MAY BE NULL: Eqs. 3-4 per comparison (LISI, augLISI)
 *   workspace            >= iqa_series_workspace_bytes(n_images, N, N_T) bytes (may be NULL when 0)
 * n_images >= 2; K * n must stay below 2^31.  Results agree with K calls of iqa_fused_tiles +
 * iqa_aggregate to fp32 rounding of the same sums (bit-identical when the same kernel serves both). */
int iqa_series_tiles(const float* const* img_ptrs_host, int n_images, int mode,
                     int N, int N_T, float C1, float C2, float C, float D,
                     float* lisi, float* auglisi, float* sum_x, float* sum_y,
                     float* lisi_num, float* auglisi_num, float* out2,
                     void* workspace, size_t workspace_bytes, void* stream);

/* Eqs. 3-4: merge n_tiles per-tile values into the whole-image pair.
 *   out2 [2] device: out2[0] = LISI, out2[1] = augLISI.  Sums are taken in double, fixed order.
 * Eq. 3 holds no D (it is inside lisi_t), so only C2 and C are needed. */
int iqa_aggregate(const float* lisi, const float* auglisi,
                  const float* sum_x, const float* sum_y, int n_tiles,
                  float C2, float C,
                  float* out2, void* stream);

/* ---- one image pair sharded over GPUs by bands of tile rows -------------------
 * Tiles are independent, so rank r computes the tiles of its band of rows with
 * iqa_fused_tiles_2d (a band is a contiguous range of rows: H = rows of the band, same pitch) and
 * nothing is exchanged for the matrices.  Only the whole-image pair of Eqs. 3-4 needs the other
 * bands: every rank reduces ITS tiles to four double sums with iqa_aggregate_partial,
 *   sums4 = { sum_t lisi_t (max(X_t, Y_t) + C2),  sum_t auglisi_t (X_t + Y_t + C),  sum_t X_t,  sum_t Y_t },
 * the ranks all-reduce (sum) these 32 bytes (NCCL), and iqa_aggregate_finish applies
 *   LISI = sums4[0] / (max(sums4[2], sums4[3]) + C2),
 *   augLISI = (sums4[1] - (n_tiles_total - 1) C) / (sums4[2] + sums4[3] + C)            (Eqs. 3-4).
 * sums4: DEVICE double[4], 8-byte aligned. */
int iqa_aggregate_partial(const float* lisi, const float* auglisi,
                          const float* sum_x, const float* sum_y, int n_tiles,
                          float C2, float C, double* sums4, void* stream);
int iqa_aggregate_finish(const double* sums4, long long n_tiles_total, float C2, float C,
                         float* out2, void* stream);

/* ---- candidate extraction ------------------------------------------------
 * The finder's output: which tiles changed.  The paper gives no decision rule -- it shows the
 * matrices (Fig. 3) and says augLISI localises "transients to tiles with fewer false positives"
 * -- so the rule is the plainest one, applied to any of the per-tile matrices (lisi or
 * auglisi; low = dissimilar).  `values` holds n_maps matrices of n_tiles values each
 * ([n_maps][n_tiles]: a batch of pairs or the comparisons of a series); values are compared as
 * the fp32 numbers they are, -0 == +0; results are exact and deterministic.
 *
 * iqa_tiles_below: tiles with value < threshold, ascending tile index.
 *   indices [n_maps * capacity]  first min(count, capacity) tile indices of each matrix (rest untouched)
 *   counts  [n_maps]             number of tiles below the threshold (may exceed capacity)
 *   threshold NaN -> IQA_ERR_PARAM; capacity may be 0 (count only; indices may then be NULL). */
int iqa_tiles_below(const float* values, int n_tiles, int n_maps, float threshold,
                    int* indices, int capacity, int* counts, void* stream);

/* iqa_tiles_bottom_k: the k tiles of lowest value of each matrix, ascending by (value, tile index).
 *   indices [n_maps * k], vals [n_maps * k] (MAY BE NULL: the values of those tiles)
 *   1 <= k <= 1024; when k > n_tiles the entries beyond n_tiles are index -1 / value +Inf. */
int iqa_tiles_bottom_k(const float* values, int n_tiles, int n_maps, int k,
                       int* indices, float* vals, void* stream);

/* iqa_series_find: the finder in ONE call (SURVEY.md 8(f)-2 + 8(f)-3) -- iqa_series_tiles followed,
 * on the same stream and inside the same call, by the candidate lists of every comparison taken from ONE of the two
 * matrices (`index`: IQA_FIND_LISI or IQA_FIND_AUGLISI).  The candidate kernels are launched behind the tile kernel
 * with programmatic dependent launch, so a caller pays no second call and no host round trip; the lists are
 * exactly those of iqa_tiles_bottom_k / iqa_tiles_below on that matrix.
 *   arguments up to `stream`   as iqa_series_tiles (K = n_images - 1 comparisons of n tiles)
 *   k, bottom_idx [K * k], bottom_val [K * k] (MAY BE NULL)   k = 0: no bottom-k list (bottom_idx may then be NULL)
 *   below_idx [K * capacity], below_counts [K]                 below_counts NULL: no threshold list
 * Either list may be left out, not both (IQA_ERR_NULL). */
#define IQA_FIND_LISI 0
#define IQA_FIND_AUGLISI 1
int iqa_series_find(const float* const* img_ptrs_host, int n_images, int mode,
                    int N, int N_T, float C1, float C2, float C, float D,
                    float* lisi, float* auglisi, float* sum_x, float* sum_y,
                    float* lisi_num, float* auglisi_num, float* out2,
                    void* workspace, size_t workspace_bytes,
                    int index, int k, int* bottom_idx, float* bottom_val,
                    float threshold, int* below_idx, int capacity, int* below_counts, void* stream);

/* iqa_series_find_2d_typed: the same for H x W images with a row pitch, edge tiles and any supported pixel type
 * (arguments as iqa_series_tiles_2d_typed, then the candidate arguments of iqa_series_find); n = ceil(H / N_T) * ceil(W / N_T). */
int iqa_series_find_2d_typed(const void* const* img_ptrs_host, int n_images, int mode, int pixel_type,
                             int H, int W, long long pitch, int N_T, float C1, float C2, float C, float D,
                             float* lisi, float* auglisi, float* sum_x, float* sum_y,
                             float* lisi_num, float* auglisi_num, float* out2,
                             void* workspace, size_t workspace_bytes,
                             int index, int k, int* bottom_idx, float* bottom_val,
                             float threshold, int* below_idx, int capacity, int* below_counts, void* stream);

/* P:66 "a larger tile formed by merging smaller ones": apply Eqs. 3-4 to every g x g block
 * of an nt x nt tile matrix, giving the (nt/g) x (nt/g) matrices of tile size g*N_T.
 *   in:  lisi, auglisi, sum_x, sum_y  [nt*nt]
 *   out: lisi_out, auglisi_out, sum_x_out, sum_y_out  [(nt/g)^2]   (nt % g == 0, g >= 1)
 * Outputs must not alias inputs. */
int iqa_merge_tiles(const float* lisi, const float* auglisi,
                    const float* sum_x, const float* sum_y, int nt, int g,
                    float C2, float C,
                    float* lisi_out, float* auglisi_out,
                    float* sum_x_out, float* sum_y_out, void* stream);

/* The same for n_maps matrices at once ([n_maps][nt*nt] in, [n_maps][(nt/g)^2] out): the comparisons of a
 * time series or the pairs of a batch -- multi-scale localisation of every comparison in one launch. */
int iqa_merge_tiles_batch(const float* lisi, const float* auglisi,
                          const float* sum_x, const float* sum_y, int nt, int g, int n_maps,
                          float C2, float C,
                          float* lisi_out, float* auglisi_out,
                          float* sum_x_out, float* sum_y_out, void* stream);

/* P:66, the whole pyramid in ONE launch: from the per-tile arrays of an nty x ntx tile matrix (any rectangle: the
 * output of iqa_fused_tiles_2d; n_maps of them stacked) every coarser level j = 1 .. L, L = iqa_pyramid_levels(nty, ntx)
 * = ceil(log2(max(nty, ntx))).  Level j merges blocks of 2^j x 2^j base tiles by Eqs. 3-4 into a
 * ceil(nty / 2^j) x ceil(ntx / 2^j) matrix, i.e. the tile matrix for tile side 2^j N_T; a block over the right / bottom
 * border merges only the tiles that exist, and Eq. 4's n is that count.  Every output tile is summed in double
 * directly from the BASE arrays (not from the rounded level below); level L is 1 x 1 and equals iqa_aggregate's pair.
 *   outputs  [n_maps][iqa_pyramid_tiles(nty, ntx)]: the levels one after the other, level j row-major at offset
 *            sum_{i<j} ceil(nty / 2^i) ceil(ntx / 2^i); may be NULL only when L == 0 (a 1 x 1 matrix).
 * Outputs must not alias inputs. */
int iqa_pyramid_levels(int nty, int ntx);
size_t iqa_pyramid_tiles(int nty, int ntx);
int iqa_pyramid(const float* lisi, const float* auglisi, const float* sum_x, const float* sum_y,
                int nty, int ntx, int n_maps, float C2, float C,
                float* lisi_out, float* auglisi_out, float* sum_x_out, float* sum_y_out, void* stream);

/* Bytes of DEVICE scratch iqa_fused_host needs for (N, N_T): both images, the four per-tile
 * arrays, out2 and the kernel workspace.  0 for invalid shapes. */
size_t iqa_host_scratch_bytes(int N, int N_T);

/* The whole hot path on HOST buffers (the call a FITS-reading front end would make):
 * copy x_host, y_host to the device, run iqa_fused_tiles + iqa_aggregate, copy the four
 * per-tile arrays and the aggregated pair back, and SYNCHRONISE the stream before returning.
 *   x_host, y_host        [N*N] host (pinned memory gives full PCIe rate; pageable works)
 *   *_host outputs        [n] each / out2_host [2]; any of them may be NULL (not copied back)
 *   dev_scratch           device buffer of >= iqa_host_scratch_bytes(N, N_T) bytes, 256-B aligned */
int iqa_fused_host(const float* x_host, const float* y_host, int N, int N_T,
                   float C1, float C2, float C, float D,
                   float* lisi_host, float* auglisi_host,
                   float* sum_x_host, float* sum_y_host, float* out2_host,
                   void* dev_scratch, size_t dev_scratch_bytes, void* stream);

/* The same, WITHOUT the final synchronisation: everything (both uploads, the kernels, the downloads) is
 * enqueued on `stream` and the call returns; the host outputs are valid, and x_host / y_host / dev_scratch
 * may be reused, once the caller has synchronised the stream.  With pinned host memory and two streams
 * (two scratch blocks) the upload of the next pair overlaps the kernels, downloads and launch gaps of
 * this one, which keeps the PCIe link busy (binding.HostPipeline; what bench.py times as `e2e`). */
int iqa_fused_host_async(const float* x_host, const float* y_host, int N, int N_T,
                         float C1, float C2, float C, float D,
                         float* lisi_host, float* auglisi_host,
                         float* sum_x_host, float* sum_y_host, float* out2_host,
                         void* dev_scratch, size_t dev_scratch_bytes, void* stream);

/* The host entry points for images of `pixel_type` pixels as a FITS file stores them ("allowing input of FITS
 * images": BITPIX 16 / 8 / 32 / -64, fp16 from a GPU imager).  The raw pixels are uploaded and computed on as they are
 * (the typed kernels of iqa_fused_tiles_2d_typed): a 16-bit plane costs half the PCIe bytes of its fp32 conversion, and
 * the host path is PCIe-bound.  Arguments as iqa_fused_host(_async); x_host, y_host [N*N] of the pixel type;
 * dev_scratch >= iqa_host_scratch_bytes_typed(N, N_T, pixel_type) bytes, 256-B aligned.  Unknown pixel_type: IQA_ERR_SHAPE. */
size_t iqa_host_scratch_bytes_typed(int N, int N_T, int pixel_type);
int iqa_fused_host_typed(const void* x_host, const void* y_host, int pixel_type, int N, int N_T,
                         float C1, float C2, float C, float D,
                         float* lisi_host, float* auglisi_host,
                         float* sum_x_host, float* sum_y_host, float* out2_host,
                         void* dev_scratch, size_t dev_scratch_bytes, void* stream);
int iqa_fused_host_typed_async(const void* x_host, const void* y_host, int pixel_type, int N, int N_T,
                               float C1, float C2, float C, float D,
                               float* lisi_host, float* auglisi_host,
                               float* sum_x_host, float* sum_y_host, float* out2_host,
                               void* dev_scratch, size_t dev_scratch_bytes, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* IQA_TILES_H */
