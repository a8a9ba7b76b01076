/*
 * tgs.h -- C ABI of the B200-native TurboGS sparse-pixel rasterisation hot path.
 *
 * The five calls follow the paper's statement of one training iteration's rasterisation
 * (PAPER.md = arxiv/paper_2606_15924 text; SURVEY.md section 8 is the scope table):
 *
 *   tgs_preprocess         EWA projection of 3D Gaussians to 2D splats      PAPER.md:62-64 (Sec. 3.1), 75
 *   tgs_bin_sort           (tile, depth)-ordered Gaussian lists per tile    PAPER.md:64   ("K(p) ... sorted by depth")
 *   tgs_sample             error-guided tile / pixel selection              PAPER.md:73, 93 (Eq. 2), 128-150 (Sec. 3.5), 156
 *   tgs_raster_fwd_sparse  Eq. 1 alpha compositing on sampled pixels only   PAPER.md:66 (Eq. 1), 154-166 (Sec. 3.6, Fig. 6)
 *   tgs_raster_bwd_sparse  its analytic backward + the projection chain     PAPER.md:69, 75, 166, 441 (Alg. 1 step 8)
 *
 * and, widening along SURVEY.md 8f (each to the same parity bar, tests/test_gpu_parity.py):
 *   tgs_loss_sparse          f1  Charbonnier + tile-level sparse NCC + lambda_ncc   PAPER.md:168-208 (Eq. 9-11), 472-481 (Eq. 17-18)
 *   tgs_sample_paper         f2  N_pix pixels in every tile: multinomial w/o         PAPER.md:128-150 (Eq. 7-8)
 *                                replacement on the error map, TopK age, remainder
 *   tgs_maps_update          f2  fp16 EMA error map, uint16 age map                  PAPER.md:97-109 (Eq. 3-4)
 *   tgs_raster_stats_sparse  f3  per-Gaussian E_i, D_i, W_i and expected depth       PAPER.md:212-223 (Eq. 12), Alg. 1 step 11
 *   tgs_lm_solve             f4  moment-damped LM solve (10x10 + 4x4 Cholesky per       PAPER.md:231-239 (Eq. 14), 483-490 (Eq. 19),
 *                                Gaussian), Adam for the higher SH coefficients         Alg. 1 steps 9-10
 *   tgs_fp32_peak                diagnostic: measured FFMA peak (roofline denominator)
 *
 * Conventions (all calls)
 *   - Plain C, no C++/torch types.  Every pointer is a DEVICE pointer unless its name ends in
 *     `_host` (then it is a HOST pointer, pinned or pageable) or it is `const tgs_camera*`
 *     (host struct, copied by value into the launch).  The caller owns every buffer; nothing is
 *     allocated per call and no pointer is retained after the call returns.
 *   - `stream` is a cudaStream_t passed as void*.  Calls only enqueue work; they do not
 *     synchronise, EXCEPT when a non-NULL `*_host` output is given (one cudaStreamSynchronize).
 *     All calls are CUDA-graph capturable when the `_host` outputs are NULL.
 *   - Every call makes the context's device current (cudaSetDevice) before it enqueues work.
 *   - A context owns 32 bytes of device scheduler counters (+ 256 scratch bytes for tgs_fp32_peak) and one side stream (+ two events): the raster calls
 *     fork their warp-per-tile kernel onto it and join before returning to `stream` (also under graph capture).
 *     The raster calls of ONE context must therefore be ordered with respect to each other (same stream, or
 *     stream-ordered by the caller); use one context per concurrently working stream.
 *   - fp32 only, 16x16 tiles only, sh_degree in {0,1,2,3}.  Anything else returns
 *     TGS_ERR_UNSUPPORTED.  There is no CPU fallback.
 *   - Return value: TGS_OK or an error code; tgs_last_error(ctx) holds a message.
 *   - Tile grid: gx = ceil(W/16), gy = ceil(H/16), T = gx*gy, tile_id = ty*gx + tx.
 *   - Pixel (x, y) is sampled at the integer point (x, y); linear pixel index = y*W + x.
 *   - Parameters are ACTIVATED: scales > 0, unit quaternions (w,x,y,z), opacities in (0,1);
 *     gradients are w.r.t. those activated values (exp / sigmoid / normalise belong to the optimiser).
 */
#ifndef TGS_H_
#define TGS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tgs_ctx tgs_ctx;

/* One pinhole view.  R, t map world to camera: t_cam = R * x_world + t (R row-major). */
typedef struct tgs_camera {
    int32_t width, height;
    float fx, fy, cx, cy;
    float R[9];
    float t[3];
    float znear; /* Gaussians with camera-space z <= znear are culled (0.2 in the 3DGS kernels) */
    float bg[3]; /* background colour added as T_final * bg */
} tgs_camera;

enum {
    TGS_OK = 0,
    TGS_ERR_INVALID_ARG = 1, /* NULL required pointer, non-positive size, bad fraction ...       */
    TGS_ERR_CAPACITY = 2,    /* a caller buffer / workspace is too small (message says how much) */
    TGS_ERR_CUDA = 3,        /* a CUDA runtime call or launch failed                             */
    TGS_ERR_UNSUPPORTED = 4  /* sh_degree > 3, T > 2^20, N or P_capacity >= 2^30, ...            */
};

enum { TGS_PIXELS_ALL = 0, TGS_PIXELS_BERNOULLI_ERR = 1 };

/* Projected splat record, 12 x 32-bit words, 48 B, one per Gaussian (float4-aligned):
 *   [0] mean2D.x  [1] mean2D.y  [2] conic A   [3] conic B
 *   [4] conic C   [5] opacity   [6] red       [7] green
 *   [8] blue      [9] depth t_z [10] rect_x = x0 | x1<<16 (uint32 bits)  [11] rect_y = y0 | y1<<16
 * conic = inverse of the dilated 2D covariance [[A,B],[B,C]]; the Gaussian covers tiles
 * x0 <= tx < x1, y0 <= ty < y1; a culled Gaussian has all 12 words zero. */
#define TGS_SPLAT_WORDS 12
/* Gradient record written by the raster half of tgs_raster_bwd_sparse, same stride:
 *   [0..1] dL/dmean2D  [2..4] dL/d(A,B,C)  [5] dL/dopacity  [6..8] dL/drgb  [9..11] unused (0) */

int tgs_create(tgs_ctx** ctx, int device);
int tgs_destroy(tgs_ctx* ctx);
const char* tgs_last_error(const tgs_ctx* ctx);
const char* tgs_version(void);
/* Number of CUDA kernels this library has launched in this process (all contexts); bench.py
 * reports the difference over its timed region as gpu_launches. */
uint64_t tgs_launch_count(void);
/* Measured FP32 peak of the device, the roofline denominator of the ALU-bound raster kernels
 * (SURVEY.md 8d): runs an FFMA-only kernel (8 independent chains per thread, every SM full) `reps`
 * times on `stream`, synchronises, and writes the best rate in TFLOP/s (2 flop per FMA) to
 * *tflops (host pointer).  Diagnostic; not on the hot path. */
int tgs_fp32_peak(tgs_ctx* ctx, int reps, double* tflops, void* stream);

/* ---- a1: projection -------------------------------------------------------
 * in : means3D[N,3] scales[N,3] quats[N,4] opacities[N] sh[N,K,3], K=(sh_degree+1)^2 (coefficient
 *      major, channel minor; sh must be 16-byte aligned).
 * out: splats[N,12] (layout above), radii[N] (int32, ceil(3 sigma_max), 0 = culled),
 *      clamped[N] (bit c set <=> colour channel c was clamped at 0).
 * The rect / depth / mean2D words are computed in a fixed, FMA-free fp32 expression order so that
 * they are bit-reproducible. */
int tgs_preprocess(tgs_ctx* ctx, const tgs_camera* cam, int N, int sh_degree,
                   const float* means3D, const float* scales, const float* quats,
                   const float* opacities, const float* sh,
                   float* splats, int32_t* radii, uint8_t* clamped, void* stream);

/* ---- a2: binning + sort ------------------------------------------------------
 * Produces the list of all (tile, Gaussian) pairs ordered by (tile_id, depth bits, Gaussian id):
 *   gid_sorted[P], tile_offsets[T+1] (CSR: tile t owns [tile_offsets[t], tile_offsets[t+1])),
 *   keys_sorted[P] = tile_id<<32 | float_bits(depth)   (optional, may be NULL).
 * tile_select[T] (nullable; as written by tgs_sample): when given, only pairs whose tile has
 * tile_select[t] != 0 are emitted; every other tile gets an empty range (the method never reads
 * the ranges of tiles it does not sample; R14).  NULL bins every tile.
 * P = number of emitted pairs is data dependent: P_dev[0] = P, P_dev[1] = 1 if P > P_capacity (then
 * the lists are invalid and, if P_host != NULL, the call returns TGS_ERR_CAPACITY).  P_host (host,
 * nullable) receives P and forces one stream synchronisation.
 * The sort is hand written (no library sort / scan): the most significant digit -- the tile id -- is a counting
 * sort (regroup by piece, ballot pair walk, per-tile counts and scan); every tile's segment is then ordered in shared
 * memory in ONE distribution step (monotone interpolation of the depth bits into ~2m buckets, members of a bucket
 * ranked by counting), ties by Gaussian id; a segment whose keys pile up in one bucket (equal depths) falls back to
 * a stable LSD radix sort on (id, depth bits) in global memory.  The result is unique, hence deterministic.
 * workspace: tgs_bin_sort_workspace_bytes (16 B per pair + 16 B per piece record + 12 B per tile), contents
 * undefined on return. */
int tgs_bin_sort_workspace_bytes(int N, int64_t P_capacity, int num_tiles, size_t* bytes);
int tgs_bin_sort(tgs_ctx* ctx, const tgs_camera* cam, int N, const float* splats,
                 const uint32_t* tile_select,
                 int64_t P_capacity, uint64_t* keys_sorted, uint32_t* gid_sorted,
                 uint32_t* tile_offsets, int64_t* P_dev, int64_t* P_host,
                 void* workspace, size_t workspace_bytes, void* stream);

/* ---- a3: error-guided sampling (BASELINE.json configs) --------------
 * Per-pixel error e(p) = err[y*W+x] if err != NULL, else sum_c |render - target| (Eq. 2).
 * Fixed point q = trunc(clamp(e,0,15.999) * 2^20); tile score = (sum q << 8) / #pixels-in-image.
 * Selects k = max(1, floor(pct_num*T/pct_den)) tiles by (score desc, tile_id asc), outputs them
 * ascending in tiles[k]; per selected tile the pixel list (ALL in-image pixels, or
 * BERNOULLI_ERR: keep iff u16(p)*S*den < num*cnt*q16(p)*2^16, at least one pixel per tile), in
 * ascending local index, concatenated in pix[n]; tile_pix_offsets[k+1] is its CSR.
 * Capacities: tile_score[T], tiles[T], tile_pix_offsets[T+1], pix[W*H].  kn_dev[0]=k, kn_dev[1]=n.
 * tile_select[T] (nullable output): 1 for a selected tile, 0 otherwise -- the mask tgs_bin_sort
 * takes to restrict binning to the sampled tiles. */
int tgs_sample_num_tiles(const tgs_camera* cam, int tile_pct_num, int tile_pct_den);
int tgs_sample_workspace_bytes(const tgs_camera* cam, size_t* bytes);
int tgs_sample(tgs_ctx* ctx, const tgs_camera* cam,
               const float* err, const float* render, const float* target,
               int tile_pct_num, int tile_pct_den, int pixel_mode,
               int pix_rate_num, int pix_rate_den, uint64_t seed,
               uint64_t* tile_score, uint32_t* tiles, uint32_t* tile_pix_offsets, uint32_t* pix,
               uint32_t* tile_select, int32_t* kn_dev, int32_t* kn_host,
               void* workspace, size_t workspace_bytes, void* stream);

/* ---- a3 without any allocation: tgs_sample for callers that cannot obtain device memory ------
 * Who this is for.  tgs_sample needs a device workspace, and every other call needs a tgs_ctx, whose creation
 * makes a small cudaMalloc.  Some hosts of this library can do neither: a plug-in whose host application hands it
 * the input and output buffers but forbids it to allocate on the GPU (the host accounts for every byte of HBM
 * itself); a step inside a training or serving loop whose latency budget rules out cudaMalloc, because it
 * synchronises the whole device and stalls every other stream; and a process in which a framework's caching
 * allocator already owns all of HBM, so that a raw cudaMalloc from a library beside it simply fails.  For them:
 *
 * tgs_sample_static computes exactly what tgs_sample computes (same kernels, same bit-exact outputs, same
 * argument meaning) but takes NO context and NO workspace.  Its scratch -- 36 B of keep mask and 4 B of selection
 * flag per tile -- is a fixed array inside the library's device image, sized for
 * TGS_SAMPLE_STATIC_MAX_TILES = 16384 tiles (any image up to 2048 x 2048, e.g. all five BASELINE.json
 * configs): 640 KiB that every GPU which loads libtgs holds until the process exits, whether or not this call is
 * ever made.  The call itself, and everything it calls, uses no cudaMalloc, cudaFree, cudaMallocAsync, stream or
 * event creation, or any library routine that allocates; inputs and outputs are the caller's, as in tgs_sample.
 *
 *   device        the CUDA device the buffers and `stream` live on; made current by the call.
 *   err_msg       (host, nullable) receives a NUL-terminated description when the return value is not TGS_OK;
 *                 err_msg_bytes is its capacity.  There is no context to ask afterwards.
 *   everything else as tgs_sample (kn_host non-NULL forces one stream synchronisation).
 *
 * Limit: an image of more than TGS_SAMPLE_STATIC_MAX_TILES tiles is refused with TGS_ERR_CAPACITY and a message
 * naming both numbers; nothing is launched.  Use tgs_sample with a workspace for such images.
 * First call on a device: looks up the device address of the scratch array (cudaGetSymbolAddress), which can make
 * the CUDA runtime load this library's device code onto that GPU.  Make that first call once per device during
 * start-up, before any stream capture begins and outside any region where an implicit synchronisation hurts;
 * later calls on that device only launch three kernels.
 * Sharing: there is ONE array per GPU and every call on that GPU uses it, from whatever thread or stream.  Calls
 * are safe one after another in the same stream (nothing needs clearing in between: a call overwrites every word
 * it later reads and never reads beyond its own tile count, so a previous call's contents are invisible).  Two
 * calls that may run on the GPU at the same time -- different streams, or different threads without ordering --
 * overwrite each other's masks and give wrong pixel lists: order them with events or use one stream. */
#define TGS_SAMPLE_STATIC_MAX_TILES 16384
int tgs_sample_static(int device, const tgs_camera* cam,
                      const float* err, const float* render, const float* target,
                      int tile_pct_num, int tile_pct_den, int pixel_mode,
                      int pix_rate_num, int pix_rate_den, uint64_t seed,
                      uint64_t* tile_score, uint32_t* tiles, uint32_t* tile_pix_offsets, uint32_t* pix,
                      uint32_t* tile_select, int32_t* kn_dev, int32_t* kn_host,
                      char* err_msg, size_t err_msg_bytes, void* stream);

/* ---- a4: sparse forward (Eq. 1, 154-166) ---------------------------------------
 * For each sampled pixel p of sampled tile tiles[i]: front-to-back over the tile's range,
 *   alpha = min(0.99, o * exp(-1/2 d^T conic d)), skipped if alpha < 1/255, stop before the
 *   Gaussian that would take T below 1e-4;  color = sum c alpha T + T_final * bg.
 * out_color[n,3], out_T[n] (T_final), n_contrib[n] (1-based position in the tile range of the last
 * Gaussian composited, 0 = none); optional work counters (NULL ok): n_walked[n] = range entries
 * visited, n_blended[n] = Gaussians actually composited (alpha >= 1/255 and not terminated).
 * k is the host-known tile count (tgs_sample_num_tiles); n is read from tile_pix_offsets[k]. */
int tgs_raster_fwd_sparse(tgs_ctx* ctx, const tgs_camera* cam, int N, const float* splats,
                          const uint32_t* tile_offsets, const uint32_t* gid_sorted,
                          int k, const uint32_t* tiles, const uint32_t* tile_pix_offsets,
                          const uint32_t* pix,
                          float* out_color, float* out_T, uint32_t* n_contrib, uint32_t* n_walked,
                          uint32_t* n_blended, void* stream);

/* ---- a5 + a6: sparse backward ----------------------------------
 * Raster half: back-to-front replay from n_contrib, accumulating into dL_dsplats[N,12] (zeroed
 * inside the call).  Projection half: chains dL_dsplats through tgs_preprocess to
 * dL_dmeans3D[N,3] dL_dscales[N,3] dL_dquats[N,4] dL_dopacities[N] dL_dsh[N,K,3]; it is skipped when
 * dL_dmeans3D == NULL (then only dL_dsplats is produced).  Derivatives are those of the forward as
 * defined: zero through an active 0.99 alpha clamp, an active colour clamp and for culled Gaussians.
 * quats, sh, dL_dquats, dL_dsh and dL_dsplats must be 16-byte aligned (a view's slice of a [V,N,K,3] buffer is, unless
 * sh_degree is 0 or 2 and N is not a multiple of 4).
 * Pixel order: the pixels of one tile may be listed in any order (in all three raster calls; the lists need not come
 * from tgs_sample).  A 256-pixel tile listed row-major, as tgs_sample writes it, takes a faster accumulation path in the
 * backward; the kernel checks the order per 32-pixel unit and any other order takes the general path, same results.
 * touched[N] (int32, nullable): SPARSE GRADIENTS.  A Gaussian that is not listed in any sampled tile (or whose raster
 * gradient record is all zero) has a zero gradient; with 5 % of the tiles sampled that is ~85 % of them.  NULL: their
 * rows of the five outputs are written as zeros.  Given: touched[i] = 1 and rows written where the record is
 * non-zero, touched[i] = 0 and the rows of i LEFT UNWRITTEN otherwise -- the mask is the `update` argument of
 * tgs_lm_solve (sparse-Adam convention), and the step's cost then follows the sampled-tile fraction
 * instead of N. */
int tgs_raster_bwd_sparse(tgs_ctx* ctx, const tgs_camera* cam, int N, int sh_degree,
                          const float* splats, const uint32_t* tile_offsets, const uint32_t* gid_sorted,
                          int k, const uint32_t* tiles, const uint32_t* tile_pix_offsets,
                          const uint32_t* pix,
                          const float* out_T, const uint32_t* n_contrib, const float* dL_dcolor,
                          const float* means3D, const float* scales, const float* quats,
                          const float* sh, const int32_t* radii, const uint8_t* clamped,
                          float* dL_dsplats,
                          float* dL_dmeans3D, float* dL_dscales, float* dL_dquats,
                          float* dL_dopacities, float* dL_dsh, int32_t* touched, void* stream);

/* ---- f1: sparse supervision (Sec. 3.7 Eq. 9-11, 472-481
 * Eq. 17-18).  Sits between the forward and the backward: from the forward's colours of the n sampled
 * pixels and the target image it writes dL_dcolor[n,3] -- the input of tgs_raster_bwd_sparse --, the
 * per-pixel error pix_err[n] = sum_c |x_c - y_c| (Eq. 2, what the error map is updated with),
 * tile_stats[k,3] = { sum_p l1(p), L_ncc^tau, lambda_tau } and (if loss != NULL) loss[2] =
 * { 1/n sum_p l1(p), 1/n sum_tau lambda_tau m_tau L_ncc^tau }, all device pointers.
 *   l1(p)      = 1/3 sum_c sqrt((x_c - y_c)^2 + eps_l1^2)                       (Charbonnier, Eq. 17 left)
 *   L_ncc^tau  = 1/3 sum_c (1 - cov_xy / sqrt(var_x var_y + eps_ncc))           (Eq. 9; population statistics
 *                over the tile's m sampled pixels, per colour channel)
 *   lambda_tau = clip(gbar_l1 / (gbar_ncc + eps_lambda), 0, 1)                   (Eq. 10 / 18; gbar = mean over the
 *                tile's pixels of the 1-norm of the per-pixel gradient; lambda is a constant for the derivative)
 *   L          = 1/n sum_p [ l1(p) + lambda_tau(p) L_ncc^tau(p) ]                (Eq. 11, pixel weighted), and
 *   dL_dcolor  = 1/n (dl1/dx + lambda_tau dL_ncc-per-pixel/dx)                   (Eq. 17-18) is its exact derivative.
 * color, dL_dcolor, pix_err are indexed like the sampled-pixel list (tile order); target is [H,W,3].
 * k = number of sampled tiles (host value, as in the raster calls); n = tile_pix_offsets[k] is read on the
 * device.  Every tile must list 1 <= m <= 256 pixels (what tgs_sample / tgs_sample_paper produce); a tile with
 * m == 0 is skipped (tile_stats = {0, 0, 0}, no contribution to loss), pixels beyond the 256th are ignored.  Enqueues two kernels, no synchronisation, no workspace. */
int tgs_loss_sparse(tgs_ctx* ctx, const tgs_camera* cam, int k, const uint32_t* tile_pix_offsets,
                    const uint32_t* pix, const float* color, const float* target,
                    float eps_l1, float eps_ncc, float eps_lambda,
                    float* dL_dcolor, float* pix_err, float* tile_stats, float* loss, void* stream);

/* ---- f3: statistics forward (Sec. 3.8 Eq. 12; Alg. 1 step 11
 * "rasterize_forward_pixels") -- the forward walk of tgs_raster_fwd_sparse (same thresholds, same stopping
 * rule) that projects per-pixel quantities back onto the Gaussians: every composited (pixel, Gaussian)
 * pair with weight w = T alpha adds
 *     stats[i][0] (E_i) += pix_err(p) w     stats[i][1] (D_i) += (d^T Sigma'^-1 d) w     stats[i][2] (W_i) += w
 * where pix_err[n] is the per-pixel error in sampled-pixel order (e.g. tgs_loss_sparse's) and
 * d^T Sigma'^-1 d the conic Mahalanobis distance between the splat centre and the pixel.
 * stats[N,4] (16-byte aligned; word 3 unused, 0) is zeroed inside the call and accumulated with fp32
 * atomics (order not deterministic).  out_depth[n] (nullable) = sum_i w z_i, the expected depth of each
 * sampled pixel.  The normalisations e_i = E_i/(W_i+eps), d_i and the score of Eq. 13 belong to the
 * density-control logic above this library. */
int tgs_raster_stats_sparse(tgs_ctx* ctx, const tgs_camera* cam, int N, const float* splats,
                            const uint32_t* tile_offsets, const uint32_t* gid_sorted,
                            int k, const uint32_t* tiles, const uint32_t* tile_pix_offsets,
                            const uint32_t* pix, const float* pix_err,
                            float* stats, float* out_depth, void* stream);

/* ---- f2: the paper's own per-tile sampler (Sec. 3.5 Eq. 7-8) and its
 * persistent maps (Eq. 3-4).  EVERY tile is sampled with N = min(n_pix, #in-image pixels)
 * pixels: min(n_hard, N) "hard" pixels by multinomial sampling WITHOUT replacement from the error prior
 * pi_E (Eq. 7), then min(n_stable, rest) "stable" pixels = TopK of the age map over the remaining pixels
 * (Eq. 8), the remainder (if n_hard + n_stable < n_pix) uniformly without replacement.
 *   E_half[H,W]  error map, IEEE fp16 bit patterns;  age[H,W] uint16.
 *   Integer decisions, identical on any machine: weight q = 1 + trunc(min(E, 15.999) * 2^16) (E <= 0 / NaN: 1);
 *   hard draw d of tile t: r = mix64(seed, t << 16 | d) mod (sum of the remaining q), the pixel whose running
 *   sum of q in ascending local index first exceeds r is taken and removed; TopK ties: lower local index;
 *   remainder draw d: the (mix64(seed ^ 0x5bd1e995a5a5a5a5, t << 16 | d) mod #remaining)-th remaining pixel.
 * Outputs as tgs_sample: tiles[T] = 0..T-1, tile_pix_offsets[T+1], pix[n] (ascending local index inside a
 * tile), kn_dev = {T, n}; kn_host nullable (given: one sync).  workspace: tgs_sample_workspace_bytes. */
int tgs_sample_paper(tgs_ctx* ctx, const tgs_camera* cam, const uint16_t* E_half, const uint16_t* age,
                     int n_pix, int n_hard, int n_stable, uint64_t seed,
                     uint32_t* tiles, uint32_t* tile_pix_offsets, uint32_t* pix,
                     int32_t* kn_dev, int32_t* kn_host, void* workspace, size_t workspace_bytes, void* stream);

/* Eq. 4 then Eq. 3: every age + 1 (saturating at 65535) and the n = kn_dev[1] sampled pixels
 * reset to 0; at the sampled pixels E <- fp16((1 - beta) E + beta pix_err[i]) (three fp32 roundings, then
 * round-to-nearest-even to fp16); every other pixel of E is left unchanged.  Updates both maps in place. */
int tgs_maps_update(tgs_ctx* ctx, const tgs_camera* cam, uint16_t* E_half, uint16_t* age, const int32_t* kn_dev,
                    const uint32_t* pix, const float* pix_err, float beta, void* stream);

/* ---- f4: the moment-damped Levenberg-Marquardt solve (Sec. 3.9 Eq. 14;
 * PAPER.md:483-490 App. A Eq. 19; Alg. 1 steps 9-10).
 * A parameter set in the layouts of tgs_preprocess / tgs_raster_bwd_sparse; five DEVICE pointers in a host struct
 * (copied by value into the launch, not retained). */
typedef struct tgs_params {
    float* means3D;   /* [N,3]   */
    float* scales;    /* [N,3]   */
    float* quats;     /* [N,4]   */
    float* opacities; /* [N]     */
    float* sh;        /* [N,K,3], K = (sh_degree+1)^2; the RGB DC term is sh[:,0,:] */
} tgs_params;

/* Per Gaussian, two blocks solved independently: geometry g = (position 3, scale 3, rotation 4) in
 * R^10 and appearance a = (RGB DC 3, opacity 1) in R^4, each by
 *     (J^T J + diag(sqrt(v) + eps)) Delta = -m                    (Eq. 14 = Eq. 19 left; Cholesky)
 * and every higher SH coefficient by  Delta = -eta_sh m_hat / (sqrt(v_hat) + eps)      (Eq. 19 right).
 *   grads   the V per-view gradients of this iteration, view major: grads->means3D is [V,N,3], ... grads->sh
 *           [V,N,K,3] (V calls of tgs_raster_bwd_sparse writing into slices of one buffer).  Read only.
 *           J ("estimated from the accumulated gradients") is the V x d matrix of the block's per-view
 *           gradients, J^T J = sum_i g_i g_i^T; the accumulated gradient is gbar = sum_i g_i (R31-R32).
 *   m, v    Adam moments in the parameter layouts, updated IN PLACE before the solve:
 *           m <- beta1 m + (1-beta1) gbar, v <- beta2 v + (1-beta2) gbar^2.  Eq. 14 takes them as printed (no bias
 *           correction); Eq. 19 right takes m_hat = m/(1-beta1^t), v_hat = v/(1-beta2^t), t >= 1.
 *   update  [N] int32, nullable: a Gaussian with update == 0 keeps its moments and gets Delta = 0 (it received no
 *           gradient; the sparse-Adam convention of Tab. 5).  NULL updates every Gaussian.
 *   view_touched  [V,N] int32, nullable: the `touched` masks of the V calls of tgs_raster_bwd_sparse (sparse
 *           gradients).  Where view_touched[v][n] == 0 the gradient of view v for Gaussian n is ZERO and its rows of
 *           grads are NOT READ (they were left unwritten); a Gaussian touched in no view is treated like
 *           update[n] == 0.  NULL: every row of grads is read.
 *   delta   nullable: receives Delta in the parameter layouts.
 *   params  nullable: Alg. 1 step 10, params <- params + Delta in place.  At least one of delta / params.
 *           Eq. 14 prints no step size: with small gradients Delta degenerates to -m/(sqrt(v)+eps), an Adam direction
 *           at unit rate, and a few such steps diverge (R37).  Pass `delta` and apply a scaled step yourself
 *           unless you want the step exactly as printed; the Python pipeline does so by default (apply=False).
 *   t       HOST scalar (t >= 1): 1 - beta^t is formed on the host (pow) and travels in the launch arguments, as do
 *           the seeds of tgs_sample / tgs_sample_paper.  A CUDA graph that captured these calls therefore replays with
 *           the t and seeds of the capture; re-capture, or update the kernel-node parameters, when they must change.
 * Arithmetic: fp32 storage.  For the two LM blocks the moment sums, J^T J and the Cholesky factorisation /
 * substitutions run in fp64 registers (the systems mix parameter groups whose gradients differ by orders of
 * magnitude: condition numbers of 1e4-1e8 would otherwise leave 1e-3-level errors in Delta); the Adam branch is
 * fp32 throughout (IEEE sqrt and division).  The system is positive definite for any J because
 * sqrt(v) + eps > 0; eps must be > 0.  NaN inputs give NaN outputs, no trap.
 * Two kernels (geometry arrays; sh + opacity arrays), no workspace, no synchronisation; V <= 64.  All sh pointers
 * 16-byte aligned. */
int tgs_lm_solve(tgs_ctx* ctx, int N, int sh_degree, int V, const tgs_params* grads, const int32_t* update,
                 const int32_t* view_touched, float beta1, float beta2, float eps, float eta_sh, int t,
                 const tgs_params* m, const tgs_params* v, const tgs_params* delta, const tgs_params* params,
                 void* stream);

#ifdef __cplusplus
}
#endif
#endif /* TGS_H_ */
