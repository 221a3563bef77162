/* nbv.h -- C ABI of libnbv: candidate-view scoring for object-aware 3D Gaussian Splatting
 * next-best-view (arxiv/paper_2602_08266), hand-written CUDA for sm_100a (NVIDIA B200).
 *
 * Citations: P:Lnnn = PAPER.md line nnn; R-n = reading n in DESIGN.md section 2.
 *
 * The library scores candidate camera poses by the confidence-weighted, block-diagonal
 * log-det information gain of the paper:
 *     IG(T,c) = f(T u c) - f(T),   f(V) = log det sum_{v in V} J_v^T J_v      (Eq. 5-6)
 *     only each Gaussian's own P x P block is kept
 *     H := J^T C J,  C_g = c_g I,  c_g = max_k(p_gk)^-a_obj sigma_g^-a_opa    (Eq. 7-9)
 *     object-centric: c_g = p_{g,obj}^-a_obj sigma_g^-a_opa if argmax_k p_gk = obj else 0 (Eq. 12)
 * J is the Jacobian of the rendered colour and depth w.r.t. the P = 14 parameters of a Gaussian
 * at SH degree 0, in this order (R-10):
 *     theta = [mu_x mu_y mu_z | logscale_x y z | quat_w x y z (raw, through q/|q|) | opacity logit | r g b]
 * A packed block holds the upper triangle row-major: entry (r,c), r <= c, at r*14 - r*(r-1)/2 + (c-r)
 * (105 floats).
 *
 * Conventions
 *  - Every function returns NBV_OK (0) or a negative nbv_status; nothing throws or aborts.
 *    nbv_last_error() gives a text for the last failure on that context.
 *  - Pointers named d_* are DEVICE pointers owned by the caller (e.g. torch tensors); the library reads or
 *    writes them during the call, on `stream`, and never frees them.  Pointers named h_* are HOST pointers.
 *    Cameras are host structs.  Everything the library allocates belongs to the context and is released
 *    by nbv_destroy().
 *  - `stream` is a cudaStream_t passed as void* (NULL = default stream).  Calls enqueue work on it; calls
 *    that size device buffers from device-side counts synchronise the stream internally (stated per call).
 *  - One context serves one GPU (the current device at nbv_create) and is not thread-safe.
 *  - There is no CPU fallback: without a CUDA device every call fails with NBV_ERR_CUDA.
 */
#ifndef NBV_H_
#define NBV_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define NBV_P 14          /* parameters per Gaussian block */
#define NBV_BLOCK 105     /* packed upper triangle of a 14 x 14 block */
#define NBV_TILE 16       /* tile edge in pixels (B: north_star "16x16 tile") */

#define NBV_CH_RGB 7      /* channel_mask bits: 1 = r, 2 = g, 4 = b, 8 = depth */
#define NBV_CH_DEPTH 8
#define NBV_CH_RGBD 15
#define NBV_CH_MASK 16    /* the object-mask output (Eq. 1-2): a context of its own, blocks of 11 + K parameters */
#define NBV_MASK_KMAX 52  /* largest number of object channels a mask context supports */
#define NBV_SH_L 59       /* parameters per block after nbv_load_sh: 11 + 3 * 16 */
#define NBV_CRIT_LOGDET 0
#define NBV_CRIT_TRACE 1
#define NBV_CRIT_DET 2

typedef enum nbv_status {
  NBV_OK = 0,
  NBV_ERR_INVALID_ARG = -1,      /* null pointer, non-positive size, bad camera (R not orthonormal within 1e-6, fx<=0 ...) */
  NBV_ERR_BAD_DATA = -2,         /* zero / non-finite quaternion, opacity outside (0,1), non-finite parameter */
  NBV_ERR_NOT_LOADED = -3,       /* a call that needs Gaussians before nbv_load_gaussians */
  NBV_ERR_EMPTY_CANDIDATES = -4, /* nbv_score_candidates with n == 0 */
  NBV_ERR_UNKNOWN_TARGET = -5,   /* target_obj >= K or < -1 */
  NBV_ERR_OOM = -6,              /* device allocation failed */
  NBV_ERR_CUDA = -7,             /* any other CUDA runtime error (text in nbv_last_error) */
  NBV_ERR_CAPACITY = -8          /* a caller-provided output buffer is too small (nbv_tile_lists) */
} nbv_status;

/* Pinhole camera, OpenCV axes (+x right, +y down, +z forward); pixel (i,j) is sampled at (i+0.5, j+0.5),
 * origin top-left (R-1).  R_cw is row-major world->camera, p_cam = R_cw p_world + t_cw. */
typedef struct nbv_camera {
  int32_t width, height;
  float fx, fy, cx, cy;
  float R_cw[9];
  float t_cw[3];
} nbv_camera;

/* Context configuration.  nbv_default_config() fills the values the oracle and DESIGN.md use. */
typedef struct nbv_config {
  float near_plane;          /* 0.01   cull z <= near (R-2) */
  float blur;                /* 0.3    px^2 added to the diagonal of Sigma2D (R-3) */
  float alpha_min;           /* 1/255  skip threshold (R-4) */
  float alpha_max;           /* 0.99   alpha cap (R-4) */
  float t_stop;              /* 1e-4   stop before T would fall below (R-4) */
  float bg[3];               /* background colour, default 0 (R-8); depth background is 0 (R-6) */
  int32_t channel_mask;      /* any non-empty subset of NBV_CH_RGBD: outputs whose Jacobians enter H (R-12); or NBV_CH_MASK */
  float channel_weight[4];   /* omega_ch, inverse noise variance per channel, default 1 (R-12) */
  int32_t opacity_coord;     /* 0 = logit (default), 1 = sigma (R-10) */
  float alpha_obj, alpha_opa;/* 0.3, 0.3 exponents of Eq. 7 / Eq. 12 */
  float p_floor, sigma_floor;/* 1e-4 floors inside Eq. 7 (R-14) */
  float prior_precision[14]; /* diagonal of Lambda (R-13), default 1.0 each */
  /* mask contexts (channel_mask == NBV_CH_MASK) only: */
  int32_t mask_bg_channel;   /* 0      object channel that receives the residual 1 - 1^T O' (Eq. 2: the background label) */
  float prior_precision_obj; /* 1.0    diagonal of Lambda on the K object logits */
  /* where the confidence c_g acts (the paper's equation and its prose differ, R-14):
   * 0 (default, R1) Eq. 9 literal, H := J^T C J for every view: IG_g = logdet(c (H_T + H_c) + L) - logdet(c H_T + L)
   * 1 (R2) "weighting each Gaussian's information gain":  IG_g = c [logdet(H_T + H_c + L) - logdet(H_T + L)]
   * 2 (R3) "scale each Jacobian ... during information gain computation", candidate only:
   *        IG_g = logdet(H_T + c H_c + L) - logdet(H_T + L).      c_g = 0 gives exactly 0 in all three. */
  int32_t weight_mode;
  /* the function f of Eq. 5, IG(T,c) = f(T u c) - f(T), on the block-diagonal H (P:L199 names the alternatives; R-17):
   * 0 (default, the paper's choice) f = log det H:  score = sum_g [logdet(c (H_T + H_c) + L) - logdet(c H_T + L)]   (Eq. 6)
   * 1 trace-based, f = 1 / trace(H^-1):  score = 1 / (S_T - D_c) - 1 / S_T with S_T = sum over ALL Gaussians of
   *        trace((c_g H_T,g + L)^-1) and D_c = the reduction of that sum by the candidate (weight_mode 0, colour / depth
   *        contexts only).  nbv_gaussian_gains then exports the per-Gaussian reductions D_g.
   * 2 determinant, f = det H: det(H_T) is a product over all Gaussians and leaves binary64 range for any real map, so
   *        the score is carried in the log domain, log(det(H_{T u c}) / det(H_T)) -- the same numbers as criterion 0,
   *        ordering the candidates exactly as the literal difference does. */
  int32_t criterion;
} nbv_config;

typedef struct nbv_ctx nbv_ctx;

/* Per-view counters of the last view processed (diagnostics and roofline accounting; host readable). */
typedef struct nbv_view_stats {
  int64_t n_visible;      /* Gaussians surviving the culls */
  int64_t n_keys;         /* total length of the tile lists (R-5) = sum of rect areas; the hot path never materialises them */
  int64_t n_entries;      /* (tile, Gaussian) list entries walked by the forward pass before the tile terminated */
  int64_t n_pairs;        /* (pixel, Gaussian) pairs composited = sum of per-pixel contributor counts */
  int64_t n_touched;      /* Gaussians with a non-zero block in this view */
  int64_t n_coarse;       /* (supertile, Gaussian) keys of the coarse binning pass */
} nbv_view_stats;

void nbv_default_config(nbv_config* cfg);

/* Create / destroy a context on the current CUDA device.  cfg == NULL -> defaults.
 * Errors: INVALID_ARG (out == NULL, non-positive thresholds, prior_precision <= 0, empty channel_mask), CUDA. */
int nbv_create(nbv_ctx** out, const nbv_config* cfg);
void nbv_destroy(nbv_ctx* ctx);
const char* nbv_last_error(const nbv_ctx* ctx);

/* Views per batch (1..16; default, chosen per call: 16 -- for images of at least 2,000 tiles only when the two sets of 16 view
 * slots, whose size grows with N x supertiles, fit a sixth of the device memory, else 8; the NBV_CONCURRENCY environment
 * variable overrides the default at nbv_create).  nbv_batch_views() returns the number a call with images of the given size
 * would use (0 on bad arguments).
 * S1-S2 of the views of a batch run concurrently on internal streams (forked from and joined back into the caller's
 * stream with events); S3, S4 and S5+S6 are ONE kernel launch each per batch (S3 and S4: persistent warps pulling
 * (view, tile) positions).  Two sets of work buffers and two internal raster streams alternate between batches.  Views are independent
 * (the arg max is over per-view gains), so this changes no result beyond the order of S4's cross-tile binary64 reductions (exact for realistic footprints)
 * (H_T is accumulated view by view in call order, and a candidate's score is summed in a fixed order).
 * views_in_flight = 0 restores the automatic choice.  Errors: INVALID_ARG outside [0, 16]. */
int nbv_set_concurrency(nbv_ctx* ctx, int32_t views_in_flight);
int32_t nbv_batch_views(const nbv_ctx* ctx, int32_t width, int32_t height);

/* S0 -- load the Gaussian map G with object vectors: device arrays, row-major, float32.
 *   d_mean N x 3, d_logscale N x 3, d_quat N x 4 (w,x,y,z; any non-zero norm), d_opacity N (sigma in (0,1)),
 *   d_rgb N x 3, d_obj_logits N x K.
 * Runs the activation kernel (s = exp l, q/|q|, M = R diag s; softmax statistics of the object logits), copies
 * what later calls need, and resets the training Hessian to zero.  Synchronises `stream` (it reads back the
 * bad-data flag).  Errors: INVALID_ARG (N <= 0, K <= 0, null), BAD_DATA, OOM, CUDA. */
int nbv_load_gaussians(nbv_ctx* ctx, int32_t N, int32_t K, const float* d_mean, const float* d_logscale,
                       const float* d_quat, const float* d_opacity, const float* d_rgb,
                       const float* d_obj_logits, void* stream);

/* View-dependent colour, SH degree 3 ("SH coefficients c in R^{3(d+1)^2}"; R-18):
 *   colour_ch(dir) = rgb_ch + sum_{j=1}^{15} B_j(dir) k_{j,ch},  dir = (mu - o) / |mu - o|, o = camera centre,
 * B_j the real spherical harmonics of degree 1..3 in the ordering and signs of the 3DGS pipeline, no clamp.
 * d_sh: N x 45 floats, coefficient-major (k_1 rgb, k_2 rgb, ..., k_15 rgb), copied.  From this call on the context works on
 * blocks of NBV_SH_L = 59 parameters [mu logscale quat opacity | rgb | k_1 .. k_15] (nbv_block_size() = 1770; the prior of
 * a coefficient is prior_precision[11 + channel]); H_T is reset.  S1 evaluates the colours per view, S3 / S4 are unchanged,
 * S5 / S6 run on 59 x 59 blocks in binary64.  Colour / depth contexts with weight_mode 0 and the log-det criterion only;
 * nbv_select_greedy re-rasterises every round in this mode.  Errors: NOT_LOADED, INVALID_ARG, OOM, CUDA. */
int nbv_load_sh(nbv_ctx* ctx, const float* d_sh, void* stream);

/* H_T <- 0, |T| <- 0. */
int nbv_reset_training(nbv_ctx* ctx, void* stream);

/* H_T += sum over the n cameras of the per-Gaussian J^T J blocks of that view (Eq. 6),
 * unweighted: confidence enters at scoring time, which is Eq. 9 because C_g = c_g I (R-14).
 * Gaussians behind a camera contribute zero.  h_cams: HOST array of n cameras.
 * Errors: NOT_LOADED, INVALID_ARG (n < 0, bad camera), OOM, CUDA. */
int nbv_accumulate_training(nbv_ctx* ctx, const nbv_camera* h_cams, int32_t n, void* stream);

/* Score n candidate cameras (S0', S1-S7):
 *   d_scores[i] = sum_g [ log det(c_g (H_T,g + H_i,g) + Lambda) - log det(c_g H_T,g + Lambda) ]   (Eq. 5, 6, 9)
 *   *d_best     = arg max_i d_scores[i], lowest index on ties (R-15)
 * target_obj = -1 scores the whole scene with Eq. 7; 0 <= target_obj < K restricts the gain to that object's
 * Gaussians with Eq. 12.  Scoring with no training view is allowed (H_T = 0).  d_scores: n floats, d_best: one
 * int32, both DEVICE.  Errors: NOT_LOADED, EMPTY_CANDIDATES (n == 0), UNKNOWN_TARGET, INVALID_ARG, OOM, CUDA. */
int nbv_score_candidates(nbv_ctx* ctx, const nbv_camera* h_cams, int32_t n, int32_t target_obj,
                         float* d_scores, int32_t* d_best, void* stream);

/* Same as nbv_score_candidates but with HOST outputs (copies back and synchronises `stream`). */
int nbv_score_candidates_host(nbv_ctx* ctx, const nbv_camera* h_cams, int32_t n, int32_t target_obj,
                              float* h_scores, int32_t* h_best, void* stream);

/* ---- view selection on top of the per-view gains ------------- */

/* Per-output normalised gains and their fusion (Eq. 10-11) for the outputs RGB, depth and (optionally)
 * object mask:
 *   raw_f[i]   = IG_f(T, c_i)                       the score nbv_score_candidates gives in the context of output f
 *   denom_f    = (1/|T|) sum_t IG_f(T, t)           the training views re-scored as candidates on top of the full H_T
 *   fused[i]   = raw_rgb[i] / denom_rgb + beta_d raw_d[i] / denom_d + beta_o raw_o[i] / denom_o
 *                (beta_d = 10, beta_o = 1 in the paper)
 *   *d_best    = arg max_i fused[i], lowest index on ties
 * ctx_rgb / ctx_depth / ctx_mask: contexts holding the SAME map, created with channel_mask = NBV_CH_RGB, NBV_CH_DEPTH and
 * NBV_CH_MASK (every output has its own Jacobian, hence its own Hessian), each with the n_train cameras of
 * h_train already accumulated.  ctx_mask may be NULL: the mask term is then left out (F = 2 outputs instead of 3).
 * h_train: HOST array of those training cameras (needed again for the denominators).
 * When ctx_rgb and ctx_depth composite with the same constants (near plane, blur, alpha_min, alpha_max, t_stop) every view goes
 * through S1-S3 once, in ctx_rgb's buffers, and is swept twice by S4-S6 (once per output): the maps of the two contexts must then
 * really hold the same values, which the call cannot check beyond N and K.
 * DEVICE outputs: d_fused n floats; d_raw F*n floats (rgb row, depth row[, mask row]; may be NULL); d_denom F floats
 * (may be NULL); d_best one int32.  A zero denominator (no training view sees anything) yields non-finite
 * fused scores, not an error.  Errors: NOT_LOADED, EMPTY_CANDIDATES (n == 0), UNKNOWN_TARGET, INVALID_ARG (null
 * pointers, n_train <= 0, contexts of different N or K, wrong channel masks, bad camera), OOM, CUDA. */
int nbv_score_candidates_fused(nbv_ctx* ctx_rgb, nbv_ctx* ctx_depth, nbv_ctx* ctx_mask, const nbv_camera* h_train,
                               int32_t n_train, const nbv_camera* h_cams, int32_t n, int32_t target_obj, float beta_d,
                               float beta_o, float* d_fused, float* d_raw, float* d_denom, int32_t* d_best, void* stream);

/* Greedy selection of `rounds` views out of n candidates without retraining (Eq. 5 applied repeatedly, P:L185;
 * P:L746 uses 6 rounds): in round r the candidates not yet selected are scored against the current H_T, the arg-max
 * (lowest index on ties) becomes h_order[r], and that view's blocks are added to H_T (Eq. 6).  On return H_T
 * contains the selected views (|T| grows by `rounds`).
 * A view's blocks do not depend on H_T, so every candidate is rasterised once (S1-S5) into a sparse pool of
 * (Gaussian, 14x14 binary64 block) entries; each round then runs only S0', S6 over the pool against the current H_T, the
 * masked arg-max and the addition of the selected view's blocks, all on the device.  The pool is limited to 4 GiB (override:
 * environment variable NBV_GREEDY_CACHE_MB at nbv_create); if the candidates' blocks do not fit, the call falls back to
 * re-rasterising the remaining candidates every round (same results, one host synchronisation per round).
 * HOST output h_order: rounds int32.  DEVICE output d_scores (may be NULL): rounds x n floats, row r = the scores of
 * round r, NaN at candidates selected in earlier rounds.  Synchronises `stream`.
 * Errors: NOT_LOADED, EMPTY_CANDIDATES, UNKNOWN_TARGET, INVALID_ARG (rounds < 1 or > n, null pointers, bad camera),
 * OOM, CUDA. */
int nbv_select_greedy(nbv_ctx* ctx, const nbv_camera* h_cams, int32_t n, int32_t rounds, int32_t target_obj,
                      int32_t* h_order, float* d_scores, void* stream);

/* Number of floats of one packed block in this context: 105 for colour/depth contexts (1770 after nbv_load_sh); L (L + 1) / 2 with L = 11 + K
 * for a loaded mask context (parameter order [mu(3) logscale(3) quat(4) opacity | object logits (K)], upper triangle
 * row-major, idx(r,c) = r L - r (r - 1) / 2 + (c - r)).  nbv_view_hessian / nbv_training_hessian use this size.
 * Returns 0 for a mask context before nbv_load_gaussians. */
int64_t nbv_block_size(const nbv_ctx* ctx);

/* Parity export of a mask context: d_mask H x W x K, the blended object vector O of Eq. 1-2 (sums to 1 per pixel). */
int nbv_render_mask(nbv_ctx* ctx, const nbv_camera* h_cam, float* d_mask, void* stream);

/* Counters of the last view processed by any call (synchronises `stream`). */
int nbv_last_view_stats(nbv_ctx* ctx, nbv_view_stats* h_out, void* stream);

/* ---- measurement ------------------------------------------------------------------------------------ */

/* Stages of one view, in stream order: S1 | depth radix sort | multi-split pass 1 (gather of the
 * splats into depth order + per-supertile counts) | count-table scan + multi-split pass 2 (keys, rects, supertile
 * ranges) | S3 (with the lazy tile-list filter) | S4 | S5 + S6. */
#define NBV_STAGE_PROJECT 0
#define NBV_STAGE_DEPTH_SORT 1
#define NBV_STAGE_BIN 2
#define NBV_STAGE_COARSE_SORT 3
#define NBV_STAGE_FORWARD 4
#define NBV_STAGE_BACKWARD 5
#define NBV_STAGE_EXPAND 6
#define NBV_N_STAGES 7

/* enable != 0: bracket every stage launch (per view for S1-S2, per batch for S3-S6) with CUDA events on the stream it
 * runs on, from now on (a few microseconds per view); clears the accumulated times.  Synchronises `stream`. 
 * Environment: NBV_TRACE_SPANS=<file> makes nbv_stage_times() also append every span it folds to <file>, one line
 * `stage views start_ms end_ms` per span (times relative to the first span since the last fold), blocks ended by `-1 0 0 0`:
 * the timeline of a call across the library's internal streams (profiles/r2_timeline_cfg2.md). */
int nbv_set_stage_timing(nbv_ctx* ctx, int32_t enable, void* stream);

/* h_ms[NBV_N_STAGES] <- milliseconds spent per stage, summed over the *h_views views processed since timing was
 * enabled (h_views may be NULL).  Synchronises `stream`. */
int nbv_stage_times(nbv_ctx* ctx, double* h_ms, int64_t* h_views, void* stream);

/* FFMA-chain microbenchmark on the current device: *h_tflops <- best of six runs of 8 independent fused multiply-add
 * chains per thread, 2 blocks of 1024 threads per SM (2 flop per FMA).  The fp32 CUDA-core peak at the clocks the GPU
 * actually holds; bench.py reports it beside the nominal SMs x 128 lanes x 2 x clock.  Synchronises `stream`. */
int nbv_measure_ffma_peak(double* h_tflops, void* stream);

/* Parity export of the decision path's exponential as the raster kernels evaluate it (exp_spec): the
 * packed routine takes its last step, bits(p) + (k << 23), as p * 2^k with 2^k from MUFU.EX2 -- bit-identical on the whole
 * domain [-80, 80] on hardware whose ex2.approx is exact at integers; tests compare it bit for bit with the oracle's
 * exp_spec so that a device where that does not hold fails loudly.  DEVICE in d_x (n floats), DEVICE out d_y (n floats);
 * elements are processed in pairs (2i, 2i + 1) as the kernels do.  Asynchronous on `stream`.  Errors: INVALID_ARG, CUDA. */
int nbv_exp_spec_pairs(const float* d_x, float* d_y, int64_t n, void* stream);

/* Number of CUDA kernels this library has launched in this process so far (all contexts). */
int64_t nbv_kernel_launches(void);

/* ---- the one call that allocates nothing ------------------------------------------------------------- */

/* Exclusive prefix sum of n 32-bit counts: d_out[i] = d_in[0] + ... + d_in[i-1] (mod 2^32), *d_total = the sum of all n --
 * the scan that turns S2's count tables into list offsets (per-tile list lengths -> the offsets of nbv_tile_lists; DESIGN.md
 * section 5, R-5), for callers that may not allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc.  The context calls keep their scratch in buffers the context allocates on demand; this call keeps the only
 * scratch the scan needs (one block sum per 2,048 elements) in a static device array of 8,192 words = 32 KB inside the library,
 * which every GPU that loads the library holds until the process exits.  It calls no cudaMalloc, cudaFree or allocating library
 * routine: at most three kernel launches on `stream` (for n == 0 one cudaMemsetAsync of the total).  The array's device address
 * is resolved on the first call on each device (cudaGetSymbolAddress, not an allocation); make that first call outside a
 * graph capture.
 *   d_in    DEVICE, n uint32 (read only);   d_out   DEVICE, n uint32, may be d_in (in place);   d_total  DEVICE, 1 uint32, or NULL
 *   n       0 <= n <= NBV_SCAN_NOALLOC_MAX; beyond that NBV_ERR_CAPACITY and nothing is launched
 *   stream  cudaStream_t; asynchronous, never synchronises.  The caller owns all three buffers.
 * EVERY call on a device shares the one array, and the array keeps the previous call's contents (a call overwrites what it
 * reads before reading it, so nothing needs clearing): calls that overlap on the GPU -- different streams without an event
 * between them, or two host threads -- race on it and return garbage; calls in one stream, or ordered by events, are safe.
 * Errors: NBV_ERR_INVALID_ARG (n < 0, null d_in / d_out with n > 0), NBV_ERR_CAPACITY (n too large), NBV_ERR_CUDA; the text of the
 * calling thread's last failure: nbv_noalloc_last_error(). */
#define NBV_SCAN_NOALLOC_MAX 16777216   /* 8,192 blocks x 2,048 elements */
int nbv_exclusive_scan_noalloc(const uint32_t* d_in, uint32_t* d_out, int64_t n, uint32_t* d_total, void* stream);
const char* nbv_noalloc_last_error(void);

/* ---- parity / debug exports (not on the timed path) ------------------------------------------------ */

/* S1 outputs of one view, indexed by Gaussian: d_visible N int32; d_rec N x 9 floats
 * (mx, my, qa, qb, qc, z, a, b, c) with power(d) = qa dx^2 + qb dx dy + qc dy^2 and Sigma2D = [[a,b],[b,c]];
 * d_rect N x 4 int32 (tx0, ty0, tx1, ty1) half-open tile rectangle.  Any output may be NULL. */
int nbv_projected(nbv_ctx* ctx, const nbv_camera* h_cam, int32_t* d_visible, float* d_rec, int32_t* d_rect,
                  void* stream);

/* S2 output of one view, materialised in full (the timed path produces each list lazily inside S3 and only as far as
 * its tile needs; this export applies the same test to the same coarse lists without stopping):
 * d_offsets (tiles+1 int64, tile t = ty*ceil(W/16)+tx lists [offsets[t], offsets[t+1]))
 * and d_ids (Gaussian indices in depth order per tile, capacity `cap` entries).  *h_total receives the number
 * of entries; if it exceeds cap, d_ids is not written and NBV_ERR_CAPACITY is returned.  Synchronises. */
int nbv_tile_lists(nbv_ctx* ctx, const nbv_camera* h_cam, int64_t* d_offsets, int32_t* d_ids, int64_t cap,
                   int64_t* h_total, void* stream);

/* What the hot path actually walked in one view: d_walked (tiles int32) = number of leading entries of each tile's
 * list that S3 consumed before all 256 pixels had terminated (a prefix of the list nbv_tile_lists returns);
 * d_last (H x W int32, may be NULL) = per pixel, 1 + the position in its tile's list of the last Gaussian composited
 * (0 if none).  Invariant: max of d_last over a tile's pixels <= d_walked[tile] <= length of the tile's list. */
int nbv_tile_walk(nbv_ctx* ctx, const nbv_camera* h_cam, int32_t* d_walked, int32_t* d_last, void* stream);

/* S3 output of one view: d_rgb H x W x 3, d_depth H x W, d_T H x W (final transmittance), d_ncontrib H x W int32
 * (number of composited Gaussians per pixel).  Any output may be NULL. */
int nbv_render(nbv_ctx* ctx, const nbv_camera* h_cam, float* d_rgb, float* d_depth, float* d_T,
               int32_t* d_ncontrib, void* stream);

/* S4+S5 output of one view: d_blocks N x 105, overwritten with that view's unweighted blocks. */
int nbv_view_hessian(nbv_ctx* ctx, const nbv_camera* h_cam, float* d_blocks, void* stream);

/* Copy of the accumulated training Hessian H_T (N x 105). */
int nbv_training_hessian(nbv_ctx* ctx, float* d_blocks, void* stream);

/* Chain rule of S5 for one camera, per Gaussian (visible or not): d_chain N x 53 floats = the 5 x 10 matrix
 * d(mx, my, a, b, c) / d(mu(3), logscale(3), quat(4)) row-major (the quaternion columns THROUGH q/|q|, R-10), then dz/dmu (3).
 * The kernel computes it in binary64 from the factor U of Sigma2D = U U^T + blur I (csrc/block_math.cuh); the export
 * exists so that a test can pin it against finite differences of nbv_projected, the library's own forward projection. */
int nbv_chain(nbv_ctx* ctx, const nbv_camera* h_cam, float* d_chain, void* stream);

/* S0' output: confidence c_g (N floats) for the given mode (Eq. 7 or Eq. 12). */
int nbv_confidence(nbv_ctx* ctx, int32_t target_obj, float* d_conf, void* stream);

/* S6 per-Gaussian terms of one candidate: d_gains N floats (zero for Gaussians the view does not touch). */
int nbv_gaussian_gains(nbv_ctx* ctx, const nbv_camera* h_cam, int32_t target_obj, float* d_gains, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* NBV_H_ */
