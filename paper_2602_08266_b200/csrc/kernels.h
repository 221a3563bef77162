// kernels.h -- host-side launchers of the CUDA kernels (internal to libnbv).
#pragma once
#include <atomic>

#include "common.cuh"

namespace nbv {

extern std::atomic<unsigned long long> g_kernel_launches;   // host-side count of kernel launches (nbv_kernel_launches)
int sm_count();                                // multiprocessors of the current device (queried once per device)

// One launch of every S1-S2 stage serves a BATCH of views (grid.y = view): the per-view device pointers travel as a
// __grid_constant__ kernel parameter, like RasterBatch below.  All views of a batch share N and the image size.
constexpr int MAX_BATCH = 16;
struct PreView {
  nbv_camera cam;
  Splat* splat;              // N, indexed by Gaussian
  uint32_t* zkey[2];         // depth keys (z bits; 0xffffffff = culled), ping-pong buffers of the radix passes
  uint32_t* ids[2];          // Gaussian ids, ping-pong; after the sort ids[0][rank]
  ushort4* rect;             // N tile rectangles, indexed by Gaussian
  float* abc;                // N x 3 Sigma2D (parity export) or nullptr
  uint32_t* hist;            // radix digit histograms (256 x radix_blocks(N)) of the current pass
  Splat* splat_sorted;       // N, indexed by depth rank
  ushort4* rect_sorted;
  uint32_t* counts;          // multi-split count table (supertiles x msplit_blocks(N)), scanned in place
  uint32_t* ckeys;           // coarse keys (supertile << rank_bits | rank)
  ushort4* crect;            // their tile rectangles
  uint2* cranges;            // 256 supertile ranges
  ViewCounters* counters;
};
struct PreBatch {
  int n;
  PreView v[MAX_BATCH];
};

// ---- sort.cu
size_t scan_temp_words(size_t n);
void exclusive_scan_u32(const uint32_t* in, uint32_t* out, size_t n, uint32_t* tmp, uint32_t* total_out, cudaStream_t st);
// in-place exclusive scans of one table of n words per view (n <= scan_batched_max(): one cluster launch for the batch)
enum ScanTable { SCAN_HIST = 0, SCAN_COUNTS = 1 };     // PreView::hist, or PreView::counts with the total in counters->n_coarse
uint32_t scan_batched_max();
void scan_batched(const PreBatch& batch, int table, size_t n, cudaStream_t st);
// one stable pass over 8 bits at `shift` of the depth sort of every view of the batch: (zkey, ids)[src] -> [src ^ 1]
void radix_pass_batched(const PreBatch& batch, int src, size_t n, int shift, cudaStream_t st);
uint32_t radix_blocks(size_t n);
size_t radix_temp_words(size_t n);      // words of PreView::hist (the table and the scratch of the long-table scan)

// ---- project.cu
struct SceneDev {            // device arrays of the loaded map
  int N, K;
  const float* mean;         // N x 3
  const float* logscale;     // N x 3
  const float* quat;         // N x 4
  const float* sigma;        // N
  const float* rgb;          // N x 3
  const float* logits;       // N x K
  float* M;                  // N x 9   R(q_hat) diag(s)            (activation output)
  float* pmax;               // N       max_k softmax
  int* amax;                 // N       argmax_k (lowest index on ties)
  float* lse;                // N       log sum exp of the logits
};
void launch_activate(const SceneDev& sc, ViewCounters* counters, cudaStream_t st);
void launch_project(const SceneDev& sc, const nbv_config& cfg, const PreBatch& batch, cudaStream_t st);

// ---- binning.cu
// stable multi-split of the depth ranks into supertile lists: pass 1 (with the gather of the splats into rank order) fills
// the supertile-major count table counts[s * msplit_blocks(N) + block]; after an exclusive scan of that table (total =
// number of coarse entries) pass 2 writes keys (supertile << rank_bits | rank), their tile rects and the supertile ranges
uint32_t msplit_blocks(int N);
void launch_msplit_count(const PreBatch& batch, int N, const TileGrid& tg, cudaStream_t st);
void launch_msplit_write(const PreBatch& batch, int N, const TileGrid& tg, int rank_bits, uint32_t cap, cudaStream_t st);
// parity export of the full tile lists: counts -> scanned offsets (+ total) -> ids
void launch_tile_counts(const uint32_t* ckeys, const ushort4* crect, const uint2* cranges, const TileGrid& tg, int rank_bits,
                        uint32_t* counts, uint32_t* scanned, uint32_t* total, uint32_t* scan_tmp, int64_t* offsets_out, cudaStream_t st);
void launch_tile_ids(const uint32_t* ckeys, const ushort4* crect, const uint2* cranges, const TileGrid& tg, int rank_bits,
                     const uint32_t* ids_sorted, const uint32_t* scanned, int32_t* ids_out, cudaStream_t st);

// ---- raster.cu
struct PixelBuf {            // per-pixel outputs of the forward pass (H x W each)
  float* rgb;                // x3
  float* depth;
  float* T;
  int32_t* ncontrib;
  int32_t* last;             // number of leading entries of the tile's list that can contribute to the pixel (every composited one does)
};
// One launch of S3 / S4 / S5+S6 serves a BATCH of views (S3, S4: launch positions interleave the views; S5+S6: grid.y = view): per-view device pointers travel as a
// __grid_constant__ kernel parameter.  All views of a batch share the image size.
constexpr int TL_CAP = 1024;    // list entries per tile S3 hands to S4 (config 2 walks 138 on average)
struct RasterView {
  const Splat* splat_sorted;
  const uint32_t* ckeys;
  const ushort4* crect;
  const uint2* cranges;
  PixelBuf pix;
  uint32_t* tile_cend;       // per tile: coarse position + 1 of the last entry some pixel of the tile passed
  uint32_t* tile_elast;      // per tile: position + 1 of that entry in the tile's list (0: nothing composited)
  uint32_t* tile_walk;       // per tile: list entries S3 consumed
  uint32_t* tlist;           // per tile TL_CAP ranks: the tile's list as S3 walked it (entry e at tlist[tile * TL_CAP + e]); S4 reads it
                             // backwards instead of filtering the supertile list again (tiles that walked more fall back to the filter)
  double* moments;           // rank r at moments + r * mom_stride (NMOM doubles: the tiles' binary32 sums are added up in binary64), zero on entry to S4 for every Gaussian
  int mom_stride;            // NMOM, or groups * NMOM in a mask context (one group of 4 object channels per S4 launch)
  uint8_t* touched_flag;     // N bytes, zero on entry to S4: S4 sets flag[rank] for every rank it adds moments to (= sum w^2 != 0),
                             // the ordered compaction reads and clears it (32x less traffic than testing moment 39 of every rank)
  uint32_t* touched;         // ranks with a non-zero block (counters->n_touched of them, in increasing rank order)
  uint32_t* touched_cnt;     // scratch of the ordered compaction: touched ranks per block of 256 ranks
  ViewCounters* counters;
};
struct RasterBatch {
  int n;
  uint32_t n_work;              // launch positions (tiles x views) of a raster launch
  uint32_t* work_fwd;           // forward: zeroed work counter of the persistent warps (nullptr: one block per position)
  uint32_t* work;               // backward: zeroed counter the persistent warps pull launch positions from (nullptr: one block per position)
  uint32_t* work_fb;            // the same for the fallback launch of S4 (tiles whose list outgrew TL_CAP)
  uint32_t* overflow;           // number of such tiles in the batch (S3 counts them; zero -> the fallback launch exits at once)
  const uint32_t* tile_order;   // launch position -> tile: tiles by increasing distance from the image centre, so the
                                // long-running central tiles of a look-at view start first and the tail is made of cheap ones
  RasterView v[MAX_BATCH];
};
void launch_forward(const RasterBatch& batch, const TileGrid& tg, int rank_bits, int W, int H, const nbv_config& cfg, bool full_pix,
                    cudaStream_t st);
void launch_backward(const RasterBatch& batch, int N, const TileGrid& tg, int rank_bits, int W, int H, const nbv_config& cfg,
                     cudaStream_t st);
// S3 + S4 of a batch in ONE persistent launch (a warp sweeps its tile forward, then backward from the registers S3 ends with),
// followed by the fallback S4 launch for tiles whose list outgrew TL_CAP; needs batch.work_fwd and the tile lists.  Opt-in
// (NBV_FUSED_RASTER=1): measured slower than the two launches
void launch_raster_fused(const RasterBatch& batch, const TileGrid& tg, int rank_bits, int W, int H, const nbv_config& cfg, cudaStream_t st);

// ---- hessian.cu (colour / depth contexts: everything after S4's binary32 per-tile moment sums is binary64)
// the touched lists (ranks with sum w^2 != 0, in rank order) of every view of the batch
void launch_touched(const RasterBatch& batch, int N, cudaStream_t st);
uint32_t touched_blocks(int N);
enum ExpandMode { EXPAND_TRAIN = 0, EXPAND_VIEW = 1, EXPAND_GAIN = 2, EXPAND_CACHE = 3 };
// EXPAND_TRAIN: H_T[id] += H ; EXPAND_VIEW: out_blocks[id] = H ; EXPAND_GAIN: gain vs H_T, summed into *score (and gains[id] if not null)
// Consumes the touched list of every view of the batch: reads the moments of every touched rank and writes zeros back
// (the moment buffers are all-zero again afterwards).
struct ExpandView {
  nbv_camera cam;
  const uint32_t* ids_sorted;
  const Splat* splat_sorted;
  const uint32_t* touched;
  double* moments;
  float* out_blocks;         // EXPAND_VIEW
  float* score;              // EXPAND_GAIN: written (not accumulated) by the last block of the view
  float* gains;              // EXPAND_GAIN, may be null
  double* partials;          // EXPAND_GAIN: per-block partial scores (expand_partials() doubles)
  ViewCounters* counters;
  // EXPAND_CACHE: the view's touched Gaussians and their unweighted blocks go to pool entries
  // [cache_span[0], cache_span[0] + cache_span[1]) (reserved by cache_reserve_kernel; span[1] = 0 on overflow)
  const uint32_t* cache_span;
};
struct ExpandBatch {
  int n;
  ExpandView v[MAX_BATCH];
};
int expand_partials();       // doubles a slot's `partials` buffer must hold
// trace_total: device scalar S_T of the trace criterion (launch_trace_total), ignored otherwise
void launch_expand(const SceneDev& sc, const nbv_config& cfg, const ExpandBatch& batch, int mode, double* H_T, const float* conf,
                   const double* trace_total, cudaStream_t st);
size_t trace_total_scratch_bytes();
void launch_trace_total(const SceneDev& sc, const nbv_config& cfg, const double* H_T, const float* conf, void* scratch, double* out,
                        cudaStream_t st);
// Sparse per-candidate block cache of greedy selection (nbv_select_greedy): pool of (Gaussian id, 105-double block) entries.
struct BlockCache {
  uint32_t* ids;             // capacity entries
  double* blocks;            // capacity x 105
  uint32_t* spans;           // per candidate: (first entry, number of entries)
  uint32_t* cursor;          // [0] entries reserved so far, [1] overflow flag
  uint32_t capacity;
};
// reserve pool space for the views of a batch (after their touched lists are known); spans_of_view[i] = spans + 2 * candidate
void launch_cache_reserve(const ExpandBatch& batch, const BlockCache& cache, int first_candidate, cudaStream_t st);
void launch_expand_cache(const SceneDev& sc, const nbv_config& cfg, const ExpandBatch& batch, const BlockCache& cache, cudaStream_t st);
// scores[c] = sum over the cached entries of candidate c of the gain against H_T (0 when taken[c] != 0); scratch:
// cached_gain_scratch_bytes(n_cand) bytes, zero on first use
size_t cached_gain_scratch_bytes(int n_cand);
void launch_cached_gain(const BlockCache& cache, const nbv_config& cfg, int n_cand, const int32_t* taken, const float* conf,
                        const double* H_T, float* scores, void* scratch, const double* trace_total, cudaStream_t st);
// H_T[g] += block for the cached entries of candidate *pick
void launch_cache_accumulate(const BlockCache& cache, const int32_t* pick, double* H_T, cudaStream_t st);
void launch_confidence(const SceneDev& sc, const nbv_config& cfg, int target, float* conf, cudaStream_t st);
void launch_export_blocks(const double* src, float* dst, size_t n, cudaStream_t st);
void launch_export_chain(const SceneDev& sc, const nbv_camera& cam, float* out, cudaStream_t st);
void launch_argmax(const float* scores, int n, int32_t* best, cudaStream_t st);

// ---- mask.cu, object-mask output (NEXT-2): groups of four object channels, blocks of L = 11 + K parameters, binary64
void launch_mask_splats(const SceneDev& sc, const Splat* splat_sorted, const uint32_t* ids_sorted, int group, int bgch, Splat* out,
                        cudaStream_t st);
void launch_expand_mask(const SceneDev& sc, const nbv_config& cfg, const ExpandBatch& batch, int mode, int groups, double* H_T,
                        const float* conf, cudaStream_t st);
void launch_mask_scatter(const float* rgb, const float* depth, size_t npx, int K, int group, int bgch, float* mask, cudaStream_t st);

// ---- sh.cu, SH degree 3 colour (NEXT-4): per-view colours in S1, 59 x 59 blocks in S5 / S6 (binary64, one warp per Gaussian)
void launch_sh_colours(const SceneDev& sc, const float* sh45, const PreBatch& batch, cudaStream_t st);
void launch_expand_sh(const SceneDev& sc, const nbv_config& cfg, const ExpandBatch& batch, int mode, const float* sh45, const float* prior59,
                      double* H_T, const float* conf, cudaStream_t st);

// ---- select.cu
// Eq. 10-11 on raw (F x n) and training (F x n_train) gains of F = 2 or 3 outputs: denominators, fused scores, arg-max
void launch_fuse(const float* raw, const float* train, int n, int n_train, int F, float beta_d, float beta_o, float* denom, float* fused,
                 int32_t* best, cudaStream_t st);
// one greedy round: row[remaining[j]] = tmp[j], NaN elsewhere; *pick = arg-max over the remaining candidates
void launch_greedy_round(const float* tmp, const int32_t* remaining, int m, int n, float* row, int32_t* pick, cudaStream_t st);
// device-resident greedy round: row[i] = taken[i] ? NaN : scores[i]; *pick = order_r[0] = arg-max over the free ones; taken[*pick] = 1
void launch_greedy_pick(const float* scores, int32_t* taken, int n, float* row, int32_t* pick, int32_t* order_r, cudaStream_t st);

}  // namespace nbv
