// nbv_api.cu -- context, per-view pipeline orchestration and the C ABI of include/nbv.h.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <utility>
#include <vector>

#include "kernels.h"

using namespace nbv;

namespace nbv {
std::atomic<unsigned long long> g_kernel_launches{0};

int sm_count() {
  static int cached[64] = {0};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) { cudaGetLastError(); return 148; }
  if (cached[dev] == 0) {
    int n = 0;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) { cudaGetLastError(); n = 148; }
    cached[dev] = n;
  }
  return cached[dev];
}
}  // namespace nbv

namespace {

struct DevBuf {
  void* p = nullptr;
  size_t cap = 0;
  template <class T> T* as() const { return reinterpret_cast<T*>(p); }
};

}  // namespace

// Work buffers of one view in flight.  Views are independent, so several slots run concurrently on their own streams
// (DESIGN.md section 5); the parity exports use slot 0 on the caller's stream.
struct ViewSlot {
  cudaStream_t st = nullptr;
  cudaEvent_t done = nullptr;
  DevBuf splat, zkey, zkey_alt, ids, ids_alt, rect, abc, splat_sorted, rect_sorted, msplit, gsplat;
  DevBuf ckeys, crect, cranges, sort_tmp, scan_tmp, tile_counts;
  DevBuf pix_rgb, pix_depth, pix_T, pix_nc, pix_last, tile_cend, tile_elast, tile_walk, tlist, moments, touched, touched_cnt, partials;
  ViewCounters* d_counters = nullptr;
  ViewCounters* h_counters = nullptr;   // pinned
  // products of the last process_view()
  TileGrid tg = {0, 0, 0, 0, 0};
  int rank_bits = 1;
  uint32_t ccap = 0;                    // capacity of the coarse key buffers
  uint32_t* ckeys_sorted = nullptr;
  bool moments_clean = false;           // the moment buffer is known to be all zero
};

// One timed interval of one stage: events a..b on the stream the stage ran on, covering `views` views.
struct Span {
  cudaEvent_t a, b;
  int stage, views;
};

struct nbv_ctx {
  nbv_config cfg;
  std::string err;
  int device = 0;
  int N = 0, K = 0;
  bool loaded = false;
  // object-mask context (channel_mask == NBV_CH_MASK): groups of four object channels, blocks of LB = L (L + 1) / 2 floats
  bool mask_mode = false;
  bool sh_mode = false;                 // SH degree 3 colour (nbv_load_sh): blocks of 59 parameters, binary64
  int mask_groups = 1;                  // 1 in colour / depth contexts (it is the moment stride in units of NMOM)
  size_t LB = NBLK;
  int n_train = 0;
  // scene
  // H_T: N x LB binary64 (LB = 105, or L (L + 1) / 2 in mask / SH contexts)
  DevBuf mean, logscale, quat, sigma, rgb, logits, M, pmax, amax, lse, H_T, conf, score_tmp, fuse_tmp, cache_ids, cache_blocks, cache_meta,
      cache_scratch, trace_buf, sh45, prior59;         // trace_buf: S_T (1 double) | scratch of launch_trace_total
  size_t greedy_cache_bytes = (size_t)4 << 30;   // budget of the block cache of nbv_select_greedy (NBV_GREEDY_CACHE_MB)
  // views in flight: S1-S2 of each view run on its slot's stream, S3-S6 of a whole batch in one launch per stage on
  // the caller's stream; two sets of `concurrency` slots alternate so the next batch's S1-S2 overlap this batch's S3-S6
  std::vector<ViewSlot*> slots;
  int concurrency = 0;                  // views per batch; 0 = automatic (auto_batch_views)
  bool fused_raster = false;            // NBV_FUSED_RASTER=1: S3 + S4 of a batch in one persistent launch (raster_kernel); measured 3% slower
  size_t dev_mem_total = 0;             // bytes of device memory (cudaMemGetInfo at nbv_create); 0 = unknown
  cudaEvent_t ev_fork = nullptr;
  cudaEvent_t ev_set_done[2] = {nullptr, nullptr};   // S3-S6 of the last batch that used slot set 0 / 1
  cudaStream_t raster_st[2] = {nullptr, nullptr};    // S3-S6 of the batches of slot set 0 / 1 (forked from / joined into the caller's stream)
  ViewSlot* last_slot = nullptr;        // slot of the last view processed (nbv_last_view_stats)
  DevBuf work_counters;                 // 3 x 128 B: work counters of the persistent backward launches
  DevBuf counters_pool;                 // ViewCounters of all 2 x MAX_BATCH slots, consecutive (one memset per batch)
  bool persistent = true;
  DevBuf tile_order;                    // centre-out launch order of the tiles of a tile_order_tx x tile_order_ty grid
  int tile_order_tx = 0, tile_order_ty = 0;
  // optional per-stage timing (nbv_set_stage_timing)
  bool timing = false;
  std::vector<Span> spans;
  size_t spans_used = 0;
  double stage_ms[NBV_N_STAGES] = {0};
  long long timed_views = 0;
};

namespace {

int fail(nbv_ctx* c, int code, const std::string& msg) {
  if (c) c->err = msg;
  return code;
}

int cuda_fail(nbv_ctx* c, cudaError_t e, const char* what) {
  cudaGetLastError();
  return fail(c, e == cudaErrorMemoryAllocation ? NBV_ERR_OOM : NBV_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

#define CK(call)                                                   \
  do {                                                             \
    cudaError_t e__ = (call);                                      \
    if (e__ != cudaSuccess) return cuda_fail(ctx, e__, #call);     \
  } while (0)

#define CKRET(expr)            \
  do {                         \
    int rc__ = (expr);         \
    if (rc__ != NBV_OK) return rc__; \
  } while (0)

int ensure(nbv_ctx* ctx, DevBuf& b, size_t bytes, bool headroom = false) {
  if (bytes <= b.cap && b.p) return NBV_OK;
  if (b.p) {
    cudaFree(b.p);
    b.p = nullptr;
    b.cap = 0;
  }
  size_t want = headroom ? bytes + bytes / 4 : bytes;
  if (want < 256) want = 256;
  cudaError_t e = cudaMalloc(&b.p, want);
  if (e != cudaSuccess && want != bytes) {
    cudaGetLastError();
    want = bytes < 256 ? 256 : bytes;
    e = cudaMalloc(&b.p, want);
  }
  if (e != cudaSuccess) {
    b.p = nullptr;
    return cuda_fail(ctx, e, "cudaMalloc");
  }
  b.cap = want;
  return NBV_OK;
}

void release(DevBuf& b) {
  if (b.p) cudaFree(b.p);
  b.p = nullptr;
  b.cap = 0;
}

int ceil_log2(size_t n) {
  int b = 0;
  while (((size_t)1 << b) < n) ++b;
  return b < 1 ? 1 : b;
}

bool valid_camera(const nbv_camera& c) {
  if (c.width <= 0 || c.height <= 0 || c.width > 65535 * TILE || c.height > 65535 * TILE) return false;
  if (!(c.fx > 0.f) || !(c.fy > 0.f) || !std::isfinite(c.fx) || !std::isfinite(c.fy) || !std::isfinite(c.cx) || !std::isfinite(c.cy))
    return false;
  for (int i = 0; i < 3; ++i) {
    if (!std::isfinite(c.t_cw[i])) return false;
    for (int j = 0; j < 3; ++j) {
      double d = 0;
      for (int k = 0; k < 3; ++k) d += (double)c.R_cw[3 * i + k] * c.R_cw[3 * j + k];
      if (!(std::fabs(d - (i == j ? 1.0 : 0.0)) <= 1e-6)) return false;
    }
  }
  return true;
}

SceneDev scene_dev(const nbv_ctx* c) {
  SceneDev s;
  s.N = c->N; s.K = c->K;
  s.mean = c->mean.as<float>(); s.logscale = c->logscale.as<float>(); s.quat = c->quat.as<float>();
  s.sigma = c->sigma.as<float>(); s.rgb = c->rgb.as<float>(); s.logits = c->logits.as<float>();
  s.M = c->M.as<float>(); s.pmax = c->pmax.as<float>(); s.amax = c->amax.as<int>(); s.lse = c->lse.as<float>();
  return s;
}

constexpr size_t MAX_SPANS = 1 << 20;       // beyond this, further spans are simply not recorded

// fold the recorded spans into ctx->stage_ms (every stream that recorded one must be idle)
void fold_timing(nbv_ctx* ctx) {
  if (const char* path = std::getenv("NBV_TRACE_SPANS")) {     // span timeline of the call(s) since the last fold: stage views start end (ms)
    if (FILE* f = ctx->spans_used ? std::fopen(path, "a") : nullptr) {
      for (size_t i = 0; i < ctx->spans_used; ++i) {
        float t0 = 0.f, t1 = 0.f;
        if (cudaEventElapsedTime(&t0, ctx->spans[0].a, ctx->spans[i].a) == cudaSuccess &&
            cudaEventElapsedTime(&t1, ctx->spans[0].a, ctx->spans[i].b) == cudaSuccess)
          std::fprintf(f, "%d %d %.4f %.4f\n", ctx->spans[i].stage, ctx->spans[i].views, t0, t1);
      }
      std::fprintf(f, "-1 0 0 0\n");
      std::fclose(f);
    }
    cudaGetLastError();
  }
  for (size_t i = 0; i < ctx->spans_used; ++i) {
    const Span& sp = ctx->spans[i];
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, sp.a, sp.b) == cudaSuccess) {
      ctx->stage_ms[sp.stage] += ms;
      if (sp.stage == NBV_STAGE_PROJECT) ctx->timed_views += sp.views;
    }
  }
  cudaGetLastError();
  ctx->spans_used = 0;
}

// open a span of `stage` on stream st; returns its index or -1 when timing is off
int span_begin(nbv_ctx* ctx, int stage, int views, cudaStream_t st) {
  if (!ctx->timing) return -1;
  if (ctx->spans_used >= MAX_SPANS) return -1;   // never recycle: callers may hold open span indices
  if (ctx->spans_used == ctx->spans.size()) {
    Span sp;
    sp.stage = 0; sp.views = 0;
    if (cudaEventCreate(&sp.a) != cudaSuccess || cudaEventCreate(&sp.b) != cudaSuccess) { cudaGetLastError(); return -1; }
    ctx->spans.push_back(sp);
  }
  const size_t i = ctx->spans_used++;
  ctx->spans[i].stage = stage;
  ctx->spans[i].views = views;
  cudaEventRecord(ctx->spans[i].a, st);
  return (int)i;
}

void span_end(nbv_ctx* ctx, int idx, cudaStream_t st) {
  if (idx >= 0) cudaEventRecord(ctx->spans[(size_t)idx].b, st);
}

// close span `idx` and open the next stage's at the same point of the stream
int span_next(nbv_ctx* ctx, int idx, int stage, int views, cudaStream_t st) {
  span_end(ctx, idx, st);
  return span_begin(ctx, stage, views, st);
}

void free_slot(ViewSlot* sl) {
  if (!sl) return;
  DevBuf* all[] = {&sl->splat, &sl->zkey, &sl->zkey_alt, &sl->ids, &sl->ids_alt, &sl->rect, &sl->abc, &sl->splat_sorted,
                   &sl->rect_sorted, &sl->msplit, &sl->gsplat, &sl->ckeys, &sl->crect, &sl->cranges, &sl->sort_tmp,
                   &sl->scan_tmp, &sl->tile_counts, &sl->pix_rgb, &sl->pix_depth, &sl->pix_T, &sl->pix_nc, &sl->pix_last,
                   &sl->tile_cend, &sl->tile_elast, &sl->tile_walk, &sl->tlist, &sl->moments, &sl->touched, &sl->touched_cnt, &sl->partials};
  for (DevBuf* b : all) release(*b);
  if (sl->h_counters) cudaFreeHost(sl->h_counters);
  if (sl->done) cudaEventDestroy(sl->done);
  if (sl->st) cudaStreamDestroy(sl->st);
  delete sl;
}

// slot i, created on first use
int get_slot(nbv_ctx* ctx, int i, ViewSlot** out) {
  while ((int)ctx->slots.size() <= i) {
    ViewSlot* sl = new ViewSlot;
    // Highest stream priority: the work distributor hands out the blocks of a queued kernel only after every earlier
    // kernel of the same priority has dispatched all of its blocks, so without it the ~30 small S1-S2 launches of the next
    // batch would sit behind the 28,800 blocks of the running raster launch instead of slipping in between them.
    int prio_least = 0, prio_greatest = 0;
    cudaDeviceGetStreamPriorityRange(&prio_least, &prio_greatest);
    bool ok = ensure(ctx, ctx->counters_pool, sizeof(ViewCounters) * 2 * MAX_BATCH) == NBV_OK &&
              cudaStreamCreateWithPriority(&sl->st, cudaStreamNonBlocking, prio_greatest) == cudaSuccess &&
              cudaEventCreateWithFlags(&sl->done, cudaEventDisableTiming) == cudaSuccess &&
              cudaMallocHost(&sl->h_counters, sizeof(ViewCounters)) == cudaSuccess;
    if (ok) sl->d_counters = ctx->counters_pool.as<ViewCounters>() + ctx->slots.size();
    if (!ok) {
      cudaGetLastError();
      free_slot(sl);
      return fail(ctx, NBV_ERR_CUDA, "cannot create a view slot (stream, event or counters)");
    }
    std::memset(sl->h_counters, 0, sizeof(ViewCounters));
    cudaMemset(sl->d_counters, 0, sizeof(ViewCounters));
    ctx->slots.push_back(sl);
  }
  *out = ctx->slots[i];
  return NBV_OK;
}

// supertile edge (in tiles, a power of two >= 8) such that the view has at most 256 supertiles
TileGrid make_grid(int W, int H) {
  TileGrid tg;
  tg.tiles_x = (W + TILE - 1) / TILE;
  tg.tiles_y = (H + TILE - 1) / TILE;
  // supertiles of 8 x 8 tiles; 4 x 4 for images of fewer than 2,000 tiles: a tile then scans a list a third as long (S3 -18% at
  // config 1) and the multi-split, which writes 2.4x the entries, is still small.  At 1280 x 720 the trade goes the other way
  // (S3 -13%, multi-split 0.11 -> 0.40 ms per 8-view batch, 1943 -> 1838 views/s at config 2).
  tg.sshift = tg.tiles_x * tg.tiles_y < 2000 ? 2 : 3;
  for (;;) {
    const int S = 1 << tg.sshift;
    tg.super_x = (tg.tiles_x + S - 1) / S;
    tg.super_y = (tg.tiles_y + S - 1) / S;
    if ((long long)tg.super_x * tg.super_y <= 256) break;
    ++tg.sshift;
  }
  return tg;
}

enum Stage { STAGE_PROJECT = 0, STAGE_BIN = 1, STAGE_FORWARD = 2, STAGE_BACKWARD = 3 };

// S1..S2 for a batch of n cameras of equal image size on stream st, in the buffers of slots sl[0..n): ONE launch per stage for
// the whole batch (grid.y = view; 16 launches instead of 16 n).  Leaves, per slot, the depth order in sl->ids, the rank-ordered
// splats and the coarse lists, and makes sure the buffers S3/S4 will need exist (upto).  Never synchronises.
int pre_batch(nbv_ctx* ctx, ViewSlot* const* sl, const nbv_camera* cams, int n, int upto, bool want_abc, bool full_pix, cudaStream_t st) {
  for (int i = 0; i < n; ++i)
    if (!valid_camera(cams[i])) return fail(ctx, NBV_ERR_INVALID_ARG, "invalid camera (size, focal length or non-orthonormal R_cw)");
  const int N = ctx->N;
  const TileGrid tg = make_grid(cams[0].width, cams[0].height);
  const int n_tiles = tg.tiles_x * tg.tiles_y, n_super = tg.super_x * tg.super_y;
  const int rank_bits = ceil_log2((size_t)N), super_bits = ceil_log2((size_t)n_super);
  if (rank_bits + super_bits > 32)
    return fail(ctx, NBV_ERR_INVALID_ARG, "N x supertiles exceeds the 32-bit (supertile | depth rank) key space");
  const unsigned long long worst = (unsigned long long)N * (unsigned long long)n_super;
  if (worst > 0x40000000ull) return fail(ctx, NBV_ERR_CAPACITY, "N x supertiles exceeds the coarse key buffer limit (2^30)");
  const uint32_t ccap = (uint32_t)worst;     // worst case: no overflow is possible, no count has to come back to the host
  const size_t n_counts = (size_t)n_super * msplit_blocks(N);
  const size_t npx = (size_t)cams[0].width * cams[0].height;
  const size_t mom_bytes = 8 * (size_t)NMOM * ctx->mask_groups * N;
  PreBatch pb;
  pb.n = n;
  for (int i = 0; i < n; ++i) {
    ViewSlot* s = sl[i];
    s->tg = tg; s->rank_bits = rank_bits; s->ccap = ccap;
    CKRET(ensure(ctx, s->splat, sizeof(Splat) * (size_t)N));
    CKRET(ensure(ctx, s->zkey, 4 * (size_t)N)); CKRET(ensure(ctx, s->zkey_alt, 4 * (size_t)N));
    CKRET(ensure(ctx, s->ids, 4 * (size_t)N)); CKRET(ensure(ctx, s->ids_alt, 4 * (size_t)N));
    CKRET(ensure(ctx, s->rect, sizeof(ushort4) * (size_t)N));
    if (want_abc) CKRET(ensure(ctx, s->abc, 12 * (size_t)N));
    CKRET(ensure(ctx, s->sort_tmp, 4 * radix_temp_words((size_t)N)));
    CKRET(ensure(ctx, s->scan_tmp, 4 * scan_temp_words(std::max((size_t)N + 1, (size_t)n_tiles + 1))));
    if (upto >= STAGE_BIN) {
      CKRET(ensure(ctx, s->splat_sorted, sizeof(Splat) * (size_t)N));
      CKRET(ensure(ctx, s->rect_sorted, sizeof(ushort4) * (size_t)N));
      CKRET(ensure(ctx, s->msplit, 4 * (n_counts + scan_temp_words(n_counts))));
      CKRET(ensure(ctx, s->ckeys, 4 * (size_t)ccap));
      CKRET(ensure(ctx, s->crect, sizeof(ushort4) * (size_t)ccap));
      CKRET(ensure(ctx, s->cranges, sizeof(uint2) * 256));
    }
    if (upto >= STAGE_FORWARD) {
      CKRET(ensure(ctx, s->pix_T, 4 * npx)); CKRET(ensure(ctx, s->pix_last, 4 * npx));
      CKRET(ensure(ctx, s->tile_cend, 4 * (size_t)n_tiles)); CKRET(ensure(ctx, s->tile_walk, 4 * (size_t)n_tiles));
      CKRET(ensure(ctx, s->tile_elast, 4 * (size_t)n_tiles));
      CKRET(ensure(ctx, s->tlist, 4 * (size_t)n_tiles * TL_CAP));
      if (full_pix) {
        CKRET(ensure(ctx, s->pix_rgb, 12 * npx)); CKRET(ensure(ctx, s->pix_depth, 4 * npx)); CKRET(ensure(ctx, s->pix_nc, 4 * npx));
      }
    }
    if (upto >= STAGE_BACKWARD) {
      if (ctx->mask_mode) CKRET(ensure(ctx, s->gsplat, sizeof(Splat) * (size_t)N));
      // the moments, then one flag byte per rank (kernels.h: touched_flag); both are all-zero between views
      if (s->moments.cap < mom_bytes + (size_t)N || !s->moments.p) s->moments_clean = false;
      CKRET(ensure(ctx, s->moments, mom_bytes + (size_t)N));
      CKRET(ensure(ctx, s->touched, 4 * (size_t)N));
      CKRET(ensure(ctx, s->touched_cnt, 4 * (size_t)touched_blocks(N)));
      CKRET(ensure(ctx, s->partials, 8 * (size_t)expand_partials()));
      if (!s->moments_clean) CK(cudaMemsetAsync(s->moments.p, 0, mom_bytes + (size_t)N, st));
      s->moments_clean = false;     // dirty until an expand kernel has consumed the touched list
    }
    PreView& v = pb.v[i];
    v.cam = cams[i];
    v.splat = s->splat.as<Splat>();
    v.zkey[0] = s->zkey.as<uint32_t>(); v.zkey[1] = s->zkey_alt.as<uint32_t>();
    v.ids[0] = s->ids.as<uint32_t>(); v.ids[1] = s->ids_alt.as<uint32_t>();
    v.rect = s->rect.as<ushort4>();
    v.abc = want_abc ? s->abc.as<float>() : nullptr;
    v.hist = s->sort_tmp.as<uint32_t>();
    v.splat_sorted = s->splat_sorted.as<Splat>(); v.rect_sorted = s->rect_sorted.as<ushort4>();
    v.counts = s->msplit.as<uint32_t>();
    v.ckeys = s->ckeys.as<uint32_t>(); v.crect = s->crect.as<ushort4>(); v.cranges = s->cranges.as<uint2>();
    v.counters = s->d_counters;
    s->ckeys_sorted = s->ckeys.as<uint32_t>();
  }
  ctx->last_slot = sl[n - 1];
  // the counters of the slots of a set are consecutive in one pool: one memset per batch
  bool consecutive = true;
  for (int i = 1; i < n; ++i) consecutive = consecutive && sl[i]->d_counters == sl[0]->d_counters + i;
  if (consecutive) {
    CK(cudaMemsetAsync(sl[0]->d_counters, 0, sizeof(ViewCounters) * (size_t)n, st));
  } else {
    for (int i = 0; i < n; ++i) CK(cudaMemsetAsync(sl[i]->d_counters, 0, sizeof(ViewCounters), st));
  }
  const SceneDev sc = scene_dev(ctx);
  int sp = span_begin(ctx, NBV_STAGE_PROJECT, n, st);
  launch_project(sc, ctx->cfg, pb, st);
  if (ctx->sh_mode) launch_sh_colours(sc, ctx->sh45.as<float>(), pb, st);      // R-18: the colour of this view direction
  CK(cudaGetLastError());
  if (upto == STAGE_PROJECT) { span_end(ctx, sp, st); return NBV_OK; }

  // depth sort: 4 stable passes of 8 bits on the z bits, Gaussian index as value (ties keep index order: R-7)
  sp = span_next(ctx, sp, NBV_STAGE_DEPTH_SORT, n, st);
  for (int pass = 0; pass < 4; ++pass) radix_pass_batched(pb, pass & 1, (size_t)N, 8 * pass, st);
  CK(cudaGetLastError());
  // coarse binning: rank-ordered splats + per-(supertile, rank block) counts | scan | keys, rects and supertile ranges
  sp = span_next(ctx, sp, NBV_STAGE_BIN, n, st);
  launch_msplit_count(pb, N, tg, st);
  sp = span_next(ctx, sp, NBV_STAGE_COARSE_SORT, n, st);
  scan_batched(pb, SCAN_COUNTS, n_counts, st);
  launch_msplit_write(pb, N, tg, rank_bits, ccap, st);
  CK(cudaGetLastError());
  span_end(ctx, sp, st);
  return NBV_OK;
}

// launch order of the tiles: by increasing distance from the image centre (ties by tile index)
int ensure_tile_order(nbv_ctx* ctx, const TileGrid& tg, cudaStream_t st) {
  if (ctx->tile_order.p && ctx->tile_order_tx == tg.tiles_x && ctx->tile_order_ty == tg.tiles_y) return NBV_OK;
  const int n = tg.tiles_x * tg.tiles_y;
  std::vector<uint32_t> order((size_t)n);
  for (int i = 0; i < n; ++i) order[(size_t)i] = (uint32_t)i;
  const double cx = 0.5 * (tg.tiles_x - 1), cy = 0.5 * (tg.tiles_y - 1);
  auto d2 = [&](uint32_t t) { const double dx = (int)(t % tg.tiles_x) - cx, dy = (int)(t / tg.tiles_x) - cy; return dx * dx + dy * dy; };
  std::stable_sort(order.begin(), order.end(), [&](uint32_t a, uint32_t b) { return d2(a) < d2(b); });
  CK(cudaDeviceSynchronize());          // a launch reading the previous table may still be queued (on either raster stream)
  CKRET(ensure(ctx, ctx->tile_order, 4 * (size_t)n));
  CK(cudaMemcpyAsync(ctx->tile_order.p, order.data(), 4 * (size_t)n, cudaMemcpyHostToDevice, st));
  CK(cudaStreamSynchronize(st));        // `order` is a pageable host buffer about to go out of scope
  ctx->tile_order_tx = tg.tiles_x; ctx->tile_order_ty = tg.tiles_y;
  return NBV_OK;
}

// configuration of the S3 / S4 launch of group gr of a mask context: slots (r, g, b | depth) <- object channels
// 4 gr .. 4 gr + 3 in the order "background channel first"; only the very first slot has a background term (Eq. 2)
nbv_config mask_group_config(const nbv_ctx* ctx, int gr) {
  nbv_config g = ctx->cfg;
  g.channel_mask = 0;
  for (int j = 0; j < 4; ++j) {
    if (4 * gr + j < ctx->K) g.channel_mask |= 1 << j;
    g.channel_weight[j] = 1.0f;
  }
  g.bg[0] = gr == 0 ? 1.0f : 0.0f;
  g.bg[1] = g.bg[2] = 0.0f;
  return g;
}

// The launch descriptor of S3 / S4 over the views in sl[0..n).  again: a further S4 pass over the lists the batch's S3 left
// (second output of a fused call): fresh work counters, S3's overflow count kept.
int fill_raster_batch(nbv_ctx* ctx, ViewSlot* const* sl, int n, bool full_pix, bool again, cudaStream_t st, RasterBatch& rb) {
  rb.n = n;
  rb.n_work = 0;
  rb.work = nullptr;
  rb.work_fwd = nullptr;
  rb.work_fb = nullptr;
  rb.overflow = nullptr;
  if (ctx->persistent) {
    // one counter per raster stream (launches on a stream are ordered); the parity exports run on the caller's stream
    const int wi = st == ctx->raster_st[0] ? 0 : st == ctx->raster_st[1] ? 1 : 2;
    rb.work = ctx->work_counters.as<uint32_t>() + 32 * wi;      // [work, work_fb, work_fwd, overflow]
    rb.work_fb = rb.work + 1;
    rb.work_fwd = rb.work + 2;
    rb.overflow = rb.work + 3;
    CK(cudaMemsetAsync(rb.work, 0, again ? 8 : 16, st));
  }
  for (int i = 0; i < n; ++i) {
    ViewSlot* s = sl[i];
    RasterView& v = rb.v[i];
    v.splat_sorted = s->splat_sorted.as<Splat>(); v.ckeys = s->ckeys_sorted; v.crect = s->crect.as<ushort4>();
    v.cranges = s->cranges.as<uint2>();
    v.pix.rgb = full_pix ? s->pix_rgb.as<float>() : nullptr;
    v.pix.depth = full_pix ? s->pix_depth.as<float>() : nullptr;
    v.pix.ncontrib = full_pix ? s->pix_nc.as<int32_t>() : nullptr;
    v.pix.T = s->pix_T.as<float>(); v.pix.last = s->pix_last.as<int32_t>();
    v.tile_cend = s->tile_cend.as<uint32_t>(); v.tile_elast = s->tile_elast.as<uint32_t>(); v.tile_walk = s->tile_walk.as<uint32_t>();
    v.tlist = s->tlist.as<uint32_t>();
    v.moments = s->moments.as<double>(); v.mom_stride = NMOM * ctx->mask_groups; v.touched = s->touched.as<uint32_t>();
    v.touched_flag = reinterpret_cast<uint8_t*>(s->moments.p) + sizeof(double) * NMOM * (size_t)ctx->mask_groups * (size_t)ctx->N;
    v.touched_cnt = s->touched_cnt.as<uint32_t>(); v.counters = s->d_counters;
  }
  CKRET(ensure_tile_order(ctx, sl[0]->tg, st));
  rb.tile_order = ctx->tile_order.as<uint32_t>();
  return NBV_OK;
}

// S3 (+ S4) for a batch of views whose S1-S2 products sit in sl[0..n): ONE launch per stage (S3, S4: persistent warps over (view, tile) positions; S5+S6: grid.y = view).
// All views share the image size (same tile grid).  Stream st must already be ordered after the slots' S1-S2.
int raster_batch(nbv_ctx* ctx, ViewSlot* const* sl, const nbv_camera* cams, int n, int upto, bool full_pix, cudaStream_t st) {
  RasterBatch rb;
  CKRET(fill_raster_batch(ctx, sl, n, full_pix, false, st, rb));
  const TileGrid tg = sl[0]->tg;
  if (ctx->fused_raster && upto == STAGE_BACKWARD && !full_pix && !ctx->mask_mode && rb.work_fwd && rb.v[0].tlist) {
    // opt-in: one launch for S3 + S4 (its time is booked under the backward stage; the forward stage then shows zero)
    const int spf = span_begin(ctx, NBV_STAGE_BACKWARD, n, st);
    launch_raster_fused(rb, tg, sl[0]->rank_bits, cams[0].width, cams[0].height, ctx->cfg, st);
    launch_touched(rb, ctx->N, st);
    CK(cudaGetLastError());
    span_end(ctx, spf, st);
    return NBV_OK;
  }
  int sp = span_begin(ctx, NBV_STAGE_FORWARD, n, st);
  launch_forward(rb, tg, sl[0]->rank_bits, cams[0].width, cams[0].height, ctx->cfg, full_pix, st);
  CK(cudaGetLastError());
  if (upto == STAGE_FORWARD) { span_end(ctx, sp, st); return NBV_OK; }
  sp = span_next(ctx, sp, NBV_STAGE_BACKWARD, n, st);
  if (!ctx->mask_mode) {
    launch_backward(rb, ctx->N, tg, sl[0]->rank_bits, cams[0].width, cams[0].height, ctx->cfg, st);
  } else {
    // one S4 launch per group of four object channels, on a copy of the splats that carries their probabilities
    const SceneDev sc = scene_dev(ctx);
    for (int gr = 0; gr < ctx->mask_groups; ++gr) {
      const nbv_config gcfg = mask_group_config(ctx, gr);
      RasterBatch gb = rb;
      for (int i = 0; i < n; ++i) {
        launch_mask_splats(sc, sl[i]->splat_sorted.as<Splat>(), sl[i]->ids.as<uint32_t>(), gr, ctx->cfg.mask_bg_channel,
                           sl[i]->gsplat.as<Splat>(), st);
        gb.v[i].splat_sorted = sl[i]->gsplat.as<Splat>();
        gb.v[i].moments = sl[i]->moments.as<double>() + (size_t)gr * NMOM;
      }
      if (gr > 0 && gb.work) CK(cudaMemsetAsync(gb.work, 0, 8, st));     // fresh work counters (main + fallback) for every launch
      launch_backward(gb, ctx->N, tg, sl[0]->rank_bits, cams[0].width, cams[0].height, gcfg, st);
    }
  }
  launch_touched(rb, ctx->N, st);            // sum w^2 of (group 0 of) every rank -> ordered touched lists
  CK(cudaGetLastError());
  span_end(ctx, sp, st);
  return NBV_OK;
}

// S4 of another output over the same views (fused scoring, Eq. 10-11): S1-S3 do not depend on the output -- `T`, `last` and the
// tile lists are the ones the batch's S3 left -- so a colour / depth context that shares the map and the compositing constants
// of ctx sweeps them again with its own channels.  The moments and flags are clean again after ctx's own S5+S6.
int backward_again(nbv_ctx* ctx, const nbv_ctx* other, ViewSlot* const* sl, const nbv_camera* cams, int n, cudaStream_t st) {
  RasterBatch rb;
  CKRET(fill_raster_batch(ctx, sl, n, false, true, st, rb));
  const int sp = span_begin(ctx, NBV_STAGE_BACKWARD, n, st);
  launch_backward(rb, ctx->N, sl[0]->tg, sl[0]->rank_bits, cams[0].width, cams[0].height, other->cfg, st);
  launch_touched(rb, ctx->N, st);
  CK(cudaGetLastError());
  span_end(ctx, sp, st);
  return NBV_OK;
}

// S5 (+S6) of the views raster_batch() left in the slots.  out_blocks / gains: single-view exports (n == 1) only.
int expand_batch(nbv_ctx* ctx, ViewSlot* const* sl, const nbv_camera* cams, int n, int mode, float* out_blocks, float* d_scores,
                 float* gains, cudaStream_t st, const BlockCache* cache = nullptr, int first_candidate = 0) {
  ExpandBatch eb;
  eb.n = n;
  for (int i = 0; i < n; ++i) {
    ViewSlot* s = sl[i];
    ExpandView& v = eb.v[i];
    v.cam = cams[i];
    v.ids_sorted = s->ids.as<uint32_t>(); v.splat_sorted = s->splat_sorted.as<Splat>(); v.touched = s->touched.as<uint32_t>();
    v.moments = s->moments.as<double>(); v.out_blocks = out_blocks; v.score = d_scores ? d_scores + i : nullptr; v.gains = gains;
    v.counters = s->d_counters; v.partials = s->partials.as<double>();
    v.cache_span = cache ? cache->spans + 2 * (size_t)(first_candidate + i) : nullptr;
  }
  const int sp = span_begin(ctx, NBV_STAGE_EXPAND, n, st);
  if (mode == EXPAND_CACHE) {
    launch_cache_reserve(eb, *cache, first_candidate, st);
    launch_expand_cache(scene_dev(ctx), ctx->cfg, eb, *cache, st);
  } else if (ctx->mask_mode) {
    launch_expand_mask(scene_dev(ctx), ctx->cfg, eb, mode, ctx->mask_groups, ctx->H_T.as<double>(), ctx->conf.as<float>(), st);
  } else if (ctx->sh_mode) {
    launch_expand_sh(scene_dev(ctx), ctx->cfg, eb, mode, ctx->sh45.as<float>(), ctx->prior59.as<float>(), ctx->H_T.as<double>(),
                     ctx->conf.as<float>(), st);
  } else {
    launch_expand(scene_dev(ctx), ctx->cfg, eb, mode, ctx->H_T.as<double>(), ctx->conf.as<float>(), ctx->trace_buf.as<double>(), st);
  }
  CK(cudaGetLastError());
  span_end(ctx, sp, st);
  for (int i = 0; i < n; ++i) sl[i]->moments_clean = true;
  return NBV_OK;
}

// one view through S1..S4 on the caller's stream in slot 0 (parity exports)
int process_view(nbv_ctx* ctx, ViewSlot* sl, const nbv_camera& cam, int upto, bool want_abc, bool full_pix, cudaStream_t st) {
  CKRET(pre_batch(ctx, &sl, &cam, 1, upto, want_abc, full_pix, st));
  if (upto >= STAGE_FORWARD) CKRET(raster_batch(ctx, &sl, &cam, 1, upto, full_pix, st));
  return NBV_OK;
}

int expand_view(nbv_ctx* ctx, ViewSlot* sl, const nbv_camera& cam, int mode, float* out_blocks, float* score, float* gains,
                cudaStream_t st) {
  return expand_batch(ctx, &sl, &cam, 1, mode, out_blocks, score, gains, st);
}

// Views per batch when the caller has not fixed it.  A batch is one S3 and one S4 launch of persistent warps; between launches the
// SMs drain, and the small launches around them (S1-S2, touched lists, S5+S6) only find room in those drains, so fewer, longer
// batches cost less: 16 views per batch instead of 8 gave +3.6% at config 2 and +3.2% at config 4.  The
// price is memory: two sets of V view slots (worst-case coarse lists, the binary64 moment rows), 9.7 GB at config 2 and 40.6 GB
// at config 4 for V = 16 -- and a fused call keeps up to three contexts alive (at config 4 the mask context alone needs 86 GB
// with V = 8).  So: 16 when the 32 slots fit a sixth of the device memory (config 2: yes, config 4: no), else 8.
int auto_batch_views(const nbv_ctx* ctx, int W, int H) {
  if (ctx->concurrency > 0) return ctx->concurrency;
  const TileGrid tg = make_grid(W, H);
  const size_t n_tiles = (size_t)tg.tiles_x * tg.tiles_y, n_super = (size_t)tg.super_x * tg.super_y, N = (size_t)ctx->N;
  if (n_tiles < 2000) return 16;                 // small images: 16 views are needed to give every resident warp several tiles
  const size_t per_slot = N * (2 * sizeof(Splat) + 2 * sizeof(ushort4) + 6 * 4 + 1 + (ctx->mask_mode ? sizeof(Splat) : 0)) +
                          N * n_super * (4 + sizeof(ushort4)) + 8 * (size_t)NMOM * ctx->mask_groups * N +
                          8 * (size_t)W * H + 4 * n_tiles * TL_CAP;
  return ctx->dev_mem_total && 2 * MAX_BATCH * per_slot <= ctx->dev_mem_total / 6 ? 16 : 8;
}

// Run S1..S6 for n cameras in batches of up to `concurrency` views of equal image size.  S1-S2 of every view run on its slot's
// stream; S3, S4 and S5+S6 of the whole batch are one launch each on the caller's stream.  Two slot sets alternate, so the
// S1-S2 work of batch b+1 overlaps the S3-S6 launches of batch b.  Everything is ordered by events: the call never blocks.
// second / d_scores2 (EXPAND_GAIN only): a second colour / depth context on the same map whose scores are wanted for the same
// views; it reuses S1-S3 of every batch (backward_again) and runs its own S4-S6 after ctx's.
int run_views(nbv_ctx* ctx, const nbv_camera* h_cams, int n, int mode, float* d_scores, cudaStream_t st, const BlockCache* cache = nullptr,
              nbv_ctx* second = nullptr, float* d_scores2 = nullptr) {
  // automatic batch size: 8 views of a 1280 x 720 image are 28,800 (view, tile) positions for the ~2,400 resident S4 warps;
  // smaller images get 16 views per batch so that every warp still draws several positions
  int V = n > 0 ? auto_batch_views(ctx, h_cams[0].width, h_cams[0].height) : 1;
  V = std::max(1, std::min(V, MAX_BATCH));
  int rc = NBV_OK;
  CK(cudaEventRecord(ctx->ev_fork, st));
  for (int s = 0; s < 2; ++s) CK(cudaStreamWaitEvent(ctx->raster_st[s], ctx->ev_fork, 0));
  auto ck = [&](cudaError_t e, const char* what) {       // event plumbing: keep enqueuing (no stream may run ahead), report the first failure
    if (e != cudaSuccess && rc == NBV_OK) rc = cuda_fail(ctx, e, what);
  };
  int batch_no = 0;
  bool set_used[2] = {false, false};
  for (int i0 = 0; i0 < n && rc == NBV_OK; ++batch_no) {
    int nb = 1;
    while (nb < V && i0 + nb < n && h_cams[i0 + nb].width == h_cams[i0].width && h_cams[i0 + nb].height == h_cams[i0].height) ++nb;
    const int set = batch_no & 1;
    // Consecutive batches raster on two different streams: the forward launch of batch b+1 fills the SMs that the
    // draining backward launch of batch b leaves idle (a launch of 28,800 one-warp blocks that each run for hundreds of
    // microseconds has a tail of about one block duration).  Batch b+2 follows batch b in stream order, which is also
    // what the reuse of the slot set requires.
    cudaStream_t rs = ctx->raster_st[set];
    ViewSlot* sl[MAX_BATCH];
    for (int i = 0; i < nb && rc == NBV_OK; ++i) rc = get_slot(ctx, set * MAX_BATCH + i, &sl[i]);
    if (rc != NBV_OK) break;
    {
      // S1-S2 of the whole batch on the high-priority stream of the set's first slot; the set's buffers are free once the
      // S3-S6 launches of the batch that last used this set have finished
      cudaStream_t ps = sl[0]->st;
      ck(cudaStreamWaitEvent(ps, set_used[set] ? ctx->ev_set_done[set] : ctx->ev_fork, 0), "cudaStreamWaitEvent(pre)");
      if (rc == NBV_OK) rc = pre_batch(ctx, sl, h_cams + i0, nb, STAGE_BACKWARD, false, false, ps);
      ck(cudaEventRecord(sl[0]->done, ps), "cudaEventRecord(pre)");
      ck(cudaStreamWaitEvent(rs, sl[0]->done, 0), "cudaStreamWaitEvent(raster)");      // join even after an error: no stream may run ahead
    }
    if (rc == NBV_OK) rc = raster_batch(ctx, sl, h_cams + i0, nb, STAGE_BACKWARD, false, rs);
    // Batches that write shared state in S5 (H_T += in view order, Eq. 6; the block pool of greedy selection) run that
    // step after the previous batch's: the sums and the pool layout do not depend on timing.  S3 / S4 still overlap.
    if ((mode == EXPAND_TRAIN || mode == EXPAND_CACHE) && set_used[set ^ 1])
      ck(cudaStreamWaitEvent(rs, ctx->ev_set_done[set ^ 1], 0), "cudaStreamWaitEvent(order)");
    if (rc == NBV_OK) rc = expand_batch(ctx, sl, h_cams + i0, nb, mode, nullptr, d_scores ? d_scores + i0 : nullptr, nullptr, rs, cache, i0);
    if (second && rc == NBV_OK) rc = backward_again(ctx, second, sl, h_cams + i0, nb, rs);
    if (second && rc == NBV_OK) {
      rc = expand_batch(second, sl, h_cams + i0, nb, mode, nullptr, d_scores2 + i0, nullptr, rs);
      if (rc != NBV_OK) ctx->err = second->err;
    }
    ck(cudaEventRecord(ctx->ev_set_done[set], rs), "cudaEventRecord(set)");
    set_used[set] = true;
    i0 += nb;
  }
  for (int s = 0; s < 2; ++s)
    if (set_used[s]) ck(cudaStreamWaitEvent(st, ctx->ev_set_done[s], 0), "cudaStreamWaitEvent(join)");
  return rc;
}

int prepare_scoring(nbv_ctx* ctx, int target, cudaStream_t st) {
  if (target < -1 || target >= ctx->K) return fail(ctx, NBV_ERR_UNKNOWN_TARGET, "target_obj must be -1 or in [0, K)");
  // S0' runs in every scoring call (Eq. 7 / Eq. 12: N numbers).  Nothing else is needed in any context: S6 factors
  // c_g H_T,g + Lambda itself, for the touched Gaussians only.
  const SceneDev sc = scene_dev(ctx);
  launch_confidence(sc, ctx->cfg, target, ctx->conf.as<float>(), st);
  if (ctx->cfg.criterion == NBV_CRIT_TRACE) {                // S_T of the trace criterion: all N blocks of the current H_T
    if (!ctx->trace_buf.p) {
      CKRET(ensure(ctx, ctx->trace_buf, 16 + trace_total_scratch_bytes()));
      CK(cudaMemsetAsync(ctx->trace_buf.p, 0, 16 + trace_total_scratch_bytes(), st));
    }
    launch_trace_total(sc, ctx->cfg, ctx->H_T.as<double>(), ctx->conf.as<float>(), ctx->trace_buf.as<char>() + 16, ctx->trace_buf.as<double>(), st);
  }
  CK(cudaGetLastError());
  return NBV_OK;
}

__global__ void export_projected_kernel(int N, const Splat* __restrict__ splat, const uint32_t* __restrict__ zkey,
                                        const ushort4* __restrict__ rect, const float* __restrict__ abc,
                                        int32_t* __restrict__ visible, float* __restrict__ rec, int32_t* __restrict__ rect_out) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= N) return;
  const Splat s = splat[g];
  if (visible) visible[g] = zkey[g] != 0xffffffffu;
  if (rec) {
    float* r = rec + 9 * (size_t)g;
    r[0] = s.mx; r[1] = s.my; r[2] = s.qa; r[3] = s.qb; r[4] = s.qc; r[5] = s.z;
    r[6] = abc[3 * (size_t)g]; r[7] = abc[3 * (size_t)g + 1]; r[8] = abc[3 * (size_t)g + 2];
  }
  if (rect_out) {
    const ushort4 q = rect[g];
    int32_t* o = rect_out + 4 * (size_t)g;
    o[0] = q.x; o[1] = q.y; o[2] = q.z; o[3] = q.w;
  }
}

}  // namespace

// =================================================================================================
extern "C" {

void nbv_default_config(nbv_config* cfg) {
  if (!cfg) return;
  std::memset(cfg, 0, sizeof(*cfg));
  cfg->near_plane = 0.01f;
  cfg->blur = 0.3f;
  cfg->alpha_min = 1.0f / 255.0f;
  cfg->alpha_max = 0.99f;
  cfg->t_stop = 1e-4f;
  cfg->channel_mask = NBV_CH_RGB;
  for (int c = 0; c < 4; ++c) cfg->channel_weight[c] = 1.0f;
  cfg->opacity_coord = 0;
  cfg->alpha_obj = 0.3f;
  cfg->alpha_opa = 0.3f;
  cfg->p_floor = 1e-4f;
  cfg->sigma_floor = 1e-4f;
  for (int k = 0; k < NBV_P; ++k) cfg->prior_precision[k] = 1.0f;
  cfg->mask_bg_channel = 0;
  cfg->prior_precision_obj = 1.0f;
  cfg->weight_mode = 0;
  cfg->criterion = NBV_CRIT_LOGDET;
}

int nbv_create(nbv_ctx** out, const nbv_config* cfg) {
  if (!out) return NBV_ERR_INVALID_ARG;
  *out = nullptr;
  nbv_config c;
  if (cfg) c = *cfg; else nbv_default_config(&c);
  const bool ok = c.near_plane > 0.f && c.blur >= 0.f && c.alpha_min >= 1.0f / 255.0f && c.alpha_max > c.alpha_min &&
                  c.alpha_max < 1.f && c.t_stop > 0.f && c.t_stop < 1.f &&
                  (c.channel_mask == NBV_CH_MASK || ((c.channel_mask & 15) != 0 && (c.channel_mask & ~15) == 0)) &&
                  c.mask_bg_channel >= 0 && c.prior_precision_obj > 0.f && std::isfinite(c.prior_precision_obj) &&
                  c.weight_mode >= 0 && c.weight_mode <= 2 && c.criterion >= NBV_CRIT_LOGDET && c.criterion <= NBV_CRIT_DET &&
                  (c.criterion != NBV_CRIT_TRACE || (c.weight_mode == 0 && c.channel_mask != NBV_CH_MASK)) &&
                  (c.opacity_coord == 0 || c.opacity_coord == 1) && c.p_floor > 0.f && c.sigma_floor > 0.f;
  if (!ok) return NBV_ERR_INVALID_ARG;
  for (int k = 0; k < NBV_P; ++k)
    if (!(c.prior_precision[k] > 0.f) || !std::isfinite(c.prior_precision[k])) return NBV_ERR_INVALID_ARG;
  for (int k = 0; k < 4; ++k)
    if (!(c.channel_weight[k] >= 0.f) || !std::isfinite(c.channel_weight[k])) return NBV_ERR_INVALID_ARG;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return NBV_ERR_CUDA; }
  nbv_ctx* ctx = new nbv_ctx;
  ctx->cfg = c;
  ctx->mask_mode = c.channel_mask == NBV_CH_MASK;
  ctx->device = dev;
  ViewSlot* s0 = nullptr;
  if (cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&ctx->ev_set_done[0], cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&ctx->ev_set_done[1], cudaEventDisableTiming) != cudaSuccess ||
      cudaStreamCreateWithFlags(&ctx->raster_st[0], cudaStreamNonBlocking) != cudaSuccess ||
      cudaStreamCreateWithFlags(&ctx->raster_st[1], cudaStreamNonBlocking) != cudaSuccess || get_slot(ctx, 0, &s0) != NBV_OK) {
    cudaGetLastError();
    nbv_destroy(ctx);
    return NBV_ERR_CUDA;
  }
  if (ensure(ctx, ctx->work_counters, 3 * 128) != NBV_OK) { nbv_destroy(ctx); return NBV_ERR_OOM; }
  {
    size_t free_b = 0, total_b = 0;
    if (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess) ctx->dev_mem_total = total_b; else cudaGetLastError();
  }
  if (const char* e = std::getenv("NBV_PERSISTENT")) ctx->persistent = std::atoi(e) != 0;
  if (const char* e = std::getenv("NBV_FUSED_RASTER")) ctx->fused_raster = std::atoi(e) != 0;
  if (const char* e = std::getenv("NBV_GREEDY_CACHE_MB")) ctx->greedy_cache_bytes = (size_t)std::max(0, std::atoi(e)) << 20;
  if (const char* e = std::getenv("NBV_CONCURRENCY")) {
    const int v = std::atoi(e);
    if (v >= 1 && v <= MAX_BATCH) ctx->concurrency = v;
  }
  *out = ctx;
  return NBV_OK;
}

void nbv_destroy(nbv_ctx* ctx) {
  if (!ctx) return;
  cudaDeviceSynchronize();
  DevBuf* all[] = {&ctx->mean, &ctx->logscale, &ctx->quat, &ctx->sigma, &ctx->rgb, &ctx->logits, &ctx->M, &ctx->pmax, &ctx->amax,
                   &ctx->lse, &ctx->H_T, &ctx->conf, &ctx->score_tmp, &ctx->fuse_tmp, &ctx->tile_order, &ctx->work_counters, &ctx->counters_pool, &ctx->cache_ids,
                   &ctx->cache_blocks, &ctx->cache_meta, &ctx->cache_scratch, &ctx->trace_buf, &ctx->sh45, &ctx->prior59};
  for (DevBuf* b : all) release(*b);
  for (ViewSlot* sl : ctx->slots) free_slot(sl);
  if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
  for (cudaEvent_t e : ctx->ev_set_done) if (e) cudaEventDestroy(e);
  for (cudaStream_t r : ctx->raster_st) if (r) cudaStreamDestroy(r);
  for (const Span& sp : ctx->spans) { cudaEventDestroy(sp.a); cudaEventDestroy(sp.b); }
  cudaGetLastError();
  delete ctx;
}

int nbv_set_concurrency(nbv_ctx* ctx, int32_t views_in_flight) {
  if (!ctx) return NBV_ERR_INVALID_ARG;
  if (views_in_flight < 0 || views_in_flight > MAX_BATCH) return fail(ctx, NBV_ERR_INVALID_ARG, "views_in_flight must be in [1, 16], or 0 for the automatic choice");
  ctx->concurrency = views_in_flight;
  return NBV_OK;
}

int32_t nbv_batch_views(const nbv_ctx* ctx, int32_t width, int32_t height) {
  if (!ctx || width <= 0 || height <= 0) return 0;
  return (int32_t)std::max(1, std::min(auto_batch_views(ctx, width, height), MAX_BATCH));
}

const char* nbv_last_error(const nbv_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }

int nbv_load_gaussians(nbv_ctx* ctx, int32_t N, int32_t K, const float* d_mean, const float* d_logscale, const float* d_quat,
                       const float* d_opacity, const float* d_rgb, const float* d_obj_logits, void* stream) {
  if (!ctx) return NBV_ERR_INVALID_ARG;
  if (N <= 0 || K <= 0 || !d_mean || !d_logscale || !d_quat || !d_opacity || !d_rgb || !d_obj_logits)
    return fail(ctx, NBV_ERR_INVALID_ARG, "nbv_load_gaussians: N, K must be positive and all pointers non-null");
  cudaStream_t st = (cudaStream_t)stream;
  ctx->loaded = false;
  if (ctx->mask_mode) {
    if (K > NBV_MASK_KMAX || ctx->cfg.mask_bg_channel >= K)
      return fail(ctx, NBV_ERR_INVALID_ARG, "mask context: K exceeds NBV_MASK_KMAX or mask_bg_channel >= K");
    const size_t L = 11 + (size_t)K;
    ctx->LB = L * (L + 1) / 2;
    ctx->mask_groups = (K + 3) / 4;
  }
  if (!ctx->mask_mode) { ctx->sh_mode = false; ctx->LB = NBLK; }
  ctx->N = N; ctx->K = K;
  const size_t n = (size_t)N;
  CKRET(ensure(ctx, ctx->mean, 12 * n)); CKRET(ensure(ctx, ctx->logscale, 12 * n)); CKRET(ensure(ctx, ctx->quat, 16 * n));
  CKRET(ensure(ctx, ctx->sigma, 4 * n)); CKRET(ensure(ctx, ctx->rgb, 12 * n)); CKRET(ensure(ctx, ctx->logits, 4 * n * K));
  CKRET(ensure(ctx, ctx->M, 36 * n)); CKRET(ensure(ctx, ctx->pmax, 4 * n)); CKRET(ensure(ctx, ctx->amax, 4 * n));
  const size_t ht_bytes = 8 * (size_t)ctx->LB * n;
  CKRET(ensure(ctx, ctx->lse, 4 * n)); CKRET(ensure(ctx, ctx->H_T, ht_bytes)); CKRET(ensure(ctx, ctx->conf, 4 * n));
  CK(cudaMemcpyAsync(ctx->mean.p, d_mean, 12 * n, cudaMemcpyDeviceToDevice, st));
  CK(cudaMemcpyAsync(ctx->logscale.p, d_logscale, 12 * n, cudaMemcpyDeviceToDevice, st));
  CK(cudaMemcpyAsync(ctx->quat.p, d_quat, 16 * n, cudaMemcpyDeviceToDevice, st));
  CK(cudaMemcpyAsync(ctx->sigma.p, d_opacity, 4 * n, cudaMemcpyDeviceToDevice, st));
  CK(cudaMemcpyAsync(ctx->rgb.p, d_rgb, 12 * n, cudaMemcpyDeviceToDevice, st));
  CK(cudaMemcpyAsync(ctx->logits.p, d_obj_logits, 4 * n * K, cudaMemcpyDeviceToDevice, st));
  CK(cudaMemsetAsync(ctx->H_T.p, 0, ht_bytes, st));
  ViewSlot* s0 = ctx->slots[0];
  CK(cudaDeviceSynchronize());             // no view of a previous scene may still be in flight
  CK(cudaMemsetAsync(s0->d_counters, 0, sizeof(ViewCounters), st));
  launch_activate(scene_dev(ctx), s0->d_counters, st);
  CK(cudaGetLastError());
  CK(cudaMemcpyAsync(s0->h_counters, s0->d_counters, sizeof(ViewCounters), cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  for (ViewSlot* sl : ctx->slots) sl->moments_clean = false;
  if (s0->h_counters->bad_data)
    return fail(ctx, NBV_ERR_BAD_DATA, "zero/non-finite quaternion, opacity outside (0,1) or non-finite parameter");
  ctx->n_train = 0;
  ctx->loaded = true;
  return NBV_OK;
}

int nbv_load_sh(nbv_ctx* ctx, const float* d_sh, void* stream) {
  if (!ctx || !d_sh) return NBV_ERR_INVALID_ARG;
  if (!ctx->loaded) return fail(ctx, NBV_ERR_NOT_LOADED, "no Gaussians loaded");
  if (ctx->mask_mode || ctx->cfg.weight_mode != 0 || ctx->cfg.criterion == NBV_CRIT_TRACE)
    return fail(ctx, NBV_ERR_INVALID_ARG, "nbv_load_sh: colour / depth contexts with weight_mode 0 and the log-det criterion only");
  cudaStream_t st = (cudaStream_t)stream;
  const size_t n = (size_t)ctx->N;
  CK(cudaDeviceSynchronize());             // no view may still be in flight on the old block size
  ctx->LB = (size_t)NBV_SH_L * (NBV_SH_L + 1) / 2;
  CKRET(ensure(ctx, ctx->sh45, 4 * 45 * n));
  CKRET(ensure(ctx, ctx->prior59, 4 * NBV_SH_L));
  CKRET(ensure(ctx, ctx->H_T, 8 * ctx->LB * n));
  CK(cudaMemcpyAsync(ctx->sh45.p, d_sh, 4 * 45 * n, cudaMemcpyDeviceToDevice, st));
  float prior[NBV_SH_L];
  for (int k = 0; k < NBV_SH_L; ++k) prior[k] = k < 14 ? ctx->cfg.prior_precision[k] : ctx->cfg.prior_precision[11 + (k - 14) % 3];
  CK(cudaMemcpyAsync(ctx->prior59.p, prior, sizeof(prior), cudaMemcpyHostToDevice, st));
  CK(cudaMemsetAsync(ctx->H_T.p, 0, 8 * ctx->LB * n, st));
  CK(cudaStreamSynchronize(st));           // `prior` is a stack buffer
  ctx->sh_mode = true;
  ctx->n_train = 0;
  return NBV_OK;
}

int nbv_reset_training(nbv_ctx* ctx, void* stream) {
  if (!ctx) return NBV_ERR_INVALID_ARG;
  if (!ctx->loaded) return fail(ctx, NBV_ERR_NOT_LOADED, "no Gaussians loaded");
  CK(cudaMemsetAsync(ctx->H_T.p, 0, 8 * (size_t)ctx->LB * ctx->N, (cudaStream_t)stream));
  ctx->n_train = 0;
  return NBV_OK;
}

int nbv_accumulate_training(nbv_ctx* ctx, const nbv_camera* h_cams, int32_t n, void* stream) {
  if (!ctx) return NBV_ERR_INVALID_ARG;
  if (!ctx->loaded) return fail(ctx, NBV_ERR_NOT_LOADED, "no Gaussians loaded");
  if (n < 0 || (n > 0 && !h_cams)) return fail(ctx, NBV_ERR_INVALID_ARG, "nbv_accumulate_training: bad camera array");
  cudaStream_t st = (cudaStream_t)stream;
  for (int i = 0; i < n; ++i)
    if (!valid_camera(h_cams[i])) return fail(ctx, NBV_ERR_INVALID_ARG, "invalid camera (size, focal length or non-orthonormal R_cw)");
  if (n == 0) return NBV_OK;
  CKRET(run_views(ctx, h_cams, n, EXPAND_TRAIN, nullptr, st));
  ctx->n_train += n;
  return NBV_OK;
}

int nbv_score_candidates(nbv_ctx* ctx, const nbv_camera* h_cams, int32_t n, int32_t target_obj, float* d_scores, int32_t* d_best,
                         void* stream) {
  if (!ctx) return NBV_ERR_INVALID_ARG;
  if (!ctx->loaded) return fail(ctx, NBV_ERR_NOT_LOADED, "no Gaussians loaded");
  if (n == 0) return fail(ctx, NBV_ERR_EMPTY_CANDIDATES, "no candidate cameras");
  if (n < 0 || !h_cams || !d_scores || !d_best) return fail(ctx, NBV_ERR_INVALID_ARG, "nbv_score_candidates: bad arguments");
  if (target_obj < -1 || target_obj >= ctx->K) return fail(ctx, NBV_ERR_UNKNOWN_TARGET, "target_obj must be -1 or in [0, K)");
  cudaStream_t st = (cudaStream_t)stream;
  for (int i = 0; i < n; ++i)
    if (!valid_camera(h_cams[i])) return fail(ctx, NBV_ERR_INVALID_ARG, "invalid camera (size, focal length or non-orthonormal R_cw)");
  CKRET(prepare_scoring(ctx, target_obj, st));
  CK(cudaMemsetAsync(d_scores, 0, 4 * (size_t)n, st));
  CKRET(run_views(ctx, h_cams, n, EXPAND_GAIN, d_scores, st));
  launch_argmax(d_scores, n, d_best, st);
  CK(cudaGetLastError());
  return NBV_OK;
}

int nbv_score_candidates_host(nbv_ctx* ctx, const nbv_camera* h_cams, int32_t n, int32_t target_obj, float* h_scores,
                              int32_t* h_best, void* stream) {
  if (!ctx) return NBV_ERR_INVALID_ARG;
  if (n == 0) return fail(ctx, NBV_ERR_EMPTY_CANDIDATES, "no candidate cameras");
  if (n < 0 || !h_scores || !h_best) return fail(ctx, NBV_ERR_INVALID_ARG, "nbv_score_candidates_host: bad arguments");
  cudaStream_t st = (cudaStream_t)stream;
  CKRET(ensure(ctx, ctx->score_tmp, 4 * (size_t)n + 16));
  float* d_scores = ctx->score_tmp.as<float>();
  int32_t* d_best = reinterpret_cast<int32_t*>(d_scores + n);
  CKRET(nbv_score_candidates(ctx, h_cams, n, target_obj, d_scores, d_best, stream));
  CK(cudaMemcpyAsync(h_scores, d_scores, 4 * (size_t)n, cudaMemcpyDeviceToHost, st));
  CK(cudaMemcpyAsync(h_best, d_best, 4, cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  return NBV_OK;
}

int nbv_score_candidates_fused(nbv_ctx* ctx_rgb, nbv_ctx* ctx_depth, nbv_ctx* ctx_mask, const nbv_camera* h_train, int32_t n_train,
                               const nbv_camera* h_cams, int32_t n, int32_t target_obj, float beta_d, float beta_o, float* d_fused,
                               float* d_raw, float* d_denom, int32_t* d_best, void* stream) {
  nbv_ctx* ctx = ctx_rgb;
  if (!ctx_rgb || !ctx_depth) return NBV_ERR_INVALID_ARG;
  if (!ctx_rgb->loaded || !ctx_depth->loaded || (ctx_mask && !ctx_mask->loaded)) return fail(ctx, NBV_ERR_NOT_LOADED, "no Gaussians loaded");
  if (n == 0) return fail(ctx, NBV_ERR_EMPTY_CANDIDATES, "no candidate cameras");
  if (n < 0 || n_train <= 0 || !h_train || !h_cams || !d_fused || !d_best || !std::isfinite(beta_d) || !std::isfinite(beta_o))
    return fail(ctx, NBV_ERR_INVALID_ARG, "nbv_score_candidates_fused: bad arguments");
  if (ctx_rgb == ctx_depth || ctx_rgb->N != ctx_depth->N || ctx_rgb->K != ctx_depth->K ||
      (ctx_mask && (ctx_mask == ctx_rgb || ctx_mask == ctx_depth || ctx_mask->N != ctx_rgb->N || ctx_mask->K != ctx_rgb->K)))
    return fail(ctx, NBV_ERR_INVALID_ARG, "nbv_score_candidates_fused: the contexts must be distinct and hold the same map");
  if ((ctx_rgb->cfg.channel_mask & ~NBV_CH_RGB) || !(ctx_rgb->cfg.channel_mask & NBV_CH_RGB) || ctx_depth->cfg.channel_mask != NBV_CH_DEPTH ||
      (ctx_mask && !ctx_mask->mask_mode))
    return fail(ctx, NBV_ERR_INVALID_ARG, "nbv_score_candidates_fused: channel masks must be RGB, DEPTH and (optionally) MASK");
  if (target_obj < -1 || target_obj >= ctx->K) return fail(ctx, NBV_ERR_UNKNOWN_TARGET, "target_obj must be -1 or in [0, K)");
  cudaStream_t st = (cudaStream_t)stream;
  const int F = ctx_mask ? 3 : 2;
  // work area in the rgb context: raw (F n) | training gains (F n_train) | denominators (F, padded to 4) | scratch arg-max (1)
  const size_t words = (size_t)F * n + (size_t)F * n_train + 8;
  CKRET(ensure(ctx, ctx->fuse_tmp, 4 * words));
  float* raw = ctx->fuse_tmp.as<float>();
  float* train = raw + (size_t)F * n;
  float* denom = train + (size_t)F * n_train;
  int32_t* scratch = reinterpret_cast<int32_t*>(denom + 4);
  nbv_ctx* cx[3] = {ctx_rgb, ctx_depth, ctx_mask};
  // RGB and depth differ in S4-S6 only: when both contexts composite with the same constants, every view goes through S1-S3 once
  const nbv_config &ca = ctx_rgb->cfg, &cb = ctx_depth->cfg;
  const bool paired = !ctx_rgb->sh_mode && !ctx_depth->sh_mode && !ctx_rgb->mask_mode && !ctx_depth->mask_mode && ca.near_plane == cb.near_plane &&
                      ca.blur == cb.blur && ca.alpha_min == cb.alpha_min && ca.alpha_max == cb.alpha_max && ca.t_stop == cb.t_stop;
  if (paired) {
    for (int i = 0; i < n + n_train; ++i)
      if (!valid_camera(i < n ? h_cams[i] : h_train[i - n]))
        return fail(ctx, NBV_ERR_INVALID_ARG, "invalid camera (size, focal length or non-orthonormal R_cw)");
    CKRET(prepare_scoring(ctx_rgb, target_obj, st));
    const int rcd = prepare_scoring(ctx_depth, target_obj, st);
    if (rcd != NBV_OK) { ctx->err = ctx_depth->err; return rcd; }
    CK(cudaMemsetAsync(raw, 0, 4 * (size_t)2 * n, st));
    CK(cudaMemsetAsync(train, 0, 4 * (size_t)2 * n_train, st));
    CKRET(run_views(ctx_rgb, h_cams, n, EXPAND_GAIN, raw, st, nullptr, ctx_depth, raw + n));
    CKRET(run_views(ctx_rgb, h_train, n_train, EXPAND_GAIN, train, st, nullptr, ctx_depth, train + n_train));
  }
  for (int f = paired ? 2 : 0; f < F; ++f) {
    int rc = nbv_score_candidates(cx[f], h_cams, n, target_obj, raw + (size_t)f * n, scratch, stream);
    if (rc == NBV_OK) rc = nbv_score_candidates(cx[f], h_train, n_train, target_obj, train + (size_t)f * n_train, scratch, stream);
    if (rc != NBV_OK) {
      if (f > 0) ctx->err = cx[f]->err;
      return rc;
    }
  }
  launch_fuse(raw, train, n, n_train, F, beta_d, beta_o, denom, d_fused, d_best, st);
  CK(cudaGetLastError());
  if (d_raw) CK(cudaMemcpyAsync(d_raw, raw, 4 * (size_t)F * n, cudaMemcpyDeviceToDevice, st));
  if (d_denom) CK(cudaMemcpyAsync(d_denom, denom, 4 * (size_t)F, cudaMemcpyDeviceToDevice, st));
  return NBV_OK;
}

// greedy selection by re-rasterising the remaining candidates every round (fallback when the block cache is too small)
static int select_greedy_rescore(nbv_ctx* ctx, const nbv_camera* h_cams, int32_t n, int32_t rounds, int32_t target_obj, int32_t* h_order,
                                 float* d_scores, cudaStream_t st) {
  // work area: scores of the remaining candidates (n) | their original indices (n) | row when d_scores == NULL (n) | pick (1)
  CKRET(ensure(ctx, ctx->fuse_tmp, 4 * (3 * (size_t)n + 4)));
  float* tmp = ctx->fuse_tmp.as<float>();
  int32_t* d_remaining = reinterpret_cast<int32_t*>(tmp + n);
  float* row_tmp = tmp + 2 * (size_t)n;
  int32_t* d_pick = reinterpret_cast<int32_t*>(tmp + 3 * (size_t)n);
  std::vector<nbv_camera> cams;
  std::vector<int32_t> remaining;
  std::vector<char> taken((size_t)n, 0);
  for (int r = 0; r < rounds; ++r) {
    cams.clear(); remaining.clear();
    for (int i = 0; i < n; ++i)
      if (!taken[(size_t)i]) { cams.push_back(h_cams[i]); remaining.push_back(i); }
    const int m = (int)cams.size();
    CKRET(nbv_score_candidates(ctx, cams.data(), m, target_obj, tmp, d_pick, (void*)st));
    CK(cudaMemcpyAsync(d_remaining, remaining.data(), 4 * (size_t)m, cudaMemcpyHostToDevice, st));
    launch_greedy_round(tmp, d_remaining, m, n, d_scores ? d_scores + (size_t)r * n : row_tmp, d_pick, st);
    CK(cudaGetLastError());
    int32_t pick = -1;
    CK(cudaMemcpyAsync(&pick, d_pick, 4, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));          // also covers the pageable `remaining` copy above
    if (pick < 0 || pick >= n || taken[(size_t)pick]) return fail(ctx, NBV_ERR_CUDA, "nbv_select_greedy: inconsistent arg-max");
    taken[(size_t)pick] = 1;
    h_order[r] = pick;
    CKRET(nbv_accumulate_training(ctx, h_cams + pick, 1, (void*)st));    // Eq. 6: H_T += H(c*)
  }
  return NBV_OK;
}

int nbv_select_greedy(nbv_ctx* ctx, const nbv_camera* h_cams, int32_t n, int32_t rounds, int32_t target_obj, int32_t* h_order,
                      float* d_scores, void* stream) {
  if (!ctx) return NBV_ERR_INVALID_ARG;
  if (!ctx->loaded) return fail(ctx, NBV_ERR_NOT_LOADED, "no Gaussians loaded");
  if (n == 0) return fail(ctx, NBV_ERR_EMPTY_CANDIDATES, "no candidate cameras");
  if (n < 0 || !h_cams || !h_order || rounds < 1 || rounds > n) return fail(ctx, NBV_ERR_INVALID_ARG, "nbv_select_greedy: bad arguments");
  if (target_obj < -1 || target_obj >= ctx->K) return fail(ctx, NBV_ERR_UNKNOWN_TARGET, "target_obj must be -1 or in [0, K)");
  for (int i = 0; i < n; ++i)
    if (!valid_camera(h_cams[i])) return fail(ctx, NBV_ERR_INVALID_ARG, "invalid camera (size, focal length or non-orthonormal R_cw)");
  cudaStream_t st = (cudaStream_t)stream;
  // A view's blocks do not depend on H_T, so every candidate is rasterised ONCE: S1-S5 leave its touched Gaussians and
  // their unweighted 14x14 blocks in a sparse pool; every round then needs only S0' (new factors), S6 over the pool,
  // the masked arg-max and H_T += (blocks of the selected view) -- all on the device, no camera and no host round trip.
  const size_t entry_bytes = 8 * (size_t)NBLK + 4;
  const size_t want = std::min((size_t)n * (size_t)ctx->N, ctx->greedy_cache_bytes / entry_bytes);
  if (want == 0 || want > 0xfffffff0ull || ctx->mask_mode || ctx->sh_mode) return select_greedy_rescore(ctx, h_cams, n, rounds, target_obj, h_order, d_scores, st);
  CKRET(ensure(ctx, ctx->cache_ids, 4 * want));
  CKRET(ensure(ctx, ctx->cache_blocks, 8 * (size_t)NBLK * want));
  CKRET(ensure(ctx, ctx->cache_scratch, cached_gain_scratch_bytes(n)));
  CK(cudaMemsetAsync(ctx->cache_scratch.p, 0, cached_gain_scratch_bytes(n), st));
  // meta: spans (2n) | cursor + overflow flag (2) | taken (n) | scores (n) | pick (1) | order (rounds)
  CKRET(ensure(ctx, ctx->cache_meta, 4 * (4 * (size_t)n + 4 + (size_t)rounds)));
  BlockCache bc;
  bc.ids = ctx->cache_ids.as<uint32_t>(); bc.blocks = ctx->cache_blocks.as<double>();
  bc.spans = ctx->cache_meta.as<uint32_t>(); bc.cursor = bc.spans + 2 * (size_t)n; bc.capacity = (uint32_t)want;
  int32_t* d_taken = reinterpret_cast<int32_t*>(bc.cursor + 2);
  float* d_round = reinterpret_cast<float*>(d_taken + n);
  int32_t* d_pick = reinterpret_cast<int32_t*>(d_round + n);
  int32_t* d_order = d_pick + 1;
  CK(cudaMemsetAsync(ctx->cache_meta.p, 0, 4 * (4 * (size_t)n + 4 + (size_t)rounds), st));
  CKRET(run_views(ctx, h_cams, n, EXPAND_CACHE, nullptr, st, &bc));
  uint32_t h_cursor[2] = {0, 0};
  CK(cudaMemcpyAsync(h_cursor, bc.cursor, 8, cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  if (h_cursor[1]) return select_greedy_rescore(ctx, h_cams, n, rounds, target_obj, h_order, d_scores, st);   // pool too small
  for (int r = 0; r < rounds; ++r) {
    CKRET(prepare_scoring(ctx, target_obj, st));
    launch_cached_gain(bc, ctx->cfg, n, d_taken, ctx->conf.as<float>(), ctx->H_T.as<double>(), d_round, ctx->cache_scratch.p,
                       ctx->trace_buf.as<double>(), st);
    launch_greedy_pick(d_round, d_taken, n, d_scores ? d_scores + (size_t)r * n : nullptr, d_pick, d_order + r, st);
    launch_cache_accumulate(bc, d_pick, ctx->H_T.as<double>(), st);      // Eq. 6: H_T += H(c*)
    CK(cudaGetLastError());
    ++ctx->n_train;
  }
  CK(cudaMemcpyAsync(h_order, d_order, 4 * (size_t)rounds, cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  return NBV_OK;
}

int nbv_last_view_stats(nbv_ctx* ctx, nbv_view_stats* h_out, void* stream) {
  if (!ctx || !h_out) return NBV_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  ViewSlot* sl = ctx->last_slot ? ctx->last_slot : ctx->slots[0];
  CK(cudaStreamSynchronize(st));           // joins the slot streams of the last call
  CK(cudaMemcpyAsync(sl->h_counters, sl->d_counters, sizeof(ViewCounters), cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  h_out->n_visible = sl->h_counters->n_visible;
  h_out->n_keys = (int64_t)sl->h_counters->n_keys;
  h_out->n_entries = (int64_t)sl->h_counters->n_entries;
  h_out->n_pairs = (int64_t)sl->h_counters->n_pairs;
  h_out->n_touched = sl->h_counters->n_touched;
  h_out->n_coarse = sl->h_counters->n_coarse;
  return NBV_OK;
}

int nbv_set_stage_timing(nbv_ctx* ctx, int32_t enable, void* stream) {
  if (!ctx) return NBV_ERR_INVALID_ARG;
  CK(cudaStreamSynchronize((cudaStream_t)stream));
  ctx->spans_used = 0;
  for (int s = 0; s < NBV_N_STAGES; ++s) ctx->stage_ms[s] = 0.0;
  ctx->timed_views = 0;
  ctx->timing = enable != 0;
  return NBV_OK;
}

int nbv_stage_times(nbv_ctx* ctx, double* h_ms, int64_t* h_views, void* stream) {
  if (!ctx || !h_ms) return NBV_ERR_INVALID_ARG;
  CK(cudaStreamSynchronize((cudaStream_t)stream));     // the slot streams are joined into the caller's stream
  for (ViewSlot* sl : ctx->slots) CK(cudaStreamSynchronize(sl->st));
  fold_timing(ctx);
  for (int s = 0; s < NBV_N_STAGES; ++s) h_ms[s] = ctx->stage_ms[s];
  if (h_views) *h_views = ctx->timed_views;
  return NBV_OK;
}

int64_t nbv_kernel_launches(void) { return (int64_t)nbv::g_kernel_launches.load(); }

int nbv_projected(nbv_ctx* ctx, const nbv_camera* h_cam, int32_t* d_visible, float* d_rec, int32_t* d_rect, void* stream) {
  if (!ctx || !h_cam) return NBV_ERR_INVALID_ARG;
  if (!ctx->loaded) return fail(ctx, NBV_ERR_NOT_LOADED, "no Gaussians loaded");
  cudaStream_t st = (cudaStream_t)stream;
  ViewSlot* sl = ctx->slots[0];
  CKRET(process_view(ctx, sl, *h_cam, STAGE_PROJECT, true, false, st));
  ++g_kernel_launches;
  export_projected_kernel<<<(ctx->N + 255) / 256, 256, 0, st>>>(ctx->N, sl->splat.as<Splat>(), sl->zkey.as<uint32_t>(),
                                                                sl->rect.as<ushort4>(), sl->abc.as<float>(), d_visible, d_rec, d_rect);
  CK(cudaGetLastError());
  return NBV_OK;
}

int nbv_tile_lists(nbv_ctx* ctx, const nbv_camera* h_cam, int64_t* d_offsets, int32_t* d_ids, int64_t cap, int64_t* h_total,
                   void* stream) {
  if (!ctx || !h_cam || !d_offsets || !h_total) return NBV_ERR_INVALID_ARG;
  if (!ctx->loaded) return fail(ctx, NBV_ERR_NOT_LOADED, "no Gaussians loaded");
  cudaStream_t st = (cudaStream_t)stream;
  ViewSlot* sl = ctx->slots[0];
  CKRET(process_view(ctx, sl, *h_cam, STAGE_BIN, false, false, st));
  const int n_tiles = sl->tg.tiles_x * sl->tg.tiles_y;
  CKRET(ensure(ctx, sl->tile_counts, 4 * (2 * (size_t)n_tiles + 4)));
  uint32_t* counts = sl->tile_counts.as<uint32_t>();
  uint32_t* scanned = counts + n_tiles;
  uint32_t* total = scanned + n_tiles;
  launch_tile_counts(sl->ckeys_sorted, sl->crect.as<ushort4>(), sl->cranges.as<uint2>(), sl->tg, sl->rank_bits, counts, scanned, total,
                     sl->scan_tmp.as<uint32_t>(), d_offsets, st);
  CK(cudaGetLastError());
  uint32_t h_tot = 0;
  CK(cudaMemcpyAsync(&h_tot, total, 4, cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  *h_total = (int64_t)h_tot;
  const bool fits = d_ids && (int64_t)h_tot <= cap;
  if (!fits && h_tot > 0) return fail(ctx, NBV_ERR_CAPACITY, "d_ids too small for the tile lists");
  if (h_tot > 0) {
    launch_tile_ids(sl->ckeys_sorted, sl->crect.as<ushort4>(), sl->cranges.as<uint2>(), sl->tg, sl->rank_bits, sl->ids.as<uint32_t>(),
                    scanned, d_ids, st);
    CK(cudaGetLastError());
    CK(cudaStreamSynchronize(st));
  }
  return NBV_OK;
}

int nbv_render(nbv_ctx* ctx, const nbv_camera* h_cam, float* d_rgb, float* d_depth, float* d_T, int32_t* d_ncontrib, void* stream) {
  if (!ctx || !h_cam) return NBV_ERR_INVALID_ARG;
  if (!ctx->loaded) return fail(ctx, NBV_ERR_NOT_LOADED, "no Gaussians loaded");
  if (ctx->mask_mode) return fail(ctx, NBV_ERR_INVALID_ARG, "nbv_render: a mask context renders with nbv_render_mask");
  cudaStream_t st = (cudaStream_t)stream;
  ViewSlot* sl = ctx->slots[0];
  CKRET(process_view(ctx, sl, *h_cam, STAGE_FORWARD, false, true, st));
  const size_t npx = (size_t)h_cam->width * h_cam->height;
  if (d_rgb) CK(cudaMemcpyAsync(d_rgb, sl->pix_rgb.p, 12 * npx, cudaMemcpyDeviceToDevice, st));
  if (d_depth) CK(cudaMemcpyAsync(d_depth, sl->pix_depth.p, 4 * npx, cudaMemcpyDeviceToDevice, st));
  if (d_T) CK(cudaMemcpyAsync(d_T, sl->pix_T.p, 4 * npx, cudaMemcpyDeviceToDevice, st));
  if (d_ncontrib) CK(cudaMemcpyAsync(d_ncontrib, sl->pix_nc.p, 4 * npx, cudaMemcpyDeviceToDevice, st));
  return NBV_OK;
}

int64_t nbv_block_size(const nbv_ctx* ctx) {
  if (!ctx) return 0;
  if (ctx->mask_mode && !ctx->loaded) return 0;
  return (int64_t)ctx->LB;
}

int nbv_render_mask(nbv_ctx* ctx, const nbv_camera* h_cam, float* d_mask, void* stream) {
  if (!ctx || !h_cam || !d_mask) return NBV_ERR_INVALID_ARG;
  if (!ctx->loaded) return fail(ctx, NBV_ERR_NOT_LOADED, "no Gaussians loaded");
  if (!ctx->mask_mode) return fail(ctx, NBV_ERR_INVALID_ARG, "nbv_render_mask needs a context created with channel_mask = NBV_CH_MASK");
  cudaStream_t st = (cudaStream_t)stream;
  ViewSlot* sl = ctx->slots[0];
  CKRET(pre_batch(ctx, &sl, h_cam, 1, STAGE_BACKWARD, false, true, st));      // S1-S2 and every buffer the raster passes use
  CKRET(ensure_tile_order(ctx, sl->tg, st));
  const size_t npx = (size_t)h_cam->width * h_cam->height;
  const SceneDev sc = scene_dev(ctx);
  for (int gr = 0; gr < ctx->mask_groups; ++gr) {
    const nbv_config gcfg = mask_group_config(ctx, gr);
    launch_mask_splats(sc, sl->splat_sorted.as<Splat>(), sl->ids.as<uint32_t>(), gr, ctx->cfg.mask_bg_channel, sl->gsplat.as<Splat>(), st);
    RasterBatch rb;
    rb.n = 1; rb.n_work = 0; rb.work = nullptr; rb.work_fwd = nullptr; rb.work_fb = nullptr; rb.overflow = nullptr;
    rb.tile_order = ctx->tile_order.as<uint32_t>();
    RasterView& v = rb.v[0];
    v.splat_sorted = sl->gsplat.as<Splat>(); v.ckeys = sl->ckeys_sorted; v.crect = sl->crect.as<ushort4>(); v.cranges = sl->cranges.as<uint2>();
    v.pix.rgb = sl->pix_rgb.as<float>(); v.pix.depth = sl->pix_depth.as<float>(); v.pix.ncontrib = sl->pix_nc.as<int32_t>();
    v.pix.T = sl->pix_T.as<float>(); v.pix.last = sl->pix_last.as<int32_t>();
    v.tile_cend = sl->tile_cend.as<uint32_t>(); v.tile_elast = sl->tile_elast.as<uint32_t>(); v.tile_walk = sl->tile_walk.as<uint32_t>();
    v.tlist = nullptr;                                   // forward pass only
    v.moments = sl->moments.as<double>(); v.mom_stride = NMOM * ctx->mask_groups; v.touched = sl->touched.as<uint32_t>();
    v.touched_flag = nullptr;                            // forward pass only
    v.touched_cnt = sl->touched_cnt.as<uint32_t>(); v.counters = sl->d_counters;
    launch_forward(rb, sl->tg, sl->rank_bits, h_cam->width, h_cam->height, gcfg, true, st);
    launch_mask_scatter(sl->pix_rgb.as<float>(), sl->pix_depth.as<float>(), npx, ctx->K, gr, ctx->cfg.mask_bg_channel, d_mask, st);
    CK(cudaGetLastError());
  }
  return NBV_OK;
}

int nbv_tile_walk(nbv_ctx* ctx, const nbv_camera* h_cam, int32_t* d_walked, int32_t* d_last, void* stream) {
  if (!ctx || !h_cam || !d_walked) return NBV_ERR_INVALID_ARG;
  if (!ctx->loaded) return fail(ctx, NBV_ERR_NOT_LOADED, "no Gaussians loaded");
  cudaStream_t st = (cudaStream_t)stream;
  ViewSlot* sl = ctx->slots[0];
  CKRET(process_view(ctx, sl, *h_cam, STAGE_FORWARD, false, false, st));
  const size_t n_tiles = (size_t)sl->tg.tiles_x * sl->tg.tiles_y;
  CK(cudaMemcpyAsync(d_walked, sl->tile_walk.p, 4 * n_tiles, cudaMemcpyDeviceToDevice, st));
  if (d_last) CK(cudaMemcpyAsync(d_last, sl->pix_last.p, 4 * (size_t)h_cam->width * h_cam->height, cudaMemcpyDeviceToDevice, st));
  return NBV_OK;
}

int nbv_view_hessian(nbv_ctx* ctx, const nbv_camera* h_cam, float* d_blocks, void* stream) {
  if (!ctx || !h_cam || !d_blocks) return NBV_ERR_INVALID_ARG;
  if (!ctx->loaded) return fail(ctx, NBV_ERR_NOT_LOADED, "no Gaussians loaded");
  cudaStream_t st = (cudaStream_t)stream;
  ViewSlot* sl = ctx->slots[0];
  CK(cudaMemsetAsync(d_blocks, 0, 4 * ctx->LB * ctx->N, st));
  CKRET(process_view(ctx, sl, *h_cam, STAGE_BACKWARD, false, false, st));
  CKRET(expand_view(ctx, sl, *h_cam, EXPAND_VIEW, d_blocks, nullptr, nullptr, st));
  return NBV_OK;
}

int nbv_training_hessian(nbv_ctx* ctx, float* d_blocks, void* stream) {
  if (!ctx || !d_blocks) return NBV_ERR_INVALID_ARG;
  if (!ctx->loaded) return fail(ctx, NBV_ERR_NOT_LOADED, "no Gaussians loaded");
  launch_export_blocks(ctx->H_T.as<double>(), d_blocks, ctx->LB * (size_t)ctx->N, (cudaStream_t)stream);
  CK(cudaGetLastError());
  return NBV_OK;
}

int nbv_chain(nbv_ctx* ctx, const nbv_camera* h_cam, float* d_chain, void* stream) {
  if (!ctx || !h_cam || !d_chain) return NBV_ERR_INVALID_ARG;
  if (!ctx->loaded) return fail(ctx, NBV_ERR_NOT_LOADED, "no Gaussians loaded");
  if (!valid_camera(*h_cam)) return fail(ctx, NBV_ERR_INVALID_ARG, "invalid camera (size, focal length or non-orthonormal R_cw)");
  launch_export_chain(scene_dev(ctx), *h_cam, d_chain, (cudaStream_t)stream);
  CK(cudaGetLastError());
  return NBV_OK;
}

int nbv_confidence(nbv_ctx* ctx, int32_t target_obj, float* d_conf, void* stream) {
  if (!ctx || !d_conf) return NBV_ERR_INVALID_ARG;
  if (!ctx->loaded) return fail(ctx, NBV_ERR_NOT_LOADED, "no Gaussians loaded");
  if (target_obj < -1 || target_obj >= ctx->K) return fail(ctx, NBV_ERR_UNKNOWN_TARGET, "target_obj must be -1 or in [0, K)");
  launch_confidence(scene_dev(ctx), ctx->cfg, target_obj, d_conf, (cudaStream_t)stream);
  CK(cudaGetLastError());
  return NBV_OK;
}

int nbv_gaussian_gains(nbv_ctx* ctx, const nbv_camera* h_cam, int32_t target_obj, float* d_gains, void* stream) {
  if (!ctx || !h_cam || !d_gains) return NBV_ERR_INVALID_ARG;
  if (!ctx->loaded) return fail(ctx, NBV_ERR_NOT_LOADED, "no Gaussians loaded");
  cudaStream_t st = (cudaStream_t)stream;
  ViewSlot* sl = ctx->slots[0];
  CKRET(prepare_scoring(ctx, target_obj, st));
  CKRET(ensure(ctx, ctx->score_tmp, 64));
  CK(cudaMemsetAsync(ctx->score_tmp.p, 0, 64, st));
  CK(cudaMemsetAsync(d_gains, 0, 4 * (size_t)ctx->N, st));
  CKRET(process_view(ctx, sl, *h_cam, STAGE_BACKWARD, false, false, st));
  CKRET(expand_view(ctx, sl, *h_cam, EXPAND_GAIN, nullptr, ctx->score_tmp.as<float>(), d_gains, st));
  return NBV_OK;
}

}  // extern "C"
