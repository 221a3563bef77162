// nbv_api.cu -- context, per-view pipeline orchestration and the C ABI of include/nbv.h.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <utility>
#include <vector>

#include "kernels.h"

using namespace nbv;

namespace nbv {
unsigned long long g_kernel_launches = 0;
}

namespace {

struct DevBuf {
  void* p = nullptr;
  size_t cap = 0;
  template <class T> T* as() const { return reinterpret_cast<T*>(p); }
};

}  // namespace

struct nbv_ctx {
  nbv_config cfg;
  std::string err;
  int device = 0;
  int N = 0, K = 0;
  bool loaded = false;
  int n_train = 0;
  // scene
  DevBuf mean, logscale, quat, sigma, rgb, logits, M, pmax, amax, lse, H_T, conf, cholT;
  // per-view work buffers
  DevBuf splat, zkey, zkey_alt, ids, ids_alt, rect, abc, splat_sorted, rect_sorted, ntiles, offsets;
  DevBuf keys, keys_alt, ranges, sort_tmp, scan_tmp, tile_counts;
  DevBuf pix_rgb, pix_depth, pix_T, pix_nc, pix_last, moments, score_tmp;
  ViewCounters* d_counters = nullptr;
  ViewCounters* h_counters = nullptr;   // pinned
  // products of the last process_view()
  int rank_bits = 1;
  size_t n_keys = 0;
  uint32_t* keys_sorted = nullptr;
  int cur_W = 0, cur_H = 0;
  int conf_target = -2;                 // target the conf / cholT buffers were prepared for (-2 = stale)
  // optional per-stage timing (nbv_set_stage_timing): one event row per view, folded on read-out
  bool timing = false;
  std::vector<cudaEvent_t> ev;          // ev[view * (NBV_N_STAGES + 1) + boundary]
  std::vector<unsigned> ev_mask;        // per view: bit b set when boundary b was recorded
  size_t ev_views = 0;
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
      if (!(std::fabs(d - (i == j ? 1.0 : 0.0)) <= 1e-4)) return false;
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

PixelBuf pixel_buf(const nbv_ctx* c) {
  PixelBuf p;
  p.rgb = c->pix_rgb.as<float>(); p.depth = c->pix_depth.as<float>(); p.T = c->pix_T.as<float>();
  p.ncontrib = c->pix_nc.as<int32_t>(); p.last = c->pix_last.as<int32_t>();
  return p;
}

constexpr int EV_ROW = NBV_N_STAGES + 1;
constexpr size_t EV_MAX_VIEWS = 1024;

// fold the recorded event rows into ctx->stage_ms (the stream must be idle)
void fold_timing(nbv_ctx* ctx) {
  for (size_t v = 0; v < ctx->ev_views; ++v) {
    const unsigned m = ctx->ev_mask[v];
    for (int s = 0; s < NBV_N_STAGES; ++s)
      if (((m >> s) & 1u) && ((m >> (s + 1)) & 1u)) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, ctx->ev[v * EV_ROW + s], ctx->ev[v * EV_ROW + s + 1]) == cudaSuccess) ctx->stage_ms[s] += ms;
      }
    if (m) ctx->timed_views++;
    ctx->ev_mask[v] = 0;
  }
  cudaGetLastError();
  ctx->ev_views = 0;
}

// start a new event row for the next view
void timing_begin_view(nbv_ctx* ctx, cudaStream_t st) {
  if (!ctx->timing) return;
  if (ctx->ev_views >= EV_MAX_VIEWS) { cudaStreamSynchronize(st); fold_timing(ctx); }
  const size_t v = ctx->ev_views++;
  if (ctx->ev.size() < (v + 1) * EV_ROW) {
    const size_t old = ctx->ev.size();
    ctx->ev.resize((v + 1) * EV_ROW);
    for (size_t i = old; i < ctx->ev.size(); ++i) cudaEventCreate(&ctx->ev[i]);
    ctx->ev_mask.resize(v + 1, 0u);
  }
  ctx->ev_mask[v] = 0;
}

// record boundary b (= start of stage b, end of stage b-1) of the current view
void mark(nbv_ctx* ctx, int b, cudaStream_t st) {
  if (!ctx->timing || ctx->ev_views == 0) return;
  const size_t v = ctx->ev_views - 1;
  cudaEventRecord(ctx->ev[v * EV_ROW + b], st);
  ctx->ev_mask[v] |= 1u << b;
}

enum Stage { STAGE_PROJECT = 0, STAGE_BIN = 1, STAGE_FORWARD = 2, STAGE_BACKWARD = 3 };

// S1..S4 for one camera.  Leaves the depth order in ctx->ids, rank-ordered splats, sorted keys, tile ranges,
// per-pixel buffers and (STAGE_BACKWARD) the moment buffer.  Synchronises the stream once (key count read-back).
int process_view(nbv_ctx* ctx, const nbv_camera& cam, int upto, bool want_abc, cudaStream_t st) {
  if (!valid_camera(cam)) return fail(ctx, NBV_ERR_INVALID_ARG, "invalid camera (size, focal length or non-orthonormal R_cw)");
  const int N = ctx->N;
  const int TX = (cam.width + TILE - 1) / TILE, TY = (cam.height + TILE - 1) / TILE;
  const int n_tiles = TX * TY;
  const int rank_bits = ceil_log2((size_t)N), tile_bits = ceil_log2((size_t)n_tiles);
  if (rank_bits + tile_bits > 32)
    return fail(ctx, NBV_ERR_INVALID_ARG, "N x tiles exceeds the 32-bit (tile | depth rank) key space");
  ctx->rank_bits = rank_bits;
  ctx->cur_W = cam.width; ctx->cur_H = cam.height;
  const SceneDev sc = scene_dev(ctx);

  CKRET(ensure(ctx, ctx->splat, sizeof(Splat) * (size_t)N));
  CKRET(ensure(ctx, ctx->zkey, 4 * (size_t)N)); CKRET(ensure(ctx, ctx->zkey_alt, 4 * (size_t)N));
  CKRET(ensure(ctx, ctx->ids, 4 * (size_t)N)); CKRET(ensure(ctx, ctx->ids_alt, 4 * (size_t)N));
  CKRET(ensure(ctx, ctx->rect, sizeof(ushort4) * (size_t)N));
  if (want_abc) CKRET(ensure(ctx, ctx->abc, 12 * (size_t)N));
  CKRET(ensure(ctx, ctx->sort_tmp, 4 * radix_temp_words((size_t)N)));
  CKRET(ensure(ctx, ctx->scan_tmp, 4 * scan_temp_words((size_t)N + 1)));

  CK(cudaMemsetAsync(ctx->d_counters, 0, sizeof(ViewCounters), st));
  timing_begin_view(ctx, st);
  mark(ctx, NBV_STAGE_PROJECT, st);
  launch_project(sc, cam, ctx->cfg, ctx->splat.as<Splat>(), ctx->zkey.as<uint32_t>(), ctx->ids.as<uint32_t>(),
                 ctx->rect.as<ushort4>(), want_abc ? ctx->abc.as<float>() : nullptr, ctx->d_counters, st);
  CK(cudaGetLastError());
  if (upto == STAGE_PROJECT) return NBV_OK;

  // depth sort: 4 stable passes of 8 bits on the z bits, Gaussian index as value (ties keep index order: R-7)
  mark(ctx, NBV_STAGE_DEPTH_SORT, st);
  {
    uint32_t *k0 = ctx->zkey.as<uint32_t>(), *k1 = ctx->zkey_alt.as<uint32_t>();
    uint32_t *v0 = ctx->ids.as<uint32_t>(), *v1 = ctx->ids_alt.as<uint32_t>();
    for (int pass = 0; pass < 4; ++pass) {
      radix_pass(k0, k1, v0, v1, (size_t)N, 8 * pass, 8, ctx->sort_tmp.as<uint32_t>(), st);
      std::swap(k0, k1);
      std::swap(v0, v1);
    }
    CK(cudaGetLastError());
  }
  mark(ctx, NBV_STAGE_BIN, st);
  CKRET(ensure(ctx, ctx->splat_sorted, sizeof(Splat) * (size_t)N));
  CKRET(ensure(ctx, ctx->rect_sorted, sizeof(ushort4) * (size_t)N));
  CKRET(ensure(ctx, ctx->ntiles, 4 * (size_t)N));
  CKRET(ensure(ctx, ctx->offsets, 4 * (size_t)N));
  launch_gather(ctx->ids.as<uint32_t>(), ctx->splat.as<Splat>(), ctx->rect.as<ushort4>(), N, ctx->splat_sorted.as<Splat>(),
                ctx->rect_sorted.as<ushort4>(), ctx->ntiles.as<uint32_t>(), st);
  exclusive_scan_u32(ctx->ntiles.as<uint32_t>(), ctx->offsets.as<uint32_t>(), (size_t)N, ctx->scan_tmp.as<uint32_t>(), nullptr, st);
  CK(cudaGetLastError());
  CK(cudaMemcpyAsync(ctx->h_counters, ctx->d_counters, sizeof(ViewCounters), cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  const unsigned long long n_keys = ctx->h_counters->n_keys;
  if (n_keys >= 0xfff00000ull) return fail(ctx, NBV_ERR_INVALID_ARG, "more than 2^32 (tile, Gaussian) keys in one view");
  ctx->n_keys = (size_t)n_keys;

  CKRET(ensure(ctx, ctx->keys, 4 * (size_t)n_keys, true));
  CKRET(ensure(ctx, ctx->keys_alt, 4 * (size_t)n_keys, true));
  CKRET(ensure(ctx, ctx->sort_tmp, 4 * radix_temp_words(std::max((size_t)n_keys, (size_t)N)), true));
  CKRET(ensure(ctx, ctx->ranges, sizeof(uint2) * (size_t)n_tiles));
  launch_emit_keys(ctx->rect_sorted.as<ushort4>(), ctx->offsets.as<uint32_t>(), N, TX, rank_bits, ctx->keys.as<uint32_t>(), st);
  mark(ctx, NBV_STAGE_TILE_SORT, st);
  {
    uint32_t *k0 = ctx->keys.as<uint32_t>(), *k1 = ctx->keys_alt.as<uint32_t>();
    const int npass = (tile_bits + 7) / 8;
    const int bits = (tile_bits + npass - 1) / npass;
    for (int pass = 0; pass < npass; ++pass) {
      radix_pass(k0, k1, nullptr, nullptr, (size_t)n_keys, rank_bits + pass * bits, bits, ctx->sort_tmp.as<uint32_t>(), st);
      std::swap(k0, k1);
    }
    ctx->keys_sorted = k0;
  }
  launch_tile_ranges(ctx->keys_sorted, (size_t)n_keys, rank_bits, ctx->ranges.as<uint2>(), n_tiles, st);
  CK(cudaGetLastError());
  mark(ctx, NBV_STAGE_FORWARD, st);
  if (upto == STAGE_BIN) return NBV_OK;

  const size_t npx = (size_t)cam.width * cam.height;
  CKRET(ensure(ctx, ctx->pix_rgb, 12 * npx)); CKRET(ensure(ctx, ctx->pix_depth, 4 * npx)); CKRET(ensure(ctx, ctx->pix_T, 4 * npx));
  CKRET(ensure(ctx, ctx->pix_nc, 4 * npx)); CKRET(ensure(ctx, ctx->pix_last, 4 * npx));
  launch_forward(ctx->splat_sorted.as<Splat>(), ctx->keys_sorted, ctx->ranges.as<uint2>(), rank_bits, cam.width, cam.height,
                 ctx->cfg, pixel_buf(ctx), ctx->d_counters, st);
  CK(cudaGetLastError());
  mark(ctx, NBV_STAGE_BACKWARD, st);
  if (upto == STAGE_FORWARD) return NBV_OK;

  CKRET(ensure(ctx, ctx->moments, 4 * (size_t)NMOM * N));
  CK(cudaMemsetAsync(ctx->moments.p, 0, 4 * (size_t)NMOM * N, st));
  launch_backward(ctx->splat_sorted.as<Splat>(), ctx->keys_sorted, ctx->ranges.as<uint2>(), rank_bits, cam.width, cam.height,
                  ctx->cfg, pixel_buf(ctx), ctx->moments.as<float>(), st);
  CK(cudaGetLastError());
  mark(ctx, NBV_STAGE_EXPAND, st);
  return NBV_OK;
}

int prepare_scoring(nbv_ctx* ctx, int target, cudaStream_t st) {
  if (target < -1 || target >= ctx->K) return fail(ctx, NBV_ERR_UNKNOWN_TARGET, "target_obj must be -1 or in [0, K)");
  if (ctx->conf_target == target) return NBV_OK;
  const SceneDev sc = scene_dev(ctx);
  launch_confidence(sc, ctx->cfg, target, ctx->conf.as<float>(), st);
  launch_prepare(sc, ctx->cfg, ctx->H_T.as<float>(), ctx->conf.as<float>(), ctx->cholT.as<float>(), st);
  CK(cudaGetLastError());
  ctx->conf_target = target;
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
}

int nbv_create(nbv_ctx** out, const nbv_config* cfg) {
  if (!out) return NBV_ERR_INVALID_ARG;
  *out = nullptr;
  nbv_config c;
  if (cfg) c = *cfg; else nbv_default_config(&c);
  const bool ok = c.near_plane > 0.f && c.blur >= 0.f && c.alpha_min >= 1.0f / 255.0f && c.alpha_max > c.alpha_min &&
                  c.alpha_max < 1.f && c.t_stop > 0.f && c.t_stop < 1.f && (c.channel_mask & 15) != 0 && (c.channel_mask & ~15) == 0 &&
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
  ctx->device = dev;
  if (cudaMalloc(&ctx->d_counters, sizeof(ViewCounters)) != cudaSuccess ||
      cudaMallocHost(&ctx->h_counters, sizeof(ViewCounters)) != cudaSuccess) {
    cudaGetLastError();
    if (ctx->d_counters) cudaFree(ctx->d_counters);
    delete ctx;
    return NBV_ERR_CUDA;
  }
  std::memset(ctx->h_counters, 0, sizeof(ViewCounters));
  *out = ctx;
  return NBV_OK;
}

void nbv_destroy(nbv_ctx* ctx) {
  if (!ctx) return;
  DevBuf* all[] = {&ctx->mean, &ctx->logscale, &ctx->quat, &ctx->sigma, &ctx->rgb, &ctx->logits, &ctx->M, &ctx->pmax, &ctx->amax,
                   &ctx->lse, &ctx->H_T, &ctx->conf, &ctx->cholT, &ctx->splat, &ctx->zkey, &ctx->zkey_alt, &ctx->ids, &ctx->ids_alt,
                   &ctx->rect, &ctx->abc, &ctx->splat_sorted, &ctx->rect_sorted, &ctx->ntiles, &ctx->offsets, &ctx->keys,
                   &ctx->keys_alt, &ctx->ranges, &ctx->sort_tmp, &ctx->scan_tmp, &ctx->tile_counts, &ctx->pix_rgb, &ctx->pix_depth,
                   &ctx->pix_T, &ctx->pix_nc, &ctx->pix_last, &ctx->moments, &ctx->score_tmp};
  for (DevBuf* b : all) release(*b);
  if (ctx->d_counters) cudaFree(ctx->d_counters);
  if (ctx->h_counters) cudaFreeHost(ctx->h_counters);
  for (cudaEvent_t e : ctx->ev) cudaEventDestroy(e);
  delete ctx;
}

const char* nbv_last_error(const nbv_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }

int nbv_load_gaussians(nbv_ctx* ctx, int32_t N, int32_t K, const float* d_mean, const float* d_logscale, const float* d_quat,
                       const float* d_opacity, const float* d_rgb, const float* d_obj_logits, void* stream) {
  if (!ctx) return NBV_ERR_INVALID_ARG;
  if (N <= 0 || K <= 0 || !d_mean || !d_logscale || !d_quat || !d_opacity || !d_rgb || !d_obj_logits)
    return fail(ctx, NBV_ERR_INVALID_ARG, "nbv_load_gaussians: N, K must be positive and all pointers non-null");
  cudaStream_t st = (cudaStream_t)stream;
  ctx->loaded = false;
  ctx->N = N; ctx->K = K;
  const size_t n = (size_t)N;
  CKRET(ensure(ctx, ctx->mean, 12 * n)); CKRET(ensure(ctx, ctx->logscale, 12 * n)); CKRET(ensure(ctx, ctx->quat, 16 * n));
  CKRET(ensure(ctx, ctx->sigma, 4 * n)); CKRET(ensure(ctx, ctx->rgb, 12 * n)); CKRET(ensure(ctx, ctx->logits, 4 * n * K));
  CKRET(ensure(ctx, ctx->M, 36 * n)); CKRET(ensure(ctx, ctx->pmax, 4 * n)); CKRET(ensure(ctx, ctx->amax, 4 * n));
  CKRET(ensure(ctx, ctx->lse, 4 * n)); CKRET(ensure(ctx, ctx->H_T, 4 * (size_t)NBLK * n)); CKRET(ensure(ctx, ctx->conf, 4 * n));
  CKRET(ensure(ctx, ctx->cholT, 4 * (size_t)NBLK * n));
  CK(cudaMemcpyAsync(ctx->mean.p, d_mean, 12 * n, cudaMemcpyDeviceToDevice, st));
  CK(cudaMemcpyAsync(ctx->logscale.p, d_logscale, 12 * n, cudaMemcpyDeviceToDevice, st));
  CK(cudaMemcpyAsync(ctx->quat.p, d_quat, 16 * n, cudaMemcpyDeviceToDevice, st));
  CK(cudaMemcpyAsync(ctx->sigma.p, d_opacity, 4 * n, cudaMemcpyDeviceToDevice, st));
  CK(cudaMemcpyAsync(ctx->rgb.p, d_rgb, 12 * n, cudaMemcpyDeviceToDevice, st));
  CK(cudaMemcpyAsync(ctx->logits.p, d_obj_logits, 4 * n * K, cudaMemcpyDeviceToDevice, st));
  CK(cudaMemsetAsync(ctx->H_T.p, 0, 4 * (size_t)NBLK * n, st));
  CK(cudaMemsetAsync(ctx->d_counters, 0, sizeof(ViewCounters), st));
  launch_activate(scene_dev(ctx), ctx->d_counters, st);
  CK(cudaGetLastError());
  CK(cudaMemcpyAsync(ctx->h_counters, ctx->d_counters, sizeof(ViewCounters), cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  if (ctx->h_counters->bad_data)
    return fail(ctx, NBV_ERR_BAD_DATA, "zero/non-finite quaternion, opacity outside (0,1) or non-finite parameter");
  ctx->n_train = 0;
  ctx->conf_target = -2;
  ctx->loaded = true;
  return NBV_OK;
}

int nbv_reset_training(nbv_ctx* ctx, void* stream) {
  if (!ctx) return NBV_ERR_INVALID_ARG;
  if (!ctx->loaded) return fail(ctx, NBV_ERR_NOT_LOADED, "no Gaussians loaded");
  CK(cudaMemsetAsync(ctx->H_T.p, 0, 4 * (size_t)NBLK * ctx->N, (cudaStream_t)stream));
  ctx->n_train = 0;
  ctx->conf_target = -2;
  return NBV_OK;
}

int nbv_accumulate_training(nbv_ctx* ctx, const nbv_camera* h_cams, int32_t n, void* stream) {
  if (!ctx) return NBV_ERR_INVALID_ARG;
  if (!ctx->loaded) return fail(ctx, NBV_ERR_NOT_LOADED, "no Gaussians loaded");
  if (n < 0 || (n > 0 && !h_cams)) return fail(ctx, NBV_ERR_INVALID_ARG, "nbv_accumulate_training: bad camera array");
  cudaStream_t st = (cudaStream_t)stream;
  for (int i = 0; i < n; ++i)
    if (!valid_camera(h_cams[i])) return fail(ctx, NBV_ERR_INVALID_ARG, "invalid camera (size, focal length or non-orthonormal R_cw)");
  for (int i = 0; i < n; ++i) {
    CKRET(process_view(ctx, h_cams[i], STAGE_BACKWARD, false, st));
    launch_expand(scene_dev(ctx), h_cams[i], ctx->cfg, ctx->ids.as<uint32_t>(), ctx->moments.as<float>(), EXPAND_TRAIN,
                  ctx->H_T.as<float>(), nullptr, nullptr, nullptr, nullptr, nullptr, ctx->d_counters, st);
    CK(cudaGetLastError());
    mark(ctx, NBV_N_STAGES, st);
    ctx->n_train++;
    ctx->conf_target = -2;
  }
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
  for (int i = 0; i < n; ++i) {
    CKRET(process_view(ctx, h_cams[i], STAGE_BACKWARD, false, st));
    launch_expand(scene_dev(ctx), h_cams[i], ctx->cfg, ctx->ids.as<uint32_t>(), ctx->moments.as<float>(), EXPAND_GAIN,
                  ctx->H_T.as<float>(), nullptr, ctx->conf.as<float>(), ctx->cholT.as<float>(), d_scores + i, nullptr,
                  ctx->d_counters, st);
    CK(cudaGetLastError());
    mark(ctx, NBV_N_STAGES, st);
  }
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

int nbv_last_view_stats(nbv_ctx* ctx, nbv_view_stats* h_out, void* stream) {
  if (!ctx || !h_out) return NBV_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  CK(cudaMemcpyAsync(ctx->h_counters, ctx->d_counters, sizeof(ViewCounters), cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  h_out->n_visible = ctx->h_counters->n_visible;
  h_out->n_keys = (int64_t)ctx->h_counters->n_keys;
  h_out->n_entries = (int64_t)ctx->h_counters->n_entries;
  h_out->n_pairs = (int64_t)ctx->h_counters->n_pairs;
  h_out->n_touched = ctx->h_counters->n_touched;
  return NBV_OK;
}

int nbv_set_stage_timing(nbv_ctx* ctx, int32_t enable, void* stream) {
  if (!ctx) return NBV_ERR_INVALID_ARG;
  CK(cudaStreamSynchronize((cudaStream_t)stream));
  ctx->ev_views = 0;
  for (auto& m : ctx->ev_mask) m = 0;
  for (int s = 0; s < NBV_N_STAGES; ++s) ctx->stage_ms[s] = 0.0;
  ctx->timed_views = 0;
  ctx->timing = enable != 0;
  return NBV_OK;
}

int nbv_stage_times(nbv_ctx* ctx, double* h_ms, int64_t* h_views, void* stream) {
  if (!ctx || !h_ms) return NBV_ERR_INVALID_ARG;
  CK(cudaStreamSynchronize((cudaStream_t)stream));
  fold_timing(ctx);
  for (int s = 0; s < NBV_N_STAGES; ++s) h_ms[s] = ctx->stage_ms[s];
  if (h_views) *h_views = ctx->timed_views;
  return NBV_OK;
}

int64_t nbv_kernel_launches(void) { return (int64_t)nbv::g_kernel_launches; }

int nbv_projected(nbv_ctx* ctx, const nbv_camera* h_cam, int32_t* d_visible, float* d_rec, int32_t* d_rect, void* stream) {
  if (!ctx || !h_cam) return NBV_ERR_INVALID_ARG;
  if (!ctx->loaded) return fail(ctx, NBV_ERR_NOT_LOADED, "no Gaussians loaded");
  cudaStream_t st = (cudaStream_t)stream;
  CKRET(process_view(ctx, *h_cam, STAGE_PROJECT, true, st));
  ++g_kernel_launches;
  export_projected_kernel<<<(ctx->N + 255) / 256, 256, 0, st>>>(ctx->N, ctx->splat.as<Splat>(), ctx->zkey.as<uint32_t>(),
                                                                ctx->rect.as<ushort4>(), ctx->abc.as<float>(), d_visible, d_rec, d_rect);
  CK(cudaGetLastError());
  return NBV_OK;
}

int nbv_tile_lists(nbv_ctx* ctx, const nbv_camera* h_cam, int64_t* d_offsets, int32_t* d_ids, int64_t cap, int64_t* h_total,
                   void* stream) {
  if (!ctx || !h_cam || !d_offsets || !h_total) return NBV_ERR_INVALID_ARG;
  if (!ctx->loaded) return fail(ctx, NBV_ERR_NOT_LOADED, "no Gaussians loaded");
  cudaStream_t st = (cudaStream_t)stream;
  CKRET(process_view(ctx, *h_cam, STAGE_BIN, false, st));
  const int n_tiles = ((h_cam->width + TILE - 1) / TILE) * ((h_cam->height + TILE - 1) / TILE);
  *h_total = (int64_t)ctx->n_keys;
  CKRET(ensure(ctx, ctx->tile_counts, 4 * (size_t)n_tiles + 4));
  CKRET(ensure(ctx, ctx->scan_tmp, 4 * scan_temp_words(std::max((size_t)n_tiles, (size_t)ctx->N + 1))));
  const bool fits = d_ids && (int64_t)ctx->n_keys <= cap;
  launch_export_lists(ctx->keys_sorted, ctx->n_keys, ctx->rank_bits, ctx->ids.as<uint32_t>(), ctx->ranges.as<uint2>(), n_tiles,
                      d_offsets, fits ? d_ids : nullptr, ctx->tile_counts.as<uint32_t>(), ctx->scan_tmp.as<uint32_t>(), st);
  CK(cudaGetLastError());
  CK(cudaStreamSynchronize(st));
  if (!fits && ctx->n_keys > 0) return fail(ctx, NBV_ERR_CAPACITY, "d_ids too small for the tile lists");
  return NBV_OK;
}

int nbv_render(nbv_ctx* ctx, const nbv_camera* h_cam, float* d_rgb, float* d_depth, float* d_T, int32_t* d_ncontrib, void* stream) {
  if (!ctx || !h_cam) return NBV_ERR_INVALID_ARG;
  if (!ctx->loaded) return fail(ctx, NBV_ERR_NOT_LOADED, "no Gaussians loaded");
  cudaStream_t st = (cudaStream_t)stream;
  CKRET(process_view(ctx, *h_cam, STAGE_FORWARD, false, st));
  const size_t npx = (size_t)h_cam->width * h_cam->height;
  if (d_rgb) CK(cudaMemcpyAsync(d_rgb, ctx->pix_rgb.p, 12 * npx, cudaMemcpyDeviceToDevice, st));
  if (d_depth) CK(cudaMemcpyAsync(d_depth, ctx->pix_depth.p, 4 * npx, cudaMemcpyDeviceToDevice, st));
  if (d_T) CK(cudaMemcpyAsync(d_T, ctx->pix_T.p, 4 * npx, cudaMemcpyDeviceToDevice, st));
  if (d_ncontrib) CK(cudaMemcpyAsync(d_ncontrib, ctx->pix_nc.p, 4 * npx, cudaMemcpyDeviceToDevice, st));
  return NBV_OK;
}

int nbv_view_hessian(nbv_ctx* ctx, const nbv_camera* h_cam, float* d_blocks, void* stream) {
  if (!ctx || !h_cam || !d_blocks) return NBV_ERR_INVALID_ARG;
  if (!ctx->loaded) return fail(ctx, NBV_ERR_NOT_LOADED, "no Gaussians loaded");
  cudaStream_t st = (cudaStream_t)stream;
  CK(cudaMemsetAsync(d_blocks, 0, 4 * (size_t)NBLK * ctx->N, st));
  CKRET(process_view(ctx, *h_cam, STAGE_BACKWARD, false, st));
  launch_expand(scene_dev(ctx), *h_cam, ctx->cfg, ctx->ids.as<uint32_t>(), ctx->moments.as<float>(), EXPAND_VIEW, nullptr, d_blocks,
                nullptr, nullptr, nullptr, nullptr, ctx->d_counters, st);
  CK(cudaGetLastError());
  return NBV_OK;
}

int nbv_training_hessian(nbv_ctx* ctx, float* d_blocks, void* stream) {
  if (!ctx || !d_blocks) return NBV_ERR_INVALID_ARG;
  if (!ctx->loaded) return fail(ctx, NBV_ERR_NOT_LOADED, "no Gaussians loaded");
  CK(cudaMemcpyAsync(d_blocks, ctx->H_T.p, 4 * (size_t)NBLK * ctx->N, cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
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
  CKRET(prepare_scoring(ctx, target_obj, st));
  CKRET(ensure(ctx, ctx->score_tmp, 64));
  CK(cudaMemsetAsync(ctx->score_tmp.p, 0, 64, st));
  CK(cudaMemsetAsync(d_gains, 0, 4 * (size_t)ctx->N, st));
  CKRET(process_view(ctx, *h_cam, STAGE_BACKWARD, false, st));
  launch_expand(scene_dev(ctx), *h_cam, ctx->cfg, ctx->ids.as<uint32_t>(), ctx->moments.as<float>(), EXPAND_GAIN, ctx->H_T.as<float>(),
                nullptr, ctx->conf.as<float>(), ctx->cholT.as<float>(), ctx->score_tmp.as<float>(), d_gains, ctx->d_counters, st);
  CK(cudaGetLastError());
  return NBV_OK;
}

}  // extern "C"
