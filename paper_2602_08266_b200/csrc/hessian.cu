// hessian.cu -- S5 (moments -> 14x14 block), S0' (confidence), S6 (log-det gain), S7 (arg-max) of colour / depth contexts.
//
// S5: for a Gaussian touched by the view, the 40 screen-space moments of S4 become
//       H_g = A Q A^T + sum_ch omega_ch [ (A x_ch) e_ch^T + e_ch (A x_ch)^T + W2 e_ch e_ch^T ]          (block_math.cuh)
//     PAPER.md L189-191 (H ~= J^T J), L210 (per-Gaussian blocks), L248.
// S6: IG_g = log det(c_g (H_T,g + H_c,g) + Lambda) - log det(c_g H_T,g + Lambda)   (Eq. 5, 6, 9; R-13, R-14)
//     as the difference of the pivots of two L D L^T factorisations, sum_j log(d1_j / d0_j).
// PRECISION: everything after the 40 binary32 moments is binary64 -- the chain rule, A Q A^T, H_T itself, the two
//     factorisations.  A block has exact null directions (R-10; single-view blocks have rank ~8 of 14) next to entries of
//     1e5-1e7: in binary32 the product A Q A^T and the storage of H_T alone leave rounding noise of eps H_kk ~ 0.1-1 on
//     pivots whose exact value is the prior, which is what limited round 1 to Lambda = 1 and 5e-3 on single gains.  In
//     binary64 the null spaces survive to 1e-9 and the plain difference form is accurate to ~1e-13 / gain.  The work is
//     ~2.5 kflop (binary64) per touched Gaussian, 1-2% of a view.
// DETERMINISM: the touched list is built in rank order (touched_count / touched_write), a thread's partial gain and a block's
//     partial score depend only on (view, block), and the last block of a view adds the partials in block order; H_T is
//     accumulated view by view without atomics.  What is left run-to-run is the order of the binary32 `red.add` of S4.
#include <algorithm>
#include <cstdlib>

#include "block_math.cuh"
#include "kernels.h"

namespace nbv {

// ---- ordered touched list: the ranks whose sum w^2 (moment 39) is non-zero, i.e. the Gaussians with at least one
// composited pixel, in increasing rank (= depth) order.  Pass 1 counts per block of 256 ranks, pass 2 offsets every block
// by the counts before it (each block sums them itself: at most a few thousand numbers) and writes its ranks in order.
constexpr int TOUCH_T = 256;

__global__ void __launch_bounds__(TOUCH_T) touched_count_kernel(const __grid_constant__ RasterBatch batch, int N) {
  const RasterView& vw = batch.v[blockIdx.y];
  const int r = blockIdx.x * TOUCH_T + threadIdx.x;
  const bool hit = r < N && vw.moments[(size_t)r * vw.mom_stride + MOM_W2] != 0.0f;
  const int c = __syncthreads_count(hit);
  if (threadIdx.x == 0) vw.touched_cnt[blockIdx.x] = (uint32_t)c;
}

__global__ void __launch_bounds__(TOUCH_T) touched_write_kernel(const __grid_constant__ RasterBatch batch, int N) {
  __shared__ uint32_t wsum[TOUCH_T / 32], wcnt[TOUCH_T / 32];
  const RasterView& vw = batch.v[blockIdx.y];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  uint32_t before = 0;
  for (uint32_t b = threadIdx.x; b < blockIdx.x; b += TOUCH_T) before += vw.touched_cnt[b];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) before += __shfl_xor_sync(0xffffffffu, before, o);
  const int r = blockIdx.x * TOUCH_T + threadIdx.x;
  const bool hit = r < N && vw.moments[(size_t)r * vw.mom_stride + MOM_W2] != 0.0f;
  const unsigned m = __ballot_sync(0xffffffffu, hit);
  if (lane == 0) { wsum[wid] = before; wcnt[wid] = (uint32_t)__popc(m); }
  __syncthreads();
  uint32_t base = 0, total = 0;
#pragma unroll
  for (int w = 0; w < TOUCH_T / 32; ++w) {
    base += wsum[w];
    if (w < wid) base += wcnt[w];
    total += wcnt[w];
  }
  if (hit) vw.touched[base + __popc(m & ((1u << lane) - 1u))] = (uint32_t)r;
  if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) {
    uint32_t all = total;
#pragma unroll
    for (int w = 0; w < TOUCH_T / 32; ++w) all += wsum[w];
    vw.counters->n_touched = all;
  }
}

void launch_touched(const RasterBatch& batch, int N, cudaStream_t st) {
  const dim3 grid((unsigned)((N + TOUCH_T - 1) / TOUCH_T), (unsigned)batch.n);
  g_kernel_launches += 2;
  touched_count_kernel<<<grid, TOUCH_T, 0, st>>>(batch, N);
  touched_write_kernel<<<grid, TOUCH_T, 0, st>>>(batch, N);
}
uint32_t touched_blocks(int N) { return (uint32_t)((N + TOUCH_T - 1) / TOUCH_T); }

// ---- S6: the gain of one block against H_T,g (R-13, R-14; the three readings of where c_g acts are in nbv.h)
__device__ double block_gain(const double* __restrict__ ht, const double* H, double c, const nbv_config& cfg) {
  const double ct = cfg.weight_mode == 0 ? c : 1.0;          // Eq. 9 literal (R1) weights H_T as well; R2 / R3 do not
  const double cb = cfg.weight_mode == 1 ? 1.0 : c;          // R2 weights the gain, R1 / R3 the candidate block
  double A[NBLK], d0[P], d1[P];
  for (int i = 0; i < NBLK; ++i) A[i] = ct * ht[i];
  for (int k = 0; k < P; ++k) A[tri(k, k)] += (double)cfg.prior_precision[k];
  ldl_pivots(A, d0);
  for (int i = 0; i < NBLK; ++i) A[i] = fma(cb, H[i], ct * ht[i]);
  for (int k = 0; k < P; ++k) A[tri(k, k)] += (double)cfg.prior_precision[k];
  ldl_pivots(A, d1);
  double gn = 0.0;
  for (int k = 0; k < P; ++k) gn += log(d1[k] / d0[k]);
  return cfg.weight_mode == 1 ? c * gn : gn;
}

// deterministic block sum of one double per thread -> thread 0
template <int THREADS>
__device__ __forceinline__ double block_sum(double v, double* ws) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = v;
  __syncthreads();
  double t = 0.0;
  if (threadIdx.x == 0)
    for (int w = 0; w < THREADS / 32; ++w) t += ws[w];
  return t;
}

constexpr int EXP_T = 64;

__global__ void __launch_bounds__(EXP_T) expand_kernel(const __grid_constant__ SceneDev sc, const __grid_constant__ nbv_config cfg,
                                                        const __grid_constant__ ExpandBatch batch, int mode, int view0,
                                                        double* __restrict__ H_T, const float* __restrict__ conf,
                                                        uint32_t* __restrict__ cache_ids, double* __restrict__ cache_blocks) {
  __shared__ double ws[EXP_T / 32];
  const ExpandView& vw = batch.v[view0 + blockIdx.y];
  const nbv_camera& cam = vw.cam;
  const uint32_t* __restrict__ ids_sorted = vw.ids_sorted;
  const Splat* __restrict__ splat_sorted = vw.splat_sorted;
  const uint32_t* __restrict__ touched = vw.touched;
  float* __restrict__ moments = vw.moments;
  const uint32_t n_touched = vw.counters->n_touched;
  double gain = 0.0;
  float omega[4];
#pragma unroll
  for (int c = 0; c < 4; ++c) omega[c] = ((cfg.channel_mask >> c) & 1) ? cfg.channel_weight[c] : 0.f;
  for (uint32_t t = blockIdx.x * blockDim.x + threadIdx.x; t < n_touched; t += gridDim.x * blockDim.x) {
    const uint32_t r = touched[t];
    const uint32_t g = ids_sorted[r];
    float4* mom4 = reinterpret_cast<float4*>(moments + (size_t)r * NMOM);
    double m[NMOM];
#pragma unroll
    for (int i = 0; i < NMOM / 4; ++i) {
      const float4 v = mom4[i];
      m[4 * i] = v.x; m[4 * i + 1] = v.y; m[4 * i + 2] = v.z; m[4 * i + 3] = v.w;
      mom4[i] = make_float4(0.f, 0.f, 0.f, 0.f);     // leave the buffer zeroed for the next view
    }
    whitened_to_u<double>(m, splat_sorted[r]);        // the conic S4 evaluated with
    Chain<double> ch;
    projection_chain<double>(cam, sc.mean + 3 * (size_t)g, sc.logscale + 3 * (size_t)g, sc.quat + 4 * (size_t)g, ch);
    const double sg = (double)sc.sigma[g];
    const double kappa = cfg.opacity_coord == 0 ? (1.0 - sg) : 1.0 / sg;       // R-10
    double H[NBLK];
    build_block<double>(m, ch, kappa, omega, H);
    if (mode == EXPAND_TRAIN) {
      double* dst = H_T + (size_t)g * NBLK;             // one launch per view, in view order: a view lists a Gaussian once
      for (int i = 0; i < NBLK; ++i) dst[i] += H[i];
    } else if (mode == EXPAND_VIEW) {
      float* dst = vw.out_blocks + (size_t)g * NBLK;
      for (int i = 0; i < NBLK; ++i) dst[i] = (float)H[i];
    } else if (mode == EXPAND_CACHE) {
      if (t < vw.cache_span[1]) {                      // span[1] = 0 when the pool overflowed: nothing is stored
        const size_t e = (size_t)vw.cache_span[0] + t;
        cache_ids[e] = g;
        double* dst = cache_blocks + e * NBLK;
        for (int i = 0; i < NBLK; ++i) dst[i] = H[i];
      }
    } else {
      const double c = (double)conf[g];
      double gn = 0.0;
      if (c > 0.0) gn = block_gain(H_T + (size_t)g * NBLK, H, c, cfg);   // c_g = 0 (Eq. 12, non-target): exactly zero gain
      if (vw.gains) vw.gains[g] = (float)gn;
      gain += gn;
    }
  }
  if (mode == EXPAND_GAIN) {
    const double tot = block_sum<EXP_T>(gain, ws);
    ordered_score(tot, vw.partials, &vw.counters->n_expanded, vw.score);
  }
}

static int expand_blocks(int N, int n_views) {
  int blocks = (N + EXP_T - 1) / EXP_T;
  const int cap = (sm_count() * 8 + n_views - 1) / n_views;
  return std::max(1, std::min(blocks, cap));
}
int expand_partials() { return sm_count() * 8; }

void launch_expand(const SceneDev& sc, const nbv_config& cfg, const ExpandBatch& batch, int mode, double* H_T, const float* conf,
                   cudaStream_t st) {
  if (mode == EXPAND_TRAIN) {
    // H_T += H(view), view after view (Eq. 6): a fixed order of binary64 additions, no atomics
    const int blocks = expand_blocks(sc.N, 1);
    for (int v = 0; v < batch.n; ++v) {
      ++g_kernel_launches;
      expand_kernel<<<dim3((unsigned)blocks, 1u), EXP_T, 0, st>>>(sc, cfg, batch, mode, v, H_T, conf, nullptr, nullptr);
    }
    return;
  }
  ++g_kernel_launches;
  expand_kernel<<<dim3((unsigned)expand_blocks(sc.N, batch.n), (unsigned)batch.n), EXP_T, 0, st>>>(sc, cfg, batch, mode, 0, H_T, conf,
                                                                                                     nullptr, nullptr);
}

// ---- sparse block cache of greedy selection ----------------------------------------------------------------------
__global__ void cache_reserve_kernel(const __grid_constant__ ExpandBatch batch, BlockCache cache, int first_candidate) {
  // one thread, views in order: the pool layout does not depend on timing
  if (threadIdx.x != 0) return;
  for (int v = 0; v < batch.n; ++v) {
    const uint32_t cnt = batch.v[v].counters->n_touched;
    const uint32_t base = cache.cursor[0];
    uint32_t* span = cache.spans + 2 * (size_t)(first_candidate + v);
    if ((unsigned long long)base + cnt > cache.capacity) {
      cache.cursor[1] = 1u;                                // overflow: the caller falls back to re-rasterising
      span[0] = 0u; span[1] = 0u;
    } else {
      span[0] = base; span[1] = cnt;
      cache.cursor[0] = base + cnt;
    }
  }
}

void launch_cache_reserve(const ExpandBatch& batch, const BlockCache& cache, int first_candidate, cudaStream_t st) {
  ++g_kernel_launches;
  cache_reserve_kernel<<<1, 32, 0, st>>>(batch, cache, first_candidate);
}

void launch_expand_cache(const SceneDev& sc, const nbv_config& cfg, const ExpandBatch& batch, const BlockCache& cache, cudaStream_t st) {
  ++g_kernel_launches;
  expand_kernel<<<dim3((unsigned)expand_blocks(sc.N, batch.n), (unsigned)batch.n), EXP_T, 0, st>>>(sc, cfg, batch, EXPAND_CACHE, 0, nullptr,
                                                                                                     nullptr, cache.ids, cache.blocks);
}

// One thread per cached (candidate, Gaussian) entry: the gain of Eq. 5/6/9 of that block against the current H_T,g.
constexpr int CG_BLOCKS = 64;
__global__ void __launch_bounds__(EXP_T) cached_gain_kernel(BlockCache cache, const __grid_constant__ nbv_config cfg,
                                                            const int32_t* __restrict__ taken, const float* __restrict__ conf,
                                                            const double* __restrict__ H_T, float* __restrict__ scores,
                                                            double* __restrict__ partials, unsigned int* __restrict__ done) {
  __shared__ double ws[EXP_T / 32];
  const int c = blockIdx.y;
  double gain = 0.0;
  if (!taken[c]) {
    const uint32_t base = cache.spans[2 * c], cnt = cache.spans[2 * c + 1];
    for (uint32_t t = blockIdx.x * blockDim.x + threadIdx.x; t < cnt; t += gridDim.x * blockDim.x) {
      const size_t e = (size_t)base + t;
      const uint32_t g = cache.ids[e];
      const double cg = (double)conf[g];
      if (cg > 0.0) gain += block_gain(H_T + (size_t)g * NBLK, cache.blocks + e * NBLK, cg, cfg);
    }
  }
  const double tot = block_sum<EXP_T>(gain, ws);
  ordered_score(tot, partials + (size_t)c * CG_BLOCKS, done + c, scores + c);
}

size_t cached_gain_scratch_bytes(int n_cand) { return (size_t)n_cand * (CG_BLOCKS * sizeof(double) + sizeof(unsigned int)); }

void launch_cached_gain(const BlockCache& cache, const nbv_config& cfg, int n_cand, const int32_t* taken, const float* conf,
                        const double* H_T, float* scores, void* scratch, cudaStream_t st) {
  ++g_kernel_launches;
  double* partials = reinterpret_cast<double*>(scratch);
  unsigned int* done = reinterpret_cast<unsigned int*>(partials + (size_t)n_cand * CG_BLOCKS);     // zero on entry, zero on exit
  cached_gain_kernel<<<dim3(CG_BLOCKS, (unsigned)n_cand), EXP_T, 0, st>>>(cache, cfg, taken, conf, H_T, scores, partials, done);
}

__global__ void __launch_bounds__(256) cache_accumulate_kernel(BlockCache cache, const int32_t* __restrict__ pick, double* __restrict__ H_T) {
  const int c = *pick;
  const uint32_t base = cache.spans[2 * c], cnt = cache.spans[2 * c + 1];
  const size_t total = (size_t)cnt * NBLK;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
    const size_t e = i / NBLK, k = i - e * NBLK;
    const uint32_t g = cache.ids[base + e];              // a view lists every Gaussian at most once: no atomics needed
    H_T[(size_t)g * NBLK + k] += cache.blocks[((size_t)base + e) * NBLK + k];
  }
}

void launch_cache_accumulate(const BlockCache& cache, const int32_t* pick, double* H_T, cudaStream_t st) {
  ++g_kernel_launches;
  cache_accumulate_kernel<<<sm_count() * 4, 256, 0, st>>>(cache, pick, H_T);
}

// S0': confidence (Eq. 7; Eq. 12)
__global__ void __launch_bounds__(256) confidence_kernel(SceneDev sc, nbv_config cfg, int target, float* __restrict__ conf) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= sc.N) return;
  const float s = fmaxf(sc.sigma[g], cfg.sigma_floor);
  float p, c;
  if (target < 0) {
    p = sc.pmax[g];
  } else {
    p = expf(sc.logits[(size_t)g * sc.K + target] - sc.lse[g]);
  }
  p = fmaxf(p, cfg.p_floor);
  c = powf(p, -cfg.alpha_obj) * powf(s, -cfg.alpha_opa);
  if (target >= 0 && sc.amax[g] != target) c = 0.f;
  conf[g] = c;
}

void launch_confidence(const SceneDev& sc, const nbv_config& cfg, int target, float* conf, cudaStream_t st) {
  ++g_kernel_launches;
  confidence_kernel<<<(sc.N + 255) / 256, 256, 0, st>>>(sc, cfg, target, conf);
}

// parity export of H_T (binary64 on the device) as the float blocks of the C ABI
__global__ void __launch_bounds__(256) export_blocks_kernel(const double* __restrict__ src, float* __restrict__ dst, size_t n) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) dst[i] = (float)src[i];
}
void launch_export_blocks(const double* src, float* dst, size_t n, cudaStream_t st) {
  ++g_kernel_launches;
  export_blocks_kernel<<<sm_count() * 8, 256, 0, st>>>(src, dst, n);
}

// parity / debug export of the chain rule of S5: per Gaussian d(mx,my,a,b,c)/d(mu,logscale,quat) (5 x 10) and dz/dmu (3)
__global__ void __launch_bounds__(128) export_chain_kernel(SceneDev sc, nbv_camera cam, float* __restrict__ out) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= sc.N) return;
  Chain<double> ch;
  projection_chain<double>(cam, sc.mean + 3 * (size_t)g, sc.logscale + 3 * (size_t)g, sc.quat + 4 * (size_t)g, ch);
  float* o = out + (size_t)g * 53;
  for (int e = 0; e < 5; ++e)
    for (int k = 0; k < 10; ++k) o[10 * e + k] = (float)ch.G[e][k];
  for (int k = 0; k < 3; ++k) o[50 + k] = (float)ch.dz[k];
}
void launch_export_chain(const SceneDev& sc, const nbv_camera& cam, float* out, cudaStream_t st) {
  ++g_kernel_launches;
  export_chain_kernel<<<(sc.N + 127) / 128, 128, 0, st>>>(sc, cam, out);
}

// S7: arg-max, lowest index on ties (R-15)
__global__ void argmax_kernel(const float* __restrict__ scores, int n, int32_t* __restrict__ best) {
  const int lane = threadIdx.x;
  float bv = -INFINITY;
  int bi = 0x7fffffff;
  for (int i = lane; i < n; i += 32) {
    const float v = scores[i];
    if (v > bv || (v == bv && i < bi)) { bv = v; bi = i; }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const float ov = __shfl_xor_sync(0xffffffffu, bv, o);
    const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
    if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
  }
  if (lane == 0) *best = bi == 0x7fffffff ? 0 : bi;
}

void launch_argmax(const float* scores, int n, int32_t* best, cudaStream_t st) {
  ++g_kernel_launches;
  argmax_kernel<<<1, 32, 0, st>>>(scores, n, best);
}

}  // namespace nbv
