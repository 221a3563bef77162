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

// ---- S5 + S6, ONE WARP PER TOUCHED GAUSSIAN, everything in shared memory (packed 105-double blocks, coalesced H_T rows).
// A thread-per-Gaussian version kept ~3 KB of dynamically indexed binary64 arrays per thread in local memory; with a few
// hundred resident threads per SM that working set fell out of the L1 and the kernel took 0.64 ms per 8-view batch for
// 2e8 binary64 operations.  Here the 32 lanes share one Gaussian: lane k computes column k of the chain rule, the 66 + 44
// entries of A Q and A x_ch and the 105 entries of H are dealt to the lanes, and the two L D L^T factorisations update the
// trailing packed entries in parallel (one __syncwarp per pivot).
constexpr int EXP_WARPS = 8;
constexpr int EXP_T = EXP_WARPS * 32;

struct WarpScratch {
  double mom[NMOM];      // S4's moments (whitened basis)
  double mu[NMOM];       // the same in the u basis
  double A[11][6];
  double AQ[11][6];
  double yv[4][11];      // sqrt(omega_ch) A x_ch
  double H[NBLK];        // the view's block
  double M[NBLK];        // the matrix being factored
  double piv0[P], piv1[P];
  double dz[4];
};

// in-place L D L^T of the packed symmetric positive definite M, all lanes; pivots -> piv
__device__ __forceinline__ void warp_ldl14(double* M, double* piv, const uint8_t* tr, const uint8_t* tc, int lane) {
  for (int j = 0; j < P; ++j) {
    __syncwarp();
    const int jj = tri(j, j);
    const double d = fmax(M[jj], 1e-300);
    if (lane == 0) piv[j] = d;
    const double inv = 1.0 / d;
    for (int t = tri(j + 1, j + 1) + lane; t < NBLK; t += 32) {          // the rows below the pivot: contiguous in packed order
      const int r = tr[t], c = tc[t];
      M[t] = fma(-(M[jj + (r - j)] * inv), M[jj + (c - j)], M[t]);
    }
  }
  __syncwarp();
}

// trace(A^-1) from the factorisation warp_ldl14 left in M / piv: lane c solves L x = e_c
__device__ __forceinline__ double warp_inverse_trace14(const double* M, const double* piv, int lane) {
  double acc = 0.0;
  if (lane < P) {
    double x[P];
    x[lane] = 1.0;
    acc = 1.0 / piv[lane];
    for (int i = lane + 1; i < P; ++i) {
      double sacc = 0.0;
      for (int j = lane; j < i; ++j) sacc = fma(M[tri(j, i)] / piv[j], x[j], sacc);
      x[i] = -sacc;
      acc = fma(sacc * sacc, 1.0 / piv[i], acc);
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  return acc;
}

// S6 for one block held in shared memory (ws.H) against H_T,g, all lanes; returns the term in every lane
__device__ double warp_block_gain(const double* __restrict__ ht, WarpScratch& ws, double c, const nbv_config& cfg, const uint8_t* tr,
                                  const uint8_t* tc, int lane) {
  const double ct = cfg.weight_mode == 0 ? c : 1.0;          // Eq. 9 literal (R1) weights H_T as well; R2 / R3 do not
  const double cb = cfg.weight_mode == 1 ? 1.0 : c;          // R2 weights the gain, R1 / R3 the candidate block
  double hreg[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int t = lane + 32 * i;
    hreg[i] = t < NBLK ? ct * ht[t] : 0.0;
    if (t < NBLK) ws.M[t] = hreg[i] + (tr[t] == tc[t] ? (double)cfg.prior_precision[tr[t]] : 0.0);
  }
  warp_ldl14(ws.M, ws.piv0, tr, tc, lane);
  const double t0 = cfg.criterion == NBV_CRIT_TRACE ? warp_inverse_trace14(ws.M, ws.piv0, lane) : 0.0;
  __syncwarp();
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int t = lane + 32 * i;
    if (t < NBLK) ws.M[t] = fma(cb, ws.H[t], hreg[i]) + (tr[t] == tc[t] ? (double)cfg.prior_precision[tr[t]] : 0.0);
  }
  warp_ldl14(ws.M, ws.piv1, tr, tc, lane);
  if (cfg.criterion == NBV_CRIT_TRACE) return t0 - warp_inverse_trace14(ws.M, ws.piv1, lane);   // this Gaussian's reduction of trace(H^-1)
  double gn = lane < P ? log(ws.piv1[lane] / ws.piv0[lane]) : 0.0;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) gn += __shfl_xor_sync(0xffffffffu, gn, o);
  return cfg.weight_mode == 1 ? c * gn : gn;
}

// one entry of the basis change u = L^-T xi (ux = p00 xi1 + p01 xi2, uy = p11 xi2):
//   sum f ux^a uy^b = p11^b sum_t C(a,t) p00^(a-t) p01^t  sum f xi1^(a-t) xi2^(t+b);   src[mono_index(i,j) - off] holds sum f xi1^i xi2^j
__device__ __forceinline__ double ubasis_entry(int a, int b, const double* src, int off, double p00, double p01, double p11) {
  const double binom[5][5] = {{1, 0, 0, 0, 0}, {1, 1, 0, 0, 0}, {1, 2, 1, 0, 0}, {1, 3, 3, 1, 0}, {1, 4, 6, 4, 1}};
  double v = 0.0, pa = 1.0;                 // pa = p01^t
  for (int t = 0; t <= a; ++t) {
    double q = binom[a][t] * pa;
    for (int e = 0; e < a - t; ++e) q *= p00;
    v = fma(q, src[mono_index(a - t, t + b) - off], v);
    pa *= p01;
  }
  for (int e = 0; e < b; ++e) v *= p11;
  return v;
}

__global__ void __launch_bounds__(EXP_T) expand_kernel(const __grid_constant__ SceneDev sc, const __grid_constant__ nbv_config cfg,
                                                        const __grid_constant__ ExpandBatch batch, int mode, int view0,
                                                        double* __restrict__ H_T, const float* __restrict__ conf,
                                                        uint32_t* __restrict__ cache_ids, double* __restrict__ cache_blocks,
                                                        const double* __restrict__ trace_total) {
  __shared__ WarpScratch scratch[EXP_WARPS];
  __shared__ uint8_t tr[NBLK], tc[NBLK];
  __shared__ double wsum[EXP_WARPS];
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  if (threadIdx.x < P) {                                      // packed index -> (row, column)
    int t = tri(threadIdx.x, threadIdx.x);
    for (int c = threadIdx.x; c < P; ++c, ++t) { tr[t] = (uint8_t)threadIdx.x; tc[t] = (uint8_t)c; }
  }
  __syncthreads();
  WarpScratch& ws = scratch[wib];
  const ExpandView& vw = batch.v[view0 + blockIdx.y];
  const uint32_t n_touched = vw.counters->n_touched;
  float omega[4];
#pragma unroll
  for (int c = 0; c < 4; ++c) omega[c] = ((cfg.channel_mask >> c) & 1) ? cfg.channel_weight[c] : 0.f;
  double gain = 0.0;
  for (uint32_t t = blockIdx.x * EXP_WARPS + wib; t < n_touched; t += gridDim.x * EXP_WARPS) {
    const uint32_t r = vw.touched[t];
    const uint32_t g = vw.ids_sorted[r];
    __syncwarp();
    if (lane < NMOM / 4) {
      float4* mom4 = reinterpret_cast<float4*>(vw.moments + (size_t)r * NMOM) + lane;
      const float4 v = *mom4;
      *mom4 = make_float4(0.f, 0.f, 0.f, 0.f);                // leave the buffer zeroed for the next view
      ws.mom[4 * lane] = v.x; ws.mom[4 * lane + 1] = v.y; ws.mom[4 * lane + 2] = v.z; ws.mom[4 * lane + 3] = v.w;
    }
    // the whitening S4 used, from the splat's conic (-2 qa, -qb, -2 qc) = Sigma2D^-1:  u = L^-T xi
    const Splat sp = vw.splat_sorted[r];
    const double cA = -2.0 * (double)sp.qa, cB = -(double)sp.qb, cC = -2.0 * (double)sp.qc, icC = 1.0 / cC;
    const double p00 = sqrt(fmax(cA * cC - cB * cB, 0.0) * icC), p11 = sqrt(cC), p01 = cB * icC * p11;
    __syncwarp();
    if (lane < 15) {                                          // monomial sums: degree n, index j within the degree
      const int n = lane < 1 ? 0 : lane < 3 ? 1 : lane < 6 ? 2 : lane < 10 ? 3 : 4;
      const int j = lane - n * (n + 1) / 2;
      ws.mu[lane] = ubasis_entry(n - j, j, ws.mom, 0, p00, p01, p11);
    }
    if (lane < 20) {                                          // cross moments of channel c: (ux, uy, ux^2, ux uy, uy^2 | 1)
      const int c = lane / 5, e = lane - 5 * c;
      const int ea[5] = {1, 0, 2, 1, 0}, eb[5] = {0, 1, 0, 1, 2};
      ws.mu[MOM_X + 6 * c + e] = ubasis_entry(ea[e], eb[e], ws.mom + MOM_X + 6 * c, 1, p00, p01, p11);
    } else if (lane < 24) {
      ws.mu[MOM_X + 6 * (lane - 20) + 5] = ws.mom[MOM_X + 6 * (lane - 20) + 5];
    } else if (lane == 24) {
      ws.mu[MOM_W2] = ws.mom[MOM_W2];
    }
    // chain rule: the prefix in every lane, column k in lane k; row k of A (14 x 6)
    {
      ChainPrefix<double> pf;
      chain_prefix<double>(vw.cam, sc.mean + 3 * (size_t)g, sc.logscale + 3 * (size_t)g, sc.quat + 4 * (size_t)g, pf);
      if (lane < 10) {
        double col[5];
        chain_column<double>(pf, lane, col);
        ws.A[lane][0] = col[0]; ws.A[lane][1] = col[1]; ws.A[lane][2] = 0.5 * col[2]; ws.A[lane][3] = col[3]; ws.A[lane][4] = 0.5 * col[4];
        ws.A[lane][5] = 0.0;
      } else if (lane == 10) {
        const double sg = (double)sc.sigma[g];
#pragma unroll
        for (int e = 0; e < 5; ++e) ws.A[10][e] = 0.0;
        ws.A[10][5] = cfg.opacity_coord == 0 ? (1.0 - sg) : 1.0 / sg;       // R-10
      } else if (lane < 14) {
        ws.dz[lane - 11] = pf.W[6 + lane - 11];
      }
    }
    __syncwarp();
    {
      const int ex[6] = {1, 0, 2, 1, 0, 0}, ey[6] = {0, 1, 0, 1, 2, 0};
      for (int idx = lane; idx < 66; idx += 32) {             // A Q
        const int k = idx / 6, j = idx - 6 * k;
        double v = 0.0;
#pragma unroll
        for (int i = 0; i < 6; ++i) v = fma(ws.A[k][i], ws.mu[mono_index(ex[i] + ex[j], ey[i] + ey[j])], v);
        ws.AQ[k][j] = v;
      }
      for (int idx = lane; idx < 44; idx += 32) {             // sqrt(omega_ch) A x_ch (S4 delivers x_ch scaled by sqrt(omega_ch))
        const int c = idx / 11, k = idx - 11 * c;
        double v = 0.0;
#pragma unroll
        for (int i = 0; i < 6; ++i) v = fma(ws.A[k][i], ws.mu[MOM_X + 6 * c + i], v);
        ws.yv[c][k] = sqrt((double)omega[c]) * v;
      }
    }
    __syncwarp();
    const double W2 = ws.mu[MOM_W2];
    for (int idx = lane; idx < NBLK; idx += 32) {             // H = A Q A^T + sum_ch [y e^T + e y^T + omega W2 e e^T]
      const int rr = tr[idx], cc = tc[idx];
      double v = 0.0;
      if (cc < 11) {
#pragma unroll
        for (int j = 0; j < 6; ++j) v = fma(ws.AQ[rr][j], ws.A[cc][j], v);
        if (omega[3] != 0.f) {                                // depth: e = (dz/dmu, 0, ...)
          const double ek = rr < 3 ? ws.dz[rr] : 0.0, el = cc < 3 ? ws.dz[cc] : 0.0;
          v += ws.yv[3][rr] * el + ek * ws.yv[3][cc] + (double)omega[3] * W2 * ek * el;
        }
      } else if (rr < 11) {
        v = omega[cc - 11] != 0.f ? ws.yv[cc - 11][rr] : 0.0;  // colour ch: e = unit vector on its parameter
      } else if (rr == cc) {
        v = (double)omega[rr - 11] * W2;
      }
      ws.H[idx] = v;
    }
    __syncwarp();
    if (mode == EXPAND_TRAIN) {
      double* dst = H_T + (size_t)g * NBLK;                   // one launch per view, in view order: a view lists a Gaussian once
      for (int idx = lane; idx < NBLK; idx += 32) dst[idx] += ws.H[idx];
    } else if (mode == EXPAND_VIEW) {
      float* dst = vw.out_blocks + (size_t)g * NBLK;
      for (int idx = lane; idx < NBLK; idx += 32) dst[idx] = (float)ws.H[idx];
    } else if (mode == EXPAND_CACHE) {
      if (t < vw.cache_span[1]) {                              // span[1] = 0 when the pool overflowed: nothing is stored
        const size_t e = (size_t)vw.cache_span[0] + t;
        if (lane == 0) cache_ids[e] = g;
        double* dst = cache_blocks + e * NBLK;
        for (int idx = lane; idx < NBLK; idx += 32) dst[idx] = ws.H[idx];
      }
    } else {
      const double c = (double)conf[g];
      double gn = 0.0;
      if (c > 0.0) gn = warp_block_gain(H_T + (size_t)g * NBLK, ws, c, cfg, tr, tc, lane);   // c_g = 0 (Eq. 12): exactly zero gain
      if (lane == 0 && vw.gains) vw.gains[g] = (float)gn;
      gain += gn;
    }
  }
  if (mode == EXPAND_GAIN) {
    if (lane == 0) wsum[wib] = gain;
    __syncthreads();
    double tot = 0.0;
    if (threadIdx.x == 0)
      for (int w = 0; w < EXP_WARPS; ++w) tot += wsum[w];
    ordered_score(tot, vw.partials, &vw.counters->n_expanded, vw.score, trace_total);
  }
}

static int expand_blocks(int N, int n_views) {
  int blocks = (N + EXP_WARPS - 1) / EXP_WARPS;
  const int cap = (sm_count() * 8 + n_views - 1) / n_views;
  return std::max(1, std::min(blocks, cap));
}
int expand_partials() { return sm_count() * 8; }

void launch_expand(const SceneDev& sc, const nbv_config& cfg, const ExpandBatch& batch, int mode, double* H_T, const float* conf,
                   const double* trace_total, cudaStream_t st) {
  if (mode == EXPAND_TRAIN) {
    // H_T += H(view), view after view (Eq. 6): a fixed order of binary64 additions, no atomics
    const int blocks = expand_blocks(sc.N, 1);
    for (int v = 0; v < batch.n; ++v) {
      ++g_kernel_launches;
      expand_kernel<<<dim3((unsigned)blocks, 1u), EXP_T, 0, st>>>(sc, cfg, batch, mode, v, H_T, conf, nullptr, nullptr, nullptr);
    }
    return;
  }
  ++g_kernel_launches;
  expand_kernel<<<dim3((unsigned)expand_blocks(sc.N, batch.n), (unsigned)batch.n), EXP_T, 0, st>>>(
      sc, cfg, batch, mode, 0, H_T, conf, nullptr, nullptr, cfg.criterion == NBV_CRIT_TRACE ? trace_total : nullptr);
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
                                                                                                     nullptr, cache.ids, cache.blocks, nullptr);
}

// One warp per cached (candidate, Gaussian) entry: the gain of Eq. 5/6/9 of that block against the current H_T,g.
constexpr int CG_BLOCKS = 64;
__global__ void __launch_bounds__(EXP_T) cached_gain_kernel(BlockCache cache, const __grid_constant__ nbv_config cfg,
                                                            const int32_t* __restrict__ taken, const float* __restrict__ conf,
                                                            const double* __restrict__ H_T, float* __restrict__ scores,
                                                            double* __restrict__ partials, unsigned int* __restrict__ done,
                                                            const double* __restrict__ trace_total) {
  __shared__ WarpScratch scratch[EXP_WARPS];
  __shared__ uint8_t tr[NBLK], tc[NBLK];
  __shared__ double wsum[EXP_WARPS];
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  if (threadIdx.x < P) {
    int t = tri(threadIdx.x, threadIdx.x);
    for (int c = threadIdx.x; c < P; ++c, ++t) { tr[t] = (uint8_t)threadIdx.x; tc[t] = (uint8_t)c; }
  }
  __syncthreads();
  WarpScratch& ws = scratch[wib];
  const int c = blockIdx.y;
  double gain = 0.0;
  if (!taken[c]) {
    const uint32_t base = cache.spans[2 * c], cnt = cache.spans[2 * c + 1];
    for (uint32_t t = blockIdx.x * EXP_WARPS + wib; t < cnt; t += gridDim.x * EXP_WARPS) {
      const size_t e = (size_t)base + t;
      const uint32_t g = cache.ids[e];
      const double cg = (double)conf[g];
      if (!(cg > 0.0)) continue;
      __syncwarp();
      for (int idx = lane; idx < NBLK; idx += 32) ws.H[idx] = cache.blocks[e * NBLK + idx];
      __syncwarp();
      gain += warp_block_gain(H_T + (size_t)g * NBLK, ws, cg, cfg, tr, tc, lane);
    }
  }
  if (lane == 0) wsum[wib] = gain;
  __syncthreads();
  double tot = 0.0;
  if (threadIdx.x == 0)
    for (int w = 0; w < EXP_WARPS; ++w) tot += wsum[w];
  ordered_score(tot, partials + (size_t)c * CG_BLOCKS, done + c, scores + c, trace_total);
}

size_t cached_gain_scratch_bytes(int n_cand) { return (size_t)n_cand * (CG_BLOCKS * sizeof(double) + sizeof(unsigned int)); }

void launch_cached_gain(const BlockCache& cache, const nbv_config& cfg, int n_cand, const int32_t* taken, const float* conf,
                        const double* H_T, float* scores, void* scratch, const double* trace_total, cudaStream_t st) {
  ++g_kernel_launches;
  double* partials = reinterpret_cast<double*>(scratch);
  unsigned int* done = reinterpret_cast<unsigned int*>(partials + (size_t)n_cand * CG_BLOCKS);     // zero on entry, zero on exit
  cached_gain_kernel<<<dim3(CG_BLOCKS, (unsigned)n_cand), EXP_T, 0, st>>>(cache, cfg, taken, conf, H_T, scores, partials, done,
                                                                          cfg.criterion == NBV_CRIT_TRACE ? trace_total : nullptr);
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

// trace criterion: S_T = sum over ALL Gaussians of trace((c_g H_T,g + Lambda)^-1), once per scoring call, summed in a fixed
// order (thread -> block -> block order).  scratch: TRACE_BLOCKS doubles + 1 counter (zero on entry) ; out: 1 double
constexpr int TRACE_BLOCKS = 592;
__global__ void __launch_bounds__(64) trace_total_kernel(int N, const __grid_constant__ nbv_config cfg, const double* __restrict__ H_T,
                                                            const float* __restrict__ conf, double* __restrict__ partials,
                                                            unsigned int* __restrict__ done, double* __restrict__ out) {
  __shared__ double ws[2];
  double prior_only = 0.0;
  for (int k = 0; k < P; ++k) prior_only += 1.0 / (double)cfg.prior_precision[k];
  double acc = 0.0;
  for (int g = blockIdx.x * blockDim.x + threadIdx.x; g < N; g += gridDim.x * blockDim.x) {
    const double c = (double)conf[g];
    if (!(c > 0.0)) { acc += prior_only; continue; }          // c_g = 0: the block is the prior alone
    double A[NBLK];
    const double* ht = H_T + (size_t)g * NBLK;
    for (int i = 0; i < NBLK; ++i) A[i] = c * ht[i];
    for (int k = 0; k < P; ++k) A[tri(k, k)] += (double)cfg.prior_precision[k];
    acc += ldl_inverse_trace(A);
  }
  const double tot = block_sum<64>(acc, ws);
  ordered_score(tot, partials, done, nullptr, nullptr, out);
}
size_t trace_total_scratch_bytes() { return TRACE_BLOCKS * sizeof(double) + 16; }
void launch_trace_total(const SceneDev& sc, const nbv_config& cfg, const double* H_T, const float* conf, void* scratch, double* out,
                        cudaStream_t st) {
  ++g_kernel_launches;
  double* partials = reinterpret_cast<double*>(scratch);
  unsigned int* done = reinterpret_cast<unsigned int*>(partials + TRACE_BLOCKS);
  trace_total_kernel<<<TRACE_BLOCKS, 64, 0, st>>>(sc.N, cfg, H_T, conf, partials, done, out);
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
