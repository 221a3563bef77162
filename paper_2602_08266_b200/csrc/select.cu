// select.cu -- view-selection arithmetic on top of the per-view gains.
//   fuse_kernel:   PAPER.md Eq. 10 (L251-257: each output's gain divided by the mean gain of the training views scored
//                  as candidates) and Eq. 11 (L261-265: IG~ = IG~_rgb + beta_d IG~_d + beta_o IG~_o), then the arg-max
//                  of Eq. 5 (lowest index on ties, R-15).
//   greedy_round_kernel: one round of greedy selection -- scatter the scores of the remaining candidates into the
//                  round's row (NaN at already selected candidates) and take the arg-max over the remaining ones.
#include <math_constants.h>

#include "kernels.h"

namespace nbv {

namespace {

constexpr int SEL_T = 256;

// block-wide (value, index) arg-max with lowest index on ties; result valid in thread 0
__device__ void block_argmax(float& bv, int& bi) {
  __shared__ float sv[SEL_T / 32];
  __shared__ int si[SEL_T / 32];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const float ov = __shfl_xor_sync(0xffffffffu, bv, o);
    const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
    if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
  }
  if ((threadIdx.x & 31) == 0) { sv[threadIdx.x >> 5] = bv; si[threadIdx.x >> 5] = bi; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < SEL_T / 32; ++w)
      if (sv[w] > bv || (sv[w] == bv && si[w] < bi)) { bv = sv[w]; bi = si[w]; }
  }
}

__device__ float block_sum(float v) {
  __shared__ float ss[SEL_T / 32];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  if ((threadIdx.x & 31) == 0) ss[threadIdx.x >> 5] = v;
  __syncthreads();
  float t = 0.f;
  for (int w = 0; w < SEL_T / 32; ++w) t += ss[w];
  __syncthreads();
  return t;                                   // same value in every thread
}

}  // namespace

// raw: F x n (rgb row, depth row[, mask row]); train: F x n_train; beta: F weights (beta[0] = 1); denom: F; fused: n; best: 1
__global__ void __launch_bounds__(SEL_T) fuse_kernel(const float* __restrict__ raw, const float* __restrict__ train, int n, int n_train,
                                                     int F, float beta_d, float beta_o, float* __restrict__ denom,
                                                     float* __restrict__ fused, int32_t* __restrict__ best) {
  float den[3] = {1.f, 1.f, 1.f};
  const float beta[3] = {1.f, beta_d, beta_o};
  for (int f = 0; f < F; ++f) {
    float s = 0.f;
    for (int t = threadIdx.x; t < n_train; t += SEL_T) s += train[(size_t)f * n_train + t];
    den[f] = block_sum(s) / (float)n_train;   // Eq. 10 denominator: (1/|T|) sum_t IG_f(T, t)
  }
  if (threadIdx.x < F) denom[threadIdx.x] = den[threadIdx.x];
  float bv = -CUDART_INF_F;
  int bi = 0x7fffffff;
  for (int i = threadIdx.x; i < n; i += SEL_T) {
    float v = 0.f;
    for (int f = 0; f < F; ++f) v += beta[f] * (raw[(size_t)f * n + i] / den[f]);     // Eq. 11
    fused[i] = v;
    if (v > bv || (v == bv && i < bi)) { bv = v; bi = i; }
  }
  block_argmax(bv, bi);
  if (threadIdx.x == 0) *best = bi == 0x7fffffff ? 0 : bi;
}

// remaining[j] (increasing) = original index of the j-th candidate scored this round; tmp[j] its score
__global__ void __launch_bounds__(SEL_T) greedy_round_kernel(const float* __restrict__ tmp, const int32_t* __restrict__ remaining, int m,
                                                             int n, float* __restrict__ row, int32_t* __restrict__ pick) {
  for (int i = threadIdx.x; i < n; i += SEL_T) row[i] = CUDART_NAN_F;
  __syncthreads();
  float bv = -CUDART_INF_F;
  int bi = 0x7fffffff;
  for (int j = threadIdx.x; j < m; j += SEL_T) {
    const float v = tmp[j];
    const int i = remaining[j];
    row[i] = v;
    if (v > bv || (v == bv && i < bi)) { bv = v; bi = i; }
  }
  block_argmax(bv, bi);
  if (threadIdx.x == 0) *pick = bi == 0x7fffffff ? remaining[0] : bi;
}

// device-resident greedy round (nbv_select_greedy with the block cache)
__global__ void __launch_bounds__(SEL_T) greedy_pick_kernel(const float* __restrict__ scores, int32_t* __restrict__ taken, int n,
                                                            float* __restrict__ row, int32_t* __restrict__ pick, int32_t* __restrict__ order_r) {
  float bv = -CUDART_INF_F;
  int bi = 0x7fffffff;
  for (int i = threadIdx.x; i < n; i += SEL_T) {
    const bool tk = taken[i] != 0;
    const float v = scores[i];
    if (row) row[i] = tk ? CUDART_NAN_F : v;
    if (!tk && (v > bv || (v == bv && i < bi))) { bv = v; bi = i; }
  }
  block_argmax(bv, bi);
  if (threadIdx.x == 0) {
    if (bi == 0x7fffffff) {                               // only non-comparable scores left: lowest free index
      for (int i = 0; i < n; ++i)
        if (!taken[i]) { bi = i; break; }
    }
    *pick = bi;
    *order_r = bi;
    taken[bi] = 1;
  }
}

void launch_greedy_pick(const float* scores, int32_t* taken, int n, float* row, int32_t* pick, int32_t* order_r, cudaStream_t st) {
  ++g_kernel_launches;
  greedy_pick_kernel<<<1, SEL_T, 0, st>>>(scores, taken, n, row, pick, order_r);
}

void launch_fuse(const float* raw, const float* train, int n, int n_train, int F, float beta_d, float beta_o, float* denom, float* fused,
                 int32_t* best, cudaStream_t st) {
  ++g_kernel_launches;
  fuse_kernel<<<1, SEL_T, 0, st>>>(raw, train, n, n_train, F, beta_d, beta_o, denom, fused, best);
}

void launch_greedy_round(const float* tmp, const int32_t* remaining, int m, int n, float* row, int32_t* pick, cudaStream_t st) {
  ++g_kernel_launches;
  greedy_round_kernel<<<1, SEL_T, 0, st>>>(tmp, remaining, m, n, row, pick);
}

}  // namespace nbv
