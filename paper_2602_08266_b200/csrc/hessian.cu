// hessian.cu -- S5 (moments -> 14x14 block), S0' (confidence), S6 (log-det gain), S7 (arg-max) of colour / depth contexts.
//
// S5: for a Gaussian touched by the view, the 40 screen-space moments of S4 become
//       H_g = A Q A^T + sum_ch omega_ch [ (A x_ch) e_ch^T + e_ch (A x_ch)^T + W2 e_ch e_ch^T ]          (block_math.cuh)
//     PAPER.md L189-191 (H ~= J^T J), L210 (per-Gaussian blocks), L248.
// S6: IG_g = log det(c_g (H_T,g + H_c,g) + Lambda) - log det(c_g H_T,g + Lambda)   (Eq. 5, 6, 9; R-13, R-14)
//     as the difference of the pivots of two L D L^T factorisations, sum_j log(d1_j / d0_j).
// PRECISION: everything after S4's binary32 per-tile moment sums is binary64 -- their sum across tiles, the chain rule, A Q A^T, H_T itself, the two
//     factorisations.  A block has exact null directions (R-10; single-view blocks have rank ~8 of 14) next to entries of
//     1e5-1e7: in binary32 the product A Q A^T and the storage of H_T alone leave rounding noise of eps H_kk ~ 0.1-1 on
//     pivots whose exact value is the prior, which is what limited round 1 to Lambda = 1 and 5e-3 on single gains.  In
//     binary64 the null spaces survive to 1e-9 and the plain difference form is accurate to ~1e-13 / gain.  The work is
//     ~2.5 kflop (binary64) per touched Gaussian, 1-2% of a view.
// DETERMINISM: the touched list is built in rank order (touched_count / touched_write), a thread's partial gain and a block's
//     partial score depend only on (view, block), and the last block of a view adds the partials in block order; H_T is
//     accumulated view by view without atomics.  What is left run-to-run is the order of S4's
//     `red.global.add.f64` across tiles, whose addends (widened binary32) sum exactly in binary64 for any realistic footprint.
#include <algorithm>
#include <cstdlib>

#include "block_math.cuh"
#include "kernels.h"

namespace nbv {

// ---- ordered touched list: the ranks S4 flagged (RasterView::touched_flag: it added moments to them, i.e. the Gaussians
// with at least one composited pixel, sum w^2 != 0), in increasing rank (= depth) order.  Pass 1 counts per block of 256 ranks, pass 2 offsets every block
// by the counts before it (each block sums them itself: at most a few thousand numbers) and writes its ranks in order.
constexpr int TOUCH_T = 256;

__global__ void __launch_bounds__(TOUCH_T) touched_count_kernel(const __grid_constant__ RasterBatch batch, int N) {
  const RasterView& vw = batch.v[blockIdx.y];
  const int r = blockIdx.x * TOUCH_T + threadIdx.x;
  const bool hit = r < N && vw.touched_flag[r] != 0;
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
  const bool hit = r < N && vw.touched_flag[r] != 0;
  if (hit) vw.touched_flag[r] = 0;                          // this is the last reader: all-zero again for the next view
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

// ---- S5 + S6, ONE THREAD PER TOUCHED GAUSSIAN, the 105-double blocks in shared memory.
// Two earlier versions -- one thread per Gaussian with its arrays in local memory, then one warp per Gaussian with the
// chain rule computed redundantly in every lane and dynamically indexed per-thread scratch -- both spent their time waiting
// on LOCAL memory (ncu, profiles/r2b_ncu_expand.md: long-scoreboard 18.7 of 26 stall cycles per issue, 870k local stores per
// view) and took 0.57 ms per 8-view batch for ~3e8 binary64 operations.  Here every array a thread indexes lives either in
// registers with compile-time indices (all loops fully unrolled) or in shared memory: a block of 64 threads owns two
// 64 x 105 binary64 arrays S0, S1 (row stride 105, odd: the 16 lanes of a 64-bit shared-memory phase hit 16 different
// bank pairs).  A thread builds its Gaussian's block into its row of S1 (its row of S0 holds the 11 x 6 chain matrix A
// meanwhile); then, per mode, the block stores the rows cooperatively and coalesced (TRAIN / VIEW / CACHE) or loads
// c H_T + Lambda into S0 and c (H_T + H) + Lambda into S1 the same way and every thread factors its two rows in place
// (GAIN): two interleaved right-looking L D L^T with the pivot row in registers.
constexpr int TPG = 64;                              // threads = Gaussians per block
constexpr int TPG_SMEM = 2 * TPG * NBLK * 8;         // bytes of dynamic shared memory

__device__ __forceinline__ double binom_d(int n, int k) {     // folds to a constant after unrolling
  return (k == 0 || k == n) ? 1.0 : (n == 2) ? 2.0 : (n == 3) ? 3.0 : (k == 2) ? 6.0 : 4.0;
}

// S4's 40 moments (whitened basis xi = L^-1 d) -> the u basis (u = L^-T xi: ux = p00 xi1 + p01 xi2, uy = p11 xi2):
//   sum f ux^a uy^b = p11^b sum_t C(a,t) p00^(a-t) p01^t  sum f xi1^(a-t) xi2^(t+b)
__device__ __forceinline__ void moments_whitened_to_u(const double (&m)[NMOM], double p00, double p01, double p11, double (&u)[NMOM]) {
  double P0[5], P1[5], P2[5];
  P0[0] = P1[0] = P2[0] = 1.0;
#pragma unroll
  for (int e = 1; e < 5; ++e) { P0[e] = P0[e - 1] * p00; P1[e] = P1[e - 1] * p01; P2[e] = P2[e - 1] * p11; }
#pragma unroll
  for (int n = 0; n <= 4; ++n)
#pragma unroll
    for (int b = 0; b <= n; ++b) {
      const int a = n - b;
      double v = 0.0;
#pragma unroll
      for (int t = 0; t <= a; ++t) v = fma(binom_d(a, t) * P0[a - t] * P1[t], m[mono_index(a - t, t + b)], v);
      u[mono_index(a, b)] = v * P2[b];
    }
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    const int o = MOM_X + 6 * c;               // (xi1, xi2, xi1^2, xi1 xi2, xi2^2, 1) -> (ux, uy, ux^2, ux uy, uy^2, 1)
    u[o + 0] = fma(p00, m[o + 0], p01 * m[o + 1]);
    u[o + 1] = p11 * m[o + 1];
    u[o + 2] = fma(P0[2], m[o + 2], fma(2.0 * p00 * p01, m[o + 3], P1[2] * m[o + 4]));
    u[o + 3] = p11 * fma(p00, m[o + 3], p01 * m[o + 4]);
    u[o + 4] = P2[2] * m[o + 4];
    u[o + 5] = m[o + 5];
  }
  u[MOM_W2] = m[MOM_W2];
}

// structural non-zeros of A (11 x 6): position rows use (ux, uy, ux^2, ux uy, uy^2), log-scale and quaternion rows only the
// quadratic monomials (they move Sigma2D, not the centre), the opacity row only the constant
__device__ __forceinline__ constexpr bool a_nz(int k, int i) { return k < 3 ? i < 5 : k < 10 ? (i >= 2 && i < 5) : i == 5; }

// S5 of one Gaussian: moments + chain rule -> packed 14 x 14 block H (row `Hrow` of S1); `Arow` (66 doubles) is scratch
__device__ __forceinline__ void tpg_build_block(const SceneDev& sc, const nbv_config& cfg, const ExpandView& vw, uint32_t r, uint32_t g,
                                                const float (&omega)[4], double* __restrict__ Arow, double* __restrict__ Hrow) {
  double u[NMOM];
  {
    double m[NMOM];
    double2* mom2 = reinterpret_cast<double2*>(vw.moments + (size_t)r * NMOM);
#pragma unroll
    for (int q = 0; q < NMOM / 2; ++q) {
      const double2 v = mom2[q];
      mom2[q] = make_double2(0.0, 0.0);                       // leave the buffer zeroed for the next view
      m[2 * q] = v.x; m[2 * q + 1] = v.y;
    }
    // the whitening S4 used, from the splat's conic (-2 qa, -qb, -2 qc) = Sigma2D^-1
    const float4 s0 = *reinterpret_cast<const float4*>(vw.splat_sorted + r);
    const float4 s1 = *(reinterpret_cast<const float4*>(vw.splat_sorted + r) + 1);
    const double cA = -2.0 * (double)s0.z, cB = -(double)s0.w, cC = -2.0 * (double)s1.x, icC = 1.0 / cC;
    const double p00 = sqrt(fmax(cA * cC - cB * cB, 0.0) * icC), p11 = sqrt(cC), p01 = cB * icC * p11;
    moments_whitened_to_u(m, p00, p01, p11, u);
  }
  double dz[3];
  {
    ChainPrefix<double> pf;
    chain_prefix<double>(vw.cam, sc.mean + 3 * (size_t)g, sc.logscale + 3 * (size_t)g, sc.quat + 4 * (size_t)g, pf);
#pragma unroll
    for (int k = 0; k < 10; ++k) {
      double col[5];
      chain_column<double>(pf, k, col);
      if (k < 3) { Arow[6 * k + 0] = col[0]; Arow[6 * k + 1] = col[1]; }
      Arow[6 * k + 2] = 0.5 * col[2]; Arow[6 * k + 3] = col[3]; Arow[6 * k + 4] = 0.5 * col[4];
    }
    const double sg = (double)sc.sigma[g];
    Arow[6 * 10 + 5] = cfg.opacity_coord == 0 ? (1.0 - sg) : 1.0 / sg;       // R-10
#pragma unroll
    for (int k = 0; k < 3; ++k) dz[k] = pf.W[6 + k];
  }
  const int ex[6] = {1, 0, 2, 1, 0, 0}, ey[6] = {0, 1, 0, 1, 2, 0};
  const double W2 = u[MOM_W2];
  const bool depth = omega[3] != 0.f;
  // y_3[l] = sqrt(omega_3) A x_3 (depth channel; S4 delivers x_ch scaled by sqrt(omega_ch)): needed for every l by the rows k < 3
  double y3[11];
  if (depth) {
    const double som = sqrt((double)omega[3]);
#pragma unroll
    for (int l = 0; l < 11; ++l) {
      double v = 0.0;
#pragma unroll
      for (int i = 0; i < 6; ++i)
        if (a_nz(l, i)) v = fma(Arow[6 * l + i], u[MOM_X + 18 + i], v);
      y3[l] = som * v;
    }
  }
#pragma unroll
  for (int k = 0; k < 11; ++k) {
    double ak[6], aq[6];
#pragma unroll
    for (int i = 0; i < 6; ++i) ak[i] = a_nz(k, i) ? Arow[6 * k + i] : 0.0;
#pragma unroll
    for (int j = 0; j < 6; ++j) {                               // row k of A Q
      double v = 0.0;
#pragma unroll
      for (int i = 0; i < 6; ++i)
        if (a_nz(k, i)) v = fma(ak[i], u[mono_index(ex[i] + ex[j], ey[i] + ey[j])], v);
      aq[j] = v;
    }
#pragma unroll
    for (int l = k; l < 11; ++l) {                              // H = A Q A^T + sum_ch [y e^T + e y^T + omega W2 e e^T]
      double v = 0.0;
#pragma unroll
      for (int j = 0; j < 6; ++j)
        if (a_nz(l, j)) v = fma(aq[j], l == k ? ak[j] : Arow[6 * l + j], v);
      if (depth && k < 3) {                                     // depth: e = (dz/dmu, 0, ...)
        const double el = l < 3 ? dz[l] : 0.0;
        v += y3[k] * el + dz[k] * y3[l] + (double)omega[3] * W2 * dz[k] * el;
      }
      Hrow[tri(k, l)] = v;
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {                               // colour ch: e = unit vector on its parameter
      double v = 0.0;
      if (omega[c] != 0.f) {
#pragma unroll
        for (int i = 0; i < 6; ++i)
          if (a_nz(k, i)) v = fma(ak[i], u[MOM_X + 6 * c + i], v);
        v *= sqrt((double)omega[c]);
      }
      Hrow[tri(k, 11 + c)] = v;
    }
  }
#pragma unroll
  for (int c = 0; c < 3; ++c)
#pragma unroll
    for (int d = c; d < 3; ++d) Hrow[tri(11 + c, 11 + d)] = c == d ? (double)omega[c] * W2 : 0.0;
}

// S6 on the thread's two rows: a0 = c H_T + Lambda, a1 = c (H_T + H) + Lambda (packed, destroyed).  Two interleaved
// right-looking L D L^T; the pivot ratios d1_j / d0_j are multiplied up in two halves (each ratio is >= 1 up to rounding
// and far below 1e20, so neither product leaves binary64 range) and enter as two logarithms.  A compiler barrier after every
// row update keeps the rows in shared memory: without it the whole packed block is promoted to registers across the
// unrolled pivot steps and spilled to local memory (2.4 KB of spill stores per thread); `volatile` rows avoid that too but
// serialise every load behind the previous store (85 us per chunk).  The row pointers are deliberately not __restrict__
// (the barrier would not apply to them).
// TRACE: this Gaussian's reduction of trace(H^-1) instead, from the same factors.
__device__ __forceinline__ double tpg_inverse_trace(const double* a) {
  // a = the rows U_j = d_j L_j^T left by the elimination; A^-1 = L^-T D^-1 L^-1, trace = sum_c sum_i x_i^2 / d_i, x = L^-1 e_c
  double inv[P];
#pragma unroll
  for (int j = 0; j < P; ++j) inv[j] = 1.0 / fmax(a[tri(j, j)], 1e-300);
  double tr = 0.0;
#pragma unroll
  for (int c = 0; c < P; ++c) {
    double x[P];
    x[c] = 1.0;
    double acc = inv[c];
#pragma unroll
    for (int i = c + 1; i < P; ++i) {
      double s = 0.0;
#pragma unroll
      for (int j = c; j < i; ++j) s = fma(a[tri(j, i)] * inv[j], x[j], s);
      x[i] = -s;
      acc = fma(s * s, inv[i], acc);
      asm volatile("" ::: "memory");
    }
    tr += acc;
  }
  return tr;
}

template <bool TRACE>
__device__ __forceinline__ double tpg_gain(double* a0, double* a1) {
  double prod_lo = 1.0, prod_hi = 1.0;
#pragma unroll
  for (int j = 0; j < P; ++j) {
    const int jj = tri(j, j);
    double r0[P], r1[P];                        // the pivot rows (compile-time indices: registers)
#pragma unroll
    for (int c = j; c < P; ++c) { r0[c] = a0[jj + c - j]; r1[c] = a1[jj + c - j]; }
    const double d0 = fmax(r0[j], 1e-300), d1 = fmax(r1[j], 1e-300);
    const double i0 = 1.0 / d0;
    if (j < P / 2) prod_lo *= d1 * i0; else prod_hi *= d1 * i0;
    if (j + 1 < P) {
      const double i1 = 1.0 / d1;
#pragma unroll
      for (int r = j + 1; r < P; ++r) {
        const double l0 = -r0[r] * i0, l1 = -r1[r] * i1;
        const int rr = tri(r, r);
#pragma unroll
        for (int c = r; c < P; ++c) {
          a0[rr + c - r] = fma(l0, r0[c], a0[rr + c - r]);
          a1[rr + c - r] = fma(l1, r1[c], a1[rr + c - r]);
        }
        asm volatile("" ::: "memory");
      }
    }
  }
  if (TRACE) return tpg_inverse_trace(a0) - tpg_inverse_trace(a1);
  return log(prod_lo) + log(prod_hi);
}

// Cooperative, coalesced walks over the block's rows: thread t owns the packed entries t and t + 64 of EVERY Gaussian of the
// chunk, so index arithmetic and the prior lookup happen once per thread, and TPG_U Gaussians' loads are in flight at a time
// (H_T is far larger than the L2: a loop that waits for one load per iteration costs a DRAM round trip per Gaussian, 64 of
// them in a row -- measured 46 us per chunk).
constexpr int TPG_U = 8;

// packed index -> prior on the diagonal, 0 elsewhere
__device__ __forceinline__ double prior_of(const nbv_config& cfg, int idx) {
  int r = 0;
#pragma unroll
  for (int q = 1; q < P; ++q) r += idx >= tri(q, q) ? 1 : 0;
  return idx == tri(r, r) ? (double)cfg.prior_precision[r] : 0.0;
}

//   S0 row i = ct H_T,g + Lambda,   S1 row i = S0 row i + cb * S1 row i      (R-14: which of the two the confidence weights)
__device__ __forceinline__ void tpg_load_combine(const double* __restrict__ H_T, const nbv_config& cfg, const uint32_t* gs, const double* cs,
                                                 int n, double* S0, double* S1) {
  const int idx0 = threadIdx.x, idx1 = threadIdx.x + TPG;
  const bool has1 = idx1 < NBLK;
  const double pr0 = prior_of(cfg, idx0), pr1 = has1 ? prior_of(cfg, idx1) : 0.0;
  for (int i0 = 0; i0 < n; i0 += TPG_U) {
    double h0[TPG_U], h1[TPG_U];
#pragma unroll
    for (int k = 0; k < TPG_U; ++k) {
      const int i = i0 + k;
      h0[k] = h1[k] = 0.0;
      if (i < n && cs[i] > 0.0) {
        const double* ht = H_T + (size_t)gs[i] * NBLK;
        h0[k] = __ldg(ht + idx0);
        if (has1) h1[k] = __ldg(ht + idx1);
      }
    }
#pragma unroll
    for (int k = 0; k < TPG_U; ++k) {
      const int i = i0 + k;
      if (i < n) {
        const double c = cs[i];
        if (c > 0.0) {
          const double ct = cfg.weight_mode == 0 ? c : 1.0;          // Eq. 9 literal (R1) weights H_T as well; R2 / R3 do not
          const double cb = cfg.weight_mode == 1 ? 1.0 : c;          // R2 weights the gain, R1 / R3 the candidate block
          const double m0 = fma(ct, h0[k], pr0);
          S0[i * NBLK + idx0] = m0;
          S1[i * NBLK + idx0] = fma(cb, S1[i * NBLK + idx0], m0);
          if (has1) {
            const double m1 = fma(ct, h1[k], pr1);
            S0[i * NBLK + idx1] = m1;
            S1[i * NBLK + idx1] = fma(cb, S1[i * NBLK + idx1], m1);
          }
        }
      }
    }
  }
}

// H_T rows += S1 rows (training accumulation; one launch per view: a view lists a Gaussian once, plain binary64 additions)
__device__ __forceinline__ void tpg_accumulate(double* __restrict__ H_T, const uint32_t* gs, int n, const double* S1) {
  const int idx0 = threadIdx.x, idx1 = threadIdx.x + TPG;
  const bool has1 = idx1 < NBLK;
  for (int i0 = 0; i0 < n; i0 += TPG_U) {
    double h0[TPG_U], h1[TPG_U];
#pragma unroll
    for (int k = 0; k < TPG_U; ++k) {
      const int i = i0 + k;
      h0[k] = h1[k] = 0.0;
      if (i < n) {
        const double* ht = H_T + (size_t)gs[i] * NBLK;
        h0[k] = ht[idx0];
        if (has1) h1[k] = ht[idx1];
      }
    }
#pragma unroll
    for (int k = 0; k < TPG_U; ++k) {
      const int i = i0 + k;
      if (i < n) {
        double* ht = H_T + (size_t)gs[i] * NBLK;
        ht[idx0] = h0[k] + S1[i * NBLK + idx0];
        if (has1) ht[idx1] = h1[k] + S1[i * NBLK + idx1];
      }
    }
  }
}

template <int MODE, bool TRACE>
__global__ void __launch_bounds__(TPG) expand_kernel(const __grid_constant__ SceneDev sc, const __grid_constant__ nbv_config cfg,
                                                      const __grid_constant__ ExpandBatch batch, int view0, double* __restrict__ H_T,
                                                      const float* __restrict__ conf, uint32_t* __restrict__ cache_ids,
                                                      double* __restrict__ cache_blocks, const double* __restrict__ trace_total) {
  extern __shared__ __align__(16) double tpg_smem[];
  double* S0 = tpg_smem;
  double* S1 = tpg_smem + TPG * NBLK;
  __shared__ uint32_t gs[TPG];
  __shared__ double cs[TPG];
  __shared__ double wsum[TPG / 32];
  const ExpandView& vw = batch.v[view0 + blockIdx.y];
  const uint32_t n_touched = vw.counters->n_touched;
  float omega[4];
#pragma unroll
  for (int c = 0; c < 4; ++c) omega[c] = ((cfg.channel_mask >> c) & 1) ? cfg.channel_weight[c] : 0.f;
  double gain = 0.0;
  for (uint32_t base = blockIdx.x * TPG; base < n_touched; base += gridDim.x * TPG) {
    const int n = (int)min((uint32_t)TPG, n_touched - base);
    const bool valid = (int)threadIdx.x < n;
    uint32_t g = 0;
    __syncthreads();                                          // the previous chunk's rows are no longer read
    if (valid) {
      const uint32_t r = vw.touched[base + threadIdx.x];
      g = vw.ids_sorted[r];
      gs[threadIdx.x] = g;
      if (MODE == EXPAND_GAIN) cs[threadIdx.x] = (double)conf[g];
      tpg_build_block(sc, cfg, vw, r, g, omega, S0 + threadIdx.x * NBLK, S1 + threadIdx.x * NBLK);
    }
    __syncthreads();
    if (MODE == EXPAND_TRAIN) {
      tpg_accumulate(H_T, gs, n, S1);
    } else if (MODE == EXPAND_VIEW) {
      for (int e = threadIdx.x; e < n * NBLK; e += TPG) {
        const int i = e / NBLK;
        vw.out_blocks[(size_t)gs[i] * NBLK + (e - i * NBLK)] = (float)S1[e];
      }
    } else if (MODE == EXPAND_CACHE) {
      // span[1] = 0 when the pool overflowed: nothing is stored
      const uint32_t span0 = vw.cache_span[0], span1 = vw.cache_span[1];
      const int m = base >= span1 ? 0 : (int)min((uint32_t)n, span1 - base);       // consecutive pool entries: one coalesced copy
      if ((int)threadIdx.x < m) cache_ids[(size_t)span0 + base + threadIdx.x] = gs[threadIdx.x];
      double* dst = cache_blocks + ((size_t)span0 + base) * NBLK;
      for (int e = threadIdx.x; e < m * NBLK; e += TPG) dst[e] = S1[e];
    } else {
      tpg_load_combine(H_T, cfg, gs, cs, n, S0, S1);
      __syncthreads();
      double gn = 0.0;
      if (valid) {
        const double c = cs[threadIdx.x];
        if (c > 0.0) {                                          // c_g = 0 (Eq. 12): exactly zero gain
          gn = tpg_gain<TRACE>(S0 + threadIdx.x * NBLK, S1 + threadIdx.x * NBLK);
          if (cfg.weight_mode == 1) gn *= c;
        }
        if (vw.gains) vw.gains[g] = (float)gn;
      }
      gain += gn;
    }
  }
  if (MODE == EXPAND_GAIN) {
    __syncthreads();
    const double tot = block_sum<TPG>(gain, wsum);
    ordered_score(tot, vw.partials, &vw.counters->n_expanded, vw.score, trace_total);
  }
}

// blocks per view: at most two resident blocks per SM over the whole batch, and never more than the partial buffers hold
static int expand_blocks(int N, int n_views) {
  const int blocks = (N + TPG - 1) / TPG;
  const int cap = std::min(expand_partials(), (sm_count() * 2 + n_views - 1) / n_views);
  return std::max(1, std::min(blocks, cap));
}
int expand_partials() { return sm_count() * 8; }

template <int MODE, bool TRACE>
static void launch_expand_mode(dim3 grid, const SceneDev& sc, const nbv_config& cfg, const ExpandBatch& batch, int view0, double* H_T,
                               const float* conf, uint32_t* cache_ids, double* cache_blocks, const double* trace_total, cudaStream_t st) {
  // the attribute is per device and per function; setting it is cheap and idempotent
  if (cudaFuncSetAttribute(expand_kernel<MODE, TRACE>, cudaFuncAttributeMaxDynamicSharedMemorySize, TPG_SMEM) != cudaSuccess) return;
  ++g_kernel_launches;
  expand_kernel<MODE, TRACE><<<grid, TPG, TPG_SMEM, st>>>(sc, cfg, batch, view0, H_T, conf, cache_ids, cache_blocks, trace_total);
}

void launch_expand(const SceneDev& sc, const nbv_config& cfg, const ExpandBatch& batch, int mode, double* H_T, const float* conf,
                   const double* trace_total, cudaStream_t st) {
  if (mode == EXPAND_TRAIN) {
    // H_T += H(view), view after view (Eq. 6): a fixed order of binary64 additions, no atomics
    const dim3 grid((unsigned)expand_blocks(sc.N, 1), 1u);
    for (int v = 0; v < batch.n; ++v)
      launch_expand_mode<EXPAND_TRAIN, false>(grid, sc, cfg, batch, v, H_T, conf, nullptr, nullptr, nullptr, st);
    return;
  }
  const dim3 grid((unsigned)expand_blocks(sc.N, batch.n), (unsigned)batch.n);
  if (mode == EXPAND_VIEW)
    launch_expand_mode<EXPAND_VIEW, false>(grid, sc, cfg, batch, 0, H_T, conf, nullptr, nullptr, nullptr, st);
  else if (cfg.criterion == NBV_CRIT_TRACE)
    launch_expand_mode<EXPAND_GAIN, true>(grid, sc, cfg, batch, 0, H_T, conf, nullptr, nullptr, trace_total, st);
  else
    launch_expand_mode<EXPAND_GAIN, false>(grid, sc, cfg, batch, 0, H_T, conf, nullptr, nullptr, nullptr, st);
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
  const dim3 grid((unsigned)expand_blocks(sc.N, batch.n), (unsigned)batch.n);
  launch_expand_mode<EXPAND_CACHE, false>(grid, sc, cfg, batch, 0, nullptr, nullptr, cache.ids, cache.blocks, nullptr, st);
}

// One thread per cached (candidate, Gaussian) entry: the gain of Eq. 5/6/9 of that block against the current H_T,g
// (the S6 of expand_kernel on blocks read back from the pool instead of rebuilt).
constexpr int CG_BLOCKS = 64;
template <bool TRACE>
__global__ void __launch_bounds__(TPG) cached_gain_kernel(BlockCache cache, const __grid_constant__ nbv_config cfg,
                                                          const int32_t* __restrict__ taken, const float* __restrict__ conf,
                                                          const double* __restrict__ H_T, float* __restrict__ scores,
                                                          double* __restrict__ partials, unsigned int* __restrict__ done,
                                                          const double* __restrict__ trace_total) {
  extern __shared__ __align__(16) double tpg_smem[];
  double* S0 = tpg_smem;
  double* S1 = tpg_smem + TPG * NBLK;
  __shared__ uint32_t gs[TPG];
  __shared__ double cs[TPG];
  __shared__ double wsum[TPG / 32];
  const int c = blockIdx.y;
  double gain = 0.0;
  if (!taken[c]) {
    const uint32_t first = cache.spans[2 * c], cnt = cache.spans[2 * c + 1];
    for (uint32_t base = blockIdx.x * TPG; base < cnt; base += gridDim.x * TPG) {
      const int n = (int)min((uint32_t)TPG, cnt - base);
      __syncthreads();
      if ((int)threadIdx.x < n) {
        const uint32_t g = cache.ids[(size_t)first + base + threadIdx.x];
        gs[threadIdx.x] = g;
        cs[threadIdx.x] = (double)conf[g];
      }
      const double* src = cache.blocks + ((size_t)first + base) * NBLK;            // n consecutive blocks: one coalesced copy
      for (int i = threadIdx.x; i < n * NBLK; i += TPG) S1[i] = src[i];
      __syncthreads();
      tpg_load_combine(H_T, cfg, gs, cs, n, S0, S1);
      __syncthreads();
      if ((int)threadIdx.x < n) {
        const double cg = cs[threadIdx.x];
        if (cg > 0.0) {
          const double gn = tpg_gain<TRACE>(S0 + threadIdx.x * NBLK, S1 + threadIdx.x * NBLK);
          gain += cfg.weight_mode == 1 ? cg * gn : gn;
        }
      }
    }
  }
  __syncthreads();
  const double tot = block_sum<TPG>(gain, wsum);
  ordered_score(tot, partials + (size_t)c * CG_BLOCKS, done + c, scores + c, trace_total);
}

size_t cached_gain_scratch_bytes(int n_cand) { return (size_t)n_cand * (CG_BLOCKS * sizeof(double) + sizeof(unsigned int)); }

void launch_cached_gain(const BlockCache& cache, const nbv_config& cfg, int n_cand, const int32_t* taken, const float* conf,
                        const double* H_T, float* scores, void* scratch, const double* trace_total, cudaStream_t st) {
  ++g_kernel_launches;
  double* partials = reinterpret_cast<double*>(scratch);
  unsigned int* done = reinterpret_cast<unsigned int*>(partials + (size_t)n_cand * CG_BLOCKS);     // zero on entry, zero on exit
  const dim3 grid(CG_BLOCKS, (unsigned)n_cand);
  if (cfg.criterion == NBV_CRIT_TRACE) {
    if (cudaFuncSetAttribute(cached_gain_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, TPG_SMEM) != cudaSuccess) return;
    cached_gain_kernel<true><<<grid, TPG, TPG_SMEM, st>>>(cache, cfg, taken, conf, H_T, scores, partials, done, trace_total);
  } else {
    if (cudaFuncSetAttribute(cached_gain_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, TPG_SMEM) != cudaSuccess) return;
    cached_gain_kernel<false><<<grid, TPG, TPG_SMEM, st>>>(cache, cfg, taken, conf, H_T, scores, partials, done, nullptr);
  }
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
