// mask.cu -- the object-mask output (NEXT-2): S5' / S6 on blocks of L = 11 + K parameters, binary64 (as the colour / depth
// contexts, and for the same reason: hessian.cu), one warp per Gaussian.
#include <algorithm>
#include <cstdlib>

#include "block_math.cuh"
#include "kernels.h"

namespace nbv {

// =====================================================================================================================
// Object-mask output (Eq. 1-2 "masks use the object vector").
//   O = sum_i softmax(o_i) alpha_i T_i + e_bg T_end : compositing of the K "colours" p_i = softmax(o_i) over the
//   background colour e_bg.  Block of a Gaussian: L = 11 + K parameters [mu, logscale, quat, opacity | logits].
//   Row of channel k at a pixel:  J_k = beta_k alpha A m6  (+)  w dp_k/do,   dp_k/do_j = p_k (delta_kj - p_j).
// S3 is shared with the other outputs; S4 is the SAME kernel, run once per group of four object channels on a copy of
// the rank-ordered splats whose (r, g, b | z) fields hold (p_t0, p_t1, p_t2 | p_t3); group 0 starts with the background
// channel (the only one with a background term, which the kernel has on its three colour slots).  Every group leaves
// 40 moments per rank: the 15 monomial sums add up over the groups (sum_k beta_k^2), the 6 cross moments x_k per
// channel stay apart.  Then, per touched Gaussian (S5'):
//   geo-geo   (11 x 11)  A Q A^T
//   geo-logit (11 x K)   sum_k (A x_k) dp_k/do_j = p_j (A x_j - sum_k p_k A x_k)
//   logit-logit (K x K)  W2 sum_k dp_k/do_j dp_k/do_l = W2 (delta_jl p_j^2 - p_j p_l (p_j + p_l) + p_j p_l sum_k p_k^2)
// and S6 is the same pivot-ratio log-det gain on L x L blocks.
// =====================================================================================================================
__host__ __device__ __forceinline__ int mask_channel_of_slot(int t, int bgch) { return t == 0 ? bgch : (t <= bgch ? t - 1 : t); }
__host__ __device__ __forceinline__ int mask_slot_of_channel(int c, int bgch) { return c == bgch ? 0 : (c < bgch ? c + 1 : c); }
__device__ __forceinline__ int triL(int r, int c, int L) { return r * L - r * (r - 1) / 2 + (c - r); }
__device__ __forceinline__ int rtri(int r) { return r * (r + 1) / 2; }      // start of row r of a row-major lower triangle

__global__ void __launch_bounds__(256) mask_splat_kernel(const Splat* __restrict__ splat_sorted, const uint32_t* __restrict__ ids_sorted,
                                                         const float* __restrict__ logits, const float* __restrict__ lse, int N, int K,
                                                         int group, int bgch, Splat* __restrict__ out) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= N) return;
  Splat s = splat_sorted[r];
  const uint32_t g = ids_sorted[r];
  float p[4];
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const int t = 4 * group + j;
    p[j] = (g < (uint32_t)N && t < K) ? expf(logits[(size_t)g * K + mask_channel_of_slot(t, bgch)] - lse[g]) : 0.f;
  }
  s.r = p[0]; s.g = p[1]; s.b = p[2]; s.z = p[3];
  out[r] = s;
}

void launch_mask_splats(const SceneDev& sc, const Splat* splat_sorted, const uint32_t* ids_sorted, int group, int bgch, Splat* out,
                        cudaStream_t st) {
  ++g_kernel_launches;
  mask_splat_kernel<<<(sc.N + 255) / 256, 256, 0, st>>>(splat_sorted, ids_sorted, sc.logits, sc.lse, sc.N, sc.K, group, bgch, out);
}

// ---- S5' + S6 of a mask context, warp-cooperative: ONE WARP PER TOUCHED GAUSSIAN, two packed symmetric L x L matrices in
// shared memory (a first version ran one thread per Gaussian over 2 x 2016 floats of local memory).  Lane l builds the columns
// l, l + 32 of the block.  S6 is the pivot-ratio form of the colour / depth contexts: M0 = c H_T + Lambda and
// M1 = c (H_T + H) + Lambda are eliminated side by side (right-looking L D L^T, one column per step, the entries of the
// trailing block dealt to the lanes one by one) and the gain is sum_j log(d1_j / d0_j).  No factor table, nothing cached
// between scoring calls.  K = 20: 12.3 KB per warp, two blocks of 8 warps per SM.
struct MaskWarpLayout {
  int LB;          // packed size of a symmetric L x L matrix
  int per_warp;    // doubles per warp
  int oH, oU, oA, oAQ, oMom, oX, oP, oMono, oPiv;
};
__host__ __device__ inline MaskWarpLayout mask_warp_layout(int K, int groups) {
  MaskWarpLayout m;
  const int L = 11 + K;
  m.LB = L * (L + 1) / 2;
  int o = 0;
  m.oH = o; o += m.LB;
  m.oU = o; o += m.LB;
  m.oA = o; o += 66;
  m.oAQ = o; o += 66;
  m.oMom = o; o += groups * NMOM;
  m.oX = o; o += K * 6;
  m.oP = o; o += K;
  m.oMono = o; o += 16;
  m.oPiv = o; o += 2 * L;
  m.per_warp = (o + 3) & ~3;
  return m;
}

__global__ void __launch_bounds__(256) expand_mask_warp_kernel(const __grid_constant__ SceneDev sc, const __grid_constant__ nbv_config cfg,
                                                                const __grid_constant__ ExpandBatch batch, int mode, int groups, int view0,
                                                                double* __restrict__ H_T, const float* __restrict__ conf) {
  extern __shared__ __align__(16) double smem[];
  const ExpandView& vw = batch.v[view0 + blockIdx.y];
  const int K = sc.K, L = 11 + K, LB = L * (L + 1) / 2, bgch = cfg.mask_bg_channel;
  const MaskWarpLayout lay = mask_warp_layout(K, groups);
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5, wpb = blockDim.x >> 5;
  double* base = smem + (size_t)wib * lay.per_warp;
  double *Hm = base + lay.oH, *Um = base + lay.oU, *As = base + lay.oA, *AQs = base + lay.oAQ, *mom = base + lay.oMom;
  double *xs = base + lay.oX, *ps = base + lay.oP, *mono = base + lay.oMono, *piv = base + lay.oPiv;
  const uint32_t n_touched = vw.counters->n_touched;
  const int stride = NMOM * groups;
  // entry e of the row-major lower triangle -> (row << 8) | column, behind the warps' areas
  uint16_t* tri = reinterpret_cast<uint16_t*>(smem + (size_t)wpb * lay.per_warp);
  for (int i = threadIdx.x; i < L - 1; i += blockDim.x)
    for (int k = 0; k <= i; ++k) tri[i * (i + 1) / 2 + k] = (uint16_t)((i << 8) | k);
  __syncthreads();
  double gain = 0.0;
  for (uint32_t t = blockIdx.x * wpb + wib; t < n_touched; t += gridDim.x * wpb) {
    const uint32_t r = vw.touched[t];
    const uint32_t g = vw.ids_sorted[r];
    __syncwarp();
    // moments of all groups -> shared memory (and zero the buffer for the next view)
    double* gm = vw.moments + (size_t)r * stride;
    for (int i = lane; i < stride; i += 32) { mom[i] = gm[i]; gm[i] = 0.0; }
    __syncwarp();
    {   // whitened basis -> u basis, one lane per group
      const Splat sp = vw.splat_sorted[r];
      for (int gr = lane; gr < groups; gr += 32) {
        double m[NMOM];
#pragma unroll
        for (int i = 0; i < NMOM; ++i) m[i] = mom[gr * NMOM + i];
        whitened_to_u<double>(m, sp);
#pragma unroll
        for (int i = 0; i < NMOM; ++i) mom[gr * NMOM + i] = m[i];
      }
    }
    __syncwarp();
    if (lane < 15) {
      double v = 0.0;
      for (int gr = 0; gr < groups; ++gr) v += mom[gr * NMOM + lane];
      mono[lane] = v;
    }
    if (lane == 15) mono[15] = mom[MOM_W2];
    for (int i = lane; i < K * 6; i += 32) {
      const int slot = i / 6, e = i - 6 * slot;
      xs[i] = mom[(slot >> 2) * NMOM + MOM_X + 6 * (slot & 3) + e];
    }
    double s2p = 0.0;
    for (int slot = lane; slot < K; slot += 32) {
      const double pv = exp(sc.logits[(size_t)g * K + mask_channel_of_slot(slot, bgch)] - sc.lse[g]);
      ps[slot] = pv;
      s2p += pv * pv;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s2p += __shfl_xor_sync(0xffffffffu, s2p, o);
    const double S2 = s2p;
    {   // chain rule (every lane, redundantly), A and A Q into shared memory for dynamic indexing
      Chain<double> ch;
      projection_chain<double>(vw.cam, sc.mean + 3 * (size_t)g, sc.logscale + 3 * (size_t)g, sc.quat + 4 * (size_t)g, ch);
      const double sg = sc.sigma[g];
      const double kappa = cfg.opacity_coord == 0 ? (1.0 - sg) : 1.0 / sg;       // R-10
      if (lane < 11) {
        double a6[6];
        if (lane < 10) {
          a6[0] = ch.G[0][lane]; a6[1] = ch.G[1][lane]; a6[2] = 0.5 * ch.G[2][lane]; a6[3] = ch.G[3][lane]; a6[4] = 0.5 * ch.G[4][lane]; a6[5] = 0.0;
        } else {
          a6[0] = a6[1] = a6[2] = a6[3] = a6[4] = 0.0; a6[5] = kappa;
        }
#pragma unroll
        for (int e = 0; e < 6; ++e) As[lane * 6 + e] = a6[e];
      }
    }
    __syncwarp();
    if (lane < 11) {
      const int ex[6] = {1, 0, 2, 1, 0, 0}, ey[6] = {0, 1, 0, 1, 2, 0};
      for (int j = 0; j < 6; ++j) {
        double v = 0.0;
        for (int i = 0; i < 6; ++i) v += As[lane * 6 + i] * mono[mono_index(ex[i] + ex[j], ey[i] + ey[j])];
        AQs[lane * 6 + j] = v;
      }
    }
    __syncwarp();
    const double W2 = mono[15];
    double xbar[6];
#pragma unroll
    for (int e = 0; e < 6; ++e) {
      double v = 0.0;
      for (int slot = 0; slot < K; ++slot) v += ps[slot] * xs[slot * 6 + e];
      xbar[e] = v;
    }
    // the upper triangle of the block, column j by lane j (and j + 32), in REVERSED packed storage: entry (i, j >= i) sits at
    // r (r + 1) / 2 + c with r = L - 1 - i, c = L - 1 - j.  In that order the trailing block of elimination step j is the prefix
    // [0, m (m + 1) / 2), m = L - 1 - j, of the array, the pivot row follows it directly, and an entry's address is its number.
    for (int j = lane; j < L; j += 32) {
      const int cj = L - 1 - j;
      if (j < 11) {
        for (int i = 0; i <= j; ++i) {
          double v = 0.0;
#pragma unroll
          for (int e = 0; e < 6; ++e) v += AQs[i * 6 + e] * As[j * 6 + e];
          Hm[rtri(L - 1 - i) + cj] = v;
        }
      } else {
        const int c = j - 11, slot = mask_slot_of_channel(c, bgch);
        const double pc = ps[slot];
        for (int i = 0; i < 11; ++i) {
          double v = 0.0;
#pragma unroll
          for (int e = 0; e < 6; ++e) v += As[i * 6 + e] * (pc * (xs[slot * 6 + e] - xbar[e]));
          Hm[rtri(L - 1 - i) + cj] = v;
        }
        for (int d = 0; d <= c; ++d) {
          const double pd = ps[mask_slot_of_channel(d, bgch)];
          double v = pc * pd * (S2 - pc - pd);
          if (d == c) v += pc * pc;
          Hm[rtri(L - 12 - d) + cj] = W2 * v;
        }
      }
    }
    __syncwarp();
    if (mode == EXPAND_TRAIN || mode == EXPAND_VIEW) {
      for (int rr = 0; rr < L; ++rr)
        for (int c = rr + lane; c < L; c += 32) {
          const size_t o = (size_t)g * LB + triL(rr, c, L);
          const double v = Hm[rtri(L - 1 - rr) + L - 1 - c];
          if (mode == EXPAND_TRAIN) H_T[o] += v;                  // one launch per view, in view order
          else vw.out_blocks[o] = (float)v;
        }
      continue;
    }
    const double cg = conf[g];
    const double ct = cfg.weight_mode == 0 ? cg : 1.0;        // Eq. 9 literal (R1) weights H_T as well; R2 / R3 do not
    const double cb = cfg.weight_mode == 1 ? 1.0 : cg;        // R2 weights the gain, R1 / R3 the candidate block
    double gn = 0.0;
    if (cg > 0.0) {
      // M0 = ct H_T + Lambda -> Um,  M1 = M0 + cb H -> Hm  (H_T is stored packed upper, row-major)
      const double* ht = H_T + (size_t)g * LB;
      for (int rr = 0; rr < L; ++rr) {
        const double pr = rr < 11 ? (double)cfg.prior_precision[rr] : (double)cfg.prior_precision_obj;
        const int rb = rtri(L - 1 - rr) + L - 1;
        for (int c = rr + lane; c < L; c += 32) {
          const double m0 = fma(ct, ht[triL(rr, c, L)], c == rr ? pr : 0.0);
          Um[rb - c] = m0;
          Hm[rb - c] = fma(cb, Hm[rb - c], m0);
        }
      }
      __syncwarp();
      // two interleaved right-looking L D L^T; the gain is the sum of log(d1_j / d0_j) over the pivots, as in the colour /
      // depth contexts (hessian.cu): 2 x L^3 / 6 multiply-adds instead of the two L^3 / 2 triangular solves + a Cholesky of
      // the solve form used while this path was binary32.  Step j: pivot row = entries [n, n + m] of the array (n = m (m + 1)
      // / 2), trailing block = entries [0, n), dealt to the lanes entry by entry through `tri` (entry -> (row, column)): a lane
      // per ROW left the lanes with 1 ... m entries each and the warp waiting for the longest row, 3 x the serial length.
      for (int j = 0; j < L; ++j) {
        const int m = L - 1 - j, n = m * (m + 1) / 2;
        const double *v0 = Um + n, *v1 = Hm + n;
        const double d0 = fmax(v0[m], 1e-300), d1 = fmax(v1[m], 1e-300);
        if (lane == 0) { piv[j] = d0; piv[L + j] = d1; }
        const double i0 = -1.0 / d0, i1 = -1.0 / d1;
#pragma unroll 2
        for (int e = lane; e < n; e += 32) {
          const int rc = tri[e], r = rc >> 8, c = rc & 255;
          Um[e] = fma(v0[r] * i0, v0[c], Um[e]);
          Hm[e] = fma(v1[r] * i1, v1[c], Hm[e]);
        }
        __syncwarp();
      }
      for (int j = lane; j < L; j += 32) gn += log(piv[L + j] / piv[j]);
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) gn += __shfl_xor_sync(0xffffffffu, gn, o);
    }
    if (cfg.weight_mode == 1) gn *= cg;
    if (lane == 0) {
      if (vw.gains) vw.gains[g] = gn;
      gain += gn;
    }
  }
  if (mode == EXPAND_GAIN) {
    __shared__ double ws[8];
    if (lane == 0) ws[wib] = gain;
    __syncthreads();
    double tsum = 0.0;
    if (threadIdx.x == 0)
      for (int w = 0; w < wpb; ++w) tsum += (double)ws[w];
    ordered_score(tsum, vw.partials, &vw.counters->n_expanded, vw.score);    // block partials added in block order
  }
}

void launch_expand_mask(const SceneDev& sc, const nbv_config& cfg, const ExpandBatch& batch, int mode, int groups, double* H_T,
                        const float* conf, cudaStream_t st) {
  const MaskWarpLayout lay = mask_warp_layout(sc.K, groups);
  int wpb = 8;
  while (wpb > 1 && (size_t)wpb * lay.per_warp * 8 > 108 * 1024) wpb >>= 1;        // two blocks per SM
  const int L = 11 + sc.K;
  const size_t smem = (size_t)wpb * lay.per_warp * 8 + (((size_t)L * (L - 1) / 2 * 2 + 15) & ~(size_t)15);
  // the attribute is per device and per function: set it whenever the launch needs more than the default 48 KB
  if (smem > 48 * 1024 &&
      cudaFuncSetAttribute(expand_mask_warp_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return;                                           // the caller's cudaGetLastError() reports it
  if (mode == EXPAND_TRAIN) {
    const int blocks = sm_count() * 2;
    for (int v = 0; v < batch.n; ++v) {
      ++g_kernel_launches;
      expand_mask_warp_kernel<<<dim3((unsigned)blocks, 1u), wpb * 32, smem, st>>>(sc, cfg, batch, mode, groups, v, H_T, conf);
    }
    return;
  }
  ++g_kernel_launches;
  const int blocks = std::max(1, (sm_count() * 2 + batch.n - 1) / batch.n);
  expand_mask_warp_kernel<<<dim3((unsigned)blocks, (unsigned)batch.n), wpb * 32, smem, st>>>(sc, cfg, batch, mode, groups, 0, H_T, conf);
}

// parity export: (rgb | depth) images of one group's forward pass -> mask channels of that group
__global__ void __launch_bounds__(256) mask_scatter_kernel(const float* __restrict__ rgb, const float* __restrict__ depth, size_t npx, int K,
                                                            int group, int bgch, float* __restrict__ mask) {
  const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= npx) return;
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const int t = 4 * group + j;
    if (t < K) mask[p * K + mask_channel_of_slot(t, bgch)] = j < 3 ? rgb[3 * p + j] : depth[p];
  }
}

void launch_mask_scatter(const float* rgb, const float* depth, size_t npx, int K, int group, int bgch, float* mask, cudaStream_t st) {
  ++g_kernel_launches;
  mask_scatter_kernel<<<(unsigned)((npx + 255) / 256), 256, 0, st>>>(rgb, depth, npx, K, group, bgch, mask);
}

}  // namespace nbv
