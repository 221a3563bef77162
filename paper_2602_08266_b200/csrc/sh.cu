// sh.cu -- view-dependent colour, SH degree 3 ("SH coefficients c in
// R^{3(d+1)^2}", L166 "raising the SH degree back to 3"; reading R-18 in DESIGN.md).
//
//   colour_ch(dir) = rgb_ch + sum_{j=1}^{15} B_j(dir) k_{j,ch},  dir = (mu - o) / |mu - o|,  o = camera centre
//   block of a Gaussian: L = 59 parameters [mu(3) logscale(3) quat(4) opacity | rgb(3) | k_1(3) .. k_15(3)]
//
// S1 evaluates the colour per (view, Gaussian) and hands it to S3 / S4 in the splat record, so the raster kernels and the 40
// moments are exactly those of the degree-0 path: per pixel the colour row is  J_ch = beta_ch alpha A m6 + w e_ch  with a
// per-(view, Gaussian) constant vector e_ch = dcolour_ch/dtheta (three position entries: the colour moves with the viewing
// direction; sixteen coefficient entries B_j, B_0 = 1), just as the depth row has e_D = (dz/dmu, 0...).  Hence
//   H = G + sum_ch [ y_ch e_ch^T + e_ch y_ch^T + omega_ch W2 e_ch e_ch^T ],   G = A Q A^T (11 x 11),  y_ch = sqrt(omega_ch) A x_ch,
// and S5' builds the 59 x 59 block from the same moments.  S6 is the pivot-ratio log-det of two L D L^T factorisations
// (c H_T + Lambda and c (H_T + H_c) + Lambda), binary64, ONE WARP PER TOUCHED GAUSSIAN with both matrices in shared memory.
#include <algorithm>

#include "block_math.cuh"
#include "kernels.h"

namespace nbv {

constexpr int SH_NB = 16;
constexpr int SH_L = NBV_SH_L;                      // 59
constexpr int SH_LB = SH_L * (SH_L + 1) / 2;        // 1770

__host__ __device__ __forceinline__ constexpr int triS(int r, int c) { return r * SH_L - r * (r - 1) / 2 + (c - r); }

// real spherical harmonics of degree 1..3 at a unit direction, 3DGS ordering and signs (B[0] = 1: the stored rgb), and
// their gradients in free (x, y, z)
template <class T>
__device__ void sh_basis(T x, T y, T z, T* B, T (*dB)[3]) {
  const T c1 = (T)0.48860251190291992, c2a = (T)1.0925484305920792, c2b = (T)0.31539156525252005, c2c = (T)0.54627421529603959;
  const T c3a = (T)0.59004358992664352, c3b = (T)2.8906114426405538, c3c = (T)0.45704579946446572, c3d = (T)0.3731763325901154,
          c3e = (T)1.4453057213202769;
  const T xx = x * x, yy = y * y, zz = z * z;
#define SH_SET(j, v, gx, gy, gz) { B[j] = (v); if (dB) { dB[j][0] = (gx); dB[j][1] = (gy); dB[j][2] = (gz); } }
  SH_SET(0, (T)1, (T)0, (T)0, (T)0)
  SH_SET(1, -c1 * y, (T)0, -c1, (T)0)
  SH_SET(2, c1 * z, (T)0, (T)0, c1)
  SH_SET(3, -c1 * x, -c1, (T)0, (T)0)
  SH_SET(4, c2a * x * y, c2a * y, c2a * x, (T)0)
  SH_SET(5, -c2a * y * z, (T)0, -c2a * z, -c2a * y)
  SH_SET(6, c2b * (2 * zz - xx - yy), -2 * c2b * x, -2 * c2b * y, 4 * c2b * z)
  SH_SET(7, -c2a * x * z, -c2a * z, (T)0, -c2a * x)
  SH_SET(8, c2c * (xx - yy), 2 * c2c * x, -2 * c2c * y, (T)0)
  SH_SET(9, -c3a * y * (3 * xx - yy), -c3a * 6 * x * y, -c3a * (3 * xx - 3 * yy), (T)0)
  SH_SET(10, c3b * x * y * z, c3b * y * z, c3b * x * z, c3b * x * y)
  SH_SET(11, -c3c * y * (4 * zz - xx - yy), c3c * 2 * x * y, -c3c * (4 * zz - xx - 3 * yy), -c3c * 8 * y * z)
  SH_SET(12, c3d * z * (2 * zz - 3 * xx - 3 * yy), -c3d * 6 * x * z, -c3d * 6 * y * z, c3d * (6 * zz - 3 * xx - 3 * yy))
  SH_SET(13, -c3c * x * (4 * zz - xx - yy), -c3c * (4 * zz - 3 * xx - yy), c3c * 2 * x * y, -c3c * 8 * x * z)
  SH_SET(14, c3e * z * (xx - yy), c3e * 2 * x * z, -c3e * 2 * y * z, c3e * (xx - yy))
  SH_SET(15, -c3a * x * (xx - 3 * yy), -c3a * (3 * xx - 3 * yy), c3a * 6 * x * y, (T)0)
#undef SH_SET
}

// camera centre o = -R^T t
template <class T>
__device__ __forceinline__ void camera_centre(const nbv_camera& cam, T* o) {
#pragma unroll
  for (int e = 0; e < 3; ++e)
    o[e] = -((T)cam.R_cw[e] * (T)cam.t_cw[0] + (T)cam.R_cw[3 + e] * (T)cam.t_cw[1] + (T)cam.R_cw[6 + e] * (T)cam.t_cw[2]);
}

// S1 add-on: the colour of every Gaussian as seen from every camera of the batch, into the splat records (value path)
__global__ void __launch_bounds__(256) sh_colour_kernel(int N, const float* __restrict__ mean, const float* __restrict__ rgb,
                                                         const float* __restrict__ sh45, const __grid_constant__ PreBatch batch) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= N) return;
  const PreView& pv = batch.v[blockIdx.y];
  float o[3];
  camera_centre<float>(pv.cam, o);
  const float rx = mean[3 * g] - o[0], ry = mean[3 * g + 1] - o[1], rz = mean[3 * g + 2] - o[2];
  const float in = rsqrtf(rx * rx + ry * ry + rz * rz);
  float B[SH_NB];
  sh_basis<float>(rx * in, ry * in, rz * in, B, nullptr);
  float c[3] = {rgb[3 * g], rgb[3 * g + 1], rgb[3 * g + 2]};
  const float* k = sh45 + (size_t)45 * g;
#pragma unroll
  for (int j = 1; j < SH_NB; ++j) {
    c[0] = fmaf(B[j], k[3 * (j - 1)], c[0]); c[1] = fmaf(B[j], k[3 * (j - 1) + 1], c[1]); c[2] = fmaf(B[j], k[3 * (j - 1) + 2], c[2]);
  }
  Splat* sp = pv.splat + g;
  sp->r = c[0]; sp->g = c[1]; sp->b = c[2];
}

void launch_sh_colours(const SceneDev& sc, const float* sh45, const PreBatch& batch, cudaStream_t st) {
  ++g_kernel_launches;
  sh_colour_kernel<<<dim3((unsigned)((sc.N + 255) / 256), (unsigned)batch.n), 256, 0, st>>>(sc.N, sc.mean, sc.rgb, sh45, batch);
}

// ---- S5' + S6, one warp per touched Gaussian ---------------------------------------------------------------------------
// shared memory per warp: Hc (the candidate / view block, then c (H_T + H) + Lambda) and Ha (c H_T + Lambda), both packed
// symmetric (1,770 doubles) in the reversed order of mask.cu -- entry (i, j >= i) at r (r + 1) / 2 + c with r = 58 - i,
// c = 58 - j, so that the trailing block of elimination step j is the prefix [0, m (m + 1) / 2), m = 58 - j, of the array and
// the pivot row follows it -- then y (4 x 11), e (4 x 59), G (11 x 11), the pivots (2 x 59).  32 KB per warp: 6 resident warps
// per SM (with full 59 x 60 storage and one factorisation after the other: 60 KB, 3 warps, 2.2 x the time).
constexpr int SH_WARP_DOUBLES = 2 * SH_LB + 4 * 11 + 4 * SH_L + 121 + 2 * SH_L + 1;
constexpr int SH_WARPS = 6;
constexpr int SH_TRI = SH_L * (SH_L - 1) / 2;          // `tri`: entry e of a row-major lower triangle -> (row << 8) | column
__device__ __forceinline__ int rtri(int r) { return r * (r + 1) / 2; }
__device__ __forceinline__ int rpk(int i, int j) { return rtri(SH_L - 1 - i) + SH_L - 1 - j; }      // i <= j

__global__ void __launch_bounds__(SH_WARPS * 32) expand_sh_kernel(const __grid_constant__ SceneDev sc, const __grid_constant__ nbv_config cfg,
                                                                    const __grid_constant__ ExpandBatch batch, int mode, int view0,
                                                                    const float* __restrict__ sh45, const float* __restrict__ prior59,
                                                                    double* __restrict__ H_T, const float* __restrict__ conf) {
  extern __shared__ __align__(16) double shm[];
  __shared__ double ws[SH_WARPS];
  __shared__ uint16_t tri[SH_TRI];
  for (int i = threadIdx.x; i < SH_L - 1; i += blockDim.x)
    for (int k = 0; k <= i; ++k) tri[i * (i + 1) / 2 + k] = (uint16_t)((i << 8) | k);
  __syncthreads();
  const ExpandView& vw = batch.v[view0 + blockIdx.y];
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  double* Hc = shm + (size_t)wib * SH_WARP_DOUBLES;
  double* Ha = Hc + SH_LB;
  double* ys = Ha + SH_LB;                 // [4][11]
  double* es = ys + 44;                    // [4][59]
  double* Gs = es + 4 * SH_L;              // [11][11]
  double* piv = Gs + 121;                  // [2][59]
  const uint32_t n_touched = vw.counters->n_touched;
  float omega[4];
#pragma unroll
  for (int c = 0; c < 4; ++c) omega[c] = ((cfg.channel_mask >> c) & 1) ? cfg.channel_weight[c] : 0.f;
  double gain = 0.0;
  for (uint32_t t = blockIdx.x * SH_WARPS + wib; t < n_touched; t += gridDim.x * SH_WARPS) {
    const uint32_t r = vw.touched[t];
    const uint32_t g = vw.ids_sorted[r];
    __syncwarp();
    // every lane reads the 40 moments (broadcast loads); lane 0 zeroes them for the next view afterwards
    double m[NMOM];
    {
      const double2* mom2 = reinterpret_cast<const double2*>(vw.moments + (size_t)r * NMOM);
#pragma unroll
      for (int i = 0; i < NMOM / 2; ++i) {
        const double2 v = mom2[i];
        m[2 * i] = v.x; m[2 * i + 1] = v.y;
      }
    }
    __syncwarp();
    if (lane < NMOM / 2) reinterpret_cast<double2*>(vw.moments + (size_t)r * NMOM)[lane] = make_double2(0.0, 0.0);
    whitened_to_u<double>(m, vw.splat_sorted[r]);
    Chain<double> ch;
    projection_chain<double>(vw.cam, sc.mean + 3 * (size_t)g, sc.logscale + 3 * (size_t)g, sc.quat + 4 * (size_t)g, ch);
    const double sg = (double)sc.sigma[g];
    const double kappa = cfg.opacity_coord == 0 ? (1.0 - sg) : 1.0 / sg;
    // lane k < 11: row k of A (11 x 6), then G row k, y_ch[k]
    if (lane < 11) {
      double a6[6];
      if (lane < 10) {
        a6[0] = ch.G[0][lane]; a6[1] = ch.G[1][lane]; a6[2] = 0.5 * ch.G[2][lane]; a6[3] = ch.G[3][lane]; a6[4] = 0.5 * ch.G[4][lane]; a6[5] = 0.0;
      } else {
        a6[0] = a6[1] = a6[2] = a6[3] = a6[4] = 0.0; a6[5] = kappa;
      }
      const int ex[6] = {1, 0, 2, 1, 0, 0}, ey[6] = {0, 1, 0, 1, 2, 0};
      double aq[6];
#pragma unroll
      for (int j = 0; j < 6; ++j) {
        double v = 0.0;
#pragma unroll
        for (int i = 0; i < 6; ++i) v += a6[i] * m[mono_index(ex[i] + ex[j], ey[i] + ey[j])];
        aq[j] = v;
      }
      // stash A row and AQ row in Ha (scratch now, overwritten later): Ha[k*12 + 0..5] = A, [6..11] = AQ
#pragma unroll
      for (int j = 0; j < 6; ++j) { Ha[lane * 12 + j] = a6[j]; Ha[lane * 12 + 6 + j] = aq[j]; }
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        double v = 0.0;
#pragma unroll
        for (int i = 0; i < 6; ++i) v += a6[i] * m[MOM_X + 6 * c + i];
        ys[c * 11 + lane] = sqrt((double)omega[c]) * v;
      }
    }
    // e_ch: colour channels from the SH model of this Gaussian seen from this camera; depth from the chain
    {
      double o[3];
      camera_centre<double>(vw.cam, o);
      const double rx = (double)sc.mean[3 * (size_t)g] - o[0], ry = (double)sc.mean[3 * (size_t)g + 1] - o[1],
                   rz = (double)sc.mean[3 * (size_t)g + 2] - o[2];
      const double in = rsqrt(rx * rx + ry * ry + rz * rz);
      const double d[3] = {rx * in, ry * in, rz * in};
      double B[SH_NB], dB[SH_NB][3];
      sh_basis<double>(d[0], d[1], d[2], B, dB);
      for (int i = lane; i < 4 * SH_L; i += 32) es[i] = 0.0;
      __syncwarp();
      if (lane < 3) {                                         // channel = lane
        const float* k = sh45 + (size_t)45 * g;
        double gr[3] = {0.0, 0.0, 0.0};
        for (int j = 1; j < SH_NB; ++j) {
          const double kj = (double)k[3 * (j - 1) + lane];
          gr[0] += kj * dB[j][0]; gr[1] += kj * dB[j][1]; gr[2] += kj * dB[j][2];
        }
        const double gd = gr[0] * d[0] + gr[1] * d[1] + gr[2] * d[2];
        for (int e = 0; e < 3; ++e) es[lane * SH_L + e] = (gr[e] - gd * d[e]) * in;
        for (int j = 0; j < SH_NB; ++j) es[lane * SH_L + 11 + 3 * j + lane] = B[j];
      } else if (lane == 3) {
        for (int e = 0; e < 3; ++e) es[3 * SH_L + e] = ch.dz[e];
      }
    }
    __syncwarp();
    if (lane < 11) {                                          // G = A Q A^T, row `lane`
      for (int l = 0; l < 11; ++l) {
        double v = 0.0;
#pragma unroll
        for (int j = 0; j < 6; ++j) v += Ha[lane * 12 + 6 + j] * Ha[l * 12 + j];
        Gs[lane * 11 + l] = v;
      }
    }
    __syncwarp();
    const double W2 = m[MOM_W2];
    // the upper triangle of the block: lane l builds columns l and 58 - l (l + 1 and 59 - l entries: 60 per lane)
    for (int half = 0; half < 2; ++half) {
      const int cc = half == 0 ? lane : SH_L - 1 - lane;
      if (lane >= 30 || (half == 1 && cc <= lane)) continue;
      double yc[4], ec[4];
#pragma unroll
      for (int c = 0; c < 4; ++c) { yc[c] = cc < 11 ? ys[c * 11 + cc] : 0.0; ec[c] = es[c * SH_L + cc]; }
      for (int rr = 0; rr <= cc; ++rr) {
        double v = cc < 11 ? Gs[rr * 11 + cc] : 0.0;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          if (omega[c] == 0.f) continue;
          const double yr = rr < 11 ? ys[c * 11 + rr] : 0.0;
          const double er = es[c * SH_L + rr];
          v += yr * ec[c] + er * yc[c] + (double)omega[c] * W2 * er * ec[c];
        }
        Hc[rpk(rr, cc)] = v;
      }
    }
    __syncwarp();
    if (mode == EXPAND_TRAIN || mode == EXPAND_VIEW) {
      for (int rr = 0; rr < SH_L; ++rr)
        for (int cc = rr + lane; cc < SH_L; cc += 32) {
          if (mode == EXPAND_TRAIN) H_T[(size_t)g * SH_LB + triS(rr, cc)] += Hc[rpk(rr, cc)];   // one launch per view, in view order
          else vw.out_blocks[(size_t)g * SH_LB + triS(rr, cc)] = (float)Hc[rpk(rr, cc)];
        }
      continue;
    }
    const double c = (double)conf[g];
    double gn = 0.0;
    if (c > 0.0) {
      // M0 = c H_T + Lambda -> Ha,  M1 = M0 + c H -> Hc, eliminated side by side (right-looking L D L^T); the gain is the sum of
      // log(d1_j / d0_j) over the pivots.  Step j: pivot row = entries [n, n + m], n = m (m + 1) / 2, trailing block = entries
      // [0, n), dealt to the lanes entry by entry through `tri`.
      const double* ht = H_T + (size_t)g * SH_LB;
      for (int rr = 0; rr < SH_L; ++rr) {
        const int rb = rpk(rr, 0);
        const double pr = (double)prior59[rr];
        for (int cc = rr + lane; cc < SH_L; cc += 32) {
          const double m0 = fma(c, ht[triS(rr, cc)], rr == cc ? pr : 0.0);
          Ha[rb - cc] = m0;
          Hc[rb - cc] = fma(c, Hc[rb - cc], m0);
        }
      }
      __syncwarp();
      for (int j = 0; j < SH_L; ++j) {
        const int m = SH_L - 1 - j, n = m * (m + 1) / 2;
        const double *v0 = Ha + n, *v1 = Hc + n;
        const double d0 = fmax(v0[m], 1e-300), d1 = fmax(v1[m], 1e-300);
        if (lane == 0) { piv[j] = d0; piv[SH_L + j] = d1; }
        const double i0 = -1.0 / d0, i1 = -1.0 / d1;
#pragma unroll 2
        for (int e = lane; e < n; e += 32) {
          const int rc = tri[e], r2 = rc >> 8, c2 = rc & 255;
          Ha[e] = fma(v0[r2] * i0, v0[c2], Ha[e]);
          Hc[e] = fma(v1[r2] * i1, v1[c2], Hc[e]);
        }
        __syncwarp();
      }
      for (int j = lane; j < SH_L; j += 32) gn += log(piv[SH_L + j] / piv[j]);
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) gn += __shfl_xor_sync(0xffffffffu, gn, o);
    }
    if (lane == 0) {
      if (vw.gains) vw.gains[g] = (float)gn;
      gain += gn;
    }
  }
  if (mode == EXPAND_GAIN) {
    if (lane == 0) ws[wib] = gain;
    __syncthreads();
    double tot = 0.0;
    if (threadIdx.x == 0)
      for (int w = 0; w < SH_WARPS; ++w) tot += ws[w];
    ordered_score(tot, vw.partials, &vw.counters->n_expanded, vw.score);
  }
}

void launch_expand_sh(const SceneDev& sc, const nbv_config& cfg, const ExpandBatch& batch, int mode, const float* sh45, const float* prior59,
                      double* H_T, const float* conf, cudaStream_t st) {
  const size_t smem = (size_t)SH_WARPS * SH_WARP_DOUBLES * sizeof(double);
  if (cudaFuncSetAttribute(expand_sh_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return;
  if (mode == EXPAND_TRAIN) {
    for (int v = 0; v < batch.n; ++v) {
      ++g_kernel_launches;
      expand_sh_kernel<<<dim3((unsigned)sm_count(), 1u), SH_WARPS * 32, smem, st>>>(sc, cfg, batch, mode, v, sh45, prior59, H_T, conf);
    }
    return;
  }
  ++g_kernel_launches;
  const int blocks = std::max(1, (sm_count() + batch.n - 1) / batch.n);
  expand_sh_kernel<<<dim3((unsigned)blocks, (unsigned)batch.n), SH_WARPS * 32, smem, st>>>(sc, cfg, batch, mode, 0, sh45, prior59, H_T, conf);
}

}  // namespace nbv
