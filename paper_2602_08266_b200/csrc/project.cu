// project.cu -- S0 activation and S1 EWA projection + 2D covariance + support rectangle.
//
// Both kernels are on the DECISION PATH (R-9): binary32, fixed operation order,
// no contraction.  What they compute follows the 3DGS conventions the paper inherits:
// Sigma3D = R S S^T R^T from scale and rotation (L131), first-order perspective projection with a
// 0.3 px^2 blur (R-3).  One thread per Gaussian; the work is ~200 flop and ~100 bytes per Gaussian per view.
#include "kernels.h"

namespace nbv {

__global__ void __launch_bounds__(256) activate_kernel(SceneDev sc, ViewCounters* counters) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= sc.N) return;
  bool bad = false;
  float s[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    float l = sc.logscale[3 * g + k];
    bad |= !isfinite(l) || !isfinite(sc.mean[3 * g + k]) || !isfinite(sc.rgb[3 * g + k]);
    l = fminf(fmaxf(l, -80.0f), 80.0f);
    s[k] = exp_spec(l);
  }
  float w = sc.quat[4 * g], x = sc.quat[4 * g + 1], y = sc.quat[4 * g + 2], z = sc.quat[4 * g + 3];
  const float n2 = add_rn(add_rn(add_rn(mul_rn(w, w), mul_rn(x, x)), mul_rn(y, y)), mul_rn(z, z));
  const float sg = sc.sigma[g];
  bad |= !(n2 > 0.0f) || !isfinite(n2) || !(sg > 0.0f) || !(sg < 1.0f);
  const float n = sqrt_rn(n2);
  w = div_rn(w, n); x = div_rn(x, n); y = div_rn(y, n); z = div_rn(z, n);
  const float xx = mul_rn(x, x), yy = mul_rn(y, y), zz = mul_rn(z, z);
  const float xy = mul_rn(x, y), xz = mul_rn(x, z), yz = mul_rn(y, z);
  const float wx = mul_rn(w, x), wy = mul_rn(w, y), wz = mul_rn(w, z);
  float R[9];
  R[0] = sub_rn(1.0f, mul_rn(2.0f, add_rn(yy, zz))); R[1] = mul_rn(2.0f, sub_rn(xy, wz)); R[2] = mul_rn(2.0f, add_rn(xz, wy));
  R[3] = mul_rn(2.0f, add_rn(xy, wz)); R[4] = sub_rn(1.0f, mul_rn(2.0f, add_rn(xx, zz))); R[5] = mul_rn(2.0f, sub_rn(yz, wx));
  R[6] = mul_rn(2.0f, sub_rn(xz, wy)); R[7] = mul_rn(2.0f, add_rn(yz, wx)); R[8] = sub_rn(1.0f, mul_rn(2.0f, add_rn(xx, yy)));
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int k = 0; k < 3; ++k) sc.M[9 * (size_t)g + 3 * i + k] = mul_rn(R[3 * i + k], s[k]);

  // softmax statistics of the object vector (p_i = softmax(o_i)); value path
  const float* lg = sc.logits + (size_t)g * sc.K;
  float mx = lg[0];
  int am = 0;
  for (int k = 1; k < sc.K; ++k) {
    float v = lg[k];
    if (v > mx) { mx = v; am = k; }   // strict: lowest index on ties (R-15)
  }
  float se = 0.0f;
  for (int k = 0; k < sc.K; ++k) {
    float v = lg[k];
    bad |= !isfinite(v);
    se += expf(v - mx);
  }
  sc.pmax[g] = 1.0f / se;
  sc.amax[g] = am;
  sc.lse[g] = mx + logf(se);
  if (bad) atomicOr(&counters->bad_data, 1u);
}

void launch_activate(const SceneDev& sc, ViewCounters* counters, cudaStream_t st) {
  ++g_kernel_launches;
  activate_kernel<<<(sc.N + 255) / 256, 256, 0, st>>>(sc, counters);
}

// Conservative upper bound of ln(255 sigma): tangent of ln at 0.75 on the mantissa.
__device__ __forceinline__ float log_bound(float sigma) {
  float x = mul_rn(255.0f, sigma);
  if (!(x > 1.0f)) x = 1.0f;
  const uint32_t u = __float_as_uint(x);
  const int e = (int)((u >> 23) & 0xffu) - 126;
  const float m = __uint_as_float((u & 0x007fffffu) | 0x3f000000u);
  const float lm = add_rn(mul_rn(m, 0x1.555556p+0f), -0x1.49a588p+0f);
  return add_rn(mul_rn((float)e, 0x1.62e43p-1f), lm);
}

__global__ void __launch_bounds__(256) project_kernel(const __grid_constant__ SceneDev sc, const __grid_constant__ nbv_config cfg,
                                                       const __grid_constant__ PreBatch batch) {
  const PreView& pv = batch.v[blockIdx.y];
  const nbv_camera& cam = pv.cam;
  Splat* __restrict__ splat = pv.splat;
  uint32_t* __restrict__ zkey = pv.zkey[0];
  uint32_t* __restrict__ ids = pv.ids[0];
  ushort4* __restrict__ rect = pv.rect;
  float* __restrict__ abc = pv.abc;
  ViewCounters* counters = pv.counters;
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  bool visible = false;
  unsigned int ntiles = 0;
  if (g < sc.N) {
    Splat sp;
    ushort4 rc = make_ushort4(0, 0, 0, 0);
    float a = 0.f, b = 0.f, c = 0.f;
    sp.mx = sp.my = sp.qa = sp.qb = sp.qc = sp.z = 0.f;
    const float sg = sc.sigma[g];
    sp.sigma = sg;
    sp.r = sc.rgb[3 * g]; sp.g = sc.rgb[3 * g + 1]; sp.b = sc.rgb[3 * g + 2];
    sp.pad = 0.f;
    sp.tau = 0.f;
    const float* W = cam.R_cw;
    const float m0 = sc.mean[3 * g], m1 = sc.mean[3 * g + 1], m2 = sc.mean[3 * g + 2];
    const float x = add_rn(add_rn(add_rn(mul_rn(W[0], m0), mul_rn(W[1], m1)), mul_rn(W[2], m2)), cam.t_cw[0]);
    const float y = add_rn(add_rn(add_rn(mul_rn(W[3], m0), mul_rn(W[4], m1)), mul_rn(W[5], m2)), cam.t_cw[1]);
    const float z = add_rn(add_rn(add_rn(mul_rn(W[6], m0), mul_rn(W[7], m1)), mul_rn(W[8], m2)), cam.t_cw[2]);
    do {
      if (!(z > cfg.near_plane)) break;
      const float iz = div_rn(1.0f, z);
      const float xz = mul_rn(x, iz), yz = mul_rn(y, iz);
      sp.mx = add_rn(mul_rn(cam.fx, xz), cam.cx);
      sp.my = add_rn(mul_rn(cam.fy, yz), cam.cy);
      sp.z = z;
      const float j00 = mul_rn(cam.fx, iz), j02 = -mul_rn(j00, xz);
      const float j11 = mul_rn(cam.fy, iz), j12 = -mul_rn(j11, yz);
      float T0[3], T1[3];
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        T0[k] = add_rn(mul_rn(j00, W[k]), mul_rn(j02, W[6 + k]));
        T1[k] = add_rn(mul_rn(j11, W[3 + k]), mul_rn(j12, W[6 + k]));
      }
      float Mm[9];
#pragma unroll
      for (int i = 0; i < 9; ++i) Mm[i] = sc.M[9 * (size_t)g + i];
      float U0[3], U1[3];
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        U0[k] = add_rn(add_rn(mul_rn(T0[0], Mm[k]), mul_rn(T0[1], Mm[3 + k])), mul_rn(T0[2], Mm[6 + k]));
        U1[k] = add_rn(add_rn(mul_rn(T1[0], Mm[k]), mul_rn(T1[1], Mm[3 + k])), mul_rn(T1[2], Mm[6 + k]));
      }
      a = add_rn(add_rn(add_rn(mul_rn(U0[0], U0[0]), mul_rn(U0[1], U0[1])), mul_rn(U0[2], U0[2])), cfg.blur);
      b = add_rn(add_rn(mul_rn(U0[0], U1[0]), mul_rn(U0[1], U1[1])), mul_rn(U0[2], U1[2]));
      c = add_rn(add_rn(add_rn(mul_rn(U1[0], U1[0]), mul_rn(U1[1], U1[1])), mul_rn(U1[2], U1[2])), cfg.blur);
      const float det = sub_rn(mul_rn(a, c), mul_rn(b, b));
      if (!(det > 0.0f) || !isfinite(det)) break;
      sp.qa = mul_rn(-0.5f, div_rn(c, det));
      sp.qb = div_rn(b, det);
      sp.qc = mul_rn(-0.5f, div_rn(a, det));
      const float L = log_bound(sg);
      sp.tau = -L - 0.01f;   // power < tau  =>  sigma exp_spec(power) < 1/255 <= alpha_min, with margin
      const float rho2 = add_rn(mul_rn(2.02f, L), 0.05f);
      float hx = add_rn(sqrt_rn(mul_rn(rho2, a)), 1.0f);
      float hy = add_rn(sqrt_rn(mul_rn(rho2, c)), 1.0f);
      if (!(fabsf(sp.mx) <= 1.0e6f) || !(fabsf(sp.my) <= 1.0e6f)) break;
      if (!(hx <= 2.0e6f)) hx = 2.0e6f;
      if (!(hy <= 2.0e6f)) hy = 2.0e6f;
      const int TX = (cam.width + TILE - 1) / TILE, TY = (cam.height + TILE - 1) / TILE;
      const float fx0 = floorf(mul_rn(sub_rn(sp.mx, hx), 0.0625f)), fx1 = add_rn(floorf(mul_rn(add_rn(sp.mx, hx), 0.0625f)), 1.0f);
      const float fy0 = floorf(mul_rn(sub_rn(sp.my, hy), 0.0625f)), fy1 = add_rn(floorf(mul_rn(add_rn(sp.my, hy), 0.0625f)), 1.0f);
      const int tx0 = (int)fminf(fmaxf(fx0, 0.0f), (float)TX), tx1 = (int)fminf(fmaxf(fx1, 0.0f), (float)TX);
      const int ty0 = (int)fminf(fmaxf(fy0, 0.0f), (float)TY), ty1 = (int)fminf(fmaxf(fy1, 0.0f), (float)TY);
      rc = make_ushort4((unsigned short)tx0, (unsigned short)ty0, (unsigned short)tx1, (unsigned short)ty1);
      if (tx1 <= tx0 || ty1 <= ty0) break;
      visible = true;
      ntiles = (unsigned)(tx1 - tx0) * (unsigned)(ty1 - ty0);
    } while (0);
    if (!visible) rc = make_ushort4(0, 0, 0, 0);   // empty rect for culled Gaussians
    splat[g] = sp;
    zkey[g] = visible ? __float_as_uint(sp.z) : 0xffffffffu;
    ids[g] = (uint32_t)g;
    rect[g] = rc;
    if (abc) { abc[3 * (size_t)g] = a; abc[3 * (size_t)g + 1] = b; abc[3 * (size_t)g + 2] = c; }
  }
  // counters: aggregated over the block (one pair of atomics per block: thousands of same-address atomics per view would
  // serialise in the L2 and cost more than the projection itself)
  __shared__ unsigned int s_vis[8];
  __shared__ unsigned long long s_nt[8];
  const unsigned vis_mask = __ballot_sync(0xffffffffu, visible);
  unsigned long long nt = ntiles;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) nt += __shfl_xor_sync(0xffffffffu, nt, o);
  const int wid = threadIdx.x >> 5;
  if ((threadIdx.x & 31) == 0) { s_vis[wid] = (unsigned)__popc(vis_mask); s_nt[wid] = nt; }
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned int v = 0;
    unsigned long long t = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) { v += s_vis[w]; t += s_nt[w]; }
    if (v) {
      atomicAdd(&counters->n_visible, v);
      atomicAdd(&counters->n_keys, t);
    }
  }
}

void launch_project(const SceneDev& sc, const nbv_config& cfg, const PreBatch& batch, cudaStream_t st) {
  ++g_kernel_launches;
  project_kernel<<<dim3((unsigned)((sc.N + 255) / 256), (unsigned)batch.n), 256, 0, st>>>(sc, cfg, batch);
}

}  // namespace nbv
