// hessian.cu -- S5 (moments -> 14x14 block), S0' (confidence), S6 (log-det gain), S7 (arg-max).
//
// S5: for a Gaussian touched by the view, the 40 screen-space moments of S4 become
//       H_g = A Q A^T + sum_ch omega_ch [ (A x_ch) e_ch^T + e_ch (A x_ch)^T + W2 e_ch e_ch^T ]
//     with Q (6x6) the monomial sums arranged by m6 = (ux,uy,ux^2,ux uy,uy^2,1), x_ch the cross moments, W2 = sum w^2,
//     e_ch = d v_ch / d theta (unit vector on the colour parameter, or (dz/dmu, 0..) for depth), and
//     A (14 x 6): rows of the chain d(mx,my,a,b,c)/d(mu,logscale,quat) (first-order EWA, through q/|q|), the
//     opacity row kappa, zero colour rows.   PAPER.md L189-191 (H ~= J^T J), L210 (per-Gaussian blocks), L248.
// S6: IG_g = log det(c_g (H_T,g + H_c,g) + Lambda) - log det(c_g H_T,g + Lambda)   (Eq. 5, 6, 9; R-13, R-14)
//     evaluated in the SOLVE FORM  log det(I + U^-T (c_g H_c,g) U^-1),  U^T U = c_g H_T,g + Lambda,
//     which is the same number without the binary32 cancellation of two log-dets of size ~100.
//     U is factored once per scoring call (prepare_kernel); per candidate one thread per touched Gaussian does the
//     two-sided triangular solve and a Cholesky of I + W whose pivots 1 + e_j enter as log1p(e_j).
#include <algorithm>
#include <cstdlib>

#include "kernels.h"

namespace nbv {

struct ChainF {
  float G[5][10];   // d(mx,my,a,b,c) / d(mu(3), logscale(3), quat(4))
  float dz[3];      // dz/dmu
};

__device__ void sandwich_f(const float* Tm, const float* S3, float& a, float& b, float& c) {
  float TS[6];
#pragma unroll
  for (int i = 0; i < 2; ++i)
#pragma unroll
    for (int k = 0; k < 3; ++k) TS[3 * i + k] = Tm[3 * i] * S3[k] + Tm[3 * i + 1] * S3[3 + k] + Tm[3 * i + 2] * S3[6 + k];
  a = TS[0] * Tm[0] + TS[1] * Tm[1] + TS[2] * Tm[2];
  b = TS[0] * Tm[3] + TS[1] * Tm[4] + TS[2] * Tm[5];
  c = TS[3] * Tm[3] + TS[4] * Tm[4] + TS[5] * Tm[5];
}

// Value-path chain rule of the projection (binary32).
__device__ void chain_f(const nbv_camera& cam, const float* mu, const float* ls, const float* q, ChainF& ch) {
  const float* W = cam.R_cw;
  const float fx = cam.fx, fy = cam.fy;
  const float x = W[0] * mu[0] + W[1] * mu[1] + W[2] * mu[2] + cam.t_cw[0];
  const float y = W[3] * mu[0] + W[4] * mu[1] + W[5] * mu[2] + cam.t_cw[1];
  const float z = W[6] * mu[0] + W[7] * mu[1] + W[8] * mu[2] + cam.t_cw[2];
  const float iz = 1.0f / z, iz2 = iz * iz;
  const float J[6] = {fx * iz, 0.f, -fx * x * iz2, 0.f, fy * iz, -fy * y * iz2};
  float Tm[6];
#pragma unroll
  for (int i = 0; i < 2; ++i)
#pragma unroll
    for (int k = 0; k < 3; ++k) Tm[3 * i + k] = J[3 * i] * W[k] + J[3 * i + 1] * W[3 + k] + J[3 * i + 2] * W[6 + k];
  const float qn = sqrtf(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
  const float iqn = 1.0f / qn;
  const float qw = q[0] * iqn, qx = q[1] * iqn, qy = q[2] * iqn, qz = q[3] * iqn;
  float R[9];
  R[0] = 1.f - 2.f * (qy * qy + qz * qz); R[1] = 2.f * (qx * qy - qw * qz);       R[2] = 2.f * (qx * qz + qw * qy);
  R[3] = 2.f * (qx * qy + qw * qz);       R[4] = 1.f - 2.f * (qx * qx + qz * qz); R[5] = 2.f * (qy * qz - qw * qx);
  R[6] = 2.f * (qx * qz - qw * qy);       R[7] = 2.f * (qy * qz + qw * qx);       R[8] = 1.f - 2.f * (qx * qx + qy * qy);
  const float s2[3] = {expf(2.f * ls[0]), expf(2.f * ls[1]), expf(2.f * ls[2])};
  float S3[9];
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j)
      S3[3 * i + j] = R[3 * i] * s2[0] * R[3 * j] + R[3 * i + 1] * s2[1] * R[3 * j + 1] + R[3 * i + 2] * s2[2] * R[3 * j + 2];
  // d/dmu
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    ch.G[0][k] = Tm[k];
    ch.G[1][k] = Tm[3 + k];
    ch.dz[k] = W[6 + k];
  }
  const float iz3 = iz2 * iz;
  const float dJ[3][6] = {{0.f, 0.f, -fx * iz2, 0.f, 0.f, 0.f},
                          {0.f, 0.f, 0.f, 0.f, 0.f, -fy * iz2},
                          {-fx * iz2, 0.f, 2.f * fx * x * iz3, 0.f, -fy * iz2, 2.f * fy * y * iz3}};
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    float dJk[6], dT[6], dTS[6];
#pragma unroll
    for (int e = 0; e < 6; ++e) dJk[e] = dJ[0][e] * W[k] + dJ[1][e] * W[3 + k] + dJ[2][e] * W[6 + k];
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
      for (int c = 0; c < 3; ++c) dT[3 * i + c] = dJk[3 * i] * W[c] + dJk[3 * i + 1] * W[3 + c] + dJk[3 * i + 2] * W[6 + c];
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
      for (int c = 0; c < 3; ++c) dTS[3 * i + c] = dT[3 * i] * S3[c] + dT[3 * i + 1] * S3[3 + c] + dT[3 * i + 2] * S3[6 + c];
    const float E00 = dTS[0] * Tm[0] + dTS[1] * Tm[1] + dTS[2] * Tm[2];
    const float E01 = dTS[0] * Tm[3] + dTS[1] * Tm[4] + dTS[2] * Tm[5];
    const float E10 = dTS[3] * Tm[0] + dTS[4] * Tm[1] + dTS[5] * Tm[2];
    const float E11 = dTS[3] * Tm[3] + dTS[4] * Tm[4] + dTS[5] * Tm[5];
    ch.G[2][k] = 2.f * E00;
    ch.G[3][k] = E01 + E10;
    ch.G[4][k] = 2.f * E11;
  }
  // d/dlogscale_k : dSigma3D = 2 s_k^2 r_k r_k^T
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const float v0 = Tm[0] * R[k] + Tm[1] * R[3 + k] + Tm[2] * R[6 + k];
    const float v1 = Tm[3] * R[k] + Tm[4] * R[3 + k] + Tm[5] * R[6 + k];
    ch.G[0][3 + k] = 0.f; ch.G[1][3 + k] = 0.f;
    ch.G[2][3 + k] = 2.f * s2[k] * v0 * v0;
    ch.G[3][3 + k] = 2.f * s2[k] * v0 * v1;
    ch.G[4][3 + k] = 2.f * s2[k] * v1 * v1;
  }
  // d/dquat through q_hat = q/|q|
  const float qh[4] = {qw, qx, qy, qz};
  float dh[4][3];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    float Dm[9];
    if (i == 0) { const float d[9] = {0.f, -2.f * qz, 2.f * qy, 2.f * qz, 0.f, -2.f * qx, -2.f * qy, 2.f * qx, 0.f}; for (int e = 0; e < 9; ++e) Dm[e] = d[e]; }
    else if (i == 1) { const float d[9] = {0.f, 2.f * qy, 2.f * qz, 2.f * qy, -4.f * qx, -2.f * qw, 2.f * qz, 2.f * qw, -4.f * qx}; for (int e = 0; e < 9; ++e) Dm[e] = d[e]; }
    else if (i == 2) { const float d[9] = {-4.f * qy, 2.f * qx, 2.f * qw, 2.f * qx, 0.f, 2.f * qz, -2.f * qw, 2.f * qz, -4.f * qy}; for (int e = 0; e < 9; ++e) Dm[e] = d[e]; }
    else { const float d[9] = {-4.f * qz, -2.f * qw, 2.f * qx, 2.f * qw, -4.f * qz, 2.f * qy, 2.f * qx, 2.f * qy, 0.f}; for (int e = 0; e < 9; ++e) Dm[e] = d[e]; }
    float dS3[9];
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        float v = 0.f;
#pragma unroll
        for (int k = 0; k < 3; ++k) v += Dm[3 * r + k] * s2[k] * R[3 * c + k] + R[3 * r + k] * s2[k] * Dm[3 * c + k];
        dS3[3 * r + c] = v;
      }
    sandwich_f(Tm, dS3, dh[i][0], dh[i][1], dh[i][2]);
  }
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    ch.G[0][6 + j] = 0.f; ch.G[1][6 + j] = 0.f;
#pragma unroll
    for (int e = 0; e < 3; ++e) {
      float v = 0.f;
#pragma unroll
      for (int i = 0; i < 4; ++i) v += dh[i][e] * ((i == j ? 1.f : 0.f) - qh[i] * qh[j]) * iqn;
      ch.G[2 + e][6 + j] = v;
    }
  }
}

// S4 accumulates the moments in the monomials xi1^i xi2^j of the whitened pixel offset xi = L^-1 (p - m),
// Sigma2D = L L^T (raster.cu).  The derivatives of alpha are monomials of u = Sigma2D^-1 d = L^-T xi, i.e.
// ux = p00 xi1 + p01 xi2, uy = p11 xi2, so each homogeneous degree is mapped by the corresponding symmetric power of
// that 2 x 2 matrix, once per touched Gaussian.  The two terms of ux are uncorrelated over the footprint (no
// cancellation), which is why the whitened basis is used rather than plain pixel offsets.
__device__ void moments_to_u_basis(float* m, float p00, float p01, float p10, float p11) {
  float out[15];
  out[0] = m[0];
#pragma unroll
  for (int n = 1; n <= 4; ++n)
#pragma unroll
    for (int j = 0; j <= n; ++j) {
      // coefficients of ux^(n-j) uy^j in xi1^(n-t) xi2^t
      float coef[5] = {1.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
      for (int sidx = 0; sidx < n; ++sidx) {
        const float a0 = sidx < n - j ? p00 : p10, a1 = sidx < n - j ? p01 : p11;
#pragma unroll
        for (int t = 4; t >= 1; --t)
          if (t <= sidx + 1) coef[t] = coef[t] * a0 + coef[t - 1] * a1;
        coef[0] *= a0;
      }
      float v = 0.f;
#pragma unroll
      for (int t = 0; t <= n; ++t) v += coef[t] * m[mono_index(n - t, t)];
      out[mono_index(n - j, j)] = v;
    }
#pragma unroll
  for (int i = 0; i < 15; ++i) m[i] = out[i];
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    float* x = m + MOM_X + 6 * c;          // (xi1, xi2, xi1^2, xi1 xi2, xi2^2, 1) -> (ux, uy, ux^2, ux uy, uy^2, 1)
    const float x0 = x[0], x1 = x[1], x2 = x[2], x3 = x[3], x4 = x[4];
    x[0] = p00 * x0 + p01 * x1;
    x[1] = p10 * x0 + p11 * x1;
    x[2] = p00 * p00 * x2 + 2.f * p00 * p01 * x3 + p01 * p01 * x4;
    x[3] = p00 * p10 * x2 + (p00 * p11 + p01 * p10) * x3 + p01 * p11 * x4;
    x[4] = p10 * p10 * x2 + 2.f * p10 * p11 * x3 + p11 * p11 * x4;
  }
}

// moments (40) + chain -> packed block H[105]
__device__ void build_block(const float* mom, const ChainF& ch, float kappa, const float* omega, float* H) {
  // A: 11 nonzero rows x 6
  float A[11][6];
#pragma unroll
  for (int k = 0; k < 10; ++k) {
    A[k][0] = ch.G[0][k]; A[k][1] = ch.G[1][k]; A[k][2] = 0.5f * ch.G[2][k]; A[k][3] = ch.G[3][k]; A[k][4] = 0.5f * ch.G[4][k]; A[k][5] = 0.f;
  }
#pragma unroll
  for (int e = 0; e < 5; ++e) A[10][e] = 0.f;
  A[10][5] = kappa;
  const int ex[6] = {1, 0, 2, 1, 0, 0}, ey[6] = {0, 1, 0, 1, 2, 0};
  float Q[6][6];
#pragma unroll
  for (int i = 0; i < 6; ++i)
#pragma unroll
    for (int j = 0; j < 6; ++j) Q[i][j] = mom[mono_index(ex[i] + ex[j], ey[i] + ey[j])];
  float AQ[11][6];
  for (int k = 0; k < 11; ++k)
#pragma unroll
    for (int j = 0; j < 6; ++j) {
      float v = 0.f;
#pragma unroll
      for (int i = 0; i < 6; ++i) v += A[k][i] * Q[i][j];
      AQ[k][j] = v;
    }
  for (int i = 0; i < NBLK; ++i) H[i] = 0.f;
  for (int k = 0; k < 11; ++k)
    for (int l = k; l < 11; ++l) {
      float v = 0.f;
#pragma unroll
      for (int j = 0; j < 6; ++j) v += AQ[k][j] * A[l][j];
      H[tri(k, l)] = v;
    }
  const float W2 = mom[MOM_W2];
  for (int c = 0; c < 4; ++c) {
    const float om = omega[c];
    if (om == 0.f) continue;
    const float som = sqrtf(om);
    float yv[11];
    for (int k = 0; k < 11; ++k) {
      float v = 0.f;
#pragma unroll
      for (int i = 0; i < 6; ++i) v += A[k][i] * mom[MOM_X + 6 * c + i];
      yv[k] = som * v;                       // S4 delivers the cross moments scaled by sqrt(omega_ch)
    }
    if (c < 3) {
      for (int k = 0; k < 11; ++k) H[tri(k, 11 + c)] += yv[k];
      H[tri(11 + c, 11 + c)] += om * W2;
    } else {
      for (int k = 0; k < 11; ++k)
        for (int l = k; l < 11; ++l) {
          const float ek = k < 3 ? ch.dz[k] : 0.f, el = l < 3 ? ch.dz[l] : 0.f;
          H[tri(k, l)] += yv[k] * el + ek * yv[l] + om * W2 * ek * el;
        }
    }
  }
}

// Upper Cholesky factor of a packed SPD 14x14, in place (row j holds U[j][j..13]).  Pivots are floored at a tiny
// positive number: with Lambda > 0 the matrix is positive definite and the floor never acts in exact arithmetic.
__device__ void cholesky_packed(float* Mx) {
  for (int j = 0; j < P; ++j) {
    float d = Mx[tri(j, j)];
    for (int k = 0; k < j; ++k) d -= Mx[tri(k, j)] * Mx[tri(k, j)];
    d = fmaxf(d, 1e-30f);
    const float inv = rsqrtf(d);
    Mx[tri(j, j)] = d * inv;
    for (int i = j + 1; i < P; ++i) {
      float v = Mx[tri(j, i)];
      for (int k = 0; k < j; ++k) v -= Mx[tri(k, j)] * Mx[tri(k, i)];
      Mx[tri(j, i)] = v * inv;
    }
  }
}

// log det(I + U^-T B U^-1) for packed symmetric PSD B (destroyed) and packed upper-triangular U.
// Step 1 is the unblocked two-sided solve (the algorithm of LAPACK's xSYGS2, itype 1, upper); step 2 a Cholesky
// of I + W that never forms 1 + e: the pivot excess e_j goes through log1p.
__device__ float gain_solve(float* B, const float* U) {
  for (int k = 0; k < P; ++k) {
    const float inv = 1.0f / U[tri(k, k)];
    const float bkk = B[tri(k, k)] * inv * inv;
    B[tri(k, k)] = bkk;
    if (k < P - 1) {
      const float ct = -0.5f * bkk;
      for (int j = k + 1; j < P; ++j) B[tri(k, j)] = fmaf(ct, U[tri(k, j)], B[tri(k, j)] * inv);
      for (int i = k + 1; i < P; ++i) {
        const float bki = B[tri(k, i)], uki = U[tri(k, i)];
        for (int j = i; j < P; ++j) B[tri(i, j)] -= bki * U[tri(k, j)] + uki * B[tri(k, j)];
      }
      for (int j = k + 1; j < P; ++j) B[tri(k, j)] = fmaf(ct, U[tri(k, j)], B[tri(k, j)]);
      // row k, columns k+1.. :  x^T <- x^T U22^-1   (forward substitution with U22^T)
      for (int j = k + 1; j < P; ++j) {
        float v = B[tri(k, j)];
        for (int i = k + 1; i < j; ++i) v -= U[tri(i, j)] * B[tri(k, i)];
        B[tri(k, j)] = v / U[tri(j, j)];
      }
    }
  }
  float ld = 0.f;
  for (int j = 0; j < P; ++j) {
    float e = B[tri(j, j)];
    for (int k = 0; k < j; ++k) e -= B[tri(k, j)] * B[tri(k, j)];
    e = fmaxf(e, 0.f);                       // W is PSD: the excess is >= 0 up to rounding
    ld += log1pf(e);
    const float inv = rsqrtf(1.0f + e);
    for (int i = j + 1; i < P; ++i) {
      float v = B[tri(j, i)];
      for (int k = 0; k < j; ++k) v -= B[tri(k, j)] * B[tri(k, i)];
      B[tri(j, i)] = v * inv;
    }
  }
  return ld;
}

__global__ void __launch_bounds__(64) expand_kernel(const __grid_constant__ SceneDev sc, const __grid_constant__ nbv_config cfg,
                                                     const __grid_constant__ ExpandBatch batch, int mode, float* __restrict__ H_T,
                                                     const float* __restrict__ conf, const float* __restrict__ cholT,
                                                     uint32_t* __restrict__ cache_ids, float* __restrict__ cache_blocks) {
  const ExpandView& vw = batch.v[blockIdx.y];
  const nbv_camera& cam = vw.cam;
  const uint32_t* __restrict__ ids_sorted = vw.ids_sorted;
  const Splat* __restrict__ splat_sorted = vw.splat_sorted;
  const uint32_t* __restrict__ touched = vw.touched;
  float* __restrict__ moments = vw.moments;
  float* __restrict__ out_blocks = vw.out_blocks;
  float* __restrict__ score = vw.score;
  float* __restrict__ gains = vw.gains;
  const uint32_t n_touched = vw.counters->n_touched;
  float gain = 0.f;
  float omega[4];
#pragma unroll
  for (int c = 0; c < 4; ++c) omega[c] = ((cfg.channel_mask >> c) & 1) ? cfg.channel_weight[c] : 0.f;
  for (uint32_t t = blockIdx.x * blockDim.x + threadIdx.x; t < n_touched; t += gridDim.x * blockDim.x) {
    const uint32_t r = touched[t];
    const uint32_t g = ids_sorted[r];
    float4* mom4 = reinterpret_cast<float4*>(moments + (size_t)r * NMOM);
    float m[NMOM];
#pragma unroll
    for (int i = 0; i < NMOM / 4; ++i) {
      const float4 v = mom4[i];
      m[4 * i] = v.x; m[4 * i + 1] = v.y; m[4 * i + 2] = v.z; m[4 * i + 3] = v.w;
      mom4[i] = make_float4(0.f, 0.f, 0.f, 0.f);     // leave the buffer zeroed for the next view
    }
    {
      const Splat sp = splat_sorted[r];                 // conic = Sigma2D^-1 = -(2 qa, qb, 2 qc), the one S4 evaluated with
      const float cA = -2.f * sp.qa, cB = -sp.qb, cC = -2.f * sp.qc, icC = 1.0f / cC;
      const float i11 = sqrtf(fmaxf(cA * cC - cB * cB, 0.0f) * icC), sh = -cB * icC, i22 = sqrtf(cC);   // as in S4
      moments_to_u_basis(m, i11, -sh * i22, 0.0f, i22);   // u = L^-T xi
    }
    ChainF ch;
    chain_f(cam, sc.mean + 3 * (size_t)g, sc.logscale + 3 * (size_t)g, sc.quat + 4 * (size_t)g, ch);
    const float sg = sc.sigma[g];
    const float kappa = cfg.opacity_coord == 0 ? (1.f - sg) : 1.f / sg;       // R-10
    float H[NBLK];
    build_block(m, ch, kappa, omega, H);
    if (mode == EXPAND_TRAIN) {
      float* dst = H_T + (size_t)g * NBLK;             // views run concurrently on several streams: atomic accumulation
      for (int i = 0; i < NBLK; ++i) atomicAdd(dst + i, H[i]);
    } else if (mode == EXPAND_VIEW) {
      float* dst = out_blocks + (size_t)g * NBLK;
      for (int i = 0; i < NBLK; ++i) dst[i] = H[i];
    } else if (mode == EXPAND_CACHE) {
      if (t < vw.cache_span[1]) {                      // span[1] = 0 when the pool overflowed: nothing is stored
        const size_t e = (size_t)vw.cache_span[0] + t;
        cache_ids[e] = g;
        float* dst = cache_blocks + e * NBLK;
        for (int i = 0; i < NBLK; ++i) dst[i] = H[i];
      }
    } else {
      const float c = conf[g];
      float gn = 0.f;
      if (c > 0.f) {                       // c_g = 0 (Eq. 12, non-target): exactly zero gain
        float U[NBLK];
        const float* ut = cholT + (size_t)g * NBLK;
        const float cb = cfg.weight_mode == 1 ? 1.0f : c;         // R2 weights the gain, R1 / R3 the candidate block
        for (int i = 0; i < NBLK; ++i) { U[i] = ut[i]; H[i] *= cb; }
        gn = gain_solve(H, U);
        if (cfg.weight_mode == 1) gn *= c;
      }
      if (gains) gains[g] = gn;
      gain += gn;
    }
  }
  if (mode == EXPAND_GAIN) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) gain += __shfl_xor_sync(0xffffffffu, gain, o);
    __shared__ float ws[2];
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = gain;
    __syncthreads();
    if (threadIdx.x == 0) {
      const float t = ws[0] + ws[1];
      if (t != 0.f) atomicAdd(score, t);
    }
  }
}

void launch_expand(const SceneDev& sc, const nbv_config& cfg, const ExpandBatch& batch, int mode, float* H_T, const float* conf,
                   const float* cholT, cudaStream_t st) {
  int blocks = (sc.N + 63) / 64;
  const int cap = (148 * 8 + batch.n - 1) / batch.n;
  if (blocks > cap) blocks = cap;
  ++g_kernel_launches;
  expand_kernel<<<dim3((unsigned)blocks, (unsigned)batch.n), 64, 0, st>>>(sc, cfg, batch, mode, H_T, conf, cholT, nullptr, nullptr);
}

// ---- sparse block cache of greedy selection ----------------------------------------------------------------------
__global__ void cache_reserve_kernel(const __grid_constant__ ExpandBatch batch, BlockCache cache, int first_candidate) {
  const int v = threadIdx.x;
  if (v >= batch.n) return;
  const uint32_t cnt = batch.v[v].counters->n_touched;
  const uint32_t base = atomicAdd(cache.cursor, cnt);
  uint32_t* span = cache.spans + 2 * (size_t)(first_candidate + v);
  if ((unsigned long long)base + cnt > cache.capacity) {
    cache.cursor[1] = 1u;                                // overflow: the caller falls back to re-rasterising
    span[0] = 0u; span[1] = 0u;
  } else {
    span[0] = base; span[1] = cnt;
  }
}

void launch_cache_reserve(const ExpandBatch& batch, const BlockCache& cache, int first_candidate, cudaStream_t st) {
  ++g_kernel_launches;
  cache_reserve_kernel<<<1, 32, 0, st>>>(batch, cache, first_candidate);
}

void launch_expand_cache(const SceneDev& sc, const nbv_config& cfg, const ExpandBatch& batch, const BlockCache& cache, cudaStream_t st) {
  int blocks = (sc.N + 63) / 64;
  const int cap = (148 * 8 + batch.n - 1) / batch.n;
  if (blocks > cap) blocks = cap;
  ++g_kernel_launches;
  expand_kernel<<<dim3((unsigned)blocks, (unsigned)batch.n), 64, 0, st>>>(sc, cfg, batch, EXPAND_CACHE, nullptr, nullptr, nullptr, cache.ids,
                                                                         cache.blocks);
}

// One thread per cached (candidate, Gaussian) entry: the gain of Eq. 5/6/9 of that block against the current factor U_g.
__global__ void __launch_bounds__(64) cached_gain_kernel(BlockCache cache, const int32_t* __restrict__ taken, const float* __restrict__ conf,
                                                         const float* __restrict__ cholT, float* __restrict__ scores, int weight_mode) {
  const int c = blockIdx.y;
  float gain = 0.f;
  if (!taken[c]) {
    const uint32_t base = cache.spans[2 * c], cnt = cache.spans[2 * c + 1];
    for (uint32_t t = blockIdx.x * blockDim.x + threadIdx.x; t < cnt; t += gridDim.x * blockDim.x) {
      const size_t e = (size_t)base + t;
      const uint32_t g = cache.ids[e];
      const float cg = conf[g];
      if (cg > 0.f) {
        float H[NBLK], U[NBLK];
        const float* hb = cache.blocks + e * NBLK;
        const float* ut = cholT + (size_t)g * NBLK;
        const float cb = weight_mode == 1 ? 1.0f : cg;
        for (int i = 0; i < NBLK; ++i) { U[i] = ut[i]; H[i] = cb * hb[i]; }
        const float gn = gain_solve(H, U);
        gain += weight_mode == 1 ? cg * gn : gn;
      }
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) gain += __shfl_xor_sync(0xffffffffu, gain, o);
  __shared__ float ws[2];
  if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = gain;
  __syncthreads();
  if (threadIdx.x == 0) {
    const float t = ws[0] + ws[1];
    if (t != 0.f) atomicAdd(scores + c, t);
  }
}

void launch_cached_gain(const BlockCache& cache, int n_cand, const int32_t* taken, const float* conf, const float* cholT, float* scores,
                        int weight_mode, cudaStream_t st) {
  ++g_kernel_launches;
  cached_gain_kernel<<<dim3(64, (unsigned)n_cand), 64, 0, st>>>(cache, taken, conf, cholT, scores, weight_mode);
}

__global__ void __launch_bounds__(256) cache_accumulate_kernel(BlockCache cache, const int32_t* __restrict__ pick, float* __restrict__ H_T) {
  const int c = *pick;
  const uint32_t base = cache.spans[2 * c], cnt = cache.spans[2 * c + 1];
  const size_t total = (size_t)cnt * NBLK;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
    const size_t e = i / NBLK, k = i - e * NBLK;
    const uint32_t g = cache.ids[base + e];              // a view lists every Gaussian at most once: no atomics needed
    H_T[(size_t)g * NBLK + k] += cache.blocks[((size_t)base + e) * NBLK + k];
  }
}

void launch_cache_accumulate(const BlockCache& cache, const int32_t* pick, float* H_T, cudaStream_t st) {
  ++g_kernel_launches;
  cache_accumulate_kernel<<<148 * 4, 256, 0, st>>>(cache, pick, H_T);
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

// once per scoring call: U_g = upper Cholesky factor of c_g H_T,g + Lambda (skipped for c_g = 0: never read)
__global__ void __launch_bounds__(64) prepare_kernel(int N, nbv_config cfg, const float* __restrict__ H_T, const float* __restrict__ conf,
                                                      float* __restrict__ cholT) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= N) return;
  const float c = conf[g];
  if (!(c > 0.f)) return;
  const float* ht = H_T + (size_t)g * NBLK;
  float H[NBLK];
  const float ct = cfg.weight_mode == 0 ? c : 1.0f;           // Eq. 9 literal (R1) weights H_T as well; R2 / R3 do not
  for (int i = 0; i < NBLK; ++i) H[i] = ct * ht[i];
  for (int k = 0; k < P; ++k) H[tri(k, k)] += cfg.prior_precision[k];
  cholesky_packed(H);
  float* dst = cholT + (size_t)g * NBLK;
  for (int i = 0; i < NBLK; ++i) dst[i] = H[i];
}

void launch_prepare(const SceneDev& sc, const nbv_config& cfg, const float* H_T, const float* conf, float* cholT, cudaStream_t st) {
  ++g_kernel_launches;
  prepare_kernel<<<(sc.N + 63) / 64, 64, 0, st>>>(sc.N, cfg, H_T, conf, cholT);
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

void launch_argmax(const float* scores, int n, int32_t* best, cudaStream_t st) { { ++g_kernel_launches; argmax_kernel<<<1, 32, 0, st>>>(scores, n, best); } }



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
// and S6 is the same solve-form log-det gain on L x L blocks.
// =====================================================================================================================
__host__ __device__ __forceinline__ int mask_channel_of_slot(int t, int bgch) { return t == 0 ? bgch : (t <= bgch ? t - 1 : t); }
__host__ __device__ __forceinline__ int mask_slot_of_channel(int c, int bgch) { return c == bgch ? 0 : (c < bgch ? c + 1 : c); }
__device__ __forceinline__ int triL(int r, int c, int L) { return r * L - r * (r - 1) / 2 + (c - r); }

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

// upper Cholesky factor of a packed SPD L x L, in place (as cholesky_packed)
__device__ void cholesky_L(float* Mx, int L) {
  for (int j = 0; j < L; ++j) {
    float d = Mx[triL(j, j, L)];
    for (int k = 0; k < j; ++k) d -= Mx[triL(k, j, L)] * Mx[triL(k, j, L)];
    d = fmaxf(d, 1e-30f);
    const float inv = rsqrtf(d);
    Mx[triL(j, j, L)] = d * inv;
    for (int i = j + 1; i < L; ++i) {
      float v = Mx[triL(j, i, L)];
      for (int k = 0; k < j; ++k) v -= Mx[triL(k, j, L)] * Mx[triL(k, i, L)];
      Mx[triL(j, i, L)] = v * inv;
    }
  }
}

// ---- S5' + S6 of a mask context, warp-cooperative: ONE WARP PER TOUCHED GAUSSIAN, the L x L block and the factor in shared
// memory.  Lane l owns the columns (or rows) l, l + 32 of the matrices, so the triangular solves and the elimination run
// on up to 63 columns at once (a first version ran one thread per Gaussian over 2 x 2016 floats of local memory).
//   W = U^-T (c H) U^-1 : (a) every lane solves U^T x = h_j for its columns j, in place; (b) every lane solves
//   U^T y = (row i of the result)^T for its rows i, in place.   log det(I + W): right-looking Cholesky on the excess
//   (pivot 1 + e_j enters as log1p(e_j), as in gain_solve), one column per step, the trailing rows updated in parallel.
struct MaskWarpLayout {
  int LS;          // row stride of H and U (odd: conflict-free column and row walks)
  int per_warp;    // floats per warp
  int oH, oU, oA, oAQ, oMom, oX, oP, oMono;
};
__host__ __device__ inline MaskWarpLayout mask_warp_layout(int K, int groups) {
  MaskWarpLayout m;
  const int L = 11 + K;
  m.LS = L | 1;
  int o = 0;
  m.oH = o; o += m.LS * L;
  m.oU = o; o += m.LS * L;
  m.oA = o; o += 66;
  m.oAQ = o; o += 66;
  m.oMom = o; o += groups * NMOM;
  m.oX = o; o += K * 6;
  m.oP = o; o += K;
  m.oMono = o; o += 16;
  m.per_warp = (o + 3) & ~3;
  return m;
}

__global__ void __launch_bounds__(256) expand_mask_warp_kernel(const __grid_constant__ SceneDev sc, const __grid_constant__ nbv_config cfg,
                                                                const __grid_constant__ ExpandBatch batch, int mode, int groups,
                                                                float* __restrict__ H_T, const float* __restrict__ conf,
                                                                const float* __restrict__ cholT) {
  extern __shared__ __align__(16) float smem[];
  const ExpandView& vw = batch.v[blockIdx.y];
  const int K = sc.K, L = 11 + K, LB = L * (L + 1) / 2, bgch = cfg.mask_bg_channel;
  const MaskWarpLayout lay = mask_warp_layout(K, groups);
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5, wpb = blockDim.x >> 5, LS = lay.LS;
  float* base = smem + (size_t)wib * lay.per_warp;
  float *Hm = base + lay.oH, *Um = base + lay.oU, *As = base + lay.oA, *AQs = base + lay.oAQ, *mom = base + lay.oMom;
  float *xs = base + lay.oX, *ps = base + lay.oP, *mono = base + lay.oMono;
  const uint32_t n_touched = vw.counters->n_touched;
  const int stride = NMOM * groups;
  float gain = 0.f;
  for (uint32_t t = blockIdx.x * wpb + wib; t < n_touched; t += gridDim.x * wpb) {
    const uint32_t r = vw.touched[t];
    const uint32_t g = vw.ids_sorted[r];
    __syncwarp();
    // moments of all groups -> shared memory (and zero the buffer for the next view)
    float* gm = vw.moments + (size_t)r * stride;
    for (int i = lane; i < stride; i += 32) { mom[i] = gm[i]; gm[i] = 0.f; }
    __syncwarp();
    {   // whitened basis -> u basis, one lane per group
      const Splat sp = vw.splat_sorted[r];
      const float cA = -2.f * sp.qa, cB = -sp.qb, cC = -2.f * sp.qc, icC = 1.0f / cC;
      const float i11 = sqrtf(fmaxf(cA * cC - cB * cB, 0.0f) * icC), sh = -cB * icC, i22 = sqrtf(cC);   // as in S4
      for (int gr = lane; gr < groups; gr += 32) {
        float m[NMOM];
#pragma unroll
        for (int i = 0; i < NMOM; ++i) m[i] = mom[gr * NMOM + i];
        moments_to_u_basis(m, i11, -sh * i22, 0.0f, i22);
#pragma unroll
        for (int i = 0; i < NMOM; ++i) mom[gr * NMOM + i] = m[i];
      }
    }
    __syncwarp();
    if (lane < 15) {
      float v = 0.f;
      for (int gr = 0; gr < groups; ++gr) v += mom[gr * NMOM + lane];
      mono[lane] = v;
    }
    if (lane == 15) mono[15] = mom[MOM_W2];
    for (int i = lane; i < K * 6; i += 32) {
      const int slot = i / 6, e = i - 6 * slot;
      xs[i] = mom[(slot >> 2) * NMOM + MOM_X + 6 * (slot & 3) + e];
    }
    float s2p = 0.f;
    for (int slot = lane; slot < K; slot += 32) {
      const float pv = expf(sc.logits[(size_t)g * K + mask_channel_of_slot(slot, bgch)] - sc.lse[g]);
      ps[slot] = pv;
      s2p += pv * pv;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s2p += __shfl_xor_sync(0xffffffffu, s2p, o);
    const float S2 = s2p;
    {   // chain rule (every lane, redundantly), A and A Q into shared memory for dynamic indexing
      ChainF ch;
      chain_f(vw.cam, sc.mean + 3 * (size_t)g, sc.logscale + 3 * (size_t)g, sc.quat + 4 * (size_t)g, ch);
      const float sg = sc.sigma[g];
      const float kappa = cfg.opacity_coord == 0 ? (1.f - sg) : 1.f / sg;       // R-10
      if (lane < 11) {
        float a6[6];
        if (lane < 10) {
          a6[0] = ch.G[0][lane]; a6[1] = ch.G[1][lane]; a6[2] = 0.5f * ch.G[2][lane]; a6[3] = ch.G[3][lane]; a6[4] = 0.5f * ch.G[4][lane]; a6[5] = 0.f;
        } else {
          a6[0] = a6[1] = a6[2] = a6[3] = a6[4] = 0.f; a6[5] = kappa;
        }
#pragma unroll
        for (int e = 0; e < 6; ++e) As[lane * 6 + e] = a6[e];
      }
    }
    __syncwarp();
    if (lane < 11) {
      const int ex[6] = {1, 0, 2, 1, 0, 0}, ey[6] = {0, 1, 0, 1, 2, 0};
      for (int j = 0; j < 6; ++j) {
        float v = 0.f;
        for (int i = 0; i < 6; ++i) v += As[lane * 6 + i] * mono[mono_index(ex[i] + ex[j], ey[i] + ey[j])];
        AQs[lane * 6 + j] = v;
      }
    }
    __syncwarp();
    const float W2 = mono[15];
    float xbar[6];
#pragma unroll
    for (int e = 0; e < 6; ++e) {
      float v = 0.f;
      for (int slot = 0; slot < K; ++slot) v += ps[slot] * xs[slot * 6 + e];
      xbar[e] = v;
    }
    // the full symmetric block, column j by lane j (and j + 32)
    for (int j = lane; j < L; j += 32) {
      if (j < 11) {
        for (int i = 0; i < 11; ++i) {
          float v = 0.f;
#pragma unroll
          for (int e = 0; e < 6; ++e) v += AQs[i * 6 + e] * As[j * 6 + e];
          Hm[i * LS + j] = v;
        }
        for (int c = 0; c < K; ++c) {
          const int slot = mask_slot_of_channel(c, bgch);
          float v = 0.f;
#pragma unroll
          for (int e = 0; e < 6; ++e) v += As[j * 6 + e] * (ps[slot] * (xs[slot * 6 + e] - xbar[e]));
          Hm[(11 + c) * LS + j] = v;
        }
      } else {
        const int c = j - 11, slot = mask_slot_of_channel(c, bgch);
        const float pc = ps[slot];
        for (int i = 0; i < 11; ++i) {
          float v = 0.f;
#pragma unroll
          for (int e = 0; e < 6; ++e) v += As[i * 6 + e] * (pc * (xs[slot * 6 + e] - xbar[e]));
          Hm[i * LS + j] = v;
        }
        for (int d = 0; d < K; ++d) {
          const float pd = ps[mask_slot_of_channel(d, bgch)];
          float v = pc * pd * (S2 - pc - pd);
          if (d == c) v += pc * pc;
          Hm[(11 + d) * LS + j] = W2 * v;
        }
      }
    }
    __syncwarp();
    if (mode == EXPAND_TRAIN || mode == EXPAND_VIEW) {
      float* dst = (mode == EXPAND_TRAIN ? H_T : vw.out_blocks) + (size_t)g * LB;
      for (int rr = 0; rr < L; ++rr)
        for (int c = rr + lane; c < L; c += 32) {
          if (mode == EXPAND_TRAIN) atomicAdd(dst + triL(rr, c, L), Hm[rr * LS + c]);
          else dst[triL(rr, c, L)] = Hm[rr * LS + c];
        }
      continue;
    }
    const float cg = conf[g];
    const float cb = cfg.weight_mode == 1 ? 1.0f : cg;
    float gn = 0.f;
    if (cg > 0.f) {
      const float* ut = cholT + (size_t)g * LB;
      for (int rr = 0; rr < L; ++rr)
        for (int c = rr + lane; c < L; c += 32) Um[rr * LS + c] = ut[triL(rr, c, L)];
      __syncwarp();
      // (a) columns: U^T x = c h_j
      for (int j = lane; j < L; j += 32)
        for (int i = 0; i < L; ++i) {
          float v = cb * Hm[i * LS + j];
#pragma unroll 4
          for (int k = 0; k < i; ++k) v -= Um[k * LS + i] * Hm[k * LS + j];
          Hm[i * LS + j] = v / Um[i * LS + i];
        }
      __syncwarp();
      // (b) rows: U^T y = (row i)^T
      for (int i = lane; i < L; i += 32)
        for (int c = 0; c < L; ++c) {
          float v = Hm[i * LS + c];
#pragma unroll 4
          for (int k = 0; k < c; ++k) v -= Um[k * LS + c] * Hm[i * LS + k];
          Hm[i * LS + c] = v / Um[c * LS + c];
        }
      __syncwarp();
      // log det(I + W): right-looking Cholesky on the excess, lower triangle
      for (int j = 0; j < L; ++j) {
        const float e = fmaxf(Hm[j * LS + j], 0.f);
        gn += log1pf(e);
        const float inv = rsqrtf(1.0f + e);
        __syncwarp();
        for (int i = j + 1 + lane; i < L; i += 32) Hm[i * LS + j] *= inv;
        __syncwarp();
        for (int i = j + 1 + lane; i < L; i += 32) {
          const float li = Hm[i * LS + j];
#pragma unroll 4
          for (int k = j + 1; k <= i; ++k) Hm[i * LS + k] -= li * Hm[k * LS + j];
        }
        __syncwarp();
      }
    }
    if (cfg.weight_mode == 1) gn *= cg;
    if (lane == 0) {
      if (vw.gains) vw.gains[g] = gn;
      gain += gn;
    }
  }
  if (mode == EXPAND_GAIN) {
    __shared__ float ws[8];
    if (lane == 0) ws[wib] = gain;
    __syncthreads();
    if (threadIdx.x == 0) {
      float tsum = 0.f;
      for (int w = 0; w < wpb; ++w) tsum += ws[w];
      if (tsum != 0.f) atomicAdd(vw.score, tsum);
    }
  }
}

void launch_expand_mask(const SceneDev& sc, const nbv_config& cfg, const ExpandBatch& batch, int mode, int groups, float* H_T,
                        const float* conf, const float* cholT, cudaStream_t st) {
  ++g_kernel_launches;
  const MaskWarpLayout lay = mask_warp_layout(sc.K, groups);
  int wpb = 8;
  while (wpb > 1 && (size_t)wpb * lay.per_warp * 4 > 200 * 1024) wpb >>= 1;
  const size_t smem = (size_t)wpb * lay.per_warp * 4;
  static size_t configured = 0;
  if (smem > configured) {
    cudaFuncSetAttribute(expand_mask_warp_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    configured = smem;
  }
  const int blocks = std::max(1, (148 * 2 + batch.n - 1) / batch.n);
  expand_mask_warp_kernel<<<dim3((unsigned)blocks, (unsigned)batch.n), wpb * 32, smem, st>>>(sc, cfg, batch, mode, groups, H_T, conf, cholT);
}

// once per scoring call of a mask context: U_g = upper Cholesky factor of c_g H_T,g + Lambda (L x L)
template <int KMAX>
__global__ void __launch_bounds__(64) prepare_mask_kernel(int N, int K, nbv_config cfg, const float* __restrict__ H_T,
                                                           const float* __restrict__ conf, float* __restrict__ cholT) {
  constexpr int LMAX = 11 + KMAX, LBMAX = LMAX * (LMAX + 1) / 2;
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= N) return;
  const float c = conf[g];
  if (!(c > 0.f)) return;
  const int L = 11 + K, LB = L * (L + 1) / 2;
  const float* ht = H_T + (size_t)g * LB;
  float H[LBMAX];
  const float ct = cfg.weight_mode == 0 ? c : 1.0f;
  for (int i = 0; i < LB; ++i) H[i] = ct * ht[i];
  for (int k = 0; k < L; ++k) H[triL(k, k, L)] += k < 11 ? cfg.prior_precision[k] : cfg.prior_precision_obj;
  cholesky_L(H, L);
  float* dst = cholT + (size_t)g * LB;
  for (int i = 0; i < LB; ++i) dst[i] = H[i];
}

void launch_prepare_mask(const SceneDev& sc, const nbv_config& cfg, const float* H_T, const float* conf, float* cholT, cudaStream_t st) {
  ++g_kernel_launches;
  if (sc.K <= 20)
    prepare_mask_kernel<20><<<(sc.N + 63) / 64, 64, 0, st>>>(sc.N, sc.K, cfg, H_T, conf, cholT);
  else
    prepare_mask_kernel<NBV_MASK_KMAX><<<(sc.N + 63) / 64, 64, 0, st>>>(sc.N, sc.K, cfg, H_T, conf, cholT);
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
