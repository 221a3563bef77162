// block_math.cuh -- per-Gaussian block arithmetic of S5 / S6, templated on the scalar type (binary64 in the colour / depth
// contexts, binary32 in the object-mask contexts).  Derived for this path from the factor the decision path already has.
//
// S1 projects a Gaussian through  Sigma2D = U U^T + blur I,   U = Jp V (2 x 3),   V = W R(q/|q|) diag(s) (3 x 3),
// W = R_cw, p = W mu + t = (x, y, z), Jp = [[fx/z, 0, -fx x/z^2], [0, fy/z, -fy y/z^2]]   (R-3), so with the
// rows u0, u1 of U:   a = |u0|^2 + blur,  b = u0 . u1,  c = |u1|^2 + blur   and for any parameter
//     da = 2 u0 . du0,    db = du0 . u1 + u0 . du1,    dc = 2 u1 . du1.
// The rows are  u0 = (fx/z) (v0 - (x/z) v2),  u1 = (fy/z) (v1 - (y/z) v2)  with v_i the rows of V.  Hence
//   position:   du0/dx = -(fx/z^2) v2,   du0/dz = -u0/z + (fx x/z^3) v2,   du0/dy = 0   (u1 alike), dp/dmu_k = W[:,k];
//   log-scale:  dV/dl_k keeps column k only, so  du_i/dl_k = u_ik e_k:   da = 2 u0k^2, db = 2 u0k u1k, dc = 2 u1k^2;
//   rotation:   R(q/|q|) = N(q) / |q|^2 with N the homogeneous quadratic form of the rotation matrix, so
//               dR/dq_j = (dN/dq_j (q_hat) - 2 q_hat_j R) / |q|   -- the derivative THROUGH the normalisation (R-10), with
//               dN/dq_j linear in q_hat; then du_i = rows of Jp W dR diag(s).
//   centre:     dm/dmu_k = (fx/z) (W0k - (x/z) W2k), (fy/z) (W1k - (y/z) W2k);   dz/dmu_k = W2k.
#pragma once
#include "common.cuh"

namespace nbv {

template <class T>
struct Chain {
  T G[5][10];   // d(mx, my, a, b, c) / d(mu(3), logscale(3), quat(4))
  T dz[3];      // dz / dmu
};

template <class T>
__device__ __forceinline__ T dot3(const T* a, const T* b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

// what every column of the chain needs (computed once per (view, Gaussian))
template <class T>
struct ChainPrefix {
  T W[9], t0[3], t1[3], u0[3], u1[3], v2[3], s[3], qh[4], in;    // in = 1 / |q|
  T ax, cx, ay, cy, iz;
  T u0v2, u1v2, u0u0, u0u1, u1u1;
};

template <class T>
__device__ void chain_prefix(const nbv_camera& cam, const float* mu_f, const float* ls_f, const float* q_f, ChainPrefix<T>& p) {
#pragma unroll
  for (int i = 0; i < 9; ++i) p.W[i] = (T)cam.R_cw[i];
  const T* W = p.W;
  const T fx = (T)cam.fx, fy = (T)cam.fy;
  const T mu[3] = {(T)mu_f[0], (T)mu_f[1], (T)mu_f[2]};
  const T x = W[0] * mu[0] + W[1] * mu[1] + W[2] * mu[2] + (T)cam.t_cw[0];
  const T y = W[3] * mu[0] + W[4] * mu[1] + W[5] * mu[2] + (T)cam.t_cw[1];
  const T z = W[6] * mu[0] + W[7] * mu[1] + W[8] * mu[2] + (T)cam.t_cw[2];
  const T iz = (T)1 / z, xz = x * iz, yz = y * iz, gx = fx * iz, gy = fy * iz;
#pragma unroll
  for (int k = 0; k < 3; ++k) p.s[k] = exp(fmin(fmax((T)ls_f[k], (T)-80), (T)80));
  const T qr[4] = {(T)q_f[0], (T)q_f[1], (T)q_f[2], (T)q_f[3]};
  const T in = rsqrt(qr[0] * qr[0] + qr[1] * qr[1] + qr[2] * qr[2] + qr[3] * qr[3]);
  const T w = qr[0] * in, i = qr[1] * in, j = qr[2] * in, k = qr[3] * in;
  p.qh[0] = w; p.qh[1] = i; p.qh[2] = j; p.qh[3] = k; p.in = in;
  // N(q_hat) = R
  const T R[9] = {w * w + i * i - j * j - k * k, 2 * (i * j - w * k), 2 * (i * k + w * j),
                  2 * (i * j + w * k), w * w - i * i + j * j - k * k, 2 * (j * k - w * i),
                  2 * (i * k - w * j), 2 * (j * k + w * i), w * w - i * i - j * j + k * k};
  // Jp W: the 2 x 3 map from world displacements to pixel displacements
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    p.t0[c] = gx * (W[c] - xz * W[6 + c]);
    p.t1[c] = gy * (W[3 + c] - yz * W[6 + c]);
  }
  // rows of U = (Jp W) R diag(s), and v2 = row 2 of V = W R diag(s)
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    p.u0[c] = (p.t0[0] * R[c] + p.t0[1] * R[3 + c] + p.t0[2] * R[6 + c]) * p.s[c];
    p.u1[c] = (p.t1[0] * R[c] + p.t1[1] * R[3 + c] + p.t1[2] * R[6 + c]) * p.s[c];
    p.v2[c] = (W[6] * R[c] + W[7] * R[3 + c] + W[8] * R[6 + c]) * p.s[c];
  }
  p.u0v2 = dot3(p.u0, p.v2); p.u1v2 = dot3(p.u1, p.v2); p.u0u0 = dot3(p.u0, p.u0); p.u0u1 = dot3(p.u0, p.u1); p.u1u1 = dot3(p.u1, p.u1);
  // du0/dx = ax v2, du0/dz = -iz u0 + cx v2;   du1/dy = ay v2, du1/dz = -iz u1 + cy v2
  p.ax = -gx * iz; p.cx = gx * xz * iz; p.ay = -gy * iz; p.cy = gy * yz * iz; p.iz = iz;
}

// column k of the chain: d(mx, my, a, b, c) / d(parameter k), k = 0..2 position, 3..5 log-scale, 6..9 raw quaternion
template <class T>
__device__ void chain_column(const ChainPrefix<T>& p, int k, T* col5) {
  if (k < 3) {
    const T wx = p.W[k], wy = p.W[3 + k], wz = p.W[6 + k];
    // du0 = (ax wx + cx wz) v2 - iz wz u0 ;  du1 = (ay wy + cy wz) v2 - iz wz u1
    const T e0 = p.ax * wx + p.cx * wz, e1 = p.ay * wy + p.cy * wz, f = -p.iz * wz;
    col5[0] = p.t0[k];
    col5[1] = p.t1[k];
    col5[2] = 2 * (e0 * p.u0v2 + f * p.u0u0);
    col5[3] = e0 * p.u1v2 + e1 * p.u0v2 + 2 * f * p.u0u1;
    col5[4] = 2 * (e1 * p.u1v2 + f * p.u1u1);
  } else if (k < 6) {
    const int m = k - 3;
    col5[0] = 0; col5[1] = 0;
    col5[2] = 2 * p.u0[m] * p.u0[m];
    col5[3] = 2 * p.u0[m] * p.u1[m];
    col5[4] = 2 * p.u1[m] * p.u1[m];
  } else {
    const int e = k - 6;
    const T w = p.qh[0], i = p.qh[1], j = p.qh[2], kk = p.qh[3];
    // D = dN/dq_e at q_hat (each entry linear in q_hat), to be doubled
    T D[9];
    if (e == 0)      { const T d[9] = {w, -kk, j, kk, w, -i, -j, i, w};   for (int n = 0; n < 9; ++n) D[n] = d[n]; }
    else if (e == 1) { const T d[9] = {i, j, kk, j, -i, -w, kk, w, -i};   for (int n = 0; n < 9; ++n) D[n] = d[n]; }
    else if (e == 2) { const T d[9] = {-j, i, w, i, j, kk, -w, kk, -j};   for (int n = 0; n < 9; ++n) D[n] = d[n]; }
    else             { const T d[9] = {-kk, -w, i, w, -kk, j, i, j, kk};  for (int n = 0; n < 9; ++n) D[n] = d[n]; }
    T d0[3], d1[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const T p0 = 2 * (p.t0[0] * D[c] + p.t0[1] * D[3 + c] + p.t0[2] * D[6 + c]) * p.s[c];
      const T p1 = 2 * (p.t1[0] * D[c] + p.t1[1] * D[3 + c] + p.t1[2] * D[6 + c]) * p.s[c];
      d0[c] = (p0 - 2 * p.qh[e] * p.u0[c]) * p.in;
      d1[c] = (p1 - 2 * p.qh[e] * p.u1[c]) * p.in;
    }
    col5[0] = 0; col5[1] = 0;
    col5[2] = 2 * dot3(p.u0, d0);
    col5[3] = dot3(d0, p.u1) + dot3(p.u0, d1);
    col5[4] = 2 * dot3(p.u1, d1);
  }
}

template <class T>
__device__ void projection_chain(const nbv_camera& cam, const float* mu_f, const float* ls_f, const float* q_f, Chain<T>& ch) {
  ChainPrefix<T> p;
  chain_prefix<T>(cam, mu_f, ls_f, q_f, p);
#pragma unroll
  for (int k = 0; k < 10; ++k) {
    T col[5];
    chain_column<T>(p, k, col);
#pragma unroll
    for (int e = 0; e < 5; ++e) ch.G[e][k] = col[e];
  }
#pragma unroll
  for (int m = 0; m < 3; ++m) ch.dz[m] = p.W[6 + m];
}

// S4 accumulates the moments in the monomials xi1^i xi2^j of the whitened pixel offset xi = L^-1 (p - m),
// Sigma2D = L L^T (raster.cu).  The derivatives of alpha are monomials of u = Sigma2D^-1 d = L^-T xi, i.e.
// ux = p00 xi1 + p01 xi2, uy = p10 xi1 + p11 xi2, so each homogeneous degree is mapped by the corresponding symmetric
// power of that 2 x 2 matrix, once per touched Gaussian.
template <class T>
__device__ void moments_to_u_basis(T* m, T p00, T p01, T p10, T p11) {
  T out[15];
  out[0] = m[0];
#pragma unroll
  for (int n = 1; n <= 4; ++n)
#pragma unroll
    for (int j = 0; j <= n; ++j) {
      // coefficients of ux^(n-j) uy^j in xi1^(n-t) xi2^t
      T coef[5] = {1, 0, 0, 0, 0};
#pragma unroll
      for (int sidx = 0; sidx < n; ++sidx) {
        const T a0 = sidx < n - j ? p00 : p10, a1 = sidx < n - j ? p01 : p11;
#pragma unroll
        for (int t = 4; t >= 1; --t)
          if (t <= sidx + 1) coef[t] = coef[t] * a0 + coef[t - 1] * a1;
        coef[0] *= a0;
      }
      T v = 0;
#pragma unroll
      for (int t = 0; t <= n; ++t) v += coef[t] * m[mono_index(n - t, t)];
      out[mono_index(n - j, j)] = v;
    }
#pragma unroll
  for (int i = 0; i < 15; ++i) m[i] = out[i];
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    T* x = m + MOM_X + 6 * c;          // (xi1, xi2, xi1^2, xi1 xi2, xi2^2, 1) -> (ux, uy, ux^2, ux uy, uy^2, 1)
    const T x0 = x[0], x1 = x[1], x2 = x[2], x3 = x[3], x4 = x[4];
    x[0] = p00 * x0 + p01 * x1;
    x[1] = p10 * x0 + p11 * x1;
    x[2] = p00 * p00 * x2 + 2 * p00 * p01 * x3 + p01 * p01 * x4;
    x[3] = p00 * p10 * x2 + (p00 * p11 + p01 * p10) * x3 + p01 * p11 * x4;
    x[4] = p10 * p10 * x2 + 2 * p10 * p11 * x3 + p11 * p11 * x4;
  }
}

// the whitening S4 used, from the splat's conic (-2 qa, -qb, -2 qc) = Sigma2D^-1:  u = L^-T xi
template <class T>
__device__ __forceinline__ void whitened_to_u(T* m, const Splat& sp) {
  const T cA = (T)-2 * (T)sp.qa, cB = -(T)sp.qb, cC = (T)-2 * (T)sp.qc, icC = (T)1 / cC;
  const T i11 = sqrt(fmax(cA * cC - cB * cB, (T)0) * icC), sh = -cB * icC, i22 = sqrt(cC);
  moments_to_u_basis<T>(m, i11, -sh * i22, (T)0, i22);
}

// moments (40, u basis) + chain -> packed 14 x 14 block
//   H = A Q A^T + sum_ch omega_ch [ (A x_ch) e_ch^T + e_ch (A x_ch)^T + W2 e_ch e_ch^T ]
// A (11 x 6): rows of the chain d(mx,my,a,b,c)/d(mu,logscale,quat) against the monomial vector (ux,uy,ux^2,ux uy,uy^2,1) of
// dalpha (the signs of dalpha/dm = -alpha u and of d = p - m cancel), the opacity row kappa; e_ch = dv_ch/dtheta.
template <class T>
__device__ void build_block(const T* mom, const Chain<T>& ch, T kappa, const float* omega, T* H) {
  T A[11][6];
#pragma unroll
  for (int k = 0; k < 10; ++k) {
    A[k][0] = ch.G[0][k]; A[k][1] = ch.G[1][k]; A[k][2] = (T)0.5 * ch.G[2][k]; A[k][3] = ch.G[3][k]; A[k][4] = (T)0.5 * ch.G[4][k]; A[k][5] = 0;
  }
#pragma unroll
  for (int e = 0; e < 5; ++e) A[10][e] = 0;
  A[10][5] = kappa;
  const int ex[6] = {1, 0, 2, 1, 0, 0}, ey[6] = {0, 1, 0, 1, 2, 0};
  T Q[6][6];
#pragma unroll
  for (int i = 0; i < 6; ++i)
#pragma unroll
    for (int j = 0; j < 6; ++j) Q[i][j] = mom[mono_index(ex[i] + ex[j], ey[i] + ey[j])];
  T AQ[11][6];
  for (int k = 0; k < 11; ++k)
#pragma unroll
    for (int j = 0; j < 6; ++j) {
      T v = 0;
#pragma unroll
      for (int i = 0; i < 6; ++i) v += A[k][i] * Q[i][j];
      AQ[k][j] = v;
    }
  for (int i = 0; i < NBLK; ++i) H[i] = 0;
  for (int k = 0; k < 11; ++k)
    for (int l = k; l < 11; ++l) {
      T v = 0;
#pragma unroll
      for (int j = 0; j < 6; ++j) v += AQ[k][j] * A[l][j];
      H[tri(k, l)] = v;
    }
  const T W2 = mom[MOM_W2];
  for (int c = 0; c < 4; ++c) {
    const T om = (T)omega[c];
    if (om == 0) continue;
    const T som = sqrt(om);
    T yv[11];
    for (int k = 0; k < 11; ++k) {
      T v = 0;
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
          const T ek = k < 3 ? ch.dz[k] : (T)0, el = l < 3 ? ch.dz[l] : (T)0;
          H[tri(k, l)] += yv[k] * el + ek * yv[l] + om * W2 * ek * el;
        }
    }
  }
}

// In-place right-looking L D L^T of a packed symmetric positive definite 14 x 14 (upper triangle, row-major); the pivots
// d_j are returned.  With Lambda > 0 the matrix is positive definite; the floor only guards against rounding.
__device__ __forceinline__ void ldl_pivots(double* Mx, double* piv) {
  for (int j = 0; j < P; ++j) {
    const double d = fmax(Mx[tri(j, j)], 1e-300);
    piv[j] = d;
    const double inv = 1.0 / d;
    for (int i = j + 1; i < P; ++i) {
      const double l = Mx[tri(j, i)] * inv;
      for (int k = i; k < P; ++k) Mx[tri(i, k)] = fma(-l, Mx[tri(j, k)], Mx[tri(i, k)]);
    }
  }
}

// trace(A^-1) of a packed symmetric positive definite 14 x 14 (destroyed): A = L D L^T, A^-1 = L^-T D^-1 L^-1, so the trace is
// sum over the columns x = L^-1 e_c of sum_i x_i^2 / d_i
__device__ __forceinline__ double ldl_inverse_trace(double* Mx) {
  double piv[P];
  ldl_pivots(Mx, piv);
  for (int j = 0; j < P; ++j) {
    const double inv = 1.0 / piv[j];
    for (int i = j + 1; i < P; ++i) Mx[tri(j, i)] *= inv;          // row j now holds L_ij, i > j
  }
  double tr = 0.0;
  for (int c = 0; c < P; ++c) {
    double x[P];
    x[c] = 1.0;
    double acc = 1.0 / piv[c];
    for (int i = c + 1; i < P; ++i) {
      double sacc = 0.0;
      for (int j = c; j < i; ++j) sacc = fma(Mx[tri(j, i)], x[j], sacc);
      x[i] = -sacc;
      acc = fma(sacc * sacc, 1.0 / piv[i], acc);
    }
    tr += acc;
  }
  return tr;
}

// every block leaves its partial in partials[blockIdx.x]; the block that finishes last adds them in block order.
// trace_total != nullptr (trace criterion): the sum D_c becomes the score 1 / (S_T - D_c) - 1 / S_T.
__device__ __forceinline__ void ordered_score(double block_total, double* partials, unsigned int* done, float* score,
                                              const double* trace_total = nullptr, double* total_out = nullptr) {
  __shared__ bool last;
  if (threadIdx.x == 0) {
    partials[blockIdx.x] = block_total;
    __threadfence();
    last = atomicAdd(done, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (last && threadIdx.x == 0) {
    __threadfence();
    double t = 0.0;
    for (unsigned b = 0; b < gridDim.x; ++b) t += __ldcg(partials + b);
    if (trace_total) { const double S = *trace_total; t = 1.0 / (S - t) - 1.0 / S; }
    if (score) *score = (float)t;
    if (total_out) *total_out = t;
    *done = 0u;
  }
}

}  // namespace nbv
