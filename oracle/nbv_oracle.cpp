// nbv_oracle.cpp -- CPU ORACLE for the candidate-view scoring hot path of
// arxiv/paper_2602_08266 (object-aware 3DGS next-best-view).
//
// THIS IS TEST INFRASTRUCTURE.  It is a plain, slow, brute-force CPU
// implementation that defines what the CUDA path must compute.  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
// may build, load or call it.  It shares no code, header, table or helper with
// paper_2602_08266_b200/csrc/ and includes nothing from there.
//
// What it follows (P:Lnnn = /root/reference/PAPER.md line nnn, S:Lnnn = SPEC.md,
// R-n = reading n in DESIGN.md "Readings of the paper"):
//   * alpha compositing, T_i = prod_{j<i}(1-alpha_j)            P:L125-129 (Eq. 1)
//   * Gaussian parameters mu, s, r, sigma, c (SH degree 0)
//   * H ~= J^T J, J = Jacobian of the rendering w.r.t. the
//     parameters of each Gaussian; only intra-Gaussian blocks
//   * f(V) = log det(sum_v J_v^T J_v)                            P:L199-205 (Eq. 6)
//   * RGB and depth share position, scale, rotation, opacity;
//     RGB adds the colour coefficients
//   * the 3DGS conventions the paper inherits silently
//     ("follows the original 3DGS pipeline"):            R-1 .. R-8
//     first-order EWA projection + 0.3 px^2 blur, alpha cap 0.99, alpha skip
//     below 1/255, stop before T would drop under 1e-4, depth = sum z a T,
//     ordering by camera-space z of the centre (ties: lower index first).
// Confidence (Eq. 7, 8, 9, 12), log-det gain (Eq. 5, 6) and arg-max are in
// oracle/nbv_oracle.py on top of numpy (library slogdet as the primitive).
//
// No tiles here.  Every pixel walks the global depth order over ALL Gaussians;
// a Gaussian is skipped early at a pixel only by its conservative pixel AABB,
// which cannot change any result (R-5).  Jacobian rows (one per output channel,
// 14 wide) are formed explicitly and J^T J is added densely -- no moment
// factorisation, no screen-space intermediate Hessian.
//
// Two arithmetic paths (R-9):
//   decision path: IEEE binary32, every operation individually rounded in the
//     order written here (compile with -ffp-contract=off; fused multiply-adds
//     only where std::fmaf is spelled out).  It yields everything that decides
//     an integer: the projected splat (centre, conic, depth), the tile rect,
//     the depth order, the per-pixel power, alpha, transmittance and the
//     skip/stop decisions -> tile lists and contributor counts.  The CUDA path
//     must reproduce these bit for bit.
//   value path: binary64.  Colour, depth, blending weights, Jacobians, Hessian
//     blocks.  It walks the contributor sets of the decision path and
//     recomputes alpha and T in double from the binary32 splat.
//   smooth mode (all binary64, contributor sets frozen) exists for the
//     finite-difference self-test only.
//
// Parity pins: tests/test_oracle_*.py (closed forms, finite differences,
// invariants, brute force).  Nothing here is "parity unpinned" except the
// overall NBV choice on the synthetic configs, for which the paper prints no
// worked example.
//
// Build: g++ -O2 -std=c++17 -fopenmp -ffp-contract=off -shared -fPIC

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <memory>
#include <numeric>
#include <vector>

#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr int P = 14;        // mu(3) logscale(3) quat(4) opacity-logit(1) rgb(3)   (R-10)
constexpr int NB = 105;      // packed upper triangle, row-major: idx(r,c)=r*14-r(r-1)/2+(c-r)
constexpr int TILE = 16;     // tile edge of the *tile list* definition only (R-5)

struct Camera {
  int32_t width, height;
  float fx, fy, cx, cy;
  float R[9];  // world->camera, row-major
  float t[3];
};

struct Config {
  float near_plane;   // 0.01
  float blur;         // 0.3
  float alpha_min;    // 1/255
  float alpha_max;    // 0.99
  float t_stop;       // 1e-4
  float power_min;    // -6: below this alpha < 1/255 for every sigma < 1
  float bg[3];        // background colour (depth background is 0)
  int32_t channel_mask;      // bit0..2 = r,g,b ; bit3 = depth
  float channel_weight[4];   // omega_ch (inverse noise variance per channel, R-12)
  int32_t opacity_coord;     // 0 = logit (default), 1 = sigma itself
};

inline int tri(int r, int c) { return r * P - r * (r - 1) / 2 + (c - r); }

// ---------------------------------------------------------------------------
// decision-path primitives (binary32)
// ---------------------------------------------------------------------------
inline uint32_t f2u(float f) { uint32_t u; std::memcpy(&u, &f, 4); return u; }
inline float u2f(uint32_t u) { float f; std::memcpy(&f, &u, 4); return f; }

// exp on [-80, 80] in binary32, fully specified (R-9): Cody-Waite reduction by
// ln2 = hi + lo, degree-6 Taylor polynomial in Horner form with fused
// multiply-adds, scaling by 2^k through the exponent field.
inline float exp_spec(float x) {
  const float LOG2E = 0x1.715476p+0f;
  const float MAGIC = 12582912.0f;        // 1.5 * 2^23: adding it rounds to an integer
  const float LN2_HI = 0x1.62e4p-1f;      // 15 significant bits -> k*LN2_HI exact
  const float LN2_LO = 0x1.7f7d1cp-20f;
  float t = std::fmaf(x, LOG2E, MAGIC);
  float kf = t - MAGIC;
  float r = std::fmaf(kf, -LN2_HI, x);
  r = std::fmaf(kf, -LN2_LO, r);
  float p = 0x1.6c16c2p-10f;              // 1/720
  p = std::fmaf(p, r, 0x1.111112p-7f);    // 1/120
  p = std::fmaf(p, r, 0x1.555556p-5f);    // 1/24
  p = std::fmaf(p, r, 0x1.555556p-3f);    // 1/6
  p = std::fmaf(p, r, 0.5f);
  p = std::fmaf(p, r, 1.0f);
  p = std::fmaf(p, r, 1.0f);
  int32_t k = (int32_t)f2u(t) - (int32_t)f2u(MAGIC);
  return u2f(f2u(p) + ((uint32_t)k << 23));
}

// Post-activation, view-independent part of one Gaussian (binary32, R-9).
struct Act {
  float M[9];   // R(q_hat) * diag(s), row-major
  float sigma;
  bool ok;
};

inline Act activate(const float* logscale, const float* quat, float sigma) {
  Act o;
  float s[3];
  for (int k = 0; k < 3; ++k) {
    float l = std::fmin(std::fmax(logscale[k], -80.0f), 80.0f);
    s[k] = exp_spec(l);
  }
  float w = quat[0], x = quat[1], y = quat[2], z = quat[3];
  float n2 = ((w * w + x * x) + y * y) + z * z;
  o.ok = (n2 > 0.0f) && std::isfinite(n2) && (sigma > 0.0f) && (sigma < 1.0f);
  float n = std::sqrt(n2);
  w = w / n; x = x / n; y = y / n; z = z / n;
  float xx = x * x, yy = y * y, zz = z * z;
  float xy = x * y, xz = x * z, yz = y * z;
  float wx = w * x, wy = w * y, wz = w * z;
  float R[9];
  R[0] = 1.0f - 2.0f * (yy + zz); R[1] = 2.0f * (xy - wz);        R[2] = 2.0f * (xz + wy);
  R[3] = 2.0f * (xy + wz);        R[4] = 1.0f - 2.0f * (xx + zz); R[5] = 2.0f * (yz - wx);
  R[6] = 2.0f * (xz - wy);        R[7] = 2.0f * (yz + wx);        R[8] = 1.0f - 2.0f * (xx + yy);
  for (int i = 0; i < 3; ++i)
    for (int k = 0; k < 3; ++k) o.M[3 * i + k] = R[3 * i + k] * s[k];
  o.sigma = sigma;
  return o;
}

// The projected splat of the decision path.
struct Splat {
  float mx, my;        // centre in pixels
  float qa, qb, qc;    // power(d) = qa dx^2 + qb dx dy + qc dy^2 ; (qa,qb,qc) = (-A/2, -B, -C/2), conic (A,B,C)
  float z;             // camera-space depth of the centre
  float sigma;
  float a, b, c;       // Sigma2D entries (diagnostic / parity)
  int32_t tx0, ty0, tx1, ty1;  // half-open tile rect
  bool visible;
};

// Conservative upper bound of ln(255 sigma) (tangent of ln at 0.75 on the mantissa), >= 0.
inline float log_bound(float sigma) {
  float x = 255.0f * sigma;
  if (!(x > 1.0f)) x = 1.0f;
  uint32_t u = f2u(x);
  int32_t e = (int32_t)((u >> 23) & 0xffu) - 126;          // x = m * 2^e, m in [0.5,1)
  float m = u2f((u & 0x007fffffu) | 0x3f000000u);
  const float LN2 = 0x1.62e43p-1f;
  float lm = m * 0x1.555556p+0f + (-0x1.49a588p+0f);       // (m - 0.75)/0.75 + ln 0.75
  return (float)e * LN2 + lm;
}

inline Splat project(const Camera& cam, const Config& cfg, const float* mu, const Act& act) {
  Splat sp{};
  sp.visible = false;
  sp.sigma = act.sigma;
  const float* W = cam.R;
  float x = ((W[0] * mu[0] + W[1] * mu[1]) + W[2] * mu[2]) + cam.t[0];
  float y = ((W[3] * mu[0] + W[4] * mu[1]) + W[5] * mu[2]) + cam.t[1];
  float z = ((W[6] * mu[0] + W[7] * mu[1]) + W[8] * mu[2]) + cam.t[2];
  if (!(z > cfg.near_plane)) return sp;                                  // R-2
  float iz = 1.0f / z;
  float xz = x * iz, yz = y * iz;
  sp.mx = cam.fx * xz + cam.cx;
  sp.my = cam.fy * yz + cam.cy;
  sp.z = z;
  // J = [[fx/z, 0, -fx x/z^2],[0, fy/z, -fy y/z^2]]   (first-order EWA, R-3)
  float j00 = cam.fx * iz, j02 = -(j00 * xz);
  float j11 = cam.fy * iz, j12 = -(j11 * yz);
  float T0[3], T1[3];
  for (int k = 0; k < 3; ++k) {
    T0[k] = j00 * W[k] + j02 * W[6 + k];
    T1[k] = j11 * W[3 + k] + j12 * W[6 + k];
  }
  float U0[3], U1[3];                                                     // U = J W R S
  for (int k = 0; k < 3; ++k) {
    U0[k] = (T0[0] * act.M[k] + T0[1] * act.M[3 + k]) + T0[2] * act.M[6 + k];
    U1[k] = (T1[0] * act.M[k] + T1[1] * act.M[3 + k]) + T1[2] * act.M[6 + k];
  }
  float a = ((U0[0] * U0[0] + U0[1] * U0[1]) + U0[2] * U0[2]) + cfg.blur;
  float b = (U0[0] * U1[0] + U0[1] * U1[1]) + U0[2] * U1[2];
  float c = ((U1[0] * U1[0] + U1[1] * U1[1]) + U1[2] * U1[2]) + cfg.blur;
  float det = a * c - b * b;
  if (!(det > 0.0f) || !std::isfinite(det)) return sp;
  sp.a = a; sp.b = b; sp.c = c;
  sp.qa = -0.5f * (c / det);
  sp.qb = b / det;
  sp.qc = -0.5f * (a / det);
  // support: {d : d^T Sigma2D^-1 d <= rho^2} has the exact AABB rho*sqrt(a) x rho*sqrt(c);
  // rho^2 is inflated so that binary32 rounding can never exclude a pixel with alpha >= 1/255.
  float rho2 = 2.02f * log_bound(act.sigma) + 0.05f;
  float hx = std::sqrt(rho2 * a) + 1.0f;
  float hy = std::sqrt(rho2 * c) + 1.0f;
  if (!(std::fabs(sp.mx) <= 1.0e6f) || !(std::fabs(sp.my) <= 1.0e6f)) return sp;
  if (!(hx <= 2.0e6f)) hx = 2.0e6f;
  if (!(hy <= 2.0e6f)) hy = 2.0e6f;
  int TX = (cam.width + TILE - 1) / TILE, TY = (cam.height + TILE - 1) / TILE;
  float fx0 = std::floor((sp.mx - hx) * 0.0625f), fx1 = std::floor((sp.mx + hx) * 0.0625f) + 1.0f;
  float fy0 = std::floor((sp.my - hy) * 0.0625f), fy1 = std::floor((sp.my + hy) * 0.0625f) + 1.0f;
  sp.tx0 = (int32_t)std::fmin(std::fmax(fx0, 0.0f), (float)TX);
  sp.tx1 = (int32_t)std::fmin(std::fmax(fx1, 0.0f), (float)TX);
  sp.ty0 = (int32_t)std::fmin(std::fmax(fy0, 0.0f), (float)TY);
  sp.ty1 = (int32_t)std::fmin(std::fmax(fy1, 0.0f), (float)TY);
  if (sp.tx1 <= sp.tx0 || sp.ty1 <= sp.ty0) return sp;
  sp.visible = true;
  return sp;
}

// Decision at one (pixel, Gaussian): returns 0 = skipped, 1 = composited, 2 = stop (not composited).
// On 1 it updates T.  alpha (binary32) and the clamp flag are returned for the value path.
inline int decide(const Config& cfg, const Splat& sp, float px, float py, float& T, bool& clamped) {
  float dx = px - sp.mx, dy = py - sp.my;
  float power = std::fmaf(dx, std::fmaf(sp.qa, dx, sp.qb * dy), (sp.qc * dy) * dy);
  if (!(power <= 0.0f) || power < cfg.power_min) return 0;   // also rejects NaN
  float g = exp_spec(power);
  float a = sp.sigma * g;
  if (a < cfg.alpha_min) return 0;                    // R-4
  clamped = a > cfg.alpha_max;
  float alpha = clamped ? cfg.alpha_max : a;
  float Tn = T * (1.0f - alpha);
  if (Tn < cfg.t_stop) return 2;                      // R-4: stop BEFORE compositing
  T = Tn;
  return 1;
}

// ---------------------------------------------------------------------------
// value path (binary64)
// ---------------------------------------------------------------------------
struct SplatV {               // what the value path reads about a projected Gaussian
  double mx, my, ca, cb, cc;  // centre, conic (A,B,C) = Sigma2D^-1
  double z, sigma;
  double rgb[3];
};

// d(mx,my,a,b,c)/d(mu,logscale,quat) (5x10) and dz/dmu, in binary64 from the raw parameters.
struct Chain {
  double G[5][10];
  double dz[3];
  // smooth-mode forward values
  double mx, my, a, b, c, z;
  bool front;
};

inline void quat_R(const double q[4], double R[9]) {
  double w = q[0], x = q[1], y = q[2], z = q[3];
  R[0] = 1 - 2 * (y * y + z * z); R[1] = 2 * (x * y - w * z);     R[2] = 2 * (x * z + w * y);
  R[3] = 2 * (x * y + w * z);     R[4] = 1 - 2 * (x * x + z * z); R[5] = 2 * (y * z - w * x);
  R[6] = 2 * (x * z - w * y);     R[7] = 2 * (y * z + w * x);     R[8] = 1 - 2 * (x * x + y * y);
}

// dR/dq_hat_j for unit quaternion (w,x,y,z)
inline void quat_dR(const double q[4], int j, double D[9]) {
  double w = q[0], x = q[1], y = q[2], z = q[3];
  switch (j) {
    case 0: { double d[9] = {0, -2 * z, 2 * y, 2 * z, 0, -2 * x, -2 * y, 2 * x, 0}; std::memcpy(D, d, sizeof d); } break;
    case 1: { double d[9] = {0, 2 * y, 2 * z, 2 * y, -4 * x, -2 * w, 2 * z, 2 * w, -4 * x}; std::memcpy(D, d, sizeof d); } break;
    case 2: { double d[9] = {-4 * y, 2 * x, 2 * w, 2 * x, 0, 2 * z, -2 * w, 2 * z, -4 * y}; std::memcpy(D, d, sizeof d); } break;
    default: { double d[9] = {-4 * z, -2 * w, 2 * x, 2 * w, -4 * z, 2 * y, 2 * x, 2 * y, 0}; std::memcpy(D, d, sizeof d); } break;
  }
}

// Sigma2D = Tm Sigma3D Tm^T (2x2 symmetric -> a,b,c) for Tm (2x3), Sigma3D symmetric 3x3 (row-major 9)
inline void sandwich(const double Tm[6], const double S3[9], double& a, double& b, double& c) {
  double TS[6];
  for (int i = 0; i < 2; ++i)
    for (int k = 0; k < 3; ++k)
      TS[3 * i + k] = Tm[3 * i] * S3[k] + Tm[3 * i + 1] * S3[3 + k] + Tm[3 * i + 2] * S3[6 + k];
  a = TS[0] * Tm[0] + TS[1] * Tm[1] + TS[2] * Tm[2];
  b = TS[0] * Tm[3] + TS[1] * Tm[4] + TS[2] * Tm[5];
  c = TS[3] * Tm[3] + TS[4] * Tm[4] + TS[5] * Tm[5];
}

// Binary64 projection and its derivatives.  mu, logscale, quat (raw, any norm) as doubles.
inline Chain chain(const Camera& cam, const Config& cfg, const double mu[3], const double ls[3], const double q[4]) {
  Chain ch{};
  double W[9], t[3];
  for (int i = 0; i < 9; ++i) W[i] = cam.R[i];
  for (int i = 0; i < 3; ++i) t[i] = cam.t[i];
  double fx = cam.fx, fy = cam.fy;
  double x = W[0] * mu[0] + W[1] * mu[1] + W[2] * mu[2] + t[0];
  double y = W[3] * mu[0] + W[4] * mu[1] + W[5] * mu[2] + t[1];
  double z = W[6] * mu[0] + W[7] * mu[1] + W[8] * mu[2] + t[2];
  ch.front = z > (double)cfg.near_plane;
  ch.z = z;
  ch.mx = fx * x / z + cam.cx;
  ch.my = fy * y / z + cam.cy;
  double J[6] = {fx / z, 0, -fx * x / (z * z), 0, fy / z, -fy * y / (z * z)};
  double Tm[6];
  for (int i = 0; i < 2; ++i)
    for (int k = 0; k < 3; ++k) Tm[3 * i + k] = J[3 * i] * W[k] + J[3 * i + 1] * W[3 + k] + J[3 * i + 2] * W[6 + k];
  double qn = std::sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
  double qh[4] = {q[0] / qn, q[1] / qn, q[2] / qn, q[3] / qn};
  double R[9];
  quat_R(qh, R);
  double s2[3] = {std::exp(2 * ls[0]), std::exp(2 * ls[1]), std::exp(2 * ls[2])};
  double S3[9];
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j)
      S3[3 * i + j] = R[3 * i] * s2[0] * R[3 * j] + R[3 * i + 1] * s2[1] * R[3 * j + 1] + R[3 * i + 2] * s2[2] * R[3 * j + 2];
  sandwich(Tm, S3, ch.a, ch.b, ch.c);
  ch.a += (double)cfg.blur;
  ch.c += (double)cfg.blur;

  // --- d/dmu ---
  // dm/dmu = J W ; dz/dmu = W[2,:]
  for (int k = 0; k < 3; ++k) {
    ch.G[0][k] = Tm[k];
    ch.G[1][k] = Tm[3 + k];
    ch.dz[k] = W[6 + k];
  }
  // dSigma2D/dmu_k = dT S3 T^T + T S3 dT^T with dT = (sum_j dJ/dp_j W[j][k]) W
  double dJ[3][6] = {
      {0, 0, -fx / (z * z), 0, 0, 0},
      {0, 0, 0, 0, 0, -fy / (z * z)},
      {-fx / (z * z), 0, 2 * fx * x / (z * z * z), 0, -fy / (z * z), 2 * fy * y / (z * z * z)}};
  for (int k = 0; k < 3; ++k) {
    double dJk[6];
    for (int e = 0; e < 6; ++e) dJk[e] = dJ[0][e] * W[k] + dJ[1][e] * W[3 + k] + dJ[2][e] * W[6 + k];
    double dT[6];
    for (int i = 0; i < 2; ++i)
      for (int c = 0; c < 3; ++c) dT[3 * i + c] = dJk[3 * i] * W[c] + dJk[3 * i + 1] * W[3 + c] + dJk[3 * i + 2] * W[6 + c];
    // E = dT S3 T^T (2x2); dSigma = E + E^T
    double dTS[6];
    for (int i = 0; i < 2; ++i)
      for (int c = 0; c < 3; ++c) dTS[3 * i + c] = dT[3 * i] * S3[c] + dT[3 * i + 1] * S3[3 + c] + dT[3 * i + 2] * S3[6 + c];
    double E00 = dTS[0] * Tm[0] + dTS[1] * Tm[1] + dTS[2] * Tm[2];
    double E01 = dTS[0] * Tm[3] + dTS[1] * Tm[4] + dTS[2] * Tm[5];
    double E10 = dTS[3] * Tm[0] + dTS[4] * Tm[1] + dTS[5] * Tm[2];
    double E11 = dTS[3] * Tm[3] + dTS[4] * Tm[4] + dTS[5] * Tm[5];
    ch.G[2][k] = 2 * E00;
    ch.G[3][k] = E01 + E10;
    ch.G[4][k] = 2 * E11;
  }
  // --- d/dlogscale_k : dSigma3D = 2 s_k^2 r_k r_k^T (r_k = column k of R) ---
  for (int k = 0; k < 3; ++k) {
    double v0 = Tm[0] * R[k] + Tm[1] * R[3 + k] + Tm[2] * R[6 + k];
    double v1 = Tm[3] * R[k] + Tm[4] * R[3 + k] + Tm[5] * R[6 + k];
    ch.G[0][3 + k] = 0; ch.G[1][3 + k] = 0;
    ch.G[2][3 + k] = 2 * s2[k] * v0 * v0;
    ch.G[3][3 + k] = 2 * s2[k] * v0 * v1;
    ch.G[4][3 + k] = 2 * s2[k] * v1 * v1;
  }
  // --- d/dquat: through q_hat = q/|q| : d/dq_j = sum_i d/dq_hat_i (delta_ij - qh_i qh_j)/|q| ---
  double dh[4][3];  // derivative of (a,b,c) w.r.t. q_hat_i
  for (int i = 0; i < 4; ++i) {
    double D[9];
    quat_dR(qh, i, D);
    double dS3[9];  // D S^2 R^T + R S^2 D^T
    for (int r = 0; r < 3; ++r)
      for (int c = 0; c < 3; ++c) {
        double v = 0;
        for (int k = 0; k < 3; ++k) v += D[3 * r + k] * s2[k] * R[3 * c + k] + R[3 * r + k] * s2[k] * D[3 * c + k];
        dS3[3 * r + c] = v;
      }
    sandwich(Tm, dS3, dh[i][0], dh[i][1], dh[i][2]);
  }
  for (int j = 0; j < 4; ++j) {
    ch.G[0][6 + j] = 0; ch.G[1][6 + j] = 0;
    for (int e = 0; e < 3; ++e) {
      double v = 0;
      for (int i = 0; i < 4; ++i) v += dh[i][e] * ((i == j ? 1.0 : 0.0) - qh[i] * qh[j]) / qn;
      ch.G[2 + e][6 + j] = v;
    }
  }
  return ch;
}

// One pixel's contributor, as the value path sees it.
struct Contrib {
  int32_t g;       // Gaussian index
  bool clamped;
};

// Value-path arithmetic for one pixel: given its ordered contributors, composite in binary64
// and (optionally) add every contributor's J^T J into H.
//   out4 = (r,g,b,depth), Tend = transmittance after the last contributor.
// Hadd(g) must return a pointer to that Gaussian's 105 packed doubles, or nullptr to skip.
template <class HAdd>
inline void pixel_value(const Config& cfg, double px, double py, const Contrib* cs, int n,
                        const SplatV* sv, const Chain* chains, double out4[4], double& Tend,
                        bool want_hessian, HAdd&& hadd) {
  const double amax = (double)cfg.alpha_max;
  // forward: alpha_i, T_i, w_i = alpha_i T_i            (Eq. 1)
  std::vector<double> al(n), Ti(n);
  double T = 1.0;
  double acc[4] = {0, 0, 0, 0};
  for (int i = 0; i < n; ++i) {
    const SplatV& s = sv[cs[i].g];
    double dx = px - s.mx, dy = py - s.my;
    double power = -0.5 * (s.ca * dx * dx + s.cc * dy * dy) - s.cb * dx * dy;
    double a = cs[i].clamped ? amax : s.sigma * std::exp(power);
    al[i] = a;
    Ti[i] = T;
    double w = a * T;
    acc[0] += s.rgb[0] * w; acc[1] += s.rgb[1] * w; acc[2] += s.rgb[2] * w; acc[3] += s.z * w;
    T *= (1.0 - a);
  }
  Tend = T;
  out4[0] = acc[0] + cfg.bg[0] * T; out4[1] = acc[1] + cfg.bg[1] * T; out4[2] = acc[2] + cfg.bg[2] * T;
  out4[3] = acc[3];                                      // R-6: depth background 0
  if (!want_hessian) return;
  // backward sweep: Splus_i = sum_{j>i} v_j w_j + v_bg T_end ; beta_i = dy/dalpha_i = T_i v_i - Splus_i/(1-alpha_i)
  double Sp[4] = {cfg.bg[0] * T, cfg.bg[1] * T, cfg.bg[2] * T, 0.0};
  for (int i = n - 1; i >= 0; --i) {
    const int g = cs[i].g;
    const SplatV& s = sv[g];
    const double v[4] = {s.rgb[0], s.rgb[1], s.rgb[2], s.z};
    const double a = al[i], w = a * Ti[i];
    double beta[4];
    for (int c = 0; c < 4; ++c) beta[c] = Ti[i] * v[c] - Sp[c] / (1.0 - a);
    for (int c = 0; c < 4; ++c) Sp[c] += v[c] * w;
    double* H = hadd(g);
    if (!H) continue;
    // dalpha/dtheta (14): zero where the 0.99 clamp is active (R-11)
    double da[P];
    for (int k = 0; k < P; ++k) da[k] = 0.0;
    if (!cs[i].clamped) {
      double dx = px - s.mx, dy = py - s.my;
      double ux = s.ca * dx + s.cb * dy, uy = s.cb * dx + s.cc * dy;   // u = Sigma2D^-1 d
      // dalpha/d(mx,my,a,b,c) = alpha (ux, uy, ux^2/2, ux uy, uy^2/2)
      const double h5[5] = {a * ux, a * uy, 0.5 * a * ux * ux, a * ux * uy, 0.5 * a * uy * uy};
      const Chain& ch = chains[g];
      for (int k = 0; k < 10; ++k) {
        double acc2 = 0;
        for (int e = 0; e < 5; ++e) acc2 += h5[e] * ch.G[e][k];
        da[k] = acc2;
      }
      da[10] = cfg.opacity_coord == 0 ? a * (1.0 - s.sigma) : a / s.sigma;   // R-10
    }
    for (int c = 0; c < 4; ++c) {
      if (!((cfg.channel_mask >> c) & 1)) continue;
      double Jr[P];
      for (int k = 0; k < P; ++k) Jr[k] = beta[c] * da[k];
      if (c < 3) Jr[11 + c] += w;                          // d colour / d rgb parameter
      else for (int k = 0; k < 3; ++k) Jr[k] += w * chains[g].dz[k];   // d z / d mu
      const double om = (double)cfg.channel_weight[c];
      for (int r = 0; r < P; ++r) {
        const double jr = om * Jr[r];
        if (jr == 0.0) continue;
        double* row = H + tri(r, r);
        for (int cc = r; cc < P; ++cc) row[cc - r] += jr * Jr[cc];
      }
    }
  }
}

// ---------------------------------------------------------------------------
// scene object
// ---------------------------------------------------------------------------
// ---------------------------------------------------------------------------
// Object-mask output.
//   O' = sum_i softmax(o_i) alpha_i T_i                                  P:L125-129 (Eq. 1)
//   O  = O' + e_bg (1 - 1^T O') = O' + e_bg T_end   (softmax sums to 1)  P:L135-139 (Eq. 2)
// "masks use the object vector" next to position, scale, rotation and opacity: the
// block of a Gaussian has L = 11 + K parameters [mu(3) logscale(3) quat(4) opacity | logits(K)],
// packed upper triangle row-major, idx(r,c) = r*L - r(r-1)/2 + (c-r).
// Row of output channel k for contributor i:
//   J_k = beta_k * dalpha_i/dtheta_geo  (+)  w_i * dp_k/do,   dp_k/do_j = p_k (delta_kj - p_j),
//   beta_k = T_i p_ik - Splus_k / (1 - alpha_i),  Splus = sum_{j>i} p_j w_j + e_bg T_end.
// Explicit rows, dense J^T J: no moment factorisation (the CUDA path has one).
// ---------------------------------------------------------------------------
inline size_t triL(int r, int c, int L) { return (size_t)r * L - (size_t)r * (r - 1) / 2 + (size_t)(c - r); }

// prob: N x K softmax probabilities (binary64).  outK: K mask values of the pixel.
// hadd(g) -> pointer to that Gaussian's L(L+1)/2 packed doubles, or nullptr to skip.
template <class HAdd>
inline void pixel_value_mask(const Config& cfg, int K, int bgch, double px, double py, const Contrib* cs, int n,
                             const SplatV* sv, const Chain* chains, const double* prob, double* outK, double& Tend,
                             bool want_hessian, HAdd&& hadd) {
  const double amax = (double)cfg.alpha_max;
  const int L = 11 + K;
  std::vector<double> al(n), Ti(n);
  double T = 1.0;
  for (int k = 0; k < K; ++k) outK[k] = 0.0;
  for (int i = 0; i < n; ++i) {
    const SplatV& s = sv[cs[i].g];
    double dx = px - s.mx, dy = py - s.my;
    double power = -0.5 * (s.ca * dx * dx + s.cc * dy * dy) - s.cb * dx * dy;
    double a = cs[i].clamped ? amax : s.sigma * std::exp(power);
    al[i] = a;
    Ti[i] = T;
    const double w = a * T;
    const double* p = prob + (size_t)cs[i].g * K;
    for (int k = 0; k < K; ++k) outK[k] += p[k] * w;
    T *= (1.0 - a);
  }
  Tend = T;
  outK[bgch] += T;                                           // Eq. 2: the residual goes to the background channel
  if (!want_hessian) return;
  std::vector<double> Sp(K, 0.0), beta(K), Jr(L), da(11);
  Sp[bgch] = T;
  for (int i = n - 1; i >= 0; --i) {
    const int g = cs[i].g;
    const SplatV& s = sv[g];
    const double* p = prob + (size_t)g * K;
    const double a = al[i], w = a * Ti[i];
    for (int k = 0; k < K; ++k) beta[k] = Ti[i] * p[k] - Sp[k] / (1.0 - a);
    for (int k = 0; k < K; ++k) Sp[k] += p[k] * w;
    double* H = hadd(g);
    if (!H) continue;
    for (int k = 0; k < 11; ++k) da[k] = 0.0;
    if (!cs[i].clamped) {                                    // R-11: zero derivative at the 0.99 clamp
      double dx = px - s.mx, dy = py - s.my;
      double ux = s.ca * dx + s.cb * dy, uy = s.cb * dx + s.cc * dy;
      const double h5[5] = {a * ux, a * uy, 0.5 * a * ux * ux, a * ux * uy, 0.5 * a * uy * uy};
      const Chain& ch = chains[g];
      for (int k = 0; k < 10; ++k) {
        double acc2 = 0;
        for (int e = 0; e < 5; ++e) acc2 += h5[e] * ch.G[e][k];
        da[k] = acc2;
      }
      da[10] = cfg.opacity_coord == 0 ? a * (1.0 - s.sigma) : a / s.sigma;   // R-10
    }
    for (int k = 0; k < K; ++k) {
      for (int r = 0; r < 11; ++r) Jr[r] = beta[k] * da[r];
      for (int j = 0; j < K; ++j) Jr[11 + j] = w * p[k] * ((j == k ? 1.0 : 0.0) - p[j]);   // softmax Jacobian
      for (int r = 0; r < L; ++r) {
        const double jr = Jr[r];
        if (jr == 0.0) continue;
        double* row = H + triL(r, r, L);
        for (int c = r; c < L; ++c) row[c - r] += jr * Jr[c];
      }
    }
  }
}

struct Scene {
  int N = 0, K = 0;
  std::vector<float> mean, logscale, quat, opacity, rgb;
  std::vector<Act> act;
  Config cfg;
  bool bad_data = false;
};

struct View {                       // decision-path products for one camera
  std::vector<Splat> sp;            // per Gaussian
  std::vector<int32_t> order;       // visible Gaussians, sorted by (z bits, index)
};

View make_view(const Scene& sc, const Camera& cam) {
  View v;
  v.sp.resize(sc.N);
#pragma omp parallel for schedule(static)
  for (int g = 0; g < sc.N; ++g) v.sp[g] = project(cam, sc.cfg, &sc.mean[3 * g], sc.act[g]);
  for (int g = 0; g < sc.N; ++g)
    if (v.sp[g].visible) v.order.push_back(g);
  std::stable_sort(v.order.begin(), v.order.end(), [&](int32_t a, int32_t b) {
    uint32_t za = f2u(v.sp[a].z), zb = f2u(v.sp[b].z);
    return za != zb ? za < zb : a < b;                                   // R-7
  });
  return v;
}

// Walk one pixel through the global depth order (decision path).  Appends contributors.
inline void walk_pixel(const Scene& sc, const View& v, int ix, int iy, std::vector<Contrib>& out, float& Tend32) {
  const float px = (float)ix + 0.5f, py = (float)iy + 0.5f;              // R-1
  const int tx = ix / TILE, ty = iy / TILE;
  float T = 1.0f;
  out.clear();
  for (int32_t g : v.order) {
    const Splat& sp = v.sp[g];
    // conservative pixel AABB (the tile rect in pixels); cannot change any result (R-5)
    if (tx < sp.tx0 || tx >= sp.tx1 || ty < sp.ty0 || ty >= sp.ty1) continue;
    bool clamped = false;
    int d = decide(sc.cfg, sp, px, py, T, clamped);
    if (d == 2) break;
    if (d == 1) out.push_back({g, clamped});
  }
  Tend32 = T;
}

void fill_splatv(const Scene& sc, const View& v, std::vector<SplatV>& sv) {
  sv.resize(sc.N);
  for (int g = 0; g < sc.N; ++g) {
    const Splat& s = v.sp[g];
    SplatV& o = sv[g];
    o.mx = s.mx; o.my = s.my;
    o.ca = -2.0 * (double)s.qa; o.cb = -(double)s.qb; o.cc = -2.0 * (double)s.qc;
    o.z = s.z; o.sigma = s.sigma;
    for (int c = 0; c < 3; ++c) o.rgb[c] = sc.rgb[3 * g + c];
  }
}

// Sparse Hessian accumulator of one BAND of image rows (chunks of Gaussians allocated on first touch; `nb` doubles
// per Gaussian).  The sum over the pixels of a view is taken band by band: every band of BAND_ROWS rows owns one
// accumulator, filled by a single thread in row-major pixel order, and the bands are added in band order.  The result
// therefore does not depend on the number of threads or on the OpenMP schedule (run-to-run deterministic).
struct HAcc {
  static constexpr int CH = 16;
  size_t nb;
  std::vector<std::unique_ptr<double[]>> chunks;
  HAcc(int N, size_t nb_) : nb(nb_), chunks((N + CH - 1) / CH) {}
  double* at(int g) {
    auto& c = chunks[g / CH];
    if (!c) { c.reset(new double[(size_t)CH * nb]); std::fill(c.get(), c.get() + (size_t)CH * nb, 0.0); }
    return c.get() + (size_t)(g % CH) * nb;
  }
};
constexpr int BAND_ROWS = 8;

// blocks += (sum over the bands, in band order): the view's sum is formed first, then added to what `blocks` held
void add_bands(const std::vector<std::unique_ptr<HAcc>>& bands, int N, size_t nb, double* blocks) {
  const int nch = (N + HAcc::CH - 1) / HAcc::CH;
#pragma omp parallel
  {
    std::vector<double> sum((size_t)HAcc::CH * nb);
#pragma omp for schedule(dynamic, 64)
    for (int c = 0; c < nch; ++c) {
      bool any = false;
      for (size_t b = 0; b < bands.size(); ++b) {
        if (!bands[b] || !bands[b]->chunks[c]) continue;
        const double* src = bands[b]->chunks[c].get();
        if (!any) { std::copy(src, src + sum.size(), sum.begin()); any = true; }
        else for (size_t i = 0; i < sum.size(); ++i) sum[i] += src[i];
      }
      if (!any) continue;
      const int g0 = c * HAcc::CH, g1 = std::min(N, g0 + HAcc::CH);
      double* dst = blocks + (size_t)g0 * nb;
      for (size_t i = 0; i < (size_t)(g1 - g0) * nb; ++i) dst[i] += sum[i];
    }
  }
}

}  // namespace

// ===========================================================================
// C interface (ctypes)
// ===========================================================================
extern "C" {

void* orc_create(int N, int K, const float* mean, const float* logscale, const float* quat,
                 const float* opacity, const float* rgb, const Config* cfg) {
  Scene* sc = new Scene;
  sc->N = N; sc->K = K;
  sc->mean.assign(mean, mean + 3 * (size_t)N);
  sc->logscale.assign(logscale, logscale + 3 * (size_t)N);
  sc->quat.assign(quat, quat + 4 * (size_t)N);
  sc->opacity.assign(opacity, opacity + (size_t)N);
  sc->rgb.assign(rgb, rgb + 3 * (size_t)N);
  sc->cfg = *cfg;
  sc->act.resize(N);
  for (int g = 0; g < N; ++g) {
    sc->act[g] = activate(&sc->logscale[3 * g], &sc->quat[4 * g], sc->opacity[g]);
    if (!sc->act[g].ok) sc->bad_data = true;
  }
  return sc;
}

void orc_destroy(void* h) { delete (Scene*)h; }
int orc_bad_data(void* h) { return ((Scene*)h)->bad_data ? 1 : 0; }
float orc_exp_spec(float x) { return exp_spec(x); }
float orc_log_bound(float s) { return log_bound(s); }

// post-activation M = R(q_hat) diag(s) per Gaussian (N x 9)
void orc_activation(void* h, float* M) {
  Scene* sc = (Scene*)h;
  for (int g = 0; g < sc->N; ++g) std::memcpy(M + 9 * (size_t)g, sc->act[g].M, 36);
}

// decision-path projection: visible (N), rec (N x 9: mx,my,qa,qb,qc,z,a,b,c), rect (N x 4: tx0,ty0,tx1,ty1)
void orc_project(void* h, const Camera* cam, int32_t* visible, float* rec, int32_t* rect) {
  Scene* sc = (Scene*)h;
  View v = make_view(*sc, *cam);
  for (int g = 0; g < sc->N; ++g) {
    const Splat& s = v.sp[g];
    visible[g] = s.visible ? 1 : 0;
    float* r = rec + 9 * (size_t)g;
    r[0] = s.mx; r[1] = s.my; r[2] = s.qa; r[3] = s.qb; r[4] = s.qc; r[5] = s.z; r[6] = s.a; r[7] = s.b; r[8] = s.c;
    int32_t* q = rect + 4 * (size_t)g;
    q[0] = s.tx0; q[1] = s.ty0; q[2] = s.tx1; q[3] = s.ty1;
  }
}

// depth order of the visible Gaussians; returns their number
int orc_depth_order(void* h, const Camera* cam, int32_t* order) {
  Scene* sc = (Scene*)h;
  View v = make_view(*sc, *cam);
  std::copy(v.order.begin(), v.order.end(), order);
  return (int)v.order.size();
}

// tile lists: tile t (row-major over ceil(W/16) x ceil(H/16)) lists the visible Gaussians whose
// rect contains t, in depth order.  offsets has tiles+1 entries.  Returns the total (even if > cap;
// ids is filled only when total <= cap).
int64_t orc_tile_lists(void* h, const Camera* cam, int64_t* offsets, int32_t* ids, int64_t cap) {
  Scene* sc = (Scene*)h;
  View v = make_view(*sc, *cam);
  int TX = (cam->width + TILE - 1) / TILE, TY = (cam->height + TILE - 1) / TILE;
  std::vector<int64_t> cnt((size_t)TX * TY + 1, 0);
  for (int32_t g : v.order) {
    const Splat& s = v.sp[g];
    for (int ty = s.ty0; ty < s.ty1; ++ty)
      for (int tx = s.tx0; tx < s.tx1; ++tx) cnt[(size_t)ty * TX + tx + 1]++;
  }
  for (size_t i = 1; i < cnt.size(); ++i) cnt[i] += cnt[i - 1];
  std::copy(cnt.begin(), cnt.end(), offsets);
  int64_t total = cnt.back();
  if (total > cap) return total;
  std::vector<int64_t> cur(cnt.begin(), cnt.end() - 1);
  for (int32_t g : v.order) {
    const Splat& s = v.sp[g];
    for (int ty = s.ty0; ty < s.ty1; ++ty)
      for (int tx = s.tx0; tx < s.tx1; ++tx) ids[cur[(size_t)ty * TX + tx]++] = g;
  }
  return total;
}

// Render.  pixel_mask (H*W bytes) selects pixels, or null for all.  Outputs (unselected pixels
// untouched): rgb (H*W*3), depth, Tfinal (binary64 value path), T32 (decision-path transmittance,
// binary32), ncontrib.  Any output pointer may be null.
void orc_render(void* h, const Camera* cam, const uint8_t* pixel_mask, double* rgb, double* depth,
                double* Tfinal, float* T32, int32_t* ncontrib) {
  Scene* sc = (Scene*)h;
  View v = make_view(*sc, *cam);
  std::vector<SplatV> sv;
  fill_splatv(*sc, v, sv);
  const int W = cam->width, H = cam->height;
#pragma omp parallel
  {
    std::vector<Contrib> cs;
#pragma omp for schedule(dynamic, 1)
    for (int iy = 0; iy < H; ++iy)
      for (int ix = 0; ix < W; ++ix) {
        size_t p = (size_t)iy * W + ix;
        if (pixel_mask && !pixel_mask[p]) continue;
        float t32;
        walk_pixel(*sc, v, ix, iy, cs, t32);
        double out4[4], Tend;
        pixel_value(sc->cfg, ix + 0.5, iy + 0.5, cs.data(), (int)cs.size(), sv.data(), nullptr, out4, Tend, false,
                    [](int) -> double* { return nullptr; });
        if (rgb) { rgb[3 * p] = out4[0]; rgb[3 * p + 1] = out4[1]; rgb[3 * p + 2] = out4[2]; }
        if (depth) depth[p] = out4[3];
        if (Tfinal) Tfinal[p] = Tend;
        if (T32) T32[p] = t32;
        if (ncontrib) ncontrib[p] = (int32_t)cs.size();
      }
  }
}

// Per-pixel contributor lists (CSR over H*W pixels).  Returns total; fills ids/clamped when total <= cap.
int64_t orc_trace(void* h, const Camera* cam, int64_t* offsets, int32_t* ids, uint8_t* clamped, int64_t cap) {
  Scene* sc = (Scene*)h;
  View v = make_view(*sc, *cam);
  const int W = cam->width, H = cam->height;
  std::vector<std::vector<Contrib>> all((size_t)W * H);
#pragma omp parallel for schedule(dynamic, 1)
  for (int iy = 0; iy < H; ++iy)
    for (int ix = 0; ix < W; ++ix) {
      float t32;
      walk_pixel(*sc, v, ix, iy, all[(size_t)iy * W + ix], t32);
    }
  int64_t total = 0;
  for (size_t p = 0; p < all.size(); ++p) { offsets[p] = total; total += (int64_t)all[p].size(); }
  offsets[all.size()] = total;
  if (total > cap) return total;
  for (size_t p = 0; p < all.size(); ++p)
    for (size_t i = 0; i < all[p].size(); ++i) {
      ids[offsets[p] + (int64_t)i] = all[p][i].g;
      clamped[offsets[p] + (int64_t)i] = all[p][i].clamped ? 1 : 0;
    }
  return total;
}

// blocks (N x 105 doubles) += sum over selected pixels and enabled channels of J^T J
// pixel_mask null = all pixels.  Blocks are complete only for Gaussians whose whole footprint is selected.
void orc_view_hessian(void* h, const Camera* cam, const uint8_t* pixel_mask, double* blocks) {
  Scene* sc = (Scene*)h;
  View v = make_view(*sc, *cam);
  std::vector<SplatV> sv;
  fill_splatv(*sc, v, sv);
  std::vector<Chain> chains(sc->N);
#pragma omp parallel for schedule(static)
  for (int g = 0; g < sc->N; ++g) {
    if (!v.sp[g].visible) continue;
    double mu[3], ls[3], q[4];
    for (int k = 0; k < 3; ++k) { mu[k] = sc->mean[3 * g + k]; ls[k] = sc->logscale[3 * g + k]; }
    for (int k = 0; k < 4; ++k) q[k] = sc->quat[4 * g + k];
    chains[g] = chain(*cam, sc->cfg, mu, ls, q);
  }
  const int W = cam->width, H = cam->height;
  const int nbands = (H + BAND_ROWS - 1) / BAND_ROWS;
  std::vector<std::unique_ptr<HAcc>> bands(nbands);
#pragma omp parallel
  {
    std::vector<Contrib> cs;
#pragma omp for schedule(dynamic, 1)
    for (int band = 0; band < nbands; ++band) {
      bands[band].reset(new HAcc(sc->N, NB));
      HAcc& acc = *bands[band];
      for (int iy = band * BAND_ROWS; iy < std::min(H, (band + 1) * BAND_ROWS); ++iy)
        for (int ix = 0; ix < W; ++ix) {
          size_t p = (size_t)iy * W + ix;
          if (pixel_mask && !pixel_mask[p]) continue;
          float t32;
          walk_pixel(*sc, v, ix, iy, cs, t32);
          double out4[4], Tend;
          pixel_value(sc->cfg, ix + 0.5, iy + 0.5, cs.data(), (int)cs.size(), sv.data(), chains.data(), out4, Tend, true,
                      [&](int g) -> double* { return acc.at(g); });
        }
    }
  }
  add_bands(bands, sc->N, NB, blocks);
}

// ---------------------------------------------------------------------------
// smooth mode (finite-difference self-test only): all binary64, contributor sets frozen.
// theta: N x 14 = [mu | logscale | quat raw | opacity logit | rgb].
// ---------------------------------------------------------------------------
static void smooth_setup(int N, const double* theta, const Camera* cam, const Config* cfg,
                         std::vector<SplatV>& sv, std::vector<Chain>& chains) {
  sv.resize(N); chains.resize(N);
  for (int g = 0; g < N; ++g) {
    const double* th = theta + (size_t)P * g;
    chains[g] = chain(*cam, *cfg, th, th + 3, th + 6);
    const Chain& ch = chains[g];
    double det = ch.a * ch.c - ch.b * ch.b;
    SplatV& o = sv[g];
    o.mx = ch.mx; o.my = ch.my;
    o.ca = ch.c / det; o.cb = -ch.b / det; o.cc = ch.a / det;
    o.z = ch.z;
    o.sigma = 1.0 / (1.0 + std::exp(-th[10]));
    o.rgb[0] = th[11]; o.rgb[1] = th[12]; o.rgb[2] = th[13];
  }
}

// out: H*W*4 (r,g,b,depth)
void orc_render_smooth(int N, const double* theta, const Camera* cam, const Config* cfg, const int64_t* offsets,
                       const int32_t* ids, const uint8_t* clamped, double* out) {
  std::vector<SplatV> sv; std::vector<Chain> chains;
  smooth_setup(N, theta, cam, cfg, sv, chains);
  const int W = cam->width, H = cam->height;
  std::vector<Contrib> cs;
  for (int iy = 0; iy < H; ++iy)
    for (int ix = 0; ix < W; ++ix) {
      size_t p = (size_t)iy * W + ix;
      cs.clear();
      for (int64_t i = offsets[p]; i < offsets[p + 1]; ++i) cs.push_back({ids[i], clamped[i] != 0});
      double Tend;
      pixel_value(*cfg, ix + 0.5, iy + 0.5, cs.data(), (int)cs.size(), sv.data(), nullptr, out + 4 * p, Tend, false,
                  [](int) -> double* { return nullptr; });
    }
}

// blocks: N x 105, overwritten.  Analytic J^T J in smooth mode (same pixel_value code as the normal mode).
void orc_view_hessian_smooth(int N, const double* theta, const Camera* cam, const Config* cfg, const int64_t* offsets,
                             const int32_t* ids, const uint8_t* clamped, double* blocks) {
  std::vector<SplatV> sv; std::vector<Chain> chains;
  smooth_setup(N, theta, cam, cfg, sv, chains);
  std::fill(blocks, blocks + (size_t)N * NB, 0.0);
  const int W = cam->width, H = cam->height;
  std::vector<Contrib> cs;
  for (int iy = 0; iy < H; ++iy)
    for (int ix = 0; ix < W; ++ix) {
      size_t p = (size_t)iy * W + ix;
      cs.clear();
      for (int64_t i = offsets[p]; i < offsets[p + 1]; ++i) cs.push_back({ids[i], clamped[i] != 0});
      double out4[4], Tend;
      pixel_value(*cfg, ix + 0.5, iy + 0.5, cs.data(), (int)cs.size(), sv.data(), chains.data(), out4, Tend, true,
                  [&](int g) -> double* { return blocks + (size_t)g * NB; });
    }
}

// binary64 projection + chain for one Gaussian (pins for geometry): out = mx,my,a,b,c,z ; G = 5x10 ; dz = 3
void orc_chain(const Camera* cam, const Config* cfg, const double* theta14, double* out6, double* G50, double* dz3) {
  Chain ch = chain(*cam, *cfg, theta14, theta14 + 3, theta14 + 6);
  out6[0] = ch.mx; out6[1] = ch.my; out6[2] = ch.a; out6[3] = ch.b; out6[4] = ch.c; out6[5] = ch.z;
  for (int e = 0; e < 5; ++e)
    for (int k = 0; k < 10; ++k) G50[10 * e + k] = ch.G[e][k];
  for (int k = 0; k < 3; ++k) dz3[k] = ch.dz[k];
}

// ---- object-mask output (NEXT-2) -------------------------------------------------------------------
// prob: N x K softmax probabilities.  out: H*W*K mask values (Eq. 1-2).
void orc_render_mask(void* h, const Camera* cam, int K, int bgch, const double* prob, double* out) {
  Scene* sc = (Scene*)h;
  View v = make_view(*sc, *cam);
  std::vector<SplatV> sv;
  fill_splatv(*sc, v, sv);
  const int W = cam->width, H = cam->height;
#pragma omp parallel
  {
    std::vector<Contrib> cs;
#pragma omp for schedule(dynamic, 1)
    for (int iy = 0; iy < H; ++iy)
      for (int ix = 0; ix < W; ++ix) {
        float t32;
        walk_pixel(*sc, v, ix, iy, cs, t32);
        double Tend;
        pixel_value_mask(sc->cfg, K, bgch, ix + 0.5, iy + 0.5, cs.data(), (int)cs.size(), sv.data(), nullptr, prob,
                         out + ((size_t)iy * W + ix) * K, Tend, false, [](int) -> double* { return nullptr; });
      }
  }
}

// blocks (N x L(L+1)/2 doubles, L = 11 + K) += sum over pixels and mask channels of J^T J.  Same band-ordered sparse
// accumulation as orc_view_hessian.
void orc_view_hessian_mask(void* h, const Camera* cam, int K, int bgch, const double* prob, double* blocks) {
  Scene* sc = (Scene*)h;
  View v = make_view(*sc, *cam);
  std::vector<SplatV> sv;
  fill_splatv(*sc, v, sv);
  std::vector<Chain> chains(sc->N);
#pragma omp parallel for schedule(static)
  for (int g = 0; g < sc->N; ++g) {
    if (!v.sp[g].visible) continue;
    double mu[3], ls[3], q[4];
    for (int k = 0; k < 3; ++k) { mu[k] = sc->mean[3 * g + k]; ls[k] = sc->logscale[3 * g + k]; }
    for (int k = 0; k < 4; ++k) q[k] = sc->quat[4 * g + k];
    chains[g] = chain(*cam, sc->cfg, mu, ls, q);
  }
  const int W = cam->width, H = cam->height, L = 11 + K;
  const size_t LB = (size_t)L * (L + 1) / 2;
  const int nbands = (H + BAND_ROWS - 1) / BAND_ROWS;
  std::vector<std::unique_ptr<HAcc>> bands(nbands);
#pragma omp parallel
  {
    std::vector<Contrib> cs;
    std::vector<double> outK(K);
#pragma omp for schedule(dynamic, 1)
    for (int band = 0; band < nbands; ++band) {
      bands[band].reset(new HAcc(sc->N, LB));
      HAcc& acc = *bands[band];
      for (int iy = band * BAND_ROWS; iy < std::min(H, (band + 1) * BAND_ROWS); ++iy)
        for (int ix = 0; ix < W; ++ix) {
          float t32;
          walk_pixel(*sc, v, ix, iy, cs, t32);
          double Tend;
          pixel_value_mask(sc->cfg, K, bgch, ix + 0.5, iy + 0.5, cs.data(), (int)cs.size(), sv.data(), chains.data(), prob,
                           outK.data(), Tend, true, [&](int g) -> double* { return acc.at(g); });
        }
    }
  }
  add_bands(bands, sc->N, LB, blocks);
}

// smooth mode (finite-difference self-test): theta N x 11 = [mu | logscale | quat raw | opacity logit], logits N x K
static void smooth_setup_mask(int N, int K, const double* theta11, const double* logits, const Camera* cam, const Config* cfg,
                              std::vector<SplatV>& sv, std::vector<Chain>& chains, std::vector<double>& prob) {
  std::vector<double> th14((size_t)N * P, 0.0);
  for (int g = 0; g < N; ++g)
    for (int k = 0; k < 11; ++k) th14[(size_t)g * P + k] = theta11[(size_t)g * 11 + k];
  smooth_setup(N, th14.data(), cam, cfg, sv, chains);
  prob.resize((size_t)N * K);
  for (int g = 0; g < N; ++g) {
    const double* o = logits + (size_t)g * K;
    double m = o[0];
    for (int k = 1; k < K; ++k) m = std::max(m, o[k]);
    double z = 0;
    for (int k = 0; k < K; ++k) z += std::exp(o[k] - m);
    for (int k = 0; k < K; ++k) prob[(size_t)g * K + k] = std::exp(o[k] - m) / z;
  }
}

void orc_render_mask_smooth(int N, int K, int bgch, const double* theta11, const double* logits, const Camera* cam,
                            const Config* cfg, const int64_t* offsets, const int32_t* ids, const uint8_t* clamped, double* out) {
  std::vector<SplatV> sv; std::vector<Chain> chains; std::vector<double> prob;
  smooth_setup_mask(N, K, theta11, logits, cam, cfg, sv, chains, prob);
  const int W = cam->width, H = cam->height;
  std::vector<Contrib> cs;
  for (int iy = 0; iy < H; ++iy)
    for (int ix = 0; ix < W; ++ix) {
      size_t p = (size_t)iy * W + ix;
      cs.clear();
      for (int64_t i = offsets[p]; i < offsets[p + 1]; ++i) cs.push_back({ids[i], clamped[i] != 0});
      double Tend;
      pixel_value_mask(*cfg, K, bgch, ix + 0.5, iy + 0.5, cs.data(), (int)cs.size(), sv.data(), nullptr, prob.data(), out + p * K,
                       Tend, false, [](int) -> double* { return nullptr; });
    }
}

void orc_view_hessian_mask_smooth(int N, int K, int bgch, const double* theta11, const double* logits, const Camera* cam,
                                  const Config* cfg, const int64_t* offsets, const int32_t* ids, const uint8_t* clamped,
                                  double* blocks) {
  std::vector<SplatV> sv; std::vector<Chain> chains; std::vector<double> prob;
  smooth_setup_mask(N, K, theta11, logits, cam, cfg, sv, chains, prob);
  const int L = 11 + K;
  const size_t LB = (size_t)L * (L + 1) / 2;
  std::fill(blocks, blocks + (size_t)N * LB, 0.0);
  const int W = cam->width, H = cam->height;
  std::vector<Contrib> cs;
  std::vector<double> outK(K);
  for (int iy = 0; iy < H; ++iy)
    for (int ix = 0; ix < W; ++ix) {
      size_t p = (size_t)iy * W + ix;
      cs.clear();
      for (int64_t i = offsets[p]; i < offsets[p + 1]; ++i) cs.push_back({ids[i], clamped[i] != 0});
      double Tend;
      pixel_value_mask(*cfg, K, bgch, ix + 0.5, iy + 0.5, cs.data(), (int)cs.size(), sv.data(), chains.data(), prob.data(),
                       outK.data(), Tend, true, [&](int g) -> double* { return blocks + (size_t)g * LB; });
    }
}

int orc_num_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"

// Later additions to the oracle (view-dependent colour) live in a separate file so that
// this one -- whose hash the stored full-size expected values (tests/golden/) carry -- stays as it was when they
// were written.  Same translation unit, same rules (test infrastructure, nothing shared with csrc/).
#include "nbv_oracle_ext.inc"
