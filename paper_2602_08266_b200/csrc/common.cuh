// common.cuh -- shared definitions of the CUDA path (sm_100a).  Not used by, and shares nothing with, oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/nbv.h"

namespace nbv {

constexpr int P = NBV_P;
constexpr int NBLK = NBV_BLOCK;
constexpr int TILE = NBV_TILE;
constexpr int NMOM = 40;        // screen-space moments per (view, Gaussian): 15 + 4*6 + 1
constexpr int MOM_X = 15;       // first cross moment
constexpr int MOM_W2 = 39;      // sum of w^2
constexpr float POWER_MIN = -6.0f;

// Projected splat, 48 bytes, stored in depth-rank order for the rasteriser.
struct __align__(16) Splat {
  float mx, my, qa, qb;      // centre (px); power(d) = qa dx^2 + qb dx dy + qc dy^2
  float qc, sigma, z, tau;   // tau: conservative lower bound of ln(alpha_min / sigma) (pre-test only, never decides)
  float r, g, b, pad;
};

struct ViewCounters {          // device-side counters of one view
  unsigned long long n_keys;   // sum of rect areas = length of all tile lists (R-5); not materialised on the hot path
  unsigned long long n_entries;// tile-list entries the forward pass walked before its tile terminated
  unsigned long long n_pairs;  // (pixel, Gaussian) pairs composited
  unsigned int n_visible;
  unsigned int n_touched;      // Gaussians with a non-zero block in this view (= length of the touched list)
  unsigned int bad_data;
  unsigned int n_coarse;       // (supertile, Gaussian) keys of the coarse binning
  unsigned int n_expanded;     // touched Gaussians consumed by the expand kernel (work-queue cursor)
  unsigned int pad[3];
};

// Tile grid of one view and its supertiles (S x S tiles, S = 1 << sshift).
struct TileGrid {
  int tiles_x, tiles_y;
  int sshift;
  int super_x, super_y;
};

// ---------------------------------------------------------------------------------------------
// Decision-path arithmetic (R-9).  Every operation individually rounded with
// the _rn intrinsics (never contracted by the compiler); fused multiply-adds only where __fmaf_rn
// is written.  Must reproduce the binary32 results of the specification bit for bit.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ float mul_rn(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ float add_rn(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ float sub_rn(float a, float b) { return __fsub_rn(a, b); }
__device__ __forceinline__ float div_rn(float a, float b) { return __fdiv_rn(a, b); }
__device__ __forceinline__ float sqrt_rn(float a) { return __fsqrt_rn(a); }

__device__ __forceinline__ float exp_spec(float x) {
  const float MAGIC = 12582912.0f;
  float t = __fmaf_rn(x, 0x1.715476p+0f, MAGIC);
  float kf = __fsub_rn(t, MAGIC);
  float r = __fmaf_rn(kf, -0x1.62e4p-1f, x);
  r = __fmaf_rn(kf, -0x1.7f7d1cp-20f, r);
  float p = 0x1.6c16c2p-10f;
  p = __fmaf_rn(p, r, 0x1.111112p-7f);
  p = __fmaf_rn(p, r, 0x1.555556p-5f);
  p = __fmaf_rn(p, r, 0x1.555556p-3f);
  p = __fmaf_rn(p, r, 0.5f);
  p = __fmaf_rn(p, r, 1.0f);
  p = __fmaf_rn(p, r, 1.0f);
  int k = __float_as_int(t) - __float_as_int(MAGIC);
  return __int_as_float(__float_as_int(p) + (k << 23));
}

// power of the Gaussian exponent at offset (dx,dy)
__device__ __forceinline__ float splat_power(float qa, float qb, float qc, float dx, float dy) {
  return __fmaf_rn(dx, __fmaf_rn(qa, dx, __fmul_rn(qb, dy)), __fmul_rn(__fmul_rn(qc, dy), dy));
}

// ---------------------------------------------------------------------------------------------
// Packed binary32 pairs (sm_100: FFMA2 / FMUL2 / FADD2 issue two operations per lane in one slot).
// Each half is rounded exactly like the scalar .rn instruction, so the decision path may use them; ptxas does
// contract a mul.rn.f32x2 feeding an add.rn.f32x2 into one FFMA2 (seen in the SASS), so the decision path never
// writes that pattern: its products feed fused multiply-adds or other products only, as the specification has it.
// ---------------------------------------------------------------------------------------------
typedef float2 f2;
__device__ __forceinline__ f2 bc2(float s) { return make_float2(s, s); }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) {
  f2 d;
  asm("{.reg .b64 ra, rb, rc, rd; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; mov.b64 rc, {%6,%7}; fma.rn.f32x2 rd, ra, rb, rc; mov.b64 {%0,%1}, rd;}"
      : "=f"(d.x), "=f"(d.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y), "f"(c.x), "f"(c.y));
  return d;
}
__device__ __forceinline__ f2 mul2(f2 a, f2 b) {
  f2 d;
  asm("{.reg .b64 ra, rb, rd; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; mul.rn.f32x2 rd, ra, rb; mov.b64 {%0,%1}, rd;}"
      : "=f"(d.x), "=f"(d.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
  return d;
}
__device__ __forceinline__ f2 add2(f2 a, f2 b) {
  f2 d;
  asm("{.reg .b64 ra, rb, rd; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; add.rn.f32x2 rd, ra, rb; mov.b64 {%0,%1}, rd;}"
      : "=f"(d.x), "=f"(d.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
  return d;
}
__device__ __forceinline__ f2 sub2(f2 a, f2 b) {
  f2 d;
  asm("{.reg .b64 ra, rb, rd; mov.b64 ra, {%2,%3}; mov.b64 rb, {%4,%5}; sub.rn.f32x2 rd, ra, rb; mov.b64 {%0,%1}, rd;}"
      : "=f"(d.x), "=f"(d.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
  return d;
}

// power of the Gaussian exponent for a pair of pixels of one column: the operations of splat_power, pair-wise
__device__ __forceinline__ f2 splat_power2(float qa, float qb, float qc, float dx, f2 dy) {
  const f2 inner = fma2(bc2(qa), bc2(dx), mul2(bc2(qb), dy));
  return fma2(bc2(dx), inner, mul2(mul2(bc2(qc), dy), dy));
}

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// exp_spec on a pair: the same operations in the same order, each half individually rounded.  The last step of exp_spec,
// bits(p) + (k << 23), is taken here as p * 2^k with 2^k from MUFU.EX2 of the integer-valued kf: on this hardware
// ex2.approx is exact at every integer in [-126, 127] and the product of p in [0.5, 2) with a power of two equals the
// exponent-field addition whenever the result is a normal number (checked exhaustively over k and on a grid of mantissas on
// the B200), i.e. for every x in [-80, 80] -- the whole domain exp_spec is specified on.  Outside it the two differ, in the
// useful direction: a NaN or -inf argument (a pixel parked at py = +inf) gives NaN instead of arbitrary bits, and NaN fails
// every `>= alpha_min` test, so the raster kernels need no separate range test to mask such lanes.  Two ALU-pipe
// operations per pixel move to the idle MUFU pipe.
__device__ __forceinline__ f2 exp_spec2(f2 x) {
  const float MAGIC = 12582912.0f;
  const f2 t = fma2(x, bc2(0x1.715476p+0f), bc2(MAGIC));
  const f2 kf = sub2(t, bc2(MAGIC));
  f2 r = fma2(kf, bc2(-0x1.62e4p-1f), x);
  r = fma2(kf, bc2(-0x1.7f7d1cp-20f), r);
  f2 p = bc2(0x1.6c16c2p-10f);
  p = fma2(p, r, bc2(0x1.111112p-7f));
  p = fma2(p, r, bc2(0x1.555556p-5f));
  p = fma2(p, r, bc2(0x1.555556p-3f));
  p = fma2(p, r, bc2(0.5f));
  p = fma2(p, r, bc2(1.0f));
  p = fma2(p, r, bc2(1.0f));
  return mul2(p, make_float2(ex2_approx(kf.x), ex2_approx(kf.y)));
}

// packed upper-triangle index, r <= c
__host__ __device__ __forceinline__ constexpr int tri(int r, int c) { return r * P - r * (r - 1) / 2 + (c - r); }

// monomial sums sum B alpha^2 ux^i uy^j, i+j <= 4, stored at mono_index(i,j)
__host__ __device__ __forceinline__ constexpr int mono_index(int i, int j) {
  // order: (0,0) | (1,0),(0,1) | (2,0),(1,1),(0,2) | (3,0),(2,1),(1,2),(0,3) | (4,0),(3,1),(2,2),(1,3),(0,4)
  return (i + j) * (i + j + 1) / 2 + j;
}

}  // namespace nbv
