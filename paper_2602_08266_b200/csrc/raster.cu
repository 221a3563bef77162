// raster.cu -- S3 front-to-back compositing and S4 back-to-front Jacobian sweep, per 16x16 tile.
//
// Mapping: ONE WARP PER TILE, each lane owns a column of 8 pixels
// (x = lane & 15, rows (lane >> 4) * 8 .. +7).  The warp streams its SUPERTILE's depth-ordered list (binning.cu),
// keeps the entries whose tile rectangle contains this tile (ballot + compaction into a shared-memory queue: this
// IS the tile list of R-5, produced lazily) and stages the splats 32 at a time in shared memory; every lane
// evaluates each splat at its 8 pixels, so the 40 moment sums of S4 are reduced over 8 pixels in registers before
// the cross-lane butterfly, and no block-level barrier exists at all.  S3 stops reading the list when all 256
// pixels have terminated and records where (tile_cend); S4 walks the same list backwards from there.
//
// S3 is on the decision path (bit-exact power / alpha / transmittance chain).
// S4 ("computes the Jacobian of the rendering with respect to Gaussian parameters", L189-191
// H ~= J^T J, L210 per-Gaussian blocks) does NOT form 14-wide rows per pixel.  With d = p - m, u = Sigma2D^-1 d,
//   dalpha/d(mx,my,a,b,c,o) = alpha (ux, uy, ux^2/2, ux uy, uy^2/2, kappa),   dy_ch/dalpha_i = beta_ch,
// the per-pixel row of channel ch is  J_ch = beta_ch * alpha * A m6 + w e_ch  with the monomial vector
// m6 = (ux, uy, ux^2, ux uy, uy^2, 1), a per-(view, Gaussian) matrix A (14 x 6, applied later in S5) and
// w = alpha T.  Hence  sum_px sum_ch omega_ch J_ch J_ch^T  needs only
//   15 sums  sum_px (sum_ch omega_ch beta_ch^2) alpha^2 ux^i uy^j, i + j <= 4
//    6 sums per channel  sum_px beta_ch w alpha m6
//    1 sum   sum_px w^2
// = 40 numbers per (tile, Gaussian) for RGB + depth.  The oracle forms explicit rows instead, so parity
// checks this algebra.
#include <algorithm>

#include "kernels.h"

namespace nbv {

constexpr int PPL = 8;                 // pixels per lane
#ifndef NBV_BWD_MIN_BLOCKS
#define NBV_BWD_MIN_BLOCKS 16          // resident warps per SM the backward kernel is compiled for (register cap)
#endif
constexpr unsigned FULL = 0xffffffffu;

struct RasterParams {
  int W, H, tiles_x, rank_bits;
  int sshift, super_x;                 // supertile = (1 << sshift)^2 tiles, super_x supertiles per row
  float alpha_min, alpha_max, t_stop;
  float bg[3];
  float omega[4];                      // channel weights, 0 for disabled channels
  float somega[4];                     // their square roots
  float ln_amax_over_amin;
};

__device__ __forceinline__ float rcp_approx(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

__device__ __forceinline__ void prefetch_l1(const void* p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }

// Can any pixel centre of the tile whose first centre is (X0 + 0.5, Y0 + 0.5) reach power >= tau?  Conservative: the
// maximum of the concave quadratic over the BOX of the 16 x 16 centres (at the centre if it lies inside, else on an
// edge, where the 1-D optimum is clamped to the edge), plus a slack that covers the binary32 rounding of both this
// evaluation and the per-pixel one.  An entry rejected here has no pixel that passes the footprint test of R-5 in
// this tile, so dropping it changes no image, count, block or gain; S3 and S4 take the identical decision.
__device__ __forceinline__ bool ellipse_reaches_tile(float mx, float my, float qa, float qb, float qc, float tau, float X0, float Y0) {
  const float ax = sub_rn(X0 + 0.5f, mx), bx = add_rn(ax, (float)(TILE - 1));
  const float ay = sub_rn(Y0 + 0.5f, my), by = add_rn(ay, (float)(TILE - 1));
  if (ax <= 0.0f && bx >= 0.0f && ay <= 0.0f && by >= 0.0f) return true;
  // the 1-D optima -qb dx / (2 qc), -qb dy / (2 qa): approximate reciprocals (MUFU) instead of two IEEE divisions -- the test
  // is conservative by the slack below, far above their 1-ulp error, and S3 / S4 still evaluate the very same expressions
  const float hb = mul_rn(-0.5f, qb);
  const float ry = mul_rn(hb, rcp_approx(qc)), rx = mul_rn(hb, rcp_approx(qa));
  const float thr = sub_rn(tau, 1e-3f);
  bool keep = false;
#pragma unroll
  for (int e = 0; e < 4; ++e) {
    float dx, dy;
    if (e < 2) { dx = e == 0 ? ax : bx; dy = fminf(fmaxf(mul_rn(ry, dx), ay), by); }
    else       { dy = e == 2 ? ay : by; dx = fminf(fmaxf(mul_rn(rx, dy), ax), bx); }
    // explicit _rn operations: S3 and S4 must take bit-identical decisions, whatever the compiler would contract
    const float t0 = mul_rn(mul_rn(qa, dx), dx), t1 = mul_rn(mul_rn(qb, dx), dy), t2 = mul_rn(mul_rn(qc, dy), dy);
    const float p = add_rn(add_rn(t0, t1), t2), mag = add_rn(add_rn(fabsf(t0), fabsf(t1)), fabsf(t2));
    keep = keep || !(add_rn(p, mul_rn(2e-5f, mag)) < thr);     // also keeps NaN / inf cases
  }
  return keep;
}

// lanes < count stage the splats of queue slots 0..count-1; slot j's coarse position + 1 rides in the pad field
__device__ __forceinline__ void stage_queue(const Splat* __restrict__ splat_sorted, const uint32_t* q_rank, const uint32_t* q_cpos,
                                            uint32_t count, float4* sm) {
  const int lane = threadIdx.x;
  if ((uint32_t)lane < count) {
    const float4* s = reinterpret_cast<const float4*>(splat_sorted + q_rank[lane]);
    sm[lane * 3 + 0] = s[0];
    sm[lane * 3 + 1] = s[1];
    float4 c = s[2];
    if (q_cpos) c.w = __uint_as_float(q_cpos[lane] + 1u);
    sm[lane * 3 + 2] = c;
  }
  __syncwarp();
}

// drop the first `count` queue slots
__device__ __forceinline__ void shift_queue(uint32_t* q_rank, uint32_t* q_cpos, uint32_t& qn, uint32_t count) {
  const int lane = threadIdx.x;
  __syncwarp();
  uint32_t r = 0, c = 0;
  const bool mv = count + lane < qn;
  if (mv) { r = q_rank[count + lane]; if (q_cpos) c = q_cpos[count + lane]; }
  __syncwarp();
  if (mv) { q_rank[lane] = r; if (q_cpos) q_cpos[lane] = c; }
  qn -= count;
  __syncwarp();
}

// FULLPIX = false is the timed path: S4 needs only the final transmittance and `last` of every pixel (it rebuilds the
// suffix sums itself), so colour, depth and the contributor count are accumulated only for the parity exports.
//
// Slot body.  A lane's 8 pixels are 4 PAIRS (row q, row 7 - q) evaluated with packed binary32 operations (FFMA2 /
// FMUL2 / FADD2: two pixels per issue slot, each half rounded like the scalar .rn operation, so the decision path is
// bit for bit the specified one).  Per pixel and entry: 19 packed-pipe operations per pair (dy, power, exp_spec, sigma G,
// 1 - alpha, T (1 - alpha)) and 8 scalar ones (the exponent bits of exp_spec, three range / alpha tests, min, two
// selects, the stop test).  Nothing else: a pixel that stops (R-4: the entry that would take T below t_stop is not
// composited, the pixel is finished) leaves its T unchanged but NEGATED, and a branch the warp takes only then -- 8 times
// per lane and tile -- retires it (py = +inf: its power fails every later range test), counts it, and records in `last`
// how many list entries precede the stop.  A pixel that never stops gets last = number of entries walked.  Every entry
// S4 must composite at a pixel lies before `last`, and S4 re-takes the same pass decisions, so it finds the same set.
// what S3 leaves in registers for an S4 sweep of the same tile by the same warp (raster_kernel): the final transmittance and
// `last` of the lane's 8 pixels (pairs as in the slot bodies) and the tile's list length
struct FwdOut {
  f2 T2[PPL / 2];
  int last[PPL];
  uint32_t elast;
};

// the shared memory of one S3 warp (2,560 bytes), one struct so that every array is an offset from one base
struct FwdSmem {
  float4 sm[32 * 3];
  uint32_t q_rank[64], q_cpos[64], p_rank[64], p_cpos[64];
};

// S3 of one launch position (view, tile) by one warp.  sm: 96 float4; q_rank, q_cpos, p_rank, p_cpos: 64 words each (p_*: rect
// hits awaiting the ellipse test, stage 2 of the tile filter).
template <bool FULLPIX>
__device__ __forceinline__ void forward_tile(const RasterBatch& batch, const RasterParams& prm, uint32_t bpos, int lane, float4* sm,
                                             uint32_t* q_rank, uint32_t* q_cpos, uint32_t* p_rank, uint32_t* p_cpos, FwdOut& fo) {
  const int vidx = (int)(bpos % (uint32_t)batch.n);
  const RasterView& vw = batch.v[vidx];
  const Splat* __restrict__ splat_sorted = vw.splat_sorted;
  const uint32_t* __restrict__ ckeys = vw.ckeys;
  const ushort4* __restrict__ crect = vw.crect;
  const uint2* __restrict__ cranges = vw.cranges;
  const PixelBuf out = vw.pix;
  ViewCounters* counters = vw.counters;
  const int tile = batch.tile_order[bpos / (uint32_t)batch.n];   // heaviest tiles first (launch order)
  const int tx = tile % prm.tiles_x, ty = tile / prm.tiles_x;
  const int x = tx * TILE + (lane & 15), y0 = ty * TILE + (lane >> 4) * PPL;
  const float px = (float)x + 0.5f;
  const float X0 = (float)(tx * TILE), Y0 = (float)(ty * TILE);
  const uint2 range = cranges[(ty >> prm.sshift) * prm.super_x + (tx >> prm.sshift)];
  const uint32_t rmask = (1u << prm.rank_bits) - 1u;
  const uint32_t lt = (1u << lane) - 1u;

  // pair q holds the pixels of rows q (.x) and 7 - q (.y)
  f2 T2[PPL / 2], py2[PPL / 2];
  float C0[PPL], C1[PPL], C2[PPL], D[PPL];
  int n[PPL], last[PPL];
  // A pixel that has terminated (or lies outside the image) gets py = +inf: its power evaluates to -inf or NaN and
  // fails `power >= tau`, so no separate done mask has to be tested in the slot body.
  int ndone = 0;
#pragma unroll
  for (int k = 0; k < PPL; ++k) {
    C0[k] = C1[k] = C2[k] = D[k] = 0.0f; n[k] = 0; last[k] = 0;
    float py = (float)(y0 + k) + 0.5f;
    if (x >= prm.W || y0 + k >= prm.H) { py = INFINITY; ++ndone; }
    if (k < PPL / 2) { T2[k].x = 1.0f; py2[k].x = py; } else { T2[PPL - 1 - k].y = 1.0f; py2[PPL - 1 - k].y = py; }
  }
  uint32_t walked = 0, cend = 0, elast = 0;
  uint32_t pos = range.x, qn = 0;
  int e_base = 0;
  bool finished = __all_sync(FULL, ndone == PPL);
  // The lazy tile filter, two stages.  Stage 1 streams the supertile list in chunks of 32 entries and keeps the ones whose rect
  // contains this tile (about one in five): rect and key are software-pipelined two chunks deep in registers, and the splat
  // record of every rect hit is requested into the L1 at once.  Stage 2 runs when 32 rect hits are pending (or the list has
  // ended): it gathers their records -- by then in the L1 -- and applies the ellipse test with all lanes busy (per chunk it
  // kept six lanes busy and cost a dependent gather each time), and the survivors enter the queue of the entry loop.
  // Until r2m the filter was one chain of dependent loads per chunk (rect -> key -> record -> ellipse test) and a third of
  // this kernel's stall samples.
  ushort4 rcA = make_ushort4(1, 1, 0, 0), rcB = rcA;       // empty rect: covers no tile
  uint32_t keyA = 0, keyB = 0;
  if (!finished) {
    if (pos + lane < range.y) { rcA = crect[pos + lane]; keyA = ckeys[pos + lane]; }
    if (pos + 32u + lane < range.y) { rcB = crect[pos + 32u + lane]; keyB = ckeys[pos + 32u + lane]; }
  }
  uint32_t pn = 0;                                         // rect hits pending for stage 2
  while (!finished) {
    // fill the queue with the next entries of the supertile list that can contribute to this tile
    while (qn < 32u) {
      while (pn < 32u && pos < range.y) {                  // stage 1
        const uint32_t i = pos + lane;
        const ushort4 rc = rcA;
        const uint32_t key = keyA;
        const bool hit = i < range.y && tx >= rc.x && tx < rc.z && ty >= rc.y && ty < rc.w;
        pos += 32;
        rcA = rcB; keyA = keyB;
        rcB = make_ushort4(1, 1, 0, 0);
        if (pos + 32u + lane < range.y) { rcB = crect[pos + 32u + lane]; keyB = ckeys[pos + 32u + lane]; }
        const unsigned m = __ballot_sync(FULL, hit);
        if (hit) {
          const uint32_t slot = pn + __popc(m & lt), r = key & rmask;
          p_rank[slot] = r;
          p_cpos[slot] = i;
          const char* rec = reinterpret_cast<const char*>(splat_sorted + r);      // 48 B: one or two sectors
          prefetch_l1(rec); prefetch_l1(rec + 16);
        }
        pn += __popc(m);
      }
      if (pn == 0) break;
      const uint32_t take = min(pn, 32u);                  // stage 2
      __syncwarp();
      bool keep = false;
      uint32_t r = 0, cp = 0;
      if ((uint32_t)lane < take) {
        r = p_rank[lane]; cp = p_cpos[lane];
        const float4* sp = reinterpret_cast<const float4*>(splat_sorted + r);
        const float4 a0 = sp[0], a1 = sp[1];
        keep = ellipse_reaches_tile(a0.x, a0.y, a0.z, a0.w, a1.x, a1.w, X0, Y0);
      }
      const unsigned m = __ballot_sync(FULL, keep);
      if (keep) {
        const uint32_t slot = qn + __popc(m & lt);
        q_rank[slot] = r;
        q_cpos[slot] = cp;
      }
      qn += __popc(m);
      shift_queue(p_rank, p_cpos, pn, take);
    }
    if (qn == 0) break;
    const uint32_t cnt = min(qn, 32u);
    __syncwarp();
    // hand the tile's list to S4: entry e_base + lane is rank q_rank[lane] (S4 reads it backwards and filters nothing)
    if (vw.tlist && (uint32_t)lane < cnt && (uint32_t)e_base + lane < (uint32_t)TL_CAP)
      vw.tlist[(size_t)tile * TL_CAP + e_base + lane] = q_rank[lane];
    stage_queue(splat_sorted, q_rank, q_cpos, cnt, sm);
    for (uint32_t j = 0; j < cnt; ++j) {
      const float4 s0 = sm[j * 3], s1 = sm[j * 3 + 1], s2 = sm[j * 3 + 2];
      const int e = e_base + (int)j;                           // position of this entry in the tile's list
      const float dx = sub_rn(px, s0.x);
      bool anypass = false;
      uint32_t neg = 0u;
      ++walked;
#pragma unroll
      for (int q = 0; q < PPL / 2; ++q) {
        const f2 dy = sub2(py2[q], bc2(s0.y));
        const f2 power = splat_power2(s0.z, s0.w, s1.x, dx, dy);
        const f2 a = mul2(bc2(s1.y), exp_spec2(power));       // NaN for a parked pixel (power = -inf or NaN): fails the alpha test
        // The lower bounds of R-5 (power >= -6) and of the splat (power >= tau) never decide: alpha_min >= 1/255 (nbv_create)
        // and sigma < 1 make sigma exp(power) >= alpha_min the stronger condition (project.cu), so the alpha test stands for both.
        const bool pass_x = power.x <= 0.0f && a.x >= prm.alpha_min;
        const bool pass_y = power.y <= 0.0f && a.y >= prm.alpha_min;
        f2 al;
        al.x = pass_x ? fminf(a.x, prm.alpha_max) : 0.0f;
        al.y = pass_y ? fminf(a.y, prm.alpha_max) : 0.0f;
        const f2 Tn = mul2(T2[q], sub2(bc2(1.0f), al));        // alpha = 0: T (1 - 0) = T exactly
        // stop BEFORE compositing (R-4).  T >= t_stop always, so Tn < t_stop happens only where the pixel passed.
        const bool stop_x = Tn.x < prm.t_stop, stop_y = Tn.y < prm.t_stop;
        if (FULLPIX) {
          const float wx = (pass_x && !stop_x) ? al.x * T2[q].x : 0.0f, wy = (pass_y && !stop_y) ? al.y * T2[q].y : 0.0f;
          const int kx = q, ky = PPL - 1 - q;
          C0[kx] = fmaf(s2.x, wx, C0[kx]); C1[kx] = fmaf(s2.y, wx, C1[kx]); C2[kx] = fmaf(s2.z, wx, C2[kx]); D[kx] = fmaf(s1.z, wx, D[kx]);
          C0[ky] = fmaf(s2.x, wy, C0[ky]); C1[ky] = fmaf(s2.y, wy, C1[ky]); C2[ky] = fmaf(s2.z, wy, C2[ky]); D[ky] = fmaf(s1.z, wy, D[ky]);
          n[kx] += (pass_x && !stop_x) ? 1 : 0;
          n[ky] += (pass_y && !stop_y) ? 1 : 0;
        }
        T2[q].x = stop_x ? -T2[q].x : Tn.x;
        T2[q].y = stop_y ? -T2[q].y : Tn.y;
        neg |= __float_as_uint(T2[q].x) | __float_as_uint(T2[q].y);
        anypass = anypass || pass_x || pass_y;
      }
      if (anypass) { cend = __float_as_uint(s2.w); elast = (uint32_t)e + 1u; }   // coarse position + 1, list position + 1
      if (neg & 0x80000000u) {                                  // some pixel of this lane stopped at this entry
#pragma unroll
        for (int q = 0; q < PPL / 2; ++q) {
          if (T2[q].x < 0.0f) { T2[q].x = -T2[q].x; py2[q].x = INFINITY; last[q] = e; ++ndone; }
          if (T2[q].y < 0.0f) { T2[q].y = -T2[q].y; py2[q].y = INFINITY; last[PPL - 1 - q] = e; ++ndone; }
        }
      }
      if (__all_sync(FULL, ndone == PPL)) { finished = true; break; }
    }
    e_base += (int)cnt;
    shift_queue(q_rank, q_cpos, qn, cnt);
  }
  unsigned pairs = 0;
#pragma unroll
  for (int k = 0; k < PPL; ++k) {
    const float pyk = k < PPL / 2 ? py2[k].x : py2[PPL - 1 - k].y;
    // never stopped: every walked entry precedes `last`; outside the image: py = inf from the start, last = 0 (and T = 1)
    const int lk = pyk == INFINITY ? last[k] : (int)walked;
    fo.last[k] = lk;
    if (x < prm.W && y0 + k < prm.H) {
      const size_t p = (size_t)(y0 + k) * prm.W + x;
      const float Tk = k < PPL / 2 ? T2[k].x : T2[PPL - 1 - k].y;
      if (FULLPIX) {
        pairs += n[k];
        out.rgb[3 * p + 0] = fmaf(prm.bg[0], Tk, C0[k]);
        out.rgb[3 * p + 1] = fmaf(prm.bg[1], Tk, C1[k]);
        out.rgb[3 * p + 2] = fmaf(prm.bg[2], Tk, C2[k]);
        out.depth[p] = D[k];
        out.ncontrib[p] = n[k];
      }
      out.T[p] = Tk;
      out.last[p] = lk;
    }
  }
#pragma unroll
  for (int q = 0; q < PPL / 2; ++q) fo.T2[q] = T2[q];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    if (FULLPIX) pairs += __shfl_xor_sync(FULL, pairs, o);
    cend = max(cend, __shfl_xor_sync(FULL, cend, o));
    elast = max(elast, __shfl_xor_sync(FULL, elast, o));
  }
  if (lane == 0) {
    vw.tile_cend[tile] = cend;
    vw.tile_elast[tile] = elast;
    vw.tile_walk[tile] = walked;
    if (elast > (uint32_t)TL_CAP && batch.overflow) atomicAdd(batch.overflow, 1u);     // S4's fallback launch takes this tile
    if (FULLPIX) {
      atomicAdd(&counters->n_entries, (unsigned long long)walked);
      atomicAdd(&counters->n_pairs, (unsigned long long)pairs);
    }
  }
  fo.elast = elast;
}

template <bool FULLPIX>
__global__ void __launch_bounds__(32, FULLPIX ? 16 : 20) forward_kernel(const __grid_constant__ RasterBatch batch, const __grid_constant__ RasterParams prm) {
  // One launch rasterises every view of the batch.  Launch position -> (view, tile): the views are
  // interleaved, so the launch starts with the central (long-running) tiles of ALL views and its tail is made of the
  // edge tiles of all views.
  // Persistent warps (batch.work_fwd != nullptr): the grid is one wave of resident warps and every warp pulls launch
  // positions from a counter until they run out, so a warp that drew a cheap tile immediately draws another one.
  __shared__ FwdSmem F;
  const int lane = threadIdx.x;
  for (uint32_t bpos = blockIdx.x;;) {
    if (batch.work_fwd) {
      if (lane == 0) bpos = atomicAdd(batch.work_fwd, 1u);
      bpos = __shfl_sync(FULL, bpos, 0);
    }
    if (bpos >= batch.n_work) return;
    __syncwarp();
    FwdOut fo;
    forward_tile<FULLPIX>(batch, prm, bpos, lane, F.sm, F.q_rank, F.q_cpos, F.p_rank, F.p_cpos, fo);
    if (!batch.work_fwd) return;
  }
}


constexpr int RED_STRIDE = 44;      // row stride (words) of the 32 x 40 reduction buffer: float4 rows, bank-conflict free

// Cross-tile sum of a Gaussian's moments, in the L2, without a return value.  Binary64: the addends are binary32 tile sums
// widened, so the sum over a few hundred tiles is exact (and the same in any order) unless their exponents span more than
// 2^29; a binary32 sum here (red.global.v4.f32.add, a quarter of the requests) left per-Gaussian gains of Gaussians a few
// pixels from the camera 2e-3 off the oracle and moving from call to call (Determinism).
__device__ __forceinline__ void red_add_f64(double* dst, double v) { asm volatile("red.global.add.f64 [%0], %1;" ::"l"(dst), "d"(v) : "memory"); }

// ---- S4 group tail.  After its slot body a lane holds, per entry, 18 column sums over its 8 pixels: F_p = sum_k f_k t_k^p
// (p <= 4), sum w^2, and G_c,p = sum_k g_c,k t_k^p (p <= 2) per channel.  Turning them into the lane's 40 moments (binomial
// shift to the Gaussian's centre line, powers of xi1) and reducing those over the 32 lanes once per entry cost as much as the
// slot body itself (ncu r2a: 41% of the kernel's instructions).  Instead the column sums of GE = 4 entries are parked in
// shared memory and ONE tail serves them all: lane l takes entry l / 8 and the four source lanes l % 8 + 8 k, assembles
// their moments (the source lane's pixel column and row block follow from its index) and accumulates them in registers;
// one shared-memory transpose then folds the eight partial sums of every entry, and the lanes issue the binary64 reductions
// into the L2 (red_add_f64 above) -- every lane assembles 4 (entry, lane) pairs instead of 4 entries x 1 lane, but the 32-row reduction per
// entry becomes an 8-row reduction per FOUR entries.
constexpr int GE = 4;

template <int NCH>
__device__ __forceinline__ void group_tail(const float4* rawA, const float2* rawB, float* red, const float4* sm, const float4* sm_wh,
                                           const float4* sm_ex, const uint32_t* q_rank, int gcount, uint32_t gpack, int tx, int ty,
                                           double* __restrict__ moments, int mom_stride, uint8_t* __restrict__ flag, int lane) {
  __syncwarp();                                            // the parked column sums are visible
  const int ge = lane >> 3, part = lane & 7;
  float acc[NMOM];
#pragma unroll
  for (int i = 0; i < NMOM; ++i) acc[i] = 0.0f;
  if (ge < gcount) {
    const int je = (int)((gpack >> (8 * ge)) & 0xffu);
    const float4 s0 = sm[je * 3], wh = sm_wh[je];
    const float h = wh.z, h2 = sm_ex[je].w;
    // The lane's 40 moments in the WHITENED coordinates xi = L^-1 (pixel - centre): xi1 = dx / l11 is the same for
    // a source lane's 8 pixels and xi2 = (dy - (l21 / l11) dx) / l22 = c1 + h t_k steps with the row, so
    // Y_b = sum_k f_k xi2_k^b follows from the F_p by a binomial shift, and the monomial sums are xi1^i Y_j.
    // (The shear keeps the column structure; the whitening keeps the later change to the u basis free of the
    // cancellation a plain pixel-offset basis has for elongated footprints.  DESIGN.md section 6.)
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int sl = part + 8 * k;                         // source lane: column sl & 15, row block sl >> 4
      const float4* ra = rawA + ge * 4 * 32 + sl;
      const float4 r0 = ra[0], r1 = ra[32], r2 = ra[64], r3 = ra[96];
      const float2 r4 = rawB[ge * 32 + sl];
      const float dx = sub_rn((float)(tx * TILE + (sl & 15)) + 0.5f, s0.x);
      const float x1 = dx * wh.x;
      const float c1 = ((((float)(ty * TILE + (sl >> 4) * PPL) + 4.0f) - s0.y) - wh.y * dx) * h;
      // Y_j = sum_p C(j, p) c1^(j - p) h^p F_p by the Pascal recurrence a_p <- c1 a_p + a_(p+1) (ten FMAs, no powers of c1)
      const float a0 = r0.x, a1 = h * r0.y, a2 = h2 * r0.z, a3 = (h2 * h) * r0.w, a4 = (h2 * h2) * r1.x;
      const float b0 = fmaf(c1, a0, a1), b1 = fmaf(c1, a1, a2), b2 = fmaf(c1, a2, a3), b3 = fmaf(c1, a3, a4);
      const float d0 = fmaf(c1, b0, b1), d1 = fmaf(c1, b1, b2), d2 = fmaf(c1, b2, b3);
      const float g0 = fmaf(c1, d0, d1), g1 = fmaf(c1, d1, d2);
      const float Y0v = a0, Y1v = b0, Y2v = d0, Y3v = g0, Y4v = fmaf(c1, g0, g1);
      const float x2 = x1 * x1, x3 = x2 * x1, x4 = x2 * x2;
      acc[0] += Y0v;
      acc[1] = fmaf(x1, Y0v, acc[1]);   acc[2] += Y1v;
      acc[3] = fmaf(x2, Y0v, acc[3]);   acc[4] = fmaf(x1, Y1v, acc[4]);   acc[5] += Y2v;
      acc[6] = fmaf(x3, Y0v, acc[6]);   acc[7] = fmaf(x2, Y1v, acc[7]);   acc[8] = fmaf(x1, Y2v, acc[8]);   acc[9] += Y3v;
      acc[10] = fmaf(x4, Y0v, acc[10]); acc[11] = fmaf(x3, Y1v, acc[11]); acc[12] = fmaf(x2, Y2v, acc[12]);
      acc[13] = fmaf(x1, Y3v, acc[13]); acc[14] += Y4v;
      const float gvv[12] = {r1.z, r1.w, r2.x, r2.y, r2.z, r2.w, r3.x, r3.y, r3.z, r3.w, r4.x, r4.y};
#pragma unroll
      for (int c = 0; c < NCH; ++c) {
        float* xm = acc + MOM_X + 6 * c;
        const float Z0 = gvv[3 * c], H1 = h * gvv[3 * c + 1], H2 = h2 * gvv[3 * c + 2];
        const float Z1 = fmaf(c1, Z0, H1);
        const float Z2 = fmaf(c1, Z1 + H1, H2);            // c1^2 Z0 + 2 c1 H1 + H2
        xm[0] = fmaf(x1, Z0, xm[0]); xm[1] += Z1; xm[2] = fmaf(x2, Z0, xm[2]); xm[3] = fmaf(x1, Z1, xm[3]); xm[4] += Z2; xm[5] += Z0;
      }
      acc[MOM_W2] += r1.y;
    }
  }
  __syncwarp();                                            // every lane has read its sources: rawA now serves as `red`
  {
    float4* row = reinterpret_cast<float4*>(red + lane * RED_STRIDE);
#pragma unroll
    for (int q = 0; q < NMOM / 4; ++q) row[q] = make_float4(acc[4 * q], acc[4 * q + 1], acc[4 * q + 2], acc[4 * q + 3]);
  }
  __syncwarp();
  // 4 entries x 10 float4 columns, each the sum of the 8 rows of its entry: columns 0..7 by all lanes, 8 and 9 by lanes 0..7.
  // No returning atomic: a returned value would tie up a scoreboard for a full L2 round trip; the touched list is built
  // afterwards from one flag byte per rank (launch_touched)
#pragma unroll
  for (int round = 0; round < 2; ++round) {
    const int e1 = round == 0 ? lane >> 3 : lane >> 1, q = round == 0 ? lane & 7 : 8 + (lane & 1);
    if ((round == 0 || lane < 8) && e1 < gcount) {
      const float* col = red + (e1 * 8) * RED_STRIDE + 4 * q;
      f2 a01 = bc2(0.f), a23 = bc2(0.f);
#pragma unroll
      for (int r = 0; r < 8; ++r) {
        const float4 x = *reinterpret_cast<const float4*>(col + r * RED_STRIDE);
        a01 = add2(a01, make_float2(x.x, x.y)); a23 = add2(a23, make_float2(x.z, x.w));
      }
      const uint32_t rank = q_rank[(gpack >> (8 * e1)) & 0xffu];
      // across the tiles a Gaussian covers the sums are taken in binary64: in binary32 their order-dependent rounding (a few 1e-7
      // of the total) was amplified to 2e-3 on the gains of Gaussians filling hundreds of tiles (near-singular moment matrices)
      double* dst = moments + (size_t)rank * mom_stride + 4 * q;
      red_add_f64(dst, (double)a01.x); red_add_f64(dst + 1, (double)a01.y); red_add_f64(dst + 2, (double)a23.x); red_add_f64(dst + 3, (double)a23.y);
      if (q == 0) flag[rank] = 1;                          // touched: the compaction of launch_touched reads these bytes
    }
  }
  __syncwarp();                                            // the buffers may be refilled
}

// S4 slot body: the lane's 8 pixels as 4 pairs (row q, row 7 - q), packed binary32 operations throughout.  With the row
// offsets t = -(3.5 - q) (.x) and +(3.5 - q) (.y), the column sums  F_p = sum_k f_k t_k^p,  G_c,p = sum_k g_c,k t_k^p  are
// accumulated per half with the broadcast weights |t|^p and folded at the end:  F_p = hi + (-1)^p lo.
// FROM_LIST: the tile's entries come from the list S3 wrote (RasterView::tlist), read backwards one chunk of 32 ranks ahead --
// no rect test, no ellipse test, no gather before the staging; tiles whose list outgrew TL_CAP are left to the instantiation
// without FROM_LIST, which filters the supertile list again as S3 did and exits at once when the batch has no such tile.
// The shared memory of one S4 warp (12,032 bytes; raster_kernel runs S3 in the same bytes):
struct BwdSmem {
  float4 sm[32 * 3];
  float4 sm_wh[32];           // per staged entry: (1/l11, l21/l11, 1/l22) of Sigma2D = L L^T, P_min
  float4 sm_ex[32];           // per staged entry: log2(sigma), P_min + P_max, P_min P_max, -
  // folded column sums of up to GE entries awaiting their group tail: values 0..15 of lane l, entry slot g at
  // rawA[(g * 4 + m) * 32 + l] (m = 0..3), values 16, 17 at rawB[g * 32 + l]; the reduction buffer of the tail aliases rawA
  float4 rawA[GE * 4 * 32];
  float2 rawB[GE * 32];
  uint32_t q_rank[64];
};

// S4 of one launch position (view, tile) by one warp.  FROM_REGS: the tile's `T`, `last` and list length come from the S3 sweep
// the same warp has just finished (fo) instead of from memory.
template <int NCH, bool FROM_LIST, bool FROM_REGS>
__device__ __forceinline__ void backward_tile(const RasterBatch& batch, const RasterParams& prm, uint32_t bpos, int lane, BwdSmem& S,
                                              const FwdOut* fo) {
  float4* sm = S.sm;
  float4* sm_wh = S.sm_wh;
  float4* sm_ex = S.sm_ex;
  float4* rawA = S.rawA;
  float2* rawB = S.rawB;
  uint32_t* q_rank = S.q_rank;
  float* red = reinterpret_cast<float*>(rawA);
  const int vidx = (int)(bpos % (uint32_t)batch.n);      // views interleaved (see forward_kernel)
  const RasterView& vw = batch.v[vidx];
  const Splat* __restrict__ splat_sorted = vw.splat_sorted;
  const uint32_t* __restrict__ ckeys = vw.ckeys;
  const ushort4* __restrict__ crect = vw.crect;
  const uint2* __restrict__ cranges = vw.cranges;
  const PixelBuf pix = vw.pix;
  double* __restrict__ moments = vw.moments;
  const int tile = batch.tile_order[bpos / (uint32_t)batch.n];   // heaviest tiles first (launch order)
  const uint32_t elast = FROM_REGS ? fo->elast : vw.tile_elast[tile];      // list position + 1 of the last entry any pixel of the tile passed
  // which instantiation owns the tile: the list holds the first TL_CAP entries only
  const bool listed = vw.tlist != nullptr && elast <= (uint32_t)TL_CAP;
  if (elast == 0u || listed != FROM_LIST) return;
  const int tx = tile % prm.tiles_x, ty = tile / prm.tiles_x;
  const int x = tx * TILE + (lane & 15), y0 = ty * TILE + (lane >> 4) * PPL;
  const float px = (float)x + 0.5f;
  const float X0 = (float)(tx * TILE), Y0 = (float)(ty * TILE);
  const uint32_t rmask = (1u << prm.rank_bits) - 1u;
  const uint32_t lt = (1u << lane) - 1u;

  // pair q: rows q (.x) and 7 - q (.y).  nS = MINUS the suffix sums, pre-scaled by sqrt(omega_ch) (see pass 2)
  f2 Tc2[PPL / 2], nS[NCH][PPL / 2];
  const float y0f = (float)y0;          // pixel centres py = y0f + (k + 0.5): small integers + 0.5, exact in binary32 (= S3's py bit for bit)
  int last_x[PPL / 2], last_y[PPL / 2];
#pragma unroll
  for (int q = 0; q < PPL / 2; ++q) {
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int k = h ? PPL - 1 - q : q;
      int l = 0;
      float T = 1.0f;
      if (FROM_REGS) {
        l = fo->last[k];
        T = h ? fo->T2[q].y : fo->T2[q].x;
      } else if (x < prm.W && y0 + k < prm.H) {
        const size_t p = (size_t)(y0 + k) * prm.W + x;
        l = pix.last[p];
        T = pix.T[p];
      }
      if (h) { last_y[q] = l; Tc2[q].y = T; } else { last_x[q] = l; Tc2[q].x = T; }
    }
#pragma unroll
    for (int c = 0; c < NCH; ++c) {
      const float b = c < 3 ? -prm.somega[c] * prm.bg[c] : 0.0f;
      nS[c][q] = make_float2(b * Tc2[q].x, b * Tc2[q].y);
    }
  }

  int e_next = (int)elast - 1;
  int gcount = 0;                      // entries parked for the group tail, and their positions j in the staged batch (8 bits each)
  uint32_t gpack = 0u;
  const float thr_near = 2e-5f * prm.ln_amax_over_amin;
  // FROM_LIST: entries elast-1, ..., 0 of the list S3 wrote, 32 at a time; the ranks of the next chunk are loaded before the
  // entry loop of this one and their splat records requested into the L1, so the staging finds them there
  const uint32_t* __restrict__ tl = FROM_LIST ? vw.tlist + (size_t)tile * TL_CAP : nullptr;
  uint32_t nrank = 0;
  if (FROM_LIST && lane <= e_next) nrank = tl[e_next - lane];
  // !FROM_LIST: walk the supertile list backwards from the last passed entry; the entries that pass the rect and ellipse tests
  // are the tile-list entries elast-1, elast-2, ..., 0 in that order
  uint32_t cbegin = 0, pos_hi = 0, qn = 0;
  ushort4 rcA = make_ushort4(1, 1, 0, 0), rcB = rcA;       // the lazy tile filter, software-pipelined two chunks deep as in forward_kernel
  uint32_t keyA = 0, keyB = 0;
  if (!FROM_LIST) {
    cbegin = cranges[(ty >> prm.sshift) * prm.super_x + (tx >> prm.sshift)].x;
    pos_hi = vw.tile_cend[tile];
    const uint32_t left = pos_hi - min(pos_hi, cbegin);
    if ((uint32_t)lane < left) { rcA = crect[pos_hi - 1u - (uint32_t)lane]; keyA = ckeys[pos_hi - 1u - (uint32_t)lane]; }
    if ((uint32_t)lane + 32u < left) { rcB = crect[pos_hi - 33u - (uint32_t)lane]; keyB = ckeys[pos_hi - 33u - (uint32_t)lane]; }
  }
  for (;;) {
    int cnt;
    if (FROM_LIST) {
      if (e_next < 0) break;
      cnt = min(32, e_next + 1);
      __syncwarp();
      if (lane < cnt) q_rank[lane] = nrank;                 // staged slot j <-> list entry e_next - j
      const int e_after = e_next - cnt;                     // first entry of the next chunk
      nrank = 0;
      if (lane <= e_after) nrank = tl[e_after - lane];
      __syncwarp();
      stage_queue(splat_sorted, q_rank, nullptr, (uint32_t)cnt, sm);
      if (lane <= e_after) {                                // 48-byte records: two sectors
        const char* nx = reinterpret_cast<const char*>(splat_sorted + nrank);
        prefetch_l1(nx); prefetch_l1(nx + 32);
      }
    } else {
      while (qn < 32u && pos_hi > cbegin) {
        const uint32_t span = min(32u, pos_hi - cbegin);
        const ushort4 rc = rcA;
        const uint32_t key = keyA;
        bool hit = (uint32_t)lane < span && tx >= rc.x && tx < rc.z && ty >= rc.y && ty < rc.w;
        pos_hi -= span;
        rcA = rcB; keyA = keyB;
        rcB = make_ushort4(1, 1, 0, 0);
        {
          const uint32_t left = pos_hi - cbegin;             // entries not yet taken; chunk A covers the first 32 of them
          if ((uint32_t)lane + 32u < left) { rcB = crect[pos_hi - 33u - (uint32_t)lane]; keyB = ckeys[pos_hi - 33u - (uint32_t)lane]; }
        }
        if (tx >= rcA.x && tx < rcA.z && ty >= rcA.y && ty < rcA.w) {
          const char* nx = reinterpret_cast<const char*>(splat_sorted + (keyA & rmask));
          prefetch_l1(nx); prefetch_l1(nx + 16);
        }
        uint32_t r = 0;
        if (hit) {
          r = key & rmask;
          const float4* sp = reinterpret_cast<const float4*>(splat_sorted + r);
          const float4 a0 = sp[0], a1 = sp[1];
          hit = ellipse_reaches_tile(a0.x, a0.y, a0.z, a0.w, a1.x, a1.w, X0, Y0);
        }
        const unsigned m = __ballot_sync(FULL, hit);
        if (hit) q_rank[qn + __popc(m & lt)] = r;
        qn += __popc(m);
      }
      if (qn == 0) break;
      cnt = (int)min(qn, 32u);
      __syncwarp();
      stage_queue(splat_sorted, q_rank, nullptr, (uint32_t)cnt, sm);
    }
    if (lane < cnt) {
      // Cholesky whitening of the footprint: xi = L^-1 d with Sigma2D = L L^T (L lower triangular), from the conic
      // Sigma2D^-1 = [[cA, cB], [cB, cC]]:  1/l22 = sqrt(cC),  1/l11 = sqrt(det(conic) / cC),  l21/l11 = -cB / cC
      const float4 q0 = sm[lane * 3], q1 = sm[lane * 3 + 1];
      const float cA = -2.0f * q0.z, cB = -q0.w, cC = -2.0f * q1.x;
      const float icC = 1.0f / cC;
      const float Pmin = __logf(prm.alpha_min / q1.y), Pmax = Pmin + prm.ln_amax_over_amin;
      sm_wh[lane] = make_float4(sqrtf(fmaxf(cA * cC - cB * cB, 0.0f) * icC), -cB * icC, sqrtf(cC), Pmin);
      sm_ex[lane] = make_float4(log2f(q1.y), Pmin + Pmax, Pmin * Pmax, cC);               // .w = h^2 = 1 / l22^2
    }
    __syncwarp();
    for (int j = 0; j <= cnt; ++j) {                         // j == cnt: only the group tail of what is still pending
      if (j < cnt) {
      const float4 s0 = sm[j * 3], s1 = sm[j * 3 + 1], s2 = sm[j * 3 + 2];
      const int e = e_next - j;
      const float dx = sub_rn(px, s0.x);
      // pass 1 (decision path): power bit-identical to S3; alpha from the fast exp (MUFU.EX2).  The two exps agree to
      // < 1e-6 relative, so they can only disagree on a decision of R-4 (contributor or not, clamped or not) when
      // `power` lies within ~1e-6 of P_min = ln(alpha_min / sigma) or P_max = ln(alpha_max / sigma).  If any pixel of the
      // tile comes within 2e-5 of either -- |(power - P_min)(power - P_max)| <= 2e-5 (P_max - P_min), two packed operations
      // -- the whole entry is evaluated with exp_spec instead, so every decision is the one S3 took.
      const float4 wh = sm_wh[j];
      const float4 ex = sm_ex[j];
      f2 pw[PPL / 2];
      bool near = false;
#pragma unroll
      for (int q = 0; q < PPL / 2; ++q) {
        const f2 dy = sub2(add2(bc2(y0f), make_float2((float)q + 0.5f, (float)(PPL - 1 - q) + 0.5f)), bc2(s0.y));
        const f2 power = splat_power2(s0.z, s0.w, s1.x, dx, dy);
        const bool in_x = e < last_x[q] && power.x <= 0.0f;        // the lower bounds never decide (see forward_kernel)
        const bool in_y = e < last_y[q] && power.y <= 0.0f;
        // outside the footprint or at / behind the entry the pixel stopped at: power = -inf, whose exp is 0 (MUFU) or NaN
        // (exp_spec); either fails `a >= alpha_min`
        pw[q].x = in_x ? power.x : -INFINITY;
        pw[q].y = in_y ? power.y : -INFINITY;
        const f2 nr = fma2(pw[q], sub2(pw[q], bc2(ex.y)), bc2(ex.z));
        near = near || fabsf(nr.x) <= thr_near || fabsf(nr.y) <= thr_near;
      }
      f2 av[PPL / 2];
      if (__any_sync(FULL, near)) {
#pragma unroll
        for (int q = 0; q < PPL / 2; ++q) av[q] = mul2(bc2(s1.y), exp_spec2(pw[q]));
      } else {
#pragma unroll
        for (int q = 0; q < PPL / 2; ++q) {
          const f2 arg = fma2(pw[q], bc2(0x1.715476p+0f), bc2(ex.x));        // sigma exp(power) in one FMA + MUFU
          av[q] = make_float2(ex2_approx(arg.x), ex2_approx(arg.y));
        }
      }
      // pass 2 (value path): with T_i = T_{i+1} / (1 - alpha_i) =: Tc * rc,
      //   beta_ch = dy_ch/dalpha_i = T_i v_i - Splus_i / (1 - alpha_i) = rc * d_ch,  d_ch = Tc v_ch - Splus_ch.
      // The channel weight enters as sqrt(omega_ch) folded into v_ch and Splus_ch (both linear), so
      // sum_ch omega_ch beta_ch^2 = rc^2 sum_ch d_ch^2 and the cross moments come out scaled by sqrt(omega_ch) (S5 applies
      // the other sqrt).
      float v[4];
      v[0] = prm.somega[0] * s2.x; v[1] = prm.somega[1] * s2.y; v[2] = prm.somega[2] * s2.z;
      v[3] = NCH == 4 ? prm.somega[3] * s1.z : 0.0f;
      f2 F0 = bc2(0.f), F1 = bc2(0.f), F2 = bc2(0.f), F3 = bc2(0.f), F4 = bc2(0.f), W2 = bc2(0.f);
      f2 G[NCH][3];
#pragma unroll
      for (int c = 0; c < NCH; ++c) G[c][0] = G[c][1] = G[c][2] = bc2(0.f);
      bool any = false;
#pragma unroll
      for (int q = 0; q < PPL / 2; ++q) {
        const f2 a = av[q];
        const bool pass_x = a.x >= prm.alpha_min, pass_y = a.y >= prm.alpha_min;     // same tests as S3 -> same contributor set
        f2 al, aa;                              // alpha (0: nothing moves), and alpha where its derivative is not zero
        al.x = pass_x ? fminf(a.x, prm.alpha_max) : 0.0f;
        al.y = pass_y ? fminf(a.y, prm.alpha_max) : 0.0f;
        aa.x = a.x > prm.alpha_max ? 0.0f : al.x;                                  // R-11: zero derivative at the 0.99 cap
        aa.y = a.y > prm.alpha_max ? 0.0f : al.y;
        const f2 om = sub2(bc2(1.0f), al);
        const f2 rc = make_float2(rcp_approx(om.x), rcp_approx(om.y));
        const f2 Ti = mul2(Tc2[q], rc);
        const f2 wm = mul2(al, Ti);
        f2 d[NCH];
#pragma unroll
        for (int c = 0; c < NCH; ++c) {
          d[c] = fma2(Tc2[q], bc2(v[c]), nS[c][q]);
          nS[c][q] = fma2(bc2(-v[c]), wm, nS[c][q]);
        }
        Tc2[q] = Ti;
        W2 = fma2(wm, wm, W2);
        f2 Dq = mul2(d[0], d[0]);
#pragma unroll
        for (int c = 1; c < NCH; ++c) Dq = fma2(d[c], d[c], Dq);
        const f2 r1 = mul2(rc, aa);                                              // rc * alpha, zero when inactive
        const f2 f = mul2(mul2(Dq, r1), r1);                                     // (sum_ch omega beta^2) alpha^2
        const f2 gw = mul2(wm, r1);                                              // beta_ch w alpha = d_ch * gw
        const float t1 = 3.5f - (float)q, t2 = t1 * t1, t3 = t2 * t1, t4 = t2 * t2;   // |t| of both rows of the pair
        F0 = add2(F0, f); F1 = fma2(f, bc2(t1), F1); F2 = fma2(f, bc2(t2), F2); F3 = fma2(f, bc2(t3), F3); F4 = fma2(f, bc2(t4), F4);
        const f2 gw1 = mul2(gw, bc2(t1)), gw2 = mul2(gw, bc2(t2));
#pragma unroll
        for (int c = 0; c < NCH; ++c) {
          G[c][0] = fma2(d[c], gw, G[c][0]); G[c][1] = fma2(d[c], gw1, G[c][1]); G[c][2] = fma2(d[c], gw2, G[c][2]);
        }
        any = any || pass_x || pass_y;
      }
      if (__any_sync(FULL, any)) {
        // fold the halves (rows q have t < 0, rows 7 - q have t > 0) and park the lane's 18 column sums; the moment assembly
        // and the cross-lane reduction happen once per GE entries (group tail below)
        const float F0s = F0.x + F0.y, F1s = F1.y - F1.x, F2s = F2.x + F2.y, F3s = F3.y - F3.x, F4s = F4.x + F4.y;
        float gv[12];
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          const int cc = c < NCH ? c : 0;
          gv[3 * c + 0] = c < NCH ? G[cc][0].x + G[cc][0].y : 0.0f;
          gv[3 * c + 1] = c < NCH ? G[cc][1].y - G[cc][1].x : 0.0f;
          gv[3 * c + 2] = c < NCH ? G[cc][2].x + G[cc][2].y : 0.0f;
        }
        float4* ra = rawA + gcount * 4 * 32 + lane;
        ra[0] = make_float4(F0s, F1s, F2s, F3s);
        ra[32] = make_float4(F4s, W2.x + W2.y, gv[0], gv[1]);
        ra[64] = make_float4(gv[2], gv[3], gv[4], gv[5]);
        ra[96] = make_float4(gv[6], gv[7], gv[8], gv[9]);
        rawB[gcount * 32 + lane] = make_float2(gv[10], gv[11]);
        gpack |= (uint32_t)j << (8 * gcount);
        ++gcount;
      }
      }  // j < cnt
      if (gcount == GE || (j == cnt && gcount > 0)) group_tail<NCH>(rawA, rawB, red, sm, sm_wh, sm_ex, q_rank, gcount, gpack, tx, ty, moments, vw.mom_stride, vw.touched_flag, lane);
      if (gcount == GE || j == cnt) { gcount = 0; gpack = 0u; }
    }
    e_next -= cnt;
    if (!FROM_LIST) shift_queue(q_rank, nullptr, qn, (uint32_t)cnt);
  }
}

template <int NCH, bool FROM_LIST>
__global__ void __launch_bounds__(32, NBV_BWD_MIN_BLOCKS) backward_kernel(const __grid_constant__ RasterBatch batch, const __grid_constant__ RasterParams prm) {
  __shared__ BwdSmem S;
  const int lane = threadIdx.x;
  // Persistent warps (batch.work != nullptr): the grid is one wave of resident warps and every warp pulls launch positions
  // from a counter until they run out, so a warp that drew a cheap tile immediately draws another one.
  uint32_t* const work = FROM_LIST ? batch.work : batch.work_fb;
  if (!FROM_LIST && batch.overflow && *batch.overflow == 0u) return;      // no tile of the batch outgrew its list
  for (uint32_t bpos = blockIdx.x;;) {
    if (work) {
      if (lane == 0) bpos = atomicAdd(work, 1u);
      bpos = __shfl_sync(FULL, bpos, 0);
    }
    if (bpos >= batch.n_work) return;
    __syncwarp();
    backward_tile<NCH, FROM_LIST, false>(batch, prm, bpos, lane, S, nullptr);
    if (!work) return;
  }
}

// OPT-IN (NBV_FUSED_RASTER=1; not the default: 1971 against 2036 views/s at config 2).
// S3 and S4 of a tile back to back by the same warp: S4 of a tile needs nothing but S3 of that tile (its `T`, `last`, and the list
// S3 wrote), so one persistent launch per batch serves both -- one drain per batch instead of two, and S4 starts from the
// registers S3 ends with instead of re-reading 8 B per pixel.  S3 still writes `T` / `last` (the fallback launch for tiles whose
// list outgrew TL_CAP and the parity exports read them).  Compiled for the register budget of S4 (16 warps per SM); the S3 part
// runs in the first 2,560 bytes of the S4 part's shared memory.
template <int NCH>
__global__ void __launch_bounds__(32, NBV_BWD_MIN_BLOCKS) raster_kernel(const __grid_constant__ RasterBatch batch, const __grid_constant__ RasterParams prm) {
  __shared__ BwdSmem S;
  const int lane = threadIdx.x;
  uint32_t* fq = reinterpret_cast<uint32_t*>(S.rawA);        // S3's four queues of 64 words in the column-sum buffer of S4
  for (uint32_t bpos = blockIdx.x;;) {
    if (lane == 0) bpos = atomicAdd(batch.work_fwd, 1u);
    bpos = __shfl_sync(FULL, bpos, 0);
    if (bpos >= batch.n_work) return;
    __syncwarp();
    FwdOut fo;
    forward_tile<false>(batch, prm, bpos, lane, S.sm, fq, fq + 64, fq + 128, fq + 192, fo);
    __syncwarp();
    backward_tile<NCH, true, true>(batch, prm, bpos, lane, S, &fo);
  }
}

static RasterParams make_params(const TileGrid& tg, int rank_bits, int W, int H, const nbv_config& cfg) {
  RasterParams p;
  p.W = W; p.H = H; p.tiles_x = tg.tiles_x; p.rank_bits = rank_bits;
  p.sshift = tg.sshift; p.super_x = tg.super_x;
  p.alpha_min = cfg.alpha_min; p.alpha_max = cfg.alpha_max; p.t_stop = cfg.t_stop;
  p.ln_amax_over_amin = logf(cfg.alpha_max / cfg.alpha_min);
  for (int c = 0; c < 3; ++c) p.bg[c] = cfg.bg[c];
  for (int c = 0; c < 4; ++c) {
    p.omega[c] = ((cfg.channel_mask >> c) & 1) ? cfg.channel_weight[c] : 0.0f;
    p.somega[c] = sqrtf(p.omega[c]);
  }
  return p;
}

void launch_forward(const RasterBatch& batch, const TileGrid& tg, int rank_bits, int W, int H, const nbv_config& cfg, bool full_pix,
                    cudaStream_t st) {
  const RasterParams p = make_params(tg, rank_bits, W, H, cfg);
  RasterBatch b = batch;
  b.n_work = (uint32_t)(tg.tiles_x * tg.tiles_y * batch.n);
  unsigned blocks = b.n_work;
  if (b.work_fwd) blocks = std::min(blocks, (unsigned)sm_count() * (full_pix ? 16u : 20u));
  const dim3 grid(blocks);
  ++g_kernel_launches;
  if (full_pix)
    forward_kernel<true><<<grid, 32, 0, st>>>(b, p);
  else
    forward_kernel<false><<<grid, 32, 0, st>>>(b, p);
}

// S3 + S4 of a batch in one persistent launch (raster_kernel), then the fallback S4 launch for tiles whose list outgrew TL_CAP.
// Needs the work counters (persistent mode) and the tile lists.
void launch_raster_fused(const RasterBatch& batch, const TileGrid& tg, int rank_bits, int W, int H, const nbv_config& cfg, cudaStream_t st) {
  const RasterParams p = make_params(tg, rank_bits, W, H, cfg);
  RasterBatch b = batch;
  b.n_work = (uint32_t)(tg.tiles_x * tg.tiles_y * batch.n);
  const dim3 grid(std::min(b.n_work, (unsigned)sm_count() * NBV_BWD_MIN_BLOCKS));
  g_kernel_launches += 2;
  if (cfg.channel_mask & NBV_CH_DEPTH) {
    raster_kernel<4><<<grid, 32, 0, st>>>(b, p);
    backward_kernel<4, false><<<grid, 32, 0, st>>>(b, p);
  } else {
    raster_kernel<3><<<grid, 32, 0, st>>>(b, p);
    backward_kernel<3, false><<<grid, 32, 0, st>>>(b, p);
  }
}

void launch_backward(const RasterBatch& batch, int N, const TileGrid& tg, int rank_bits, int W, int H, const nbv_config& cfg,
                     cudaStream_t st) {
  const RasterParams p = make_params(tg, rank_bits, W, H, cfg);
  RasterBatch b = batch;
  b.n_work = (uint32_t)(tg.tiles_x * tg.tiles_y * batch.n);
  unsigned blocks = b.n_work;
  if (b.work) blocks = std::min(blocks, (unsigned)sm_count() * NBV_BWD_MIN_BLOCKS);
  const dim3 grid(blocks);
  ++g_kernel_launches;
  // main launch: the tiles whose list S3 handed over; fallback launch: the tiles that outgrew it (exits at once if none did)
  if (cfg.channel_mask & NBV_CH_DEPTH) {
    backward_kernel<4, true><<<grid, 32, 0, st>>>(b, p);
    backward_kernel<4, false><<<grid, 32, 0, st>>>(b, p);
  } else {
    backward_kernel<3, true><<<grid, 32, 0, st>>>(b, p);
    backward_kernel<3, false><<<grid, 32, 0, st>>>(b, p);
  }
  ++g_kernel_launches;
  (void)N;
}

}  // namespace nbv
