// binning.cu -- S2 tile binning around the radix passes of sort.cu.
//
// Two-level binning.  After the depth sort (rank r <-> Gaussian ids_sorted[r]) the splats are
// gathered into rank order and every rank is duplicated into the SUPERTILES (S x S tiles, S a power of two chosen so
// that there are at most 256 of them) its tile rectangle touches, by a stable multi-split (count, scan, write): per
// supertile, the keys (supertile << rank_bits | rank) come out in rank = depth order.
// The tile list of tile t (R-5: the visible Gaussians whose rect contains t, in depth order) is the sub-sequence of
// its supertile's list that passes the rect test.  The rasteriser applies that test on the fly and only as far as the
// tile needs (until all 256 pixels have terminated), so the ~98% of the (tile, Gaussian) pairs that lie behind the
// termination depth in the dense configs are never materialised.  nbv_tile_lists materialises the full lists with the
// same test (count, scan, write) for the bit-exact parity check.
#include <algorithm>

#include "kernels.h"

namespace nbv {

__device__ __forceinline__ uint32_t coarse_count(ushort4 rc, int sshift) {
  if (rc.z <= rc.x || rc.w <= rc.y) return 0u;
  const uint32_t sx0 = rc.x >> sshift, sx1 = ((uint32_t)rc.z - 1u) >> sshift;
  const uint32_t sy0 = rc.y >> sshift, sy1 = ((uint32_t)rc.w - 1u) >> sshift;
  return (sx1 - sx0 + 1u) * (sy1 - sy0 + 1u);
}

// tile rect -> inclusive supertile rect (x0, y0, x1, y1); an empty tile rect gives x0 > x1 (covers nothing)
__device__ __forceinline__ uint4 super_rect(ushort4 rc, int sshift) {
  if (rc.z <= rc.x || rc.w <= rc.y) return make_uint4(1u, 1u, 0u, 0u);
  return make_uint4(rc.x >> sshift, rc.y >> sshift, ((uint32_t)rc.z - 1u) >> sshift, ((uint32_t)rc.w - 1u) >> sshift);
}
__device__ __forceinline__ bool covers_super(uint4 sr, uint32_t sx, uint32_t sy) {
  return sx >= sr.x && sx <= sr.z && sy >= sr.y && sy <= sr.w;
}
// bit s of the result = the supertile rect touches supertile s (row-major index); for grids of at most 64 supertiles the
// per-supertile loops below test one bit instead of four comparisons
__device__ __forceinline__ unsigned long long super_mask64(uint4 sr, int super_x) {
  unsigned long long m = 0ull;
  if (sr.x > sr.z) return m;
  const unsigned long long row = ((2ull << (sr.z - sr.x)) - 1ull) << sr.x;      // columns x0..x1 of one row
  for (uint32_t sy = sr.y; sy <= sr.w; ++sy) m |= row << (sy * (uint32_t)super_x);
  return m;
}

// Stable multi-split of the ranks into supertile lists, without materialising unsorted keys: block b owns the ranks
// [b * MS_T, (b + 1) * MS_T).  Pass 1 (this kernel, fused with the gather of the splats into rank order) counts, per
// supertile, the block's ranks that touch it; an exclusive scan of the (supertile-major) count table gives the start of
// every (supertile, block) segment; pass 2 writes each (supertile, rank) key and its tile rect at
// segment start + (number of earlier ranks of the block touching the same supertile), found with warp ballots.
// Rank order inside a supertile is preserved by construction: the lists are in depth order.
constexpr int MS_T = 1024;
constexpr int MS_W = MS_T / 32;

__global__ void __launch_bounds__(MS_T) msplit_count_kernel(const __grid_constant__ PreBatch batch, int N, int sshift, int super_x,
                                                            int n_super, uint32_t nblk) {
  __shared__ uint32_t cnt[256];
  const PreView& pv = batch.v[blockIdx.y];
  const uint32_t* __restrict__ ids_sorted = pv.ids[0];
  const Splat* __restrict__ splat = pv.splat;
  const ushort4* __restrict__ rect = pv.rect;
  Splat* __restrict__ splat_sorted = pv.splat_sorted;
  ushort4* __restrict__ rect_sorted = pv.rect_sorted;
  uint32_t* __restrict__ counts = pv.counts;
  const int r = blockIdx.x * MS_T + threadIdx.x, lane = threadIdx.x & 31;
  if (threadIdx.x < 256) cnt[threadIdx.x] = 0;
  __syncthreads();
  ushort4 rc = make_ushort4(0, 0, 0, 0);
  if (r < N) {
    const uint32_t g = ids_sorted[r];
    rc = rect[g];
    rect_sorted[r] = rc;
    const float4* src = reinterpret_cast<const float4*>(splat + g);
    float4* dst = reinterpret_cast<float4*>(splat_sorted + r);
    dst[0] = src[0];
    dst[1] = src[1];
    dst[2] = src[2];
  }
  const uint4 sr = super_rect(rc, sshift);
  if (n_super <= 64) {
    const unsigned long long cm = super_mask64(sr, super_x);
    for (int s = 0; s < n_super; ++s) {
      const unsigned m = __ballot_sync(0xffffffffu, (cm >> s) & 1ull);
      if (lane == 0 && m) atomicAdd(&cnt[s], (uint32_t)__popc(m));
    }
  } else {
    for (int s = 0, sx = 0, sy = 0; s < n_super; ++s) {          // (sx, sy) walk the supertiles row-major: no division
      const unsigned m = __ballot_sync(0xffffffffu, covers_super(sr, (uint32_t)sx, (uint32_t)sy));
      if (lane == 0 && m) atomicAdd(&cnt[s], (uint32_t)__popc(m));
      if (++sx == super_x) { sx = 0; ++sy; }
    }
  }
  __syncthreads();
  if ((int)threadIdx.x < n_super) counts[(size_t)threadIdx.x * nblk + blockIdx.x] = cnt[threadIdx.x];
}

__global__ void __launch_bounds__(MS_T) msplit_write_kernel(const __grid_constant__ PreBatch batch, int N, int sshift, int super_x,
                                                            int n_super, int rank_bits, uint32_t nblk, uint32_t cap) {
  const PreView& pv = batch.v[blockIdx.y];
  const ushort4* __restrict__ rect_sorted = pv.rect_sorted;
  const uint32_t* __restrict__ scanned = pv.counts;
  const uint32_t* __restrict__ d_total = &pv.counters->n_coarse;
  uint32_t* __restrict__ keys = pv.ckeys;
  ushort4* __restrict__ crect = pv.crect;
  uint2* __restrict__ ranges = pv.cranges;
  __shared__ uint16_t wc[256][MS_W];         // per supertile: ranks of warp w touching it, then the exclusive prefix over warps
  __shared__ uint32_t seg[256];              // start of this block's segment in every supertile list (one global load each,
                                             // up front: a load inside the write loop would stall every iteration on the L2)
  const int r = blockIdx.x * MS_T + threadIdx.x, lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const uint32_t lt = (1u << lane) - 1u;
  const ushort4 rc = r < N ? rect_sorted[r] : make_ushort4(0, 0, 0, 0);
  const uint4 sr = super_rect(rc, sshift);
  const bool small = n_super <= 64;
  const unsigned long long cm = small ? super_mask64(sr, super_x) : 0ull;
  for (int s = 0, sx = 0, sy = 0; s < n_super; ++s) {
    const bool c = small ? ((cm >> s) & 1ull) != 0ull : covers_super(sr, (uint32_t)sx, (uint32_t)sy);
    const unsigned m = __ballot_sync(0xffffffffu, c);
    if (lane == 0) wc[s][w] = (uint16_t)__popc(m);
    if (!small && ++sx == super_x) { sx = 0; ++sy; }
  }
  __syncthreads();
  if ((int)threadIdx.x < n_super) {
    seg[threadIdx.x] = scanned[(size_t)threadIdx.x * nblk + blockIdx.x];
    uint32_t run = 0;
    for (int k = 0; k < MS_W; ++k) {
      const uint32_t c = wc[threadIdx.x][k];
      wc[threadIdx.x][k] = (uint16_t)run;
      run += c;
    }
    if (blockIdx.x == 0) {                    // supertile ranges: [start of (s, block 0), start of (s + 1, block 0))
      const uint32_t b = scanned[(size_t)threadIdx.x * nblk];
      const uint32_t e = ((int)threadIdx.x + 1 < n_super) ? scanned[(size_t)(threadIdx.x + 1) * nblk] : min(*d_total, cap);
      ranges[threadIdx.x] = make_uint2(b, e);
    }
  }
  __syncthreads();
  for (int s = 0, sx = 0, sy = 0; s < n_super; ++s) {
    const bool c = small ? ((cm >> s) & 1ull) != 0ull : covers_super(sr, (uint32_t)sx, (uint32_t)sy);
    const unsigned m = __ballot_sync(0xffffffffu, c);
    if (!small && ++sx == super_x) { sx = 0; ++sy; }
    if (c) {
      const uint32_t pos = seg[s] + wc[s][w] + __popc(m & lt);
      if (pos < cap) {
        keys[pos] = ((uint32_t)s << rank_bits) | (uint32_t)r;
        crect[pos] = rc;
      }
    }
  }
}

uint32_t msplit_blocks(int N) { return (uint32_t)((N + MS_T - 1) / MS_T); }

void launch_msplit_count(const PreBatch& batch, int N, const TileGrid& tg, cudaStream_t st) {
  const uint32_t nblk = msplit_blocks(N);
  ++g_kernel_launches;
  msplit_count_kernel<<<dim3(nblk, (unsigned)batch.n), MS_T, 0, st>>>(batch, N, tg.sshift, tg.super_x, tg.super_x * tg.super_y, nblk);
}

void launch_msplit_write(const PreBatch& batch, int N, const TileGrid& tg, int rank_bits, uint32_t cap, cudaStream_t st) {
  const uint32_t nblk = msplit_blocks(N);
  ++g_kernel_launches;
  msplit_write_kernel<<<dim3(nblk, (unsigned)batch.n), MS_T, 0, st>>>(batch, N, tg.sshift, tg.super_x, tg.super_x * tg.super_y, rank_bits, nblk,
                                                                      cap);
}

// ---- parity export: the full tile lists (R-5), by the same rect test the rasteriser applies on the fly.
// One warp per tile; pass 0 counts, pass 1 writes Gaussian ids at the scanned offsets.
__global__ void __launch_bounds__(32) tile_list_kernel(const uint32_t* __restrict__ ckeys, const ushort4* __restrict__ crect,
                                                        const uint2* __restrict__ cranges, TileGrid tg, uint32_t rmask,
                                                        const uint32_t* __restrict__ ids_sorted, const uint32_t* __restrict__ offsets,
                                                        uint32_t* __restrict__ counts, int32_t* __restrict__ ids_out) {
  const int tile = blockIdx.x, lane = threadIdx.x;
  const int tx = tile % tg.tiles_x, ty = tile / tg.tiles_x;
  const uint2 range = cranges[(ty >> tg.sshift) * tg.super_x + (tx >> tg.sshift)];
  uint32_t n = 0;
  const uint32_t base = ids_out ? offsets[tile] : 0u;
  for (uint32_t pos = range.x; pos < range.y; pos += 32) {
    const uint32_t i = pos + lane;
    bool hit = false;
    if (i < range.y) {
      const ushort4 rc = crect[i];
      hit = tx >= rc.x && tx < rc.z && ty >= rc.y && ty < rc.w;
    }
    const unsigned m = __ballot_sync(0xffffffffu, hit);
    if (hit && ids_out) ids_out[base + n + __popc(m & ((1u << lane) - 1u))] = (int32_t)ids_sorted[ckeys[i] & rmask];
    n += __popc(m);
  }
  if (lane == 0 && counts) counts[tile] = n;
}

__global__ void export_offsets_kernel(const uint32_t* __restrict__ scanned, int n_tiles, const uint32_t* __restrict__ total,
                                      int64_t* __restrict__ offsets) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t < n_tiles) offsets[t] = (int64_t)scanned[t];
  if (t == n_tiles) offsets[t] = (int64_t)*total;
}

void launch_tile_counts(const uint32_t* ckeys, const ushort4* crect, const uint2* cranges, const TileGrid& tg, int rank_bits,
                        uint32_t* counts, uint32_t* scanned, uint32_t* total, uint32_t* scan_tmp, int64_t* offsets_out, cudaStream_t st) {
  const int n_tiles = tg.tiles_x * tg.tiles_y;
  ++g_kernel_launches;
  tile_list_kernel<<<n_tiles, 32, 0, st>>>(ckeys, crect, cranges, tg, (1u << rank_bits) - 1u, nullptr, nullptr, counts, nullptr);
  exclusive_scan_u32(counts, scanned, (size_t)n_tiles, scan_tmp, total, st);
  ++g_kernel_launches;
  export_offsets_kernel<<<(n_tiles + 1 + 255) / 256, 256, 0, st>>>(scanned, n_tiles, total, offsets_out);
}

void launch_tile_ids(const uint32_t* ckeys, const ushort4* crect, const uint2* cranges, const TileGrid& tg, int rank_bits,
                     const uint32_t* ids_sorted, const uint32_t* scanned, int32_t* ids_out, cudaStream_t st) {
  const int n_tiles = tg.tiles_x * tg.tiles_y;
  ++g_kernel_launches;
  tile_list_kernel<<<n_tiles, 32, 0, st>>>(ckeys, crect, cranges, tg, (1u << rank_bits) - 1u, ids_sorted, scanned, nullptr, ids_out);
}

}  // namespace nbv
