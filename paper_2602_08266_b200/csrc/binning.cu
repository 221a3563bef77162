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

// tile rect -> inclusive supertile rect (x0, y0, x1, y1); an empty tile rect gives x0 > x1 (covers nothing)
__device__ __forceinline__ uint4 super_rect(ushort4 rc, int sshift) {
  if (rc.z <= rc.x || rc.w <= rc.y) return make_uint4(1u, 1u, 0u, 0u);
  return make_uint4(rc.x >> sshift, rc.y >> sshift, ((uint32_t)rc.z - 1u) >> sshift, ((uint32_t)rc.w - 1u) >> sshift);
}
// Coverage of a supertile rect as a bit mask over the (at most 256) supertiles, row-major: bit s of word s / 32.
constexpr int MS_WORDS = 8;
__device__ __forceinline__ void super_mask(uint4 sr, int super_x, int words, uint32_t (&cm)[MS_WORDS]) {
#pragma unroll
  for (int w = 0; w < MS_WORDS; ++w) cm[w] = 0u;
  if (sr.x > sr.z) return;
  const uint32_t len = sr.z - sr.x + 1u;
  for (uint32_t sy = sr.y; sy <= sr.w; ++sy) {
    const uint32_t lo = sy * (uint32_t)super_x + sr.x, hi = lo + len;       // bits [lo, hi)
#pragma unroll
    for (int w = 0; w < MS_WORDS; ++w) {
      if (w < words) {
        const uint32_t a = max(lo, 32u * w), e = min(hi, 32u * w + 32u);
        if (a < e) cm[w] |= (e - a == 32u ? 0xffffffffu : ((1u << (e - a)) - 1u) << (a - 32u * w));
      }
    }
  }
}

// 32 x 32 bit-matrix transpose across the warp: lane i gives row i and receives column i (bit c of the result = bit i of
// lane c's input).  Applied to the lanes' coverage words it yields, in lane i, the ballot "which lanes touch supertile
// 32 w + i" -- 5 shuffles per 32 supertiles instead of 32 votes.
__device__ __forceinline__ uint32_t transpose32(uint32_t x, int lane) {
#pragma unroll
  for (int j = 16; j > 0; j >>= 1) {
    const uint32_t m = j == 16 ? 0x0000ffffu : j == 8 ? 0x00ff00ffu : j == 4 ? 0x0f0f0f0fu : j == 2 ? 0x33333333u : 0x55555555u;
    const uint32_t y = __shfl_xor_sync(0xffffffffu, x, j);
    x = (lane & j) ? ((x & ~m) | ((y >> j) & m)) : ((x & m) | ((y << j) & ~m));
  }
  return x;
}

// Stable multi-split of the ranks into supertile lists, without materialising unsorted keys: block b owns the ranks
// [b * MS_T, (b + 1) * MS_T).  Pass 1 (this kernel, fused with the gather of the splats into rank order) counts, per
// supertile, the block's ranks that touch it; an exclusive scan of the (supertile-major) count table gives the start of
// every (supertile, block) segment; pass 2 writes each (supertile, rank) key and its tile rect at
// segment start + (number of earlier ranks of the block touching the same supertile).
// Rank order inside a supertile is preserved by construction: the lists are in depth order.
// Both passes were issue-bound on one vote per (warp, supertile) (ncu r2c: 64-106 M warp instructions per 8-view batch);
// now a warp transposes its 32 coverage masks, which gives every per-supertile lane mask at once.
constexpr int MS_T = 1024;
constexpr int MS_W = MS_T / 32;

__global__ void __launch_bounds__(MS_T) msplit_count_kernel(const __grid_constant__ PreBatch batch, int N, int sshift, int super_x,
                                                            int n_super, uint32_t nblk) {
  __shared__ uint16_t wc[256][MS_W + 2];     // [supertile][warp]; row stride 34 halves = 17 words (odd): conflict-free column sums
  const PreView& pv = batch.v[blockIdx.y];
  const uint32_t* __restrict__ ids_sorted = pv.ids[0];
  const Splat* __restrict__ splat = pv.splat;
  const ushort4* __restrict__ rect = pv.rect;
  Splat* __restrict__ splat_sorted = pv.splat_sorted;
  ushort4* __restrict__ rect_sorted = pv.rect_sorted;
  uint32_t* __restrict__ counts = pv.counts;
  const int r = blockIdx.x * MS_T + threadIdx.x, lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int words = (n_super + 31) >> 5;
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
  uint32_t cm[MS_WORDS];
  super_mask(super_rect(rc, sshift), super_x, words, cm);
#pragma unroll
  for (int k = 0; k < MS_WORDS; ++k)
    if (k < words) wc[32 * k + lane][w] = (uint16_t)__popc(transpose32(cm[k], lane));
  __syncthreads();
  if ((int)threadIdx.x < n_super) {
    uint32_t c = 0;
#pragma unroll
    for (int k = 0; k < MS_W; ++k) c += wc[threadIdx.x][k];
    counts[(size_t)threadIdx.x * nblk + blockIdx.x] = c;
  }
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
  extern __shared__ __align__(16) uint32_t ms_smem[];
  // per supertile: start of this block's segment in its list + the ranks of earlier warps touching it (seg), and per
  // (warp, supertile) the lanes of that warp touching it (bm)
  uint32_t* seg = ms_smem;                              // [n_super]
  uint32_t* bm = ms_smem + 256;                         // [MS_W][n_super]
  uint16_t* wc = reinterpret_cast<uint16_t*>(bm + MS_W * n_super);      // [n_super][MS_W + 2]
  const int r = blockIdx.x * MS_T + threadIdx.x, lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int words = (n_super + 31) >> 5;
  const uint32_t lt = (1u << lane) - 1u;
  const ushort4 rc = r < N ? rect_sorted[r] : make_ushort4(0, 0, 0, 0);
  // this block's row of the scanned count table (supertile-major: one sector per supertile), needed after the first barrier
  const uint32_t seg0 = (int)threadIdx.x < n_super ? scanned[(size_t)threadIdx.x * nblk + blockIdx.x] : 0u;
  uint32_t cm[MS_WORDS];
  super_mask(super_rect(rc, sshift), super_x, words, cm);
#pragma unroll
  for (int k = 0; k < MS_WORDS; ++k)
    if (k < words) {                                    // uniform over the warp: the shuffles inside are warp-wide
      const uint32_t m = transpose32(cm[k], lane);
      if (32 * k + lane < n_super) {
        bm[w * n_super + 32 * k + lane] = m;
        wc[(32 * k + lane) * (MS_W + 2) + w] = (uint16_t)__popc(m);
      }
    }
  __syncthreads();
  if ((int)threadIdx.x < n_super) {
    seg[threadIdx.x] = seg0;
    uint16_t* row = wc + threadIdx.x * (MS_W + 2);
    uint32_t before = 0;
#pragma unroll
    for (int k = 0; k < MS_W; ++k) {                    // exclusive prefix over the warps (a block holds 1024 ranks: fits 16 bits)
      const uint32_t c = row[k];
      row[k] = (uint16_t)before;
      before += c;
    }
    if (blockIdx.x == 0) {                    // supertile ranges: [start of (s, block 0), start of (s + 1, block 0))
      const uint32_t b = scanned[(size_t)threadIdx.x * nblk];
      const uint32_t e = ((int)threadIdx.x + 1 < n_super) ? scanned[(size_t)(threadIdx.x + 1) * nblk] : min(*d_total, cap);
      ranges[threadIdx.x] = make_uint2(b, e);
    }
  }
  __syncthreads();
  // every lane walks the supertiles of its own rect
#pragma unroll
  for (int k = 0; k < MS_WORDS; ++k) {
    if (k >= words) break;
    uint32_t bits = cm[k];
    while (bits) {
      const int s = 32 * k + __ffs((int)bits) - 1;
      bits &= bits - 1u;
      const uint32_t pos = seg[s] + wc[s * (MS_W + 2) + w] + __popc(bm[w * n_super + s] & lt);
      if (pos < cap) {
        keys[pos] = ((uint32_t)s << rank_bits) | (uint32_t)r;
        crect[pos] = rc;
      }
    }
  }
}

static size_t msplit_write_smem(int n_super) {
  return (size_t)256 * 4 + (size_t)MS_W * n_super * 4 + (size_t)n_super * (MS_W + 2) * 2;
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
  const int n_super = tg.super_x * tg.super_y;
  const size_t smem = msplit_write_smem(n_super);
  if (smem > 48 * 1024 && cudaFuncSetAttribute(msplit_write_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return;                                             // the caller's cudaGetLastError() reports it
  msplit_write_kernel<<<dim3(nblk, (unsigned)batch.n), MS_T, smem, st>>>(batch, N, tg.sshift, tg.super_x, n_super, rank_bits, nblk, cap);
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
