// binning.cu -- S2 tile binning around the radix passes of sort.cu.
//
// Two-level binning.  After the depth sort (rank r <-> Gaussian ids_sorted[r]) the splats are
// gathered into rank order and every rank is duplicated into the SUPERTILES (S x S tiles, S a power of two chosen so
// that there are at most 256 of them) its tile rectangle touches: keys (supertile << rank_bits | rank) are emitted
// rank-major, so one stable radix pass on the supertile digit yields, per supertile, the ranks in depth order.
// The tile list of tile t (R-5: the visible Gaussians whose rect contains t, in depth order) is the sub-sequence of
// its supertile's list that passes the rect test.  The rasteriser applies that test on the fly and only as far as the
// tile needs (until all 256 pixels have terminated), so the ~98% of the (tile, Gaussian) pairs that lie behind the
// termination depth in the dense configs are never materialised.  nbv_tile_lists materialises the full lists with the
// same test (count, scan, write) for the bit-exact parity check.
#include "kernels.h"

namespace nbv {

__device__ __forceinline__ uint32_t coarse_count(ushort4 rc, int sshift) {
  if (rc.z <= rc.x || rc.w <= rc.y) return 0u;
  const uint32_t sx0 = rc.x >> sshift, sx1 = ((uint32_t)rc.z - 1u) >> sshift;
  const uint32_t sy0 = rc.y >> sshift, sy1 = ((uint32_t)rc.w - 1u) >> sshift;
  return (sx1 - sx0 + 1u) * (sy1 - sy0 + 1u);
}

__global__ void __launch_bounds__(256) gather_kernel(const uint32_t* __restrict__ ids_sorted, const Splat* __restrict__ splat,
                                                      const ushort4* __restrict__ rect, int N, int sshift,
                                                      Splat* __restrict__ splat_sorted, ushort4* __restrict__ rect_sorted,
                                                      uint32_t* __restrict__ ncoarse_sorted) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= N) return;
  const uint32_t g = ids_sorted[r];
  const ushort4 rc = rect[g];
  rect_sorted[r] = rc;
  ncoarse_sorted[r] = coarse_count(rc, sshift);
  const float4* src = reinterpret_cast<const float4*>(splat + g);
  float4* dst = reinterpret_cast<float4*>(splat_sorted + r);
  dst[0] = src[0];
  dst[1] = src[1];
  dst[2] = src[2];
}

void launch_gather(const uint32_t* ids_sorted, const Splat* splat, const ushort4* rect, int N, int sshift, Splat* splat_sorted,
                   ushort4* rect_sorted, uint32_t* ncoarse_sorted, cudaStream_t st) {
  ++g_kernel_launches;
  gather_kernel<<<(N + 255) / 256, 256, 0, st>>>(ids_sorted, splat, rect, N, sshift, splat_sorted, rect_sorted, ncoarse_sorted);
}

// 8 ranks per warp (4 lanes each): a rank touches a handful of supertiles
__global__ void __launch_bounds__(256) emit_coarse_kernel(const ushort4* __restrict__ rect_sorted, const uint32_t* __restrict__ offsets,
                                                           int N, int sshift, int super_x, int rank_bits, uint32_t cap,
                                                           uint32_t* __restrict__ keys) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  const int r = t >> 2, sub = t & 3;
  if (r >= N) return;
  const ushort4 rc = rect_sorted[r];
  if (rc.z <= rc.x || rc.w <= rc.y) return;
  const uint32_t sx0 = rc.x >> sshift, sx1 = ((uint32_t)rc.z - 1u) >> sshift;
  const uint32_t sy0 = rc.y >> sshift, sy1 = ((uint32_t)rc.w - 1u) >> sshift;
  const uint32_t w = sx1 - sx0 + 1u, n = w * (sy1 - sy0 + 1u);
  const uint32_t off = offsets[r];
  for (uint32_t i = sub; i < n; i += 4) {
    const uint32_t sy = sy0 + i / w, sx = sx0 + i % w;
    if (off + i < cap) keys[off + i] = ((sy * (uint32_t)super_x + sx) << rank_bits) | (uint32_t)r;
  }
}

void launch_emit_coarse(const ushort4* rect_sorted, const uint32_t* offsets, int N, int sshift, int super_x, int rank_bits,
                        uint32_t cap, uint32_t* keys, cudaStream_t st) {
  const long long threads = (long long)N * 4;
  ++g_kernel_launches;
  emit_coarse_kernel<<<(unsigned)((threads + 255) / 256), 256, 0, st>>>(rect_sorted, offsets, N, sshift, super_x, rank_bits, cap, keys);
}

// After the single stable pass on the supertile digit the scanned histogram holds every digit's start:
// range of supertile s = [hist[s * nb], hist[(s + 1) * nb]) (the last one ends at n).
__global__ void __launch_bounds__(256) coarse_ranges_kernel(const uint32_t* __restrict__ hist_scanned, uint32_t nb, int n_super,
                                                             int n_digits, const uint32_t* __restrict__ d_n, uint32_t cap,
                                                             uint2* __restrict__ ranges) {
  const int s = threadIdx.x;
  if (s >= n_super) return;
  const uint32_t n = min(*d_n, cap);
  const uint32_t b = hist_scanned[(size_t)s * nb];
  const uint32_t e = (s + 1 < n_digits) ? hist_scanned[(size_t)(s + 1) * nb] : n;
  ranges[s] = make_uint2(b, e);
}

void launch_coarse_ranges(const uint32_t* hist_scanned, uint32_t nb, int n_super, int n_digits, const uint32_t* d_n, uint32_t cap,
                          uint2* ranges, cudaStream_t st) {
  ++g_kernel_launches;
  coarse_ranges_kernel<<<1, 256, 0, st>>>(hist_scanned, nb, n_super, n_digits, d_n, cap, ranges);
}

// rect of every sorted coarse entry, in list order (coalesced reads for the rasteriser's rect test)
__global__ void __launch_bounds__(256) coarse_rect_kernel(const uint32_t* __restrict__ keys, const uint32_t* __restrict__ d_n, uint32_t cap,
                                                           uint32_t rmask, const ushort4* __restrict__ rect_sorted,
                                                           ushort4* __restrict__ crect) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= min(*d_n, cap)) return;
  crect[i] = rect_sorted[keys[i] & rmask];
}

void launch_coarse_rect(const uint32_t* keys, const uint32_t* d_n, uint32_t cap, int rank_bits, const ushort4* rect_sorted,
                        ushort4* crect, cudaStream_t st) {
  if (cap == 0) return;
  ++g_kernel_launches;
  coarse_rect_kernel<<<(cap + 255) / 256, 256, 0, st>>>(keys, d_n, cap, (1u << rank_bits) - 1u, rect_sorted, crect);
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
