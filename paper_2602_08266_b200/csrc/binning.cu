// binning.cu -- S2 tile binning around the radix passes of sort.cu.
//
// After the depth sort (rank r <-> Gaussian ids_sorted[r]): gather the splats into rank order, count the tiles of
// every rank, scan, emit keys (tile << rank_bits | rank) rank-major (so the low digits are already sorted), sort
// the tile digit with stable passes, and find each tile's [begin, end) range.
#include "kernels.h"

namespace nbv {

__global__ void __launch_bounds__(256) gather_kernel(const uint32_t* __restrict__ ids_sorted, const Splat* __restrict__ splat,
                                                      const ushort4* __restrict__ rect, int N, Splat* __restrict__ splat_sorted,
                                                      ushort4* __restrict__ rect_sorted, uint32_t* __restrict__ ntiles_sorted) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= N) return;
  const uint32_t g = ids_sorted[r];
  const ushort4 rc = rect[g];
  rect_sorted[r] = rc;
  ntiles_sorted[r] = (uint32_t)(rc.z - rc.x) * (uint32_t)(rc.w - rc.y);
  const float4* src = reinterpret_cast<const float4*>(splat + g);
  float4* dst = reinterpret_cast<float4*>(splat_sorted + r);
  dst[0] = src[0];
  dst[1] = src[1];
  dst[2] = src[2];
}

void launch_gather(const uint32_t* ids_sorted, const Splat* splat, const ushort4* rect, int N, Splat* splat_sorted,
                   ushort4* rect_sorted, uint32_t* ntiles_sorted, cudaStream_t st) {
  ++g_kernel_launches;
  gather_kernel<<<(N + 255) / 256, 256, 0, st>>>(ids_sorted, splat, rect, N, splat_sorted, rect_sorted, ntiles_sorted);
}

// one warp per rank; lanes stride over the rect's tiles (row-major inside the rect): coalesced key writes
__global__ void __launch_bounds__(256) emit_keys_kernel(const ushort4* __restrict__ rect_sorted, const uint32_t* __restrict__ offsets,
                                                         int N, int tiles_x, int rank_bits, uint32_t* __restrict__ keys) {
  const int r = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (r >= N) return;
  const ushort4 rc = rect_sorted[r];
  const uint32_t w = rc.z - rc.x, h = rc.w - rc.y;
  const uint32_t n = w * h;
  if (n == 0) return;
  const uint32_t off = offsets[r];
  for (uint32_t i = lane; i < n; i += 32) {
    const uint32_t ty = rc.y + i / w, tx = rc.x + i % w;
    keys[off + i] = ((ty * (uint32_t)tiles_x + tx) << rank_bits) | (uint32_t)r;
  }
}

void launch_emit_keys(const ushort4* rect_sorted, const uint32_t* offsets, int N, int tiles_x, int rank_bits,
                      uint32_t* keys, cudaStream_t st) {
  const long long threads = (long long)N * 32;
  ++g_kernel_launches;
  emit_keys_kernel<<<(unsigned)((threads + 255) / 256), 256, 0, st>>>(rect_sorted, offsets, N, tiles_x, rank_bits, keys);
}

__global__ void __launch_bounds__(256) tile_ranges_kernel(const uint32_t* __restrict__ keys, uint32_t n, int rank_bits,
                                                           uint2* __restrict__ ranges) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t t = keys[i] >> rank_bits;
  if (i == 0 || (keys[i - 1] >> rank_bits) != t) ranges[t].x = i;
  if (i == n - 1 || (keys[i + 1] >> rank_bits) != t) ranges[t].y = i + 1;
}

void launch_tile_ranges(const uint32_t* keys, size_t n_keys, int rank_bits, uint2* ranges, int n_tiles, cudaStream_t st) {
  cudaMemsetAsync(ranges, 0, sizeof(uint2) * (size_t)n_tiles, st);
  if (n_keys == 0) return;
  ++g_kernel_launches;
  tile_ranges_kernel<<<(unsigned)((n_keys + 255) / 256), 256, 0, st>>>(keys, (uint32_t)n_keys, rank_bits, ranges);
}

// ---- parity export: per-tile offsets (int64) and Gaussian ids
__global__ void range_counts_kernel(const uint2* __restrict__ ranges, int n_tiles, uint32_t* __restrict__ counts) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t < n_tiles) counts[t] = ranges[t].y - ranges[t].x;
}

__global__ void export_offsets_kernel(const uint32_t* __restrict__ scanned, int n_tiles, uint32_t total, int64_t* __restrict__ offsets) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t < n_tiles) offsets[t] = (int64_t)scanned[t];
  if (t == n_tiles) offsets[t] = (int64_t)total;
}

__global__ void export_ids_kernel(const uint32_t* __restrict__ keys, uint32_t n, int rank_bits, const uint32_t* __restrict__ ids_sorted,
                                  int32_t* __restrict__ ids_out) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) ids_out[i] = (int32_t)ids_sorted[keys[i] & ((1u << rank_bits) - 1u)];
}

void launch_export_lists(const uint32_t* keys, size_t n_keys, int rank_bits, const uint32_t* ids_sorted, const uint2* ranges,
                         int n_tiles, int64_t* offsets, int32_t* ids_out, uint32_t* tmp_counts, uint32_t* scan_tmp, cudaStream_t st) {
  // the sorted keys are already grouped by ascending tile, so offsets are the scanned counts
  ++g_kernel_launches;
  range_counts_kernel<<<(n_tiles + 255) / 256, 256, 0, st>>>(ranges, n_tiles, tmp_counts);
  exclusive_scan_u32(tmp_counts, tmp_counts, (size_t)n_tiles, scan_tmp, nullptr, st);
  ++g_kernel_launches;
  export_offsets_kernel<<<(n_tiles + 1 + 255) / 256, 256, 0, st>>>(tmp_counts, n_tiles, (uint32_t)n_keys, offsets);
  if (ids_out && n_keys) {
    ++g_kernel_launches;
    export_ids_kernel<<<(unsigned)((n_keys + 255) / 256), 256, 0, st>>>(keys, (uint32_t)n_keys, rank_bits, ids_sorted, ids_out);
  }
}

}  // namespace nbv
