// sort.cu -- S2 primitives: device exclusive scan and a stable LSD radix sort pass (hand-written, sm_100a).
//
// The (tile, depth) sort of B: north_star is done as an LSD radix sort whose least significant digits (the
// depth key) are sorted BEFORE the Gaussians are duplicated into tiles: N 32-bit depth keys with their
// Gaussian index (4 passes of 8 bits), then keys (tile << rank_bits | depth_rank) are emitted in depth-rank
// order and only the tile digit is sorted, by stable passes.  Stability makes the result identical to a full
// sort on (tile, z bits, index) -- the definition of the tile lists (R-5, R-7).
#include <cooperative_groups.h>

#include "kernels.h"

namespace nbv {

// ------------------------------------------------------------------------------------------------
// exclusive scan (uint32), any length < 2^32: reduce -> (recursive) scan of block sums -> downsweep
// ------------------------------------------------------------------------------------------------
constexpr int SCAN_T = 256;
constexpr int SCAN_I = 8;
constexpr int SCAN_TILE = SCAN_T * SCAN_I;

// exclusive prefix of v over the block; total = block sum.  sm must hold 32 words.
__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t* sm, uint32_t& total) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
  uint32_t x = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
    if (lane >= o) x += y;
  }
  if (lane == 31) sm[wid] = x;
  __syncthreads();
  if (wid == 0) {
    uint32_t w = lane < nw ? sm[lane] : 0u;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      uint32_t y = __shfl_up_sync(0xffffffffu, w, o);
      if (lane >= o) w += y;
    }
    sm[lane] = w;
  }
  __syncthreads();
  uint32_t woff = wid > 0 ? sm[wid - 1] : 0u;
  total = sm[nw - 1];
  __syncthreads();
  return woff + x - v;
}

__global__ void __launch_bounds__(SCAN_T) scan_reduce_kernel(const uint32_t* __restrict__ in, uint32_t n,
                                                              uint32_t* __restrict__ sums) {
  __shared__ uint32_t sm[32];
  const uint32_t base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_I;
  uint32_t s = 0;
#pragma unroll
  for (int i = 0; i < SCAN_I; ++i) {
    uint32_t idx = base + i;
    s += idx < n ? in[idx] : 0u;
  }
  uint32_t total;
  block_exclusive_scan(s, sm, total);
  if (threadIdx.x == 0) sums[blockIdx.x] = total;
}

// out[i] = offsets[block] + exclusive prefix within the block.  offsets == nullptr -> 0.
// If total_out != nullptr the last block also writes the grand total there (as uint32).
__global__ void __launch_bounds__(SCAN_T) scan_downsweep_kernel(const uint32_t* in, uint32_t* out,
                                                                 uint32_t n, const uint32_t* __restrict__ offsets,
                                                                 uint32_t* __restrict__ total_out) {
  __shared__ uint32_t sm[32];
  const uint32_t base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_I;
  uint32_t v[SCAN_I];
  uint32_t s = 0;
#pragma unroll
  for (int i = 0; i < SCAN_I; ++i) {
    uint32_t idx = base + i;
    v[i] = idx < n ? in[idx] : 0u;
    s += v[i];
  }
  uint32_t total;
  uint32_t ex = block_exclusive_scan(s, sm, total);
  uint32_t off = (offsets ? offsets[blockIdx.x] : 0u) + ex;
#pragma unroll
  for (int i = 0; i < SCAN_I; ++i) {
    uint32_t idx = base + i;
    if (idx < n) out[idx] = off;
    off += v[i];
  }
  if (total_out && blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) *total_out = (offsets ? offsets[blockIdx.x] : 0u) + total;
}

// Whole scan in ONE launch of ONE thread-block cluster (n up to 64k: the digit histograms of the depth sort and the
// multi-split count table), so that a radix pass is three dependent launches instead of five: the S1-S2 chain of a batch is
// latency bound.  Eight CTAs on eight SMs each stage an eighth of the input in shared memory
// (coalesced in, coalesced out), scan it, publish their total, and read the totals of the lower-ranked CTAs through
// distributed shared memory after one cluster barrier.
constexpr int SCAN1_T = 1024;
constexpr int SCAN1_CTAS = 8;
constexpr uint32_t SCAN1_PER_CTA = 8192;
constexpr uint32_t SCAN1_MAX = SCAN1_CTAS * SCAN1_PER_CTA;

__global__ void __cluster_dims__(SCAN1_CTAS, 1, 1) __launch_bounds__(SCAN1_T)
scan_cluster_kernel(const uint32_t* in, uint32_t* out, uint32_t n, uint32_t* __restrict__ total_out) {
  namespace cg = cooperative_groups;
  cg::cluster_group cluster = cg::this_cluster();
  __shared__ uint32_t sdata[SCAN1_PER_CTA];
  __shared__ uint32_t sm[32];
  __shared__ uint32_t cta_total;
  const uint32_t rank = cluster.block_rank();
  const uint32_t per = (n + SCAN1_CTAS - 1) / SCAN1_CTAS;
  const uint32_t g0 = min(rank * per, n), g1 = min(g0 + per, n), m = g1 - g0;
  for (uint32_t i = threadIdx.x; i < m; i += SCAN1_T) sdata[i] = in[g0 + i];
  __syncthreads();
  // thread t owns the contiguous chunk [t c, (t + 1) c), c odd: the chunk walks of a warp fall into distinct banks
  const uint32_t c = ((m + SCAN1_T - 1) / SCAN1_T) | 1u;
  const uint32_t i0 = min(threadIdx.x * c, m), i1 = min(i0 + c, m);
  uint32_t s = 0;
  for (uint32_t i = i0; i < i1; ++i) s += sdata[i];
  uint32_t total;
  uint32_t off = block_exclusive_scan(s, sm, total);
  for (uint32_t i = i0; i < i1; ++i) {
    const uint32_t v = sdata[i];
    sdata[i] = off;
    off += v;
  }
  if (threadIdx.x == 0) cta_total = total;
  cluster.sync();
  uint32_t base = 0;
  for (uint32_t r = 0; r < rank; ++r) base += *cluster.map_shared_rank(&cta_total, r);
  for (uint32_t i = threadIdx.x; i < m; i += SCAN1_T) out[g0 + i] = base + sdata[i];
  if (total_out && rank == SCAN1_CTAS - 1 && threadIdx.x == 0) *total_out = base + total;
  cluster.sync();                            // no CTA may exit while its shared memory can still be read
}

// the same scan for one table per view of a batch (grid.y = view), in place
__global__ void __cluster_dims__(SCAN1_CTAS, 1, 1) __launch_bounds__(SCAN1_T)
scan_cluster_batched_kernel(const __grid_constant__ PreBatch batch, int table, uint32_t n) {
  namespace cg = cooperative_groups;
  cg::cluster_group cluster = cg::this_cluster();
  __shared__ uint32_t sdata[SCAN1_PER_CTA];
  __shared__ uint32_t sm[32];
  __shared__ uint32_t cta_total;
  const PreView& pv = batch.v[blockIdx.y];
  uint32_t* data = table == SCAN_HIST ? pv.hist : pv.counts;
  uint32_t* total_out = table == SCAN_COUNTS ? &pv.counters->n_coarse : nullptr;
  const uint32_t rank = cluster.block_rank();
  const uint32_t per = (n + SCAN1_CTAS - 1) / SCAN1_CTAS;
  const uint32_t g0 = min(rank * per, n), g1 = min(g0 + per, n), m = g1 - g0;
  for (uint32_t i = threadIdx.x; i < m; i += SCAN1_T) sdata[i] = data[g0 + i];
  __syncthreads();
  const uint32_t c = ((m + SCAN1_T - 1) / SCAN1_T) | 1u;
  const uint32_t i0 = min(threadIdx.x * c, m), i1 = min(i0 + c, m);
  uint32_t s = 0;
  for (uint32_t i = i0; i < i1; ++i) s += sdata[i];
  uint32_t total;
  uint32_t off = block_exclusive_scan(s, sm, total);
  for (uint32_t i = i0; i < i1; ++i) {
    const uint32_t v = sdata[i];
    sdata[i] = off;
    off += v;
  }
  if (threadIdx.x == 0) cta_total = total;
  cluster.sync();
  uint32_t base = 0;
  for (uint32_t r = 0; r < rank; ++r) base += *cluster.map_shared_rank(&cta_total, r);
  for (uint32_t i = threadIdx.x; i < m; i += SCAN1_T) data[g0 + i] = base + sdata[i];
  if (total_out && rank == SCAN1_CTAS - 1 && threadIdx.x == 0) *total_out = base + total;
  cluster.sync();                            // no CTA may exit while its shared memory can still be read
}

size_t scan_temp_words(size_t n) {
  size_t words = 0;
  while (n > (size_t)SCAN_TILE) {
    n = (n + SCAN_TILE - 1) / SCAN_TILE;
    words += n;
  }
  return words + 1;
}

void exclusive_scan_u32(const uint32_t* in, uint32_t* out, size_t n, uint32_t* tmp, uint32_t* total_out, cudaStream_t st) {
  if (n == 0) {
    if (total_out) cudaMemsetAsync(total_out, 0, 4, st);
    return;
  }
  const uint32_t nb = (uint32_t)((n + SCAN_TILE - 1) / SCAN_TILE);
  if (nb > 1 && n <= SCAN1_MAX) {
    ++g_kernel_launches;
    scan_cluster_kernel<<<SCAN1_CTAS, SCAN1_T, 0, st>>>(in, out, (uint32_t)n, total_out);
    return;
  }
  if (nb == 1) {
    ++g_kernel_launches;
    scan_downsweep_kernel<<<1, SCAN_T, 0, st>>>(in, out, (uint32_t)n, nullptr, total_out);
    return;
  }
  uint32_t* sums = tmp;
  ++g_kernel_launches;
  scan_reduce_kernel<<<nb, SCAN_T, 0, st>>>(in, (uint32_t)n, sums);
  exclusive_scan_u32(sums, sums, nb, tmp + nb, nullptr, st);
  ++g_kernel_launches;
  scan_downsweep_kernel<<<nb, SCAN_T, 0, st>>>(in, out, (uint32_t)n, sums, total_out);
}

uint32_t scan_batched_max() { return SCAN1_MAX; }

void scan_batched(const PreBatch& batch, int table, size_t n, cudaStream_t st) {
  if (n == 0) return;
  if (n > SCAN1_MAX) {                       // long tables: the general multi-level scan, view by view (scratch follows the table)
    for (int v = 0; v < batch.n; ++v) {
      uint32_t* data = table == SCAN_HIST ? batch.v[v].hist : batch.v[v].counts;
      exclusive_scan_u32(data, data, n, data + n, table == SCAN_COUNTS ? &batch.v[v].counters->n_coarse : nullptr, st);
    }
    return;
  }
  ++g_kernel_launches;
  scan_cluster_batched_kernel<<<dim3(SCAN1_CTAS, (unsigned)batch.n), SCAN1_T, 0, st>>>(batch, table, (uint32_t)n);
}

// ------------------------------------------------------------------------------------------------
// one stable radix pass on `bits` (<= 8) bits at `shift`
// ------------------------------------------------------------------------------------------------
constexpr int RS_T = 256;
// keys per thread: 16 (4096 keys per block) for long inputs, 4 (1024 per block) for short ones -- a pass over 200,000
// keys is one partial wave of blocks either way, so its time is one block's critical path: shorter blocks, shorter pass
constexpr int RS_I_LONG = 16, RS_I_SHORT = 4;
constexpr size_t RS_SHORT_MAX = 256 * 1024;
__host__ __device__ constexpr int rs_tile(int rs_i) { return RS_T * rs_i; }
static int rs_i_for(size_t n) { return n <= RS_SHORT_MAX ? RS_I_SHORT : RS_I_LONG; }   // <= 256 blocks up to 2^20 keys: one cluster scan
constexpr int RS_W = RS_T / 32;        // 8 warps, 512 consecutive keys each

template <int RS_I>
__global__ void __launch_bounds__(RS_T) radix_hist_kernel(const __grid_constant__ PreBatch batch, int src, uint32_t n, int shift,
                                                           uint32_t mask, uint32_t nblocks) {
  constexpr int RS_TILE = RS_T * RS_I;
  __shared__ uint32_t h[256];
  const PreView& pv = batch.v[blockIdx.y];
  const uint32_t* __restrict__ keys = pv.zkey[src];
  uint32_t* __restrict__ hist = pv.hist;
  h[threadIdx.x] = 0;
  __syncthreads();
  const uint32_t base = blockIdx.x * RS_TILE;
#pragma unroll
  for (int i = 0; i < RS_I; ++i) {
    uint32_t idx = base + i * RS_T + threadIdx.x;
    if (idx < n) atomicAdd(&h[(keys[idx] >> shift) & mask], 1u);
  }
  __syncthreads();
  if (threadIdx.x <= mask) hist[(size_t)threadIdx.x * nblocks + blockIdx.x] = h[threadIdx.x];
}

template <int RS_I>
__global__ void __launch_bounds__(RS_T) radix_scatter_kernel(const __grid_constant__ PreBatch batch, int src, uint32_t n, int shift,
                                                              uint32_t mask, uint32_t nblocks) {
  constexpr int RS_TILE = RS_T * RS_I;
  constexpr bool HAS_VALS = true;
  const PreView& pv = batch.v[blockIdx.y];
  const uint32_t* __restrict__ keys_in = pv.zkey[src];
  uint32_t* __restrict__ keys_out = pv.zkey[src ^ 1];
  const uint32_t* __restrict__ vals_in = pv.ids[src];
  uint32_t* __restrict__ vals_out = pv.ids[src ^ 1];
  const uint32_t* __restrict__ hist_scanned = pv.hist;
  if (blockIdx.x * RS_TILE >= n) return;
  __shared__ uint32_t wh[RS_W][256];     // per-warp digit counts, then per-warp digit bases
  __shared__ uint32_t dstart[256];       // block-local start of each digit's run
  __shared__ uint32_t gofs[256];         // global position of local slot i with digit d = gofs[d] + i
  __shared__ uint32_t sm_scan[32];
  __shared__ uint32_t skeys[RS_TILE];
  __shared__ uint32_t svals[HAS_VALS ? RS_TILE : 1];

  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const uint32_t lt = (1u << lane) - 1u;
  for (int i = tid; i < RS_W * 256; i += RS_T) (&wh[0][0])[i] = 0;
  __syncthreads();

  const uint32_t base = blockIdx.x * RS_TILE + w * (RS_TILE / RS_W);
  uint32_t k[RS_I];
  uint32_t rk[RS_I];
  // all of the thread's keys first: the ranking loop below synchronises the warp in every iteration, and a load issued
  // inside it would cost one DRAM round trip per key (ncu at 1M keys: long scoreboard 22 of 40 stall cycles per issue)
  uint32_t v[RS_I];
#pragma unroll
  for (int r = 0; r < RS_I; ++r) {
    const uint32_t idx = base + r * 32 + lane;
    k[r] = idx < n ? keys_in[idx] : 0xffffffffu;
    v[r] = (HAS_VALS && idx < n) ? vals_in[idx] : 0u;
  }
  // this block's row of the scanned histogram (digit-major table: 256 separate sectors), needed only in phase 2
  const uint32_t hscan = (uint32_t)tid <= mask ? hist_scanned[(size_t)tid * nblocks + blockIdx.x] : 0u;
  // phase 1: rank every key among the keys of its warp with the same digit, in memory order
#pragma unroll
  for (int r = 0; r < RS_I; ++r) {
    const uint32_t idx = base + r * 32 + lane;
    const bool valid = idx < n;
    const uint32_t d = valid ? ((k[r] >> shift) & mask) : 0x100u;
    const uint32_t peers = __match_any_sync(0xffffffffu, d);
    const uint32_t pre = valid ? wh[w][d] : 0u;
    __syncwarp();
    rk[r] = pre + __popc(peers & lt);
    if (valid && lane == __ffs(peers) - 1) wh[w][d] = pre + __popc(peers);
    __syncwarp();
  }
  __syncthreads();
  // phase 2: per digit, prefix over warps; then prefix over digits
  uint32_t bt = 0;
  if ((uint32_t)tid <= mask) {
#pragma unroll
    for (int w2 = 0; w2 < RS_W; ++w2) {
      uint32_t t = wh[w2][tid];
      wh[w2][tid] = bt;
      bt += t;
    }
  }
  uint32_t total;
  uint32_t ds = block_exclusive_scan(bt, sm_scan, total);
  if ((uint32_t)tid <= mask) {
    dstart[tid] = ds;
    gofs[tid] = hscan - ds;
  }
  __syncthreads();
  // phase 3: stage in shared memory in sorted order
#pragma unroll
  for (int r = 0; r < RS_I; ++r) {
    const uint32_t idx = base + r * 32 + lane;
    if (idx < n) {
      const uint32_t d = (k[r] >> shift) & mask;
      const uint32_t lpos = dstart[d] + wh[w][d] + rk[r];
      skeys[lpos] = k[r];
      if (HAS_VALS) svals[lpos] = v[r];
    }
  }
  __syncthreads();
  // phase 4: coalesced runs to global
  for (uint32_t i = tid; i < total; i += RS_T) {
    const uint32_t key = skeys[i];
    const uint32_t pos = gofs[(key >> shift) & mask] + i;
    keys_out[pos] = key;
    if (HAS_VALS) vals_out[pos] = svals[i];
  }
}

uint32_t radix_blocks(size_t n) { const size_t t = (size_t)rs_tile(rs_i_for(n)); return (uint32_t)((n + t - 1) / t); }

size_t radix_temp_words(size_t n) { const size_t h = 256 * (size_t)radix_blocks(n); return h + scan_temp_words(h); }

void radix_pass_batched(const PreBatch& batch, int src, size_t n, int shift, cudaStream_t st) {
  if (n == 0) return;
  const uint32_t nb = radix_blocks(n);
  const bool shrt = rs_i_for(n) == RS_I_SHORT;
  const uint32_t mask = 255u;
  const dim3 grid(nb, (unsigned)batch.n);
  ++g_kernel_launches;
  if (shrt) radix_hist_kernel<RS_I_SHORT><<<grid, RS_T, 0, st>>>(batch, src, (uint32_t)n, shift, mask, nb);
  else radix_hist_kernel<RS_I_LONG><<<grid, RS_T, 0, st>>>(batch, src, (uint32_t)n, shift, mask, nb);
  scan_batched(batch, SCAN_HIST, 256 * (size_t)nb, st);
  ++g_kernel_launches;
  if (shrt) radix_scatter_kernel<RS_I_SHORT><<<grid, RS_T, 0, st>>>(batch, src, (uint32_t)n, shift, mask, nb);
  else radix_scatter_kernel<RS_I_LONG><<<grid, RS_T, 0, st>>>(batch, src, (uint32_t)n, shift, mask, nb);
}

}  // namespace nbv
