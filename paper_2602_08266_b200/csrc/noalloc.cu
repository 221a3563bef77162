// noalloc.cu -- nbv_exclusive_scan_noalloc: S2's exclusive scan (count table -> list offsets; R-5) for callers
// that may not allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// The library's own scan (sort.cu: exclusive_scan_u32) keeps the block sums of long inputs in a scratch buffer the context
// allocates with cudaMalloc.  This variant keeps them in a file-scope `static __device__` array instead: NA_MAX_BLOCKS words
// (32 KB) that every GPU which loads the library holds until the process exits.  Consequences, all stated in include/nbv.h:
//   - n is limited to NBV_SCAN_NOALLOC_MAX = NA_MAX_BLOCKS x NA_TILE elements; larger inputs are rejected;
//   - every call on a device shares the array, so calls that OVERLAP on that GPU (different streams, no ordering) race;
//   - the array keeps the last call's contents; nothing has to start at zero here, because a call writes entry b (kernel 1,
//     all of its nb blocks) before anything reads it (kernels 2 and 3 read entries < nb only);
//   - the call makes no cudaMalloc / cudaFree / allocating library call: three launches (one for n <= NA_TILE) and, for
//     n == 0, one cudaMemsetAsync of the total.
// In host code `g_scan_sums` is only the host-side stand-in of the symbol, not a device address: its address on the current
// device comes from cudaGetSymbolAddress (once per device, cached) and is what the kernels are given.
#include <cstdio>
#include <mutex>

#include "kernels.h"

namespace nbv {
namespace {

constexpr int NA_T = 256;                          // threads per block
constexpr int NA_I = 8;                            // consecutive elements per thread
constexpr int NA_TILE = NA_T * NA_I;               // 2,048 elements per block
constexpr int NA_MAX_BLOCKS = 8192;                // = 1,024 threads x NA_I of the single block that scans the block sums
constexpr int64_t NA_MAX_N = (int64_t)NA_MAX_BLOCKS * NA_TILE;
static_assert(NA_MAX_N == NBV_SCAN_NOALLOC_MAX, "include/nbv.h states the limit");

static __device__ __align__(256) uint32_t g_scan_sums[NA_MAX_BLOCKS];      // block sums, then their exclusive prefix

// exclusive prefix of v over the block (blockDim.x a multiple of 32, at most 1024); total = block sum.  sm: 32 words.
__device__ __forceinline__ uint32_t na_block_scan(uint32_t v, uint32_t* sm, uint32_t& total) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
  uint32_t x = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
    if (lane >= o) x += y;
  }
  if (lane == 31) sm[wid] = x;
  __syncthreads();
  if (wid == 0) {
    uint32_t w = lane < nw ? sm[lane] : 0u;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t y = __shfl_up_sync(0xffffffffu, w, o);
      if (lane >= o) w += y;
    }
    sm[lane] = w;
  }
  __syncthreads();
  const uint32_t before = wid > 0 ? sm[wid - 1] : 0u;
  total = sm[nw - 1];
  __syncthreads();
  return before + x - v;
}

// kernel 1: sums[b] = sum of the block's NA_TILE elements
__global__ void __launch_bounds__(NA_T) na_block_sums_kernel(const uint32_t* __restrict__ in, uint32_t n, uint32_t* __restrict__ sums) {
  __shared__ uint32_t sm[32];
  const uint32_t base = blockIdx.x * NA_TILE + threadIdx.x * NA_I;
  uint32_t s = 0;
#pragma unroll
  for (int i = 0; i < NA_I; ++i) s += base + i < n ? in[base + i] : 0u;
  uint32_t total;
  na_block_scan(s, sm, total);
  if (threadIdx.x == 0) sums[blockIdx.x] = total;
}

// kernel 2: one block of 1,024 threads turns the nb <= NA_MAX_BLOCKS block sums into their exclusive prefix, in place
__global__ void __launch_bounds__(1024) na_scan_sums_kernel(uint32_t* sums, uint32_t nb) {
  __shared__ uint32_t sm[32];
  const uint32_t base = threadIdx.x * NA_I;
  uint32_t v[NA_I], s = 0;
#pragma unroll
  for (int i = 0; i < NA_I; ++i) {
    v[i] = base + i < nb ? sums[base + i] : 0u;
    s += v[i];
  }
  uint32_t total;
  uint32_t off = na_block_scan(s, sm, total);
#pragma unroll
  for (int i = 0; i < NA_I; ++i) {
    if (base + i < nb) sums[base + i] = off;
    off += v[i];
  }
}

// kernel 3: out[i] = offsets[block] + exclusive prefix inside the block (offsets == nullptr: one block, no offsets).  A thread
// reads its NA_I inputs before it writes its NA_I outputs and no other thread touches them: out may be in.
__global__ void __launch_bounds__(NA_T) na_apply_kernel(const uint32_t* in, uint32_t* out, uint32_t n, const uint32_t* offsets,
                                                        uint32_t* __restrict__ total_out) {
  __shared__ uint32_t sm[32];
  const uint32_t base = blockIdx.x * NA_TILE + threadIdx.x * NA_I;
  uint32_t v[NA_I], s = 0;
#pragma unroll
  for (int i = 0; i < NA_I; ++i) {
    v[i] = base + i < n ? in[base + i] : 0u;
    s += v[i];
  }
  uint32_t total;
  const uint32_t block_off = offsets ? offsets[blockIdx.x] : 0u;
  uint32_t off = block_off + na_block_scan(s, sm, total);
#pragma unroll
  for (int i = 0; i < NA_I; ++i) {
    if (base + i < n) out[base + i] = off;
    off += v[i];
  }
  if (total_out && blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) *total_out = block_off + total;
}

// ---- set-up: the array's address on the current device, resolved once per device -----------------------------------------
constexpr int NA_MAX_DEVICES = 64;
std::mutex g_na_mutex;
uint32_t* g_na_ptr[NA_MAX_DEVICES] = {};
thread_local char g_na_err[256] = "";

int na_fail(int code, const char* fmt, long long a = 0, long long b = 0) {
  std::snprintf(g_na_err, sizeof(g_na_err), fmt, a, b);
  return code;
}

// the current device's copy of g_scan_sums (nullptr + error text on failure)
uint32_t* na_scratch() {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess || dev < 0 || dev >= NA_MAX_DEVICES) {
    cudaGetLastError();
    na_fail(NBV_ERR_CUDA, "nbv_exclusive_scan_noalloc: no current CUDA device (cudaGetDevice: %lld, device %lld)", (long long)e, dev);
    return nullptr;
  }
  std::lock_guard<std::mutex> lock(g_na_mutex);
  if (!g_na_ptr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_scan_sums);           // with device `dev` current: its instance of the array
    if (e != cudaSuccess || !p) {
      cudaGetLastError();
      na_fail(NBV_ERR_CUDA, "nbv_exclusive_scan_noalloc: cudaGetSymbolAddress failed (error %lld) on device %lld", (long long)e, dev);
      return nullptr;
    }
    g_na_ptr[dev] = static_cast<uint32_t*>(p);
  }
  return g_na_ptr[dev];
}

}  // namespace
}  // namespace nbv

extern "C" const char* nbv_noalloc_last_error(void) { return nbv::g_na_err; }

extern "C" int nbv_exclusive_scan_noalloc(const uint32_t* d_in, uint32_t* d_out, int64_t n, uint32_t* d_total, void* stream) {
  using namespace nbv;
  cudaStream_t st = (cudaStream_t)stream;
  if (n < 0 || (n > 0 && (!d_in || !d_out)))
    return na_fail(NBV_ERR_INVALID_ARG, "nbv_exclusive_scan_noalloc: n = %lld must be >= 0 and d_in, d_out non-null", (long long)n);
  if (n > NA_MAX_N)
    return na_fail(NBV_ERR_CAPACITY,
                   "nbv_exclusive_scan_noalloc: n = %lld exceeds NBV_SCAN_NOALLOC_MAX = %lld (the static scratch holds one block sum per "
                   "2048 elements); use the context calls, which allocate",
                   (long long)n, (long long)NA_MAX_N);
  uint32_t* sums = na_scratch();                           // also on the n == 0 path: set-up happens on the first call of any size
  if (!sums) return NBV_ERR_CUDA;
  if (n == 0) {
    if (d_total && cudaMemsetAsync(d_total, 0, 4, st) != cudaSuccess) {
      cudaGetLastError();
      return na_fail(NBV_ERR_CUDA, "nbv_exclusive_scan_noalloc: cudaMemsetAsync of the total failed");
    }
    return NBV_OK;
  }
  const uint32_t nb = (uint32_t)((n + NA_TILE - 1) / NA_TILE);
  if (nb == 1) {
    ++g_kernel_launches;
    na_apply_kernel<<<1, NA_T, 0, st>>>(d_in, d_out, (uint32_t)n, nullptr, d_total);
  } else {
    g_kernel_launches += 3;
    na_block_sums_kernel<<<nb, NA_T, 0, st>>>(d_in, (uint32_t)n, sums);
    na_scan_sums_kernel<<<1, 1024, 0, st>>>(sums, nb);
    na_apply_kernel<<<nb, NA_T, 0, st>>>(d_in, d_out, (uint32_t)n, sums, d_total);
  }
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return na_fail(NBV_ERR_CUDA, "nbv_exclusive_scan_noalloc: kernel launch failed (CUDA error %lld)", (long long)e);
  return NBV_OK;
}
