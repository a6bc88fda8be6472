// common.cuh -- shared host/device helpers of libbits_b200 (sm_100a only).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>

#include "../../include/bits.h"

namespace bits {

constexpr int kWarp = 32;
constexpr uint32_t kFullMask = 0xffffffffu;

// Number of kernel launches made by the library (bits_launch_count()).
extern std::atomic<unsigned long long> g_launches;

#define BITS_CUDA_TRY(expr)                              \
  do {                                                   \
    cudaError_t e__ = (expr);                            \
    if (e__ != cudaSuccess) { (void)cudaGetLastError(); return BITS_ERR_CUDA; } \
  } while (0)

#define BITS_LAUNCH_CHECK()                              \
  do {                                                   \
    ++::bits::g_launches;                                \
    cudaError_t e__ = cudaGetLastError();                \
    if (e__ != cudaSuccess) return BITS_ERR_CUDA;        \
  } while (0)

#define BITS_TRY(expr)                                   \
  do {                                                   \
    int s__ = (expr);                                    \
    if (s__ != BITS_OK) return s__;                      \
  } while (0)

__host__ __device__ inline uint64_t align_up(uint64_t x, uint64_t a) { return (x + a - 1) / a * a; }
__host__ __device__ inline uint64_t ceil_div(uint64_t x, uint64_t a) { return (x + a - 1) / a; }

// Programmatic dependent launch: a kernel launched with the programmatic-stream-serialization attribute may be
// scheduled while its predecessor on the stream drains; it must not touch what the predecessor wrote (or overwrite
// what it reads) before grid_dependency_wait().  A no-op in a plain launch.
__device__ __forceinline__ void grid_dependency_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void grid_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// 64-bit warp sum (all 32 lanes participate; every lane gets the total).
__device__ __forceinline__ uint64_t warp_sum_u64(uint64_t v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFullMask, v, o);
  return v;
}

// Block sum of per-thread uint64 partials, then ONE atomicAdd per block (the
// O(|A|) "combining the results" step).  `red` is shared scratch of >= blockDim.x/32 uint64.
__device__ __forceinline__ void block_sum_atomic(uint64_t v, uint64_t* red, unsigned long long* out) {
  v = warp_sum_u64(v);
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  if (lane == 0) red[w] = v;
  __syncthreads();
  if (w == 0) {
    const int nw = (blockDim.x + 31) >> 5;
    uint64_t t = lane < nw ? red[lane] : 0;
    t = warp_sum_u64(t);
    if (lane == 0 && t != 0) atomicAdd(out, (unsigned long long)t);
  }
}

}  // namespace bits
