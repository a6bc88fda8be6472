// enumerate.cuh -- the enumeration sub-problem (sub-problem 4): emit every pair
// <a, b> with a.start <= b.end and a.end >= b.start.
//
// "The size of I(B, a_i) also serves as the termination condition for enumerating
// intersections that was missing in the naive binary search solution."  So: per-interval counts
// first (ICOUNT, Algorithm 1), an exclusive scan gives every a_i its slice of the output, and a_i
// then walks B in start order downwards from its `first` (= #{b.start <= a.end}) position,
// emitting every b whose end reaches a.start, until c(a_i) pairs are out.
//
// The walk needs B's ends and original indices IN START ORDER.  The sorts of this library are
// keys-only, so that order is rebuilt by ranking: interval j goes to position
//   #{keys of B_S < b_j.start} + (its arrival number among the intervals with the same start),
// which is a valid position of b_j.start in B_S whatever the arrival order is.
#pragma once
#include "common.cuh"
#include "search.cuh"

namespace bits {
namespace enu {

// #{keys < q}
__device__ __forceinline__ uint32_t rank_lt(const SortedSet& s, uint32_t q) { return q == 0 ? 0u : rank_le(s, q - 1u); }

// ends and original indices of B in start order.  tie[] is zero on entry (one counter per position).
__global__ void __launch_bounds__(256) start_order_kernel(const uint32_t* __restrict__ b_start, const uint32_t* __restrict__ b_end,
                                                          uint32_t n_b, SortedSet bs, uint32_t* tie,
                                                          uint32_t* __restrict__ end_by_start, uint32_t* __restrict__ idx_by_start) {
  grid_dependency_wait();
  for (uint64_t j = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; j < n_b; j += (uint64_t)gridDim.x * blockDim.x) {
    const uint32_t p = rank_lt(bs, b_start[j]);
    const uint32_t pos = p + atomicAdd(&tie[p], 1u);
    end_by_start[pos] = b_end[j];
    idx_by_start[pos] = (uint32_t)j;
  }
}

// Exclusive scan of uint32 counts into uint64 offsets, three small kernels (blocks of kScanTile).
constexpr int kScanThreads = 256, kScanPer = 16, kScanTile = kScanThreads * kScanPer;

__global__ void __launch_bounds__(kScanThreads) scan_tile_sums_kernel(const uint32_t* __restrict__ counts, uint32_t n,
                                                                      unsigned long long* __restrict__ tile_sums) {
  __shared__ uint64_t s_red[kScanThreads / 32];
  grid_dependency_wait();
  const uint64_t base = (uint64_t)blockIdx.x * kScanTile;
  uint64_t sum = 0;
  for (int j = 0; j < kScanPer; ++j) {
    const uint64_t i = base + threadIdx.x + (uint64_t)j * kScanThreads;
    if (i < n) sum += counts[i];
  }
  sum = warp_sum_u64(sum);
  if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = sum;
  __syncthreads();
  if (threadIdx.x == 0) {
    uint64_t t = 0;
    for (int w = 0; w < kScanThreads / 32; ++w) t += s_red[w];
    tile_sums[blockIdx.x] = t;
  }
}

// one block: tile_sums -> exclusive prefixes in place; the grand total goes to *total
__global__ void __launch_bounds__(1024) scan_tile_prefix_kernel(unsigned long long* tile_sums, uint32_t n_tiles,
                                                                unsigned long long* total) {
  __shared__ uint64_t s_w[32];
  __shared__ uint64_t s_carry;
  grid_dependency_wait();
  if (threadIdx.x == 0) s_carry = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  for (uint32_t t0 = 0; t0 < n_tiles; t0 += 1024) {
    const uint32_t i = t0 + threadIdx.x;
    const uint64_t v = i < n_tiles ? tile_sums[i] : 0ull;
    uint64_t incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const uint64_t t = __shfl_up_sync(kFullMask, incl, o); if (lane >= o) incl += t; }
    if (lane == 31) s_w[w] = incl;
    __syncthreads();
    uint64_t before = 0;
    for (int k = 0; k < w; ++k) before += s_w[k];
    const uint64_t carry = s_carry;
    if (i < n_tiles) tile_sums[i] = carry + before + incl - v;
    __syncthreads();
    if (threadIdx.x == 1023) s_carry = carry + before + incl;
    __syncthreads();
  }
  if (threadIdx.x == 0 && total) *total = s_carry;
}

// offsets[i] = tile prefix + exclusive prefix inside the tile (one thread per kScanPer consecutive counts)
__global__ void __launch_bounds__(kScanThreads) scan_apply_kernel(const uint32_t* __restrict__ counts, uint32_t n,
                                                                  const unsigned long long* __restrict__ tile_prefix,
                                                                  unsigned long long* __restrict__ offsets) {
  __shared__ uint64_t s_w[kScanThreads / 32];
  grid_dependency_wait();
  const uint64_t i0 = (uint64_t)blockIdx.x * kScanTile + (uint64_t)threadIdx.x * kScanPer;
  uint32_t c[kScanPer];
  uint64_t sum = 0;
#pragma unroll
  for (int j = 0; j < kScanPer; ++j) { c[j] = i0 + j < n ? counts[i0 + j] : 0u; sum += c[j]; }
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  uint64_t incl = sum;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const uint64_t t = __shfl_up_sync(kFullMask, incl, o); if (lane >= o) incl += t; }
  if (lane == 31) s_w[w] = incl;
  __syncthreads();
  uint64_t run = tile_prefix[blockIdx.x] + incl - sum;
  for (int k = 0; k < w; ++k) run += s_w[k];
#pragma unroll
  for (int j = 0; j < kScanPer; ++j) {
    if (i0 + j < n) offsets[i0 + j] = run;
    run += c[j];
  }
}

// Largest end of every run of 32 / 1,024 / 32,768 consecutive positions of end_by_start (three levels of
// fan-out 32).  They bound the walk below: a run whose largest end lies before a.start holds no
// intersection and is skipped whole.  Without them ONE long interval with a small start (a
// chromosome-wide feature) would make every query that meets it scan all of B below its `first` --
// the linear scan PAPER.md:63-67 warns about.  max3 is zero on entry.  1,024 threads per block.
constexpr int kSkip1 = 5, kSkip2 = 10, kSkip3 = 15;
__global__ void __launch_bounds__(1024) end_maxima_kernel(const uint32_t* __restrict__ end_by_start, uint32_t n_b,
                                                          uint32_t* __restrict__ max1, uint32_t* __restrict__ max2, uint32_t* max3) {
  __shared__ uint32_t s_m[32];
  grid_dependency_wait();
  const uint64_t i = (uint64_t)blockIdx.x * 1024 + threadIdx.x;
  uint32_t m = i < n_b ? end_by_start[i] : 0u;
  m = __reduce_max_sync(kFullMask, m);
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  if (lane == 0) { s_m[w] = m; if (i < n_b) max1[i >> kSkip1] = m; }
  __syncthreads();
  if (w == 0) {
    m = __reduce_max_sync(kFullMask, s_m[lane]);
    if (lane == 0) { max2[blockIdx.x] = m; atomicMax(&max3[blockIdx.x >> (kSkip3 - kSkip2)], m); }
  }
}

// One query per thread: walk B in start order downwards from `first`, emit until c(a) pairs are out; runs of 32,
// 1,024 and 32,768 positions none of whose ends reaches a.start are stepped over through the maxima above, so
// the walk costs O(32 * 3 + n_b / 32,768) steps per emitted pair at worst instead of O(n_b).
__global__ void __launch_bounds__(256) emit_pairs_kernel(const uint32_t* __restrict__ a_start, const uint32_t* __restrict__ a_end,
                                                         uint32_t n_a, SortedSet bs, const uint32_t* __restrict__ counts,
                                                         const unsigned long long* __restrict__ offsets,
                                                         const uint32_t* __restrict__ end_by_start,
                                                         const uint32_t* __restrict__ idx_by_start,
                                                         const uint32_t* __restrict__ max1, const uint32_t* __restrict__ max2,
                                                         const uint32_t* __restrict__ max3,
                                                         uint32_t* __restrict__ pair_a, uint32_t* __restrict__ pair_b,
                                                         unsigned long long capacity) {
  grid_dependency_wait();
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_a; i += (uint64_t)gridDim.x * blockDim.x) {
    uint32_t left = counts[i];
    if (left == 0) continue;
    const uint32_t s = a_start[i];
    unsigned long long out = offsets[i];
    uint32_t p = rank_le(bs, a_end[i]);            // = first: every b below it starts at or before a.end
    while (left && p) {
      if ((p & 31u) == 0) {                        // at a run boundary: may the run(s) just below be skipped?
        if ((p & 1023u) == 0) {
          if ((p & 32767u) == 0 && max3[(p >> kSkip3) - 1u] < s) { p -= 32768u; continue; }
          if (max2[(p >> kSkip2) - 1u] < s) { p -= 1024u; continue; }
        }
        if (max1[(p >> kSkip1) - 1u] < s) { p -= 32u; continue; }
      }
      --p;
      if (end_by_start[p] >= s) {                  // ... and this one also ends at or after a.start: <a, b> is in I(A, B)
        if (out < capacity) { pair_a[out] = (uint32_t)i; pair_b[out] = idx_by_start[p]; }
        ++out; --left;
      }
    }
  }
}

}  // namespace enu
}  // namespace bits
