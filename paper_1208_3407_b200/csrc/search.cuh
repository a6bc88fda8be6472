// search.cuh -- the "search" and "reduce" steps.
//
// PAPER.md:93-99 (Algorithm 1 ICOUNT): first = BSEARCH(B_S, a.end), last = BSEARCH(B_E, a.start),
// c = first - last, with the ranks fixed by the set definitions L and R (PAPER.md:83-89,
// :103-107; reading R1):  first = #{b.start <= a.end}, last = #{b.end < a.start}.
// Both are "count of keys <= x": last = (a.start == 0) ? 0 : #{b.end <= a.start - 1}.
// PAPER.md:127-131 (Sec. 2.3): one independent ICOUNT per thread, no communication -- here
// four queries (eight rank look-ups) per thread for memory-level parallelism.
//
// Search structure (not in the paper): a bucket index over each sorted array,
//   idx[h] = #{keys < h << shift},  h = 0 .. 2^(32-shift),
// so a look-up is one index read plus one or two 32-byte sectors of keys, instead of ~log2|B|
// dependent probes.  Sorted arrays are padded with 16 keys of 0xffffffff.
#pragma once
#include "common.cuh"
#include "philox_place.cuh"

namespace bits {

constexpr int kPad = 16;   // sentinel keys after the last real key of a sorted array

struct SortedSet {
  const uint32_t* keys;   // ascending, 32-byte aligned, padded with kPad x 0xffffffff
  const uint32_t* idx;    // uint32[(1 << (32 - shift)) + 1]
  uint32_t n;
  uint32_t shift;         // 1..31
};

inline uint32_t index_shift_for(uint64_t n) {
  // about one bucket per four keys, between 2 and 2^24 buckets; per eight keys once keys + index
  // outgrow the L2 (measured on config 4: 303 -> 283 us; on config 3, which stays L2-resident, the
  // finer index is the faster one: 47.6 against 52.8 us)
  const uint64_t per = n > (4ull << 20) ? 8 : 4;
  uint32_t bits = 1;
  while (bits < 24 && (1ull << bits) < n / per) ++bits;
  return 32 - bits;
}
inline uint64_t index_entries(uint32_t shift) { return (1ull << (32 - shift)) + 1; }

__device__ __forceinline__ uint32_t count_le8(const uint4& a, const uint4& b, uint32_t q) {
  return (a.x <= q) + (a.y <= q) + (a.z <= q) + (a.w <= q) + (b.x <= q) + (b.y <= q) + (b.z <= q) + (b.w <= q);
}

// #{keys <= q}
__device__ __forceinline__ uint32_t rank_le(const SortedSet& s, uint32_t q) {
  const uint32_t h = q >> s.shift;
  const uint32_t pos = __ldg(s.idx + h);
  uint32_t base = pos & ~7u;      // every key before `pos` is < h << shift <= q
  const uint4* p = reinterpret_cast<const uint4*>(s.keys + base);
  uint32_t c = count_le8(__ldg(p), __ldg(p + 1), q);
  if (c == 8) {
    base += 8;
    c = count_le8(__ldg(p + 2), __ldg(p + 3), q);
    if (c == 8) {                 // long bucket: finish with a binary search inside it
      uint32_t lo = base + 8, hi = __ldg(s.idx + h + 1);
      while (lo < hi) {
        const uint32_t mid = lo + ((hi - lo) >> 1);
        if (__ldg(s.keys + mid) <= q) lo = mid + 1; else hi = mid;
      }
      return min(lo, s.n);
    }
  }
  return min(base + c, s.n);
}

// c(a) = #{b.start <= a.end} - #{b.end < a.start}
__device__ __forceinline__ uint32_t icount(const SortedSet& bs, const SortedSet& be, uint32_t a_start, uint32_t a_end) {
  const uint32_t first = rank_le(bs, a_end);
  const uint32_t last = a_start == 0 ? 0u : rank_le(be, a_start - 1u);
  return first - last;
}

// ---------------------------------------------------------------------------------------------
// Index build.  One thread per position i in [0, n]: fills idx[(key[i-1] >> s) + 1 .. key[i] >> s]
// with i (key[-1] = "-1", key[n] = "2^32").  Long gaps are filled by the whole warp.  Also writes
// the kPad sentinels.  grid.y = array (0: starts, 1: ends).
struct IndexArgs {
  uint32_t* keys[2];      // sorted; sentinels are written at keys[n .. n+kPad)
  uint32_t* idx[2];
  uint32_t n;
  uint32_t shift;
  uint64_t total;           // threads' worth of work: four positions each, a multiple of the block size
  const uint32_t* run_if;   // null: always; else dev uint32[2]: run only if one of them is non-zero (fallback behind binned_count.cuh)
};

__global__ void __launch_bounds__(256) build_index_kernel(IndexArgs a) {
  uint32_t* __restrict__ keys = blockIdx.y ? a.keys[1] : a.keys[0];
  uint32_t* __restrict__ idx = blockIdx.y ? a.idx[1] : a.idx[0];
  const uint32_t n = a.n, s = a.shift;
  const uint32_t H = 1u << (32 - s);
  grid_dependency_wait();
  if (a.run_if && (a.run_if[0] | a.run_if[1]) == 0u) return;
  const uint64_t gid0 = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
  const uint32_t lane = threadIdx.x & 31;
  {
    // idx[(key[n-1] >> s) + 1 .. H] = n: the entries above the largest key (for a genome that ends well
    // below 2^32 that is a long run) are filled by the whole grid, not by one thread
    const uint64_t tail_lo = n ? (uint64_t)(keys[n - 1] >> s) + 1u : 0u;
    for (uint64_t h = tail_lo + gid0; h <= H; h += stride) idx[h] = n;
  }
  // four consecutive positions per thread (one 16-byte load; the arrays are 32-byte aligned and padded);
  // a.total is a multiple of the block size, so warps are never partly out of range
  for (uint64_t gid = gid0; gid < a.total; gid += stride) {
    if (gid < kPad) keys[(uint64_t)n + gid] = 0xffffffffu;
    const uint64_t i0 = gid << 2;
    uint32_t k[4] = {0, 0, 0, 0};
    uint32_t prev = 0;
    if (i0 < n) {
      if (i0 + 3 < n) {
        const uint4 v = *reinterpret_cast<const uint4*>(keys + i0);
        k[0] = v.x; k[1] = v.y; k[2] = v.z; k[3] = v.w;
      } else {
#pragma unroll
        for (int j = 0; j < 4; ++j) k[j] = i0 + j < n ? keys[i0 + j] : 0u;
      }
      if (i0) prev = keys[i0 - 1];
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const uint32_t i = (uint32_t)i0 + j;
      uint32_t lo = 1, hi = 0;   // fill idx[lo..hi] = i  (empty by default)
      if (i0 + j < n) {
        lo = (i == 0) ? 0u : (prev >> s) + 1u;
        hi = k[j] >> s;
      }
      prev = k[j];
      const bool some = lo <= hi;
      const uint32_t len = some ? hi - lo + 1u : 0u;
      if (some && len <= 4)
        for (uint32_t h = lo; h <= hi; ++h) idx[h] = i;
      uint32_t big = __ballot_sync(kFullMask, len > 4);
      while (big) {
        const int src = __ffs(big) - 1;
        big &= big - 1;
        const uint32_t l = __shfl_sync(kFullMask, lo, src), hh = __shfl_sync(kFullMask, hi, src);
        const uint32_t v = __shfl_sync(kFullMask, i, src);
        for (uint64_t h = (uint64_t)l + lane; h <= hh; h += 32) idx[h] = v;
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// Search designs of the count kernel (bits_set_option "search_variant"; DESIGN.md section 5 has the numbers):
//   kSearchIndex   bucket index over the sorted array: one index word + two 32-byte sectors per look-up [default]
//   kSearchPlain   the paper's design: a binary search over the whole sorted
//                  array, nothing staged, ~log2|B| dependent probes (fixed trip count, no divergence)
//   kSearchStaged  the top 11 levels staged in shared memory (2,048 evenly spaced keys per array, 16 KB),
//                  then a binary search inside one 1/2048th of the array
enum { kSearchIndex = 0, kSearchPlain = 1, kSearchStaged = 2 };
constexpr int kStagedLevels = 11, kStaged = 1 << kStagedLevels;

// #{keys <= q} by a fixed-trip binary search over keys[lo .. lo + len)
__device__ __forceinline__ uint32_t rank_le_range(const uint32_t* __restrict__ keys, uint32_t lo, uint32_t len, uint32_t q) {
  while (len > 0) {
    const uint32_t half = len >> 1;
    const bool right = __ldg(keys + lo + half) <= q;
    lo = right ? lo + half + 1 : lo;
    len = right ? len - half - 1 : half;
  }
  return lo;
}

// block j of the staged search = keys[(j * n) >> 11 .. ((j + 1) * n) >> 11); s_top[j] = its last key
__device__ __forceinline__ uint32_t staged_bound(uint32_t j, uint32_t n) { return (uint32_t)(((uint64_t)j * n) >> kStagedLevels); }
__device__ __forceinline__ void stage_top_levels(const SortedSet& s, uint32_t* s_top) {
  for (uint32_t j = threadIdx.x; j < (uint32_t)kStaged; j += blockDim.x) {
    const uint32_t e = staged_bound(j + 1, s.n);
    s_top[j] = e ? __ldg(s.keys + e - 1) : 0u;       // (an empty block repeats a smaller key or 0: harmless)
  }
}
__device__ __forceinline__ uint32_t rank_le_staged(const SortedSet& s, const uint32_t* s_top, uint32_t q) {
  uint32_t j = 0;                                   // #{blocks whose last key <= q}
#pragma unroll
  for (uint32_t step = kStaged >> 1; step > 0; step >>= 1) j += (s_top[j + step - 1] <= q) ? step : 0u;
  j += (j < (uint32_t)kStaged && s_top[j] <= q) ? 1u : 0u;
  if (j >= (uint32_t)kStaged) return s.n;
  const uint32_t lo = staged_bound(j, s.n);
  return rank_le_range(s.keys, lo, staged_bound(j + 1, s.n) - lo, q);
}

// Count kernel: queries in input order, four per thread.  Writes per-interval counts if
// counts != nullptr; adds the block's sum to *total if total != nullptr.
template <bool kVec, int kSearch>
__global__ void __launch_bounds__(256) count_kernel(const uint32_t* __restrict__ a_start,
                                                    const uint32_t* __restrict__ a_end, uint32_t n_a,
                                                    SortedSet bs, SortedSet be,
                                                    uint32_t* __restrict__ counts, unsigned long long* total,
                                                    const uint32_t* run_if) {
  __shared__ uint64_t s_red[8];
  __shared__ uint32_t s_top[kSearch == kSearchStaged ? 2 * kStaged : 1];
  grid_dependency_wait();
  if (run_if && (run_if[0] | run_if[1]) == 0u) return;   // (fallback behind binned_count.cuh: runs only if the MSD sort fell back)
  if (kSearch == kSearchStaged) {
    stage_top_levels(bs, s_top);
    stage_top_levels(be, s_top + kStaged);
    __syncthreads();
  }
  uint64_t sum = 0;
  const uint64_t n4 = ((uint64_t)n_a + 3) >> 2;
  for (uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; t < n4; t += (uint64_t)gridDim.x * blockDim.x) {
    const uint64_t i0 = t << 2;
    uint32_t qs[4], qe[4], c[4];
    const bool full = i0 + 3 < n_a;
    if (kVec && full) {
      const uint4 s4 = __ldcs(reinterpret_cast<const uint4*>(a_start) + t);
      const uint4 e4 = __ldcs(reinterpret_cast<const uint4*>(a_end) + t);
      qs[0] = s4.x; qs[1] = s4.y; qs[2] = s4.z; qs[3] = s4.w;
      qe[0] = e4.x; qe[1] = e4.y; qe[2] = e4.z; qe[3] = e4.w;
    } else {
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const bool ok = i0 + j < n_a;
        qs[j] = ok ? a_start[i0 + j] : 0u;
        qe[j] = ok ? a_end[i0 + j] : 0u;
      }
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      if (kSearch == kSearchIndex) {
        c[j] = icount(bs, be, qs[j], qe[j]);
      } else if (kSearch == kSearchPlain) {
        c[j] = rank_le_range(bs.keys, 0, bs.n, qe[j]) - (qs[j] == 0 ? 0u : rank_le_range(be.keys, 0, be.n, qs[j] - 1u));
      } else {
        c[j] = rank_le_staged(bs, s_top, qe[j]) - (qs[j] == 0 ? 0u : rank_le_staged(be, s_top + kStaged, qs[j] - 1u));
      }
    }
    if (!full) {
#pragma unroll
      for (int j = 0; j < 4; ++j) if (i0 + j >= n_a) c[j] = 0;
    }
    if (counts) {
      if (kVec && full) {
        __stcs(reinterpret_cast<uint4*>(counts) + t, make_uint4(c[0], c[1], c[2], c[3]));
      } else {
#pragma unroll
        for (int j = 0; j < 4; ++j) if (i0 + j < n_a) counts[i0 + j] = c[j];
      }
    }
    sum += (uint64_t)c[0] + c[1] + c[2] + c[3];
  }
  if (total) block_sum_atomic(sum, s_red, total);
}

// ---------------------------------------------------------------------------------------------
// Decision problem (PAPER.md:47, sub-problem 1; :91 "with the size of I(B, a_i) we can directly answer
// the decision problem"): *any = 1 iff some a in A has c(a) > 0.  Same look-ups as the count kernel;
// a block stops as soon as anybody has found an intersection.  *any is zero on entry.
__global__ void __launch_bounds__(256) decide_kernel(const uint32_t* __restrict__ a_start, const uint32_t* __restrict__ a_end,
                                                     uint32_t n_a, SortedSet bs, SortedSet be, uint32_t* any) {
  // (whole warps iterate together; one lane reports for the warp, and only if nobody has yet: a store
  // from every thread that finds an intersection would serialise on the one word)
  grid_dependency_wait();
  const uint64_t n_pad = ((uint64_t)n_a + 31) & ~31ull;
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_pad; i += (uint64_t)gridDim.x * blockDim.x) {
    if (*reinterpret_cast<volatile uint32_t*>(any)) return;
    const bool hit = i < n_a && icount(bs, be, a_start[i], a_end[i]) != 0;
    if (__any_sync(kFullMask, hit)) {
      if ((threadIdx.x & 31) == 0) *any = 1u;
      return;
    }
  }
}

// ---------------------------------------------------------------------------------------------
// Plain rank look-ups for SORTED queries (the per-round search when B is re-placed: A's ends and
// A's starts are sorted once per call, so neighbouring threads walk neighbouring keys and the
// probes coalesce).  sum_first = sum_q #{keys <= q};  sum_last = sum_q #{keys < q}.
// The round total is sum_first(B_S; A ends) - sum_last(B_E; A starts): integer sums commute, so
// this equals sum_a (first - last) bit for bit.
template <bool kStrict>
__device__ __forceinline__ uint32_t rank_plain(const uint32_t* __restrict__ keys, uint32_t n, uint32_t q) {
  uint32_t lo = 0, len = n;
  while (len > 0) {
    const uint32_t half = len >> 1;
    const uint32_t k = __ldg(keys + lo + half);
    const bool right = kStrict ? (k < q) : (k <= q);
    lo = right ? lo + half + 1 : lo;
    len = right ? len - half - 1 : half;
  }
  return lo;
}

__global__ void __launch_bounds__(256) sorted_query_total_kernel(const uint32_t* __restrict__ q_end_sorted,
                                                                 const uint32_t* __restrict__ q_start_sorted, uint32_t n_q,
                                                                 const uint32_t* __restrict__ b_s, const uint32_t* __restrict__ b_e,
                                                                 uint32_t n_b, unsigned long long* total) {
  __shared__ uint64_t s_red[8];
  // two's-complement accumulation: the final sum is exact modulo 2^64 and non-negative
  uint64_t sum = 0;
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_q; i += (uint64_t)gridDim.x * blockDim.x) {
    const uint32_t first = rank_plain<false>(b_s, n_b, __ldg(q_end_sorted + i));
    const uint32_t last = rank_plain<true>(b_e, n_b, __ldg(q_start_sorted + i));
    sum += (uint64_t)first - (uint64_t)last;
  }
  block_sum_atomic(sum, s_red, total);
}

// ---------------------------------------------------------------------------------------------
// Fused Monte Carlo kernel for re-placed QUERIES (BITS_PERMUTE_A): place -> search -> reduce with
// no intermediate arrays.  grid = (tiles of 1024 queries, rounds in this launch).
struct McAArgs {
  const uint32_t* spans;     // dev uint32[n_a], padded to a multiple of 4 with zeros
  uint32_t n_a;
  uint32_t tag;              // Philox stream of the re-placed set (0: A, 1: B searched the other way round)
  uint32_t round0;           // first round of this launch
  PhiloxKeys key;
  ChromTable chrom;
  SortedSet bs, be;
  unsigned long long* round_counts;   // indexed by out0 + round of the launch
  uint32_t out0;
  uint32_t rpb;              // rounds per block: gridDim.y = ceil(n_launch / rpb)
  uint32_t n_launch;         // rounds of this launch
};

__global__ void __launch_bounds__(256) mc_permute_a_rounds_kernel(McAArgs a) {
  __shared__ uint32_t s_off[kMaxChromSmem];
  __shared__ __align__(16) uint16_t s_lut[kLutSize];
  const ChromView off = stage_chrom_table(a.chrom, s_off, s_lut);
  const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
  const uint32_t i0 = t << 2;
  const bool active = i0 < a.n_a;
  const uint4 d4 = active ? __ldg(reinterpret_cast<const uint4*>(a.spans) + t) : make_uint4(0, 0, 0, 0);
  const uint32_t d[4] = {d4.x, d4.y, d4.z, d4.w};
  // a block serves the same query tile for a.rpb consecutive rounds: the staged chromosome table and the spans are
  // paid once; one atomicAdd per warp and round (no block barrier inside the loop)
  const uint32_t r_first = blockIdx.y * a.rpb;
  const uint32_t r_end = min(r_first + a.rpb, a.n_launch);
  for (uint32_t r = r_first; r < r_end; ++r) {
    uint64_t sum = 0;
    if (active) {
      uint32_t st[4];
      place4(i0, a.round0 + r, a.tag, a.key, d, off, a.chrom, st);
#pragma unroll
      for (int j = 0; j < 4; ++j)
        if (i0 + j < a.n_a) sum += icount(a.bs, a.be, st[j], st[j] + d[j]);
    }
    sum = warp_sum_u64(sum);
    if ((threadIdx.x & 31) == 0 && sum) atomicAdd(a.round_counts + a.out0 + r, (unsigned long long)sum);
  }
}

// One round per block (grid = (query tiles, rounds)): for launches too small to give every block several rounds.
__global__ void __launch_bounds__(256) mc_permute_a_kernel(McAArgs a) {
  __shared__ uint32_t s_off[kMaxChromSmem];
  __shared__ __align__(16) uint16_t s_lut[kLutSize];
  __shared__ uint64_t s_red[8];
  const ChromView off = stage_chrom_table(a.chrom, s_off, s_lut);
  const uint32_t round = a.round0 + blockIdx.y;
  const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
  const uint32_t i0 = t << 2;
  uint64_t sum = 0;
  if (i0 < a.n_a) {
    const uint4 d4 = __ldg(reinterpret_cast<const uint4*>(a.spans) + t);
    const uint32_t d[4] = {d4.x, d4.y, d4.z, d4.w};
    uint32_t st[4];
    place4(i0, round, a.tag, a.key, d, off, a.chrom, st);
#pragma unroll
    for (int j = 0; j < 4; ++j)
      if (i0 + j < a.n_a) sum += icount(a.bs, a.be, st[j], st[j] + d[j]);
  }
  block_sum_atomic(sum, s_red, a.round_counts + a.out0 + blockIdx.y);
}

}  // namespace bits
