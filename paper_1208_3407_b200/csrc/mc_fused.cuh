// mc_fused.cuh -- the Monte Carlo round when the SEARCHED set is re-placed (BITS_PERMUTE_B;
// "a random interval set is generated and placed into the associated data
// structure" every round), as three launches:
//
//   place_scatter_kernel   place (Philox4x32-10 -> start', end') fused with the first pass of the
//                          MSD sort (msd_sort.cuh): the fresh keys never go to HBM unsorted, they
//                          are ranked in shared memory and written straight into per-bin slabs.
//                          The bins are fixed per call (bin = key >> shift, chosen from the genome
//                          size and the set size), so no histogram is needed first: re-placed
//                          intervals are uniform over the valid starts by construction.
//   slab_plan_kernel       exclusive scan of the bin counts = where every bin's keys end up.
//   bucket_sort_kernel<true, true>  (msd_sort.cuh) sorts every bin in shared memory, writes the
//                          sorted arrays B_S / B_E, and -- while the bin is still in shared
//                          memory -- answers the queries that fall into it (search + reduce).
//
// A slab that overflows or a crowded sub-bucket raises the round's flag; the host redoes flagged
// rounds with the general path (place_kernel -> sort_arrays -> sorted_query_total_kernel).
#pragma once
#include "msd_sort.cuh"
#include "philox_place.cuh"

namespace bits {
namespace mcf {

constexpr int kMaxBins = msd::kBins;     // 4096
constexpr int kPsThreads = 512;
constexpr int kPsIpt = 16;               // intervals per thread and tile (four groups of four consecutive ones)
constexpr int kPsTile = kPsThreads * kPsIpt;   // 8192 intervals
constexpr size_t kPsSmem = (size_t)(kPsTile + 2 * kMaxBins + kMaxChromSmem) * sizeof(uint32_t);

struct PlaceScatterArgs {
  const uint32_t* spans;     // dev uint32[n], padded to a multiple of 4 with zeros, 16-byte aligned
  uint32_t n;
  uint32_t tile;             // intervals per tile: a multiple of 4, <= kPsTile (balanced over the grid by the host)
  uint32_t n_tiles;
  uint32_t round;
  uint32_t tag;
  PhiloxKeys key;
  ChromTable chrom;
  uint32_t shift;            // bin = key >> shift
  uint32_t n_bins;           // <= kMaxBins
  uint32_t slab;             // keys per slab
  uint32_t* slab_keys[2];    // [n_bins * slab] starts, ends
  uint32_t* cursor[2];       // [n_bins] keys written so far (zero at the start of the round)
  uint32_t* flag;            // round flag: msd::kFlagBucketTooBig on slab overflow
};

// Rank the tile's keys of one array by bin, reserve slab space, stage and write.  Called by all
// threads; key[] are this thread's kPsIpt keys, valid[] marks real intervals.
__device__ __forceinline__ void scatter_tile(const uint32_t (&key)[kPsIpt], uint32_t valid_mask, uint32_t shift, uint32_t n_bins,
                                             uint32_t slab, uint32_t* __restrict__ slab_keys, uint32_t* cursor, uint32_t* flag,
                                             uint32_t* s_stage, uint32_t* s_cnt, uint32_t* s_delta, uint32_t* s_w, uint32_t tile_count) {
  constexpr int kPer = kMaxBins / kPsThreads;   // 8 counters per thread
  const int tid = threadIdx.x;
  uint32_t r[kPsIpt];
#pragma unroll
  for (int j = 0; j < kPsIpt; ++j)
    if ((valid_mask >> j) & 1u) r[j] = atomicAdd(&s_cnt[key[j] >> shift], 1u);
  __syncthreads();
  uint32_t c[kPer], ga[kPer], lb[kPer];
  {
    const uint4 v0 = reinterpret_cast<const uint4*>(s_cnt)[2 * tid], v1 = reinterpret_cast<const uint4*>(s_cnt)[2 * tid + 1];
    c[0] = v0.x; c[1] = v0.y; c[2] = v0.z; c[3] = v0.w; c[4] = v1.x; c[5] = v1.y; c[6] = v1.z; c[7] = v1.w;
    uint32_t sum = 0;
#pragma unroll
    for (int j = 0; j < kPer; ++j) sum += c[j];
    uint32_t run = msd::block_excl_scan<kPsThreads>(sum, s_w);
    bool over = false;
#pragma unroll
    for (int j = 0; j < kPer; ++j) {
      const uint32_t b = tid * kPer + j;
      lb[j] = run;
      ga[j] = 0;
      if (c[j]) {
        const uint32_t g = atomicAdd(&cursor[b], c[j]);
        if (g + c[j] > slab) { over = true; ga[j] = 0xffffffffu; } else ga[j] = b * slab + g - run;
      }
      run += c[j];
    }
    if (over) atomicOr(flag, msd::kFlagBucketTooBig);
    reinterpret_cast<uint4*>(s_cnt)[2 * tid] = make_uint4(lb[0], lb[1], lb[2], lb[3]);
    reinterpret_cast<uint4*>(s_cnt)[2 * tid + 1] = make_uint4(lb[4], lb[5], lb[6], lb[7]);
  }
  __syncthreads();
#pragma unroll
  for (int j = 0; j < kPsIpt; ++j)
    if ((valid_mask >> j) & 1u) s_stage[s_cnt[key[j] >> shift] + r[j]] = key[j];
  reinterpret_cast<uint4*>(s_delta)[2 * tid] = make_uint4(ga[0], ga[1], ga[2], ga[3]);
  reinterpret_cast<uint4*>(s_delta)[2 * tid + 1] = make_uint4(ga[4], ga[5], ga[6], ga[7]);
  __syncthreads();
  reinterpret_cast<uint4*>(s_cnt)[2 * tid] = make_uint4(0, 0, 0, 0);
  reinterpret_cast<uint4*>(s_cnt)[2 * tid + 1] = make_uint4(0, 0, 0, 0);
#pragma unroll
  for (int j = 0; j < kPsIpt; ++j) {
    const uint32_t i = tid + j * kPsThreads;
    if (i < tile_count) {
      const uint32_t k = s_stage[i];
      const uint32_t dl = s_delta[k >> shift];
      if (dl != 0xffffffffu) slab_keys[dl + i] = k;
    }
  }
  __syncthreads();   // s_stage, s_cnt and s_delta are free again
  (void)n_bins;
}

__global__ void __launch_bounds__(kPsThreads, 2) place_scatter_kernel(PlaceScatterArgs a) {
  extern __shared__ __align__(16) uint8_t smem_raw[];
  uint32_t* s_stage = reinterpret_cast<uint32_t*>(smem_raw);   // [kPsTile]
  uint32_t* s_cnt = s_stage + kPsTile;                         // [kMaxBins]
  uint32_t* s_delta = s_cnt + kMaxBins;                        // [kMaxBins]
  uint32_t* s_off = s_delta + kMaxBins;                        // [kMaxChromSmem]
  __shared__ uint32_t s_w[32];
  const int tid = threadIdx.x;
  for (int i = tid; i < kMaxBins; i += kPsThreads) s_cnt[i] = 0;
  const uint32_t* off = stage_chrom_table(a.chrom, s_off);     // barrier inside
  for (uint32_t tile = blockIdx.x; tile < a.n_tiles; tile += gridDim.x) {
    const uint32_t base = tile * a.tile;
    const uint32_t tile_count = min(a.tile, a.n - base);
    uint32_t st[kPsIpt];
    uint32_t valid = 0;
#pragma unroll
    for (int g = 0; g < kPsIpt / 4; ++g) {
      const uint32_t l0 = 4u * (tid + g * kPsThreads);           // four consecutive intervals of the tile
      const uint32_t i0 = base + l0;
      if (l0 < tile_count) {
        const uint4 d4 = __ldg(reinterpret_cast<const uint4*>(a.spans + i0));
        const uint32_t dd[4] = {d4.x, d4.y, d4.z, d4.w};
        uint32_t ss[4];
        place4(i0, a.round, a.tag, a.key, dd, off, a.chrom, ss);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          st[4 * g + j] = ss[j];
          if (l0 + j < tile_count) valid |= 1u << (4 * g + j);
        }
      }
    }
    scatter_tile(st, valid, a.shift, a.n_bins, a.slab, a.slab_keys[0], a.cursor[0], a.flag, s_stage, s_cnt, s_delta, s_w, tile_count);
#pragma unroll
    for (int g = 0; g < kPsIpt / 4; ++g) {                       // end' = start' + span (spans re-read: L1/L2 hits)
      const uint32_t l0 = 4u * (tid + g * kPsThreads);
      if (l0 < tile_count) {
        const uint4 d4 = __ldg(reinterpret_cast<const uint4*>(a.spans + base + l0));
        st[4 * g] += d4.x; st[4 * g + 1] += d4.y; st[4 * g + 2] += d4.z; st[4 * g + 3] += d4.w;
      }
    }
    scatter_tile(st, valid, a.shift, a.n_bins, a.slab, a.slab_keys[1], a.cursor[1], a.flag, s_stage, s_cnt, s_delta, s_w, tile_count);
  }
}

// ---------------------------------------------------------------------------------------------
// Exclusive scan of the bin counts of both arrays (gridDim.x = 2, 1024 threads); clears the
// cursors for the next round; accounts for the queries beyond the last bin.
struct SlabPlanArgs {
  uint32_t* cursor[2];          // [kMaxBins] in: counts; cleared
  uint32_t* bucket_start[2];    // [kMaxBins + 1] out
  uint32_t* n_buckets;          // [2] out: n_bins
  uint32_t n_bins;
  uint32_t slab;
  uint32_t n_keys;              // keys per array (for the consistency check)
  uint32_t* flag;               // round flag
  uint32_t* msd_flag;           // [2] per-array flag words read by bucket_sort_kernel (written here)
  const uint32_t* qb[2];        // [n_bins + 1] query ranges per bin; queries from qb[n_bins] on lie beyond the last bin:
  uint32_t n_q;                 //   each of them counts every key (rank = n_keys)
  unsigned long long* round_total;
};

__global__ void __launch_bounds__(1024) slab_plan_kernel(SlabPlanArgs a) {
  __shared__ uint32_t s_w[32];
  const int arr = blockIdx.x, t = threadIdx.x;
  uint32_t* cursor = arr ? a.cursor[1] : a.cursor[0];
  uint32_t* bstart = arr ? a.bucket_start[1] : a.bucket_start[0];
  uint32_t c[4], sum = 0;
  bool over = false;
  {
    const uint4 v = reinterpret_cast<const uint4*>(cursor)[t];
    c[0] = v.x; c[1] = v.y; c[2] = v.z; c[3] = v.w;
    reinterpret_cast<uint4*>(cursor)[t] = make_uint4(0, 0, 0, 0);
  }
#pragma unroll
  for (int j = 0; j < 4; ++j) { over |= c[j] > a.slab; sum += c[j]; }
  uint32_t total;
  uint32_t run = msd::block_excl_scan<1024>(sum, s_w, &total);
#pragma unroll
  for (int j = 0; j < 4; ++j) { const uint32_t b = 4 * t + j; if (b <= a.n_bins) bstart[b] = run; run += c[j]; }
  over |= total != a.n_keys;
  const int any_over = __syncthreads_or(over);
  if (t == 0) {
    a.n_buckets[arr] = a.n_bins;
    a.msd_flag[arr] = any_over ? msd::kFlagBucketTooBig : 0u;
    if (any_over) atomicOr(a.flag, msd::kFlagBucketTooBig);
    const unsigned long long beyond = (unsigned long long)(a.n_q - (arr ? a.qb[1] : a.qb[0])[a.n_bins]) * a.n_keys;
    if (beyond) atomicAdd(a.round_total, arr ? (0ull - beyond) : beyond);
  }
}

// ---------------------------------------------------------------------------------------------
// Query ranges per bin, once per call: qb[b] = #{sorted queries < b << shift}, b = 0 .. n_bins.
struct QueryBinsArgs {
  const uint32_t* q_sorted[2];   // [n_q] each (A's ends for the start array, A's starts for the end array)
  uint32_t* qb[2];               // [kMaxBins + 1]
  uint32_t n_q;
  uint32_t n_bins;
  uint32_t shift;
};

__global__ void __launch_bounds__(256) query_bins_kernel(QueryBinsArgs a) {
  const uint32_t b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b > a.n_bins) return;
  const uint32_t* __restrict__ q = blockIdx.y ? a.q_sorted[1] : a.q_sorted[0];
  const uint64_t bound = (uint64_t)b << a.shift;
  uint32_t lo = 0, hi = a.n_q;
  while (lo < hi) {
    const uint32_t mid = lo + ((hi - lo) >> 1);
    if ((uint64_t)q[mid] < bound) lo = mid + 1; else hi = mid;
  }
  (blockIdx.y ? a.qb[1] : a.qb[0])[b] = lo;
}

}  // namespace mcf
}  // namespace bits
