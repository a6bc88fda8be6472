// msd_sort.cuh -- the "sort" step, fast path: most-significant-digit bucket sort of uint32 keys.
//
// PAPER.md:117-125 (Algorithm 2): Sort(B_S), Sort(B_E); keys only, so any correct sort gives the
// same array (reading R16).  The paper's sort is a library LSD radix sort of its day
// (PAPER.md:131, :159).  On sm_100a a stable LSD pass is bound by its ranking instruction
// (MATCH.ANY costs ~60 SM-cycles per warp, profiles/r1a_*), so this path is built around ranks
// that need NOT be stable and can come from shared-memory atomics (4 SM-cycles per warp):
//
//   1. bin histogram     top kBinBits bits of every key (fused into the placement kernel inside
//                        the Monte Carlo loop, place_kernels.cuh).
//   2. plan_kernel       exclusive scan of the bins = where each bin's keys go; consecutive bins
//                        are grouped into buckets of at most kBucketCap keys.
//   3. scatter_kernel    one pass: tile-local ranks by atomicAdd on per-bin counters, one global
//                        reservation per (tile, bin), keys staged through shared memory so the
//                        writes of a bin are contiguous.  Afterwards every bucket's keys are in
//                        their final range, unordered inside.
//   4. bucket_sort_kernel  one bucket at a time per block, entirely in shared memory: sub-bucket
//                        by the next kSubBits bits of (key - min) with atomics, exclusive scan,
//                        stage; the few keys that share a sub-bucket are ordered by a tiny
//                        insertion sort; coalesced write-out.
//
// Two passes over HBM instead of the four of an 8-bit LSD sort.  It assumes nothing about the
// input: when a bucket would not fit (plan) or a sub-bucket is crowded (bucket sort) a flag is set
// on the device and the stable LSD sort of radix_sort.cuh, launched right behind, redoes the job;
// otherwise those launches exit at once.
#pragma once
#include "common.cuh"

namespace bits {
namespace msd {

constexpr int kBinBits = 12;
constexpr int kBins = 1 << kBinBits;          // 4096
constexpr int kBinShift = 32 - kBinBits;

// scatter: 16 keys per thread; the block shape is a template configuration (ScatterCfg below)
constexpr int kScKpt = 16;

// bucket sort: 512 threads x 16 keys, two blocks per SM
constexpr int kBkThreads = 512;
constexpr int kBkKpt = 16;
constexpr int kBucketCap = kBkThreads * kBkKpt;   // 8192 keys
constexpr int kSubBits = 12;
constexpr int kSub = 1 << kSubBits;
constexpr int kSubLimit = 64;                     // a sub-bucket with more keys raises the flag
constexpr int kWl = kBucketCap / 2;               // groups of >= 2 keys: at most n / 2
constexpr size_t kBkSmem = (size_t)(2 * (kBucketCap + 4) + kSub + kWl) * sizeof(uint32_t);

constexpr uint32_t kFlagBucketTooBig = 1u, kFlagSubCrowded = 2u;

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
  const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async4(void* smem_dst, const void* gsrc) {
  const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// Copy `count` keys into shared memory asynchronously.  16-byte copies need src and s_dst
// congruent modulo 16 bytes: the caller passes s_dst already offset by (src & 15) / 4 words.
template <int kThreads>
__device__ __forceinline__ void prefetch_keys(uint32_t* s_dst, const uint32_t* src, uint32_t count) {
  const uint32_t head = min(count, (uint32_t)((16u - ((uintptr_t)src & 15u)) & 15u) >> 2);
  if (threadIdx.x < head) cp_async4(s_dst + threadIdx.x, src + threadIdx.x);
  const uint32_t body = (count - head) >> 2;
  for (uint32_t i = threadIdx.x; i < body; i += kThreads) cp_async16(s_dst + head + 4 * i, src + head + 4 * i);
  const uint32_t done = head + 4 * body;
  if (threadIdx.x < count - done) cp_async4(s_dst + done + threadIdx.x, src + done + threadIdx.x);
}
__device__ __forceinline__ uint32_t misalign_words(const uint32_t* p) { return (uint32_t)(((uintptr_t)p & 15u) >> 2); }

// Exclusive prefix of one value per thread over the block; `total` of the block in *total_out
// (may be null).  One barrier inside; s_w is scratch of 32 words.  Call from all threads.
template <int kThreads>
__device__ __forceinline__ uint32_t block_excl_scan(uint32_t v, uint32_t* s_w, uint32_t* total_out = nullptr) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  uint32_t incl = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(kFullMask, incl, o); if (lane >= o) incl += t; }
  if (lane == 31) s_w[w] = incl;
  __syncthreads();
  uint32_t x = lane < kThreads / 32 ? s_w[lane] : 0u;      // every warp scans the warp totals itself
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(kFullMask, x, o); if (lane >= o) x += t; }
  const uint32_t before = __shfl_sync(kFullMask, x, (w + 31) & 31);
  if (total_out) *total_out = __shfl_sync(kFullMask, x, 31);
  return incl - v + (w ? before : 0u);
}

// ---------------------------------------------------------------------------------------------
// 1. histogram of the top kBinBits bits (stand-alone version).  gridDim.y = arrays.
struct BinHistArgs {
  const uint32_t* keys[3];   // [2]: an extra key array histogrammed in the same launch (the query ends of binned_count.cuh)
  uint32_t* hist[3];         // uint32[kBins] each, zero on entry (plan_kernel leaves them zero)
  uint32_t n[3];
};

__global__ void __launch_bounds__(512) bin_hist_kernel(BinHistArgs a) {
  __shared__ uint32_t s_h[kBins];
  grid_dependency_wait();
  for (int i = threadIdx.x; i < kBins; i += blockDim.x) s_h[i] = 0;
  __syncthreads();
  const uint32_t* __restrict__ keys = blockIdx.y == 0 ? a.keys[0] : (blockIdx.y == 1 ? a.keys[1] : a.keys[2]);
  const uint32_t n = blockIdx.y == 0 ? a.n[0] : (blockIdx.y == 1 ? a.n[1] : a.n[2]);
  const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
  if (((uintptr_t)keys & 15) == 0) {
    const uint32_t n4 = n >> 2;
    const uint4* k4 = reinterpret_cast<const uint4*>(keys);
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += stride) {
      const uint4 k = __ldg(k4 + i);
      atomicAdd(&s_h[k.x >> kBinShift], 1u); atomicAdd(&s_h[k.y >> kBinShift], 1u);
      atomicAdd(&s_h[k.z >> kBinShift], 1u); atomicAdd(&s_h[k.w >> kBinShift], 1u);
    }
    if (blockIdx.x == 0 && threadIdx.x < (n & 3u)) atomicAdd(&s_h[keys[(n & ~3u) + threadIdx.x] >> kBinShift], 1u);
  } else {
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
      atomicAdd(&s_h[keys[i] >> kBinShift], 1u);
  }
  __syncthreads();
  uint32_t* g = blockIdx.y == 0 ? a.hist[0] : (blockIdx.y == 1 ? a.hist[1] : a.hist[2]);
  for (int i = threadIdx.x; i < kBins; i += blockDim.x) if (s_h[i]) atomicAdd(&g[i], s_h[i]);
}

// ---------------------------------------------------------------------------------------------
// 2. plan.  Bucket = run of consecutive bins whose exclusive prefix count falls into the same
// multiple of `target` = kBucketCap - (largest bin) + 1, so a bucket holds at most kBucketCap keys
// whenever the largest bin does.  Buckets get dense ids 0 .. n_buckets-1 (<= kBins).
// One block of 1024 threads per array (gridDim.x = arrays).
struct PlanArr {
  uint32_t* hist;           // [kBins] in; cleared for the next use
  uint32_t* bin_cursor;     // [kBins] out: exclusive prefix of hist = #{keys < bin << 20} (read by binned_count.cuh)
  uint32_t* bucket_start;   // [kBins + 1] out: bucket d occupies [bucket_start[d], bucket_start[d+1])
  uint32_t* n_buckets;      // [1] out
  uint32_t* flag;           // [1] out: kFlagBucketTooBig or 0 (plain store: this also resets it)
  uint32_t* lsd_hist;       // [1024] cleared here for the fallback sort's digit histograms (may be null)
  uint32_t* lsd_ticket;     // [4] cleared here: the fallback sort's tile tickets, one per pass (may be null)
  uint16_t* bucket_of_bin;  // [kBins] out: the bucket every bin belongs to (the scatter pass writes by bucket; binned_count.cuh)
  uint32_t* bucket_cursor;  // [kBins] out: = bucket_start (advanced by the scatter pass, one reservation per tile and bucket)
  uint32_t* bucket_lo;      // [kBins + 1] out (may be null): first bin of bucket d; bucket_lo[n_buckets] = kBins
};
// Plan of a query set that is to be brought into the order of array 0's buckets (binned_count.cuh), made by the
// block that plans array 0: queries per bucket from the queries' own bin histogram.
struct QueryPlan {
  uint32_t* bin_hist;       // [kBins] in: histogram of the queries' bins (null: no queries); cleared for the next use
  uint32_t* off;            // [kBins + 1] out: where each bucket's queries start; off[n_buckets] = number of queries
  uint32_t* cursor;         // [kBins] out: = off (advanced by the scatter pass)
  uint32_t* item_off;       // [kBins + 1] out: exclusive prefix of the work items per bucket; [kBins] = their number
  uint16_t* item_bucket;    // out: the bucket of every work item
  uint32_t chunk;           // queries per work item
};
struct PlanArgs {
  PlanArr p[2];
  QueryPlan q;
  uint32_t pack_cap;        // 0: buckets by the prefix / target rule; else consecutive bins are packed greedily up to this many keys
};

__global__ void __launch_bounds__(1024) plan_kernel(PlanArgs a) {
  static_assert(kBins == 4096, "4 bins per thread");
  __shared__ uint32_t s_w[32];
  __shared__ uint32_t s_raw[kBins + kBins / 32 + 2];
  __shared__ uint32_t s_start[kBins + 1];
  const PlanArr P = blockIdx.x ? a.p[1] : a.p[0];
  const int t = threadIdx.x;
  grid_dependency_wait();
  if (P.lsd_hist) P.lsd_hist[t] = 0;
  if (P.lsd_ticket && t < 4) P.lsd_ticket[t] = 0;
  uint32_t h[4], ex[4];
  {
    const uint4 v = reinterpret_cast<const uint4*>(P.hist)[t];
    h[0] = v.x; h[1] = v.y; h[2] = v.z; h[3] = v.w;
    reinterpret_cast<uint4*>(P.hist)[t] = make_uint4(0, 0, 0, 0);
  }
  uint32_t sum = 0, big = 0;
#pragma unroll
  for (int j = 0; j < 4; ++j) { ex[j] = sum; sum += h[j]; big = max(big, h[j]); }
  big = __reduce_max_sync(kFullMask, big);
  if ((t & 31) == 0) s_raw[t >> 5] = big;
  uint32_t total;
  const uint32_t before = block_excl_scan<1024>(sum, s_w, &total);     // barrier inside: s_raw[0..31] visible
  big = __reduce_max_sync(kFullMask, s_raw[t & 31]);
  __syncthreads();
  const uint32_t target = big < (uint32_t)kBucketCap ? (uint32_t)kBucketCap - big + 1u : 1u;
#pragma unroll
  for (int j = 0; j < 4; ++j) ex[j] += before;
  reinterpret_cast<uint4*>(P.bin_cursor)[t] = make_uint4(ex[0], ex[1], ex[2], ex[3]);
  uint32_t first[4], nf = 0, fex[4];
  if (a.pack_cap) {
    // greedy packing: a bucket takes consecutive bins while it stays within pack_cap keys (fuller buckets than the
    // rule below: fewer of them, fewer fixed costs per bucket).  Sequential inside chunks of 64 bins, one thread per
    // chunk; a chunk boundary always starts a bucket.
    // (prefixes are read with a stride of 64 words by the chunk threads: one pad word per 32 keeps them off one bank;
    // a chunk's 64 "starts a bucket" flags travel as one 64-bit mask)
    uint32_t* s_pad = s_raw;                              // [kBins + kBins / 32 + 2]
    __shared__ unsigned long long s_mask[kBins / 64];
    auto pad = [](uint32_t i) { return i + (i >> 5); };
#pragma unroll
    for (int j = 0; j < 4; ++j) s_pad[pad(4 * t + j)] = ex[j];
    if (t == 0) s_pad[pad(kBins)] = total;
    __syncthreads();
    if (t < kBins / 64) {
      uint32_t from = s_pad[pad(64 * t)];
      unsigned long long mask = 1ull;
      for (int b = 64 * t + 1; b < 64 * t + 64; ++b) {
        const bool brk = s_pad[pad(b + 1)] - from > a.pack_cap;
        if (brk) { from = s_pad[pad(b)]; mask |= 1ull << (b & 63); }
      }
      s_mask[t] = mask;
    }
    __syncthreads();
    const unsigned long long m = s_mask[t >> 4];
#pragma unroll
    for (int j = 0; j < 4; ++j) { first[j] = (uint32_t)(m >> ((4 * t + j) & 63)) & 1u; fex[j] = nf; nf += first[j]; }
  } else {
#pragma unroll
    for (int j = 0; j < 4; ++j) s_raw[4 * t + j + 1] = ex[j] / target;
    if (t == 0) s_raw[0] = 0xffffffffu;
    __syncthreads();
#pragma unroll
    for (int j = 0; j < 4; ++j) { first[j] = s_raw[4 * t + j + 1] != s_raw[4 * t + j]; fex[j] = nf; nf += first[j]; }
  }
  uint32_t nb;
  const uint32_t fbefore = block_excl_scan<1024>(nf, s_w, &nb);
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const uint32_t d = fbefore + fex[j] + first[j] - 1u;       // bucket of bin 4t + j (bin 0 always starts one)
    if (first[j]) { P.bucket_start[d] = ex[j]; P.bucket_cursor[d] = ex[j]; s_start[d] = ex[j]; if (P.bucket_lo) P.bucket_lo[d] = 4u * t + j; }
    P.bucket_of_bin[4 * t + j] = (uint16_t)d;
  }
  if (t == 0) { P.bucket_start[nb] = total; s_start[nb] = total; *P.n_buckets = nb; if (P.bucket_lo) P.bucket_lo[nb] = (uint32_t)kBins; }
  if (blockIdx.x == 0 && a.q.bin_hist) {
    // queries per bucket: the exclusive prefix of the queries' bin histogram, read at the buckets' first bins
    uint32_t* s_qoff = s_raw;                             // (s_raw is free: the barrier of the scan above lies behind its last use)
    const uint4 qv = reinterpret_cast<const uint4*>(a.q.bin_hist)[t];
    reinterpret_cast<uint4*>(a.q.bin_hist)[t] = make_uint4(0, 0, 0, 0);
    const uint32_t qh[4] = {qv.x, qv.y, qv.z, qv.w};
    uint32_t qtotal;
    __syncthreads();
    uint32_t qrun = block_excl_scan<1024>(qh[0] + qh[1] + qh[2] + qh[3], s_w, &qtotal);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      if (first[j]) { const uint32_t d = fbefore + fex[j]; s_qoff[d] = qrun; a.q.off[d] = qrun; a.q.cursor[d] = qrun; }
      qrun += qh[j];
    }
    if (t == 0) { s_qoff[nb] = qtotal; a.q.off[nb] = qtotal; }
    __syncthreads();
    uint32_t items[4], isum = 0;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const uint32_t d = 4u * t + j;
      items[j] = d < nb ? (s_qoff[d + 1] - s_qoff[d] + a.q.chunk - 1u) / a.q.chunk : 0u;
      isum += items[j];
    }
    uint32_t itotal;
    uint32_t irun = block_excl_scan<1024>(isum, s_w, &itotal);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      a.q.item_off[4 * t + j] = irun;
      for (uint32_t k = 0; k < items[j]; ++k) a.q.item_bucket[irun + k] = (uint16_t)(4 * t + j);
      irun += items[j];
    }
    if (t == 0) a.q.item_off[kBins] = itotal;
  }
  __syncthreads();
  bool bad = false;
  for (uint32_t d = t; d < nb; d += 1024) bad |= (s_start[d + 1] - s_start[d]) > (uint32_t)kBucketCap;
  const int any_bad = __syncthreads_or(bad);
  if (t == 0) *P.flag = any_bad ? kFlagBucketTooBig : 0u;
}

// ---------------------------------------------------------------------------------------------
// 3. scatter by BUCKET (unstable; the bins of a bucket need no order among themselves: the per-bucket sort
// orders the whole bucket).  Fewer, longer runs per tile than a scatter by bin: a 16,384-key tile spreads over
// ~1,650 buckets instead of ~3,400 bins on config 4.  Persistent blocks: grid = (blocks, arrays); block b takes
// tiles b, b + gridDim.x, ...; the next tile is prefetched with cp.async while this one is ranked.
struct ScatterArr {
  const uint32_t* src;
  uint32_t* dst;
  const uint16_t* bucket_of_bin;   // [kBins]
  uint32_t* bucket_cursor;         // [kBins]: advanced by atomicAdd, one reservation per (tile, bucket)
  const uint32_t* flag;
};
struct ScatterArgs { ScatterArr arr[2]; uint32_t n; uint32_t n_tiles; };

// Shape: kT threads x kScKpt keys per tile, kB resident blocks per SM (1,024 x 1: 16,384-key tiles, longer runs per bin;
// 512 x 2: 8,192-key tiles, two blocks hide each other's barriers).
template <int kT, int kB>
struct ScatterCfg {
  static constexpr int kThreads = kT, kBlocksPerSm = kB;
  static constexpr int kTile = kT * kScKpt;
  static constexpr size_t kSmem = (size_t)(2 * (kTile + 4) + 2 * kBins) * sizeof(uint32_t) + (size_t)kBins * sizeof(uint16_t);
};

template <class C>
__global__ void __launch_bounds__(C::kThreads, C::kBlocksPerSm) scatter_kernel(ScatterArgs a) {
  constexpr int kThreads = C::kThreads, kTile = C::kTile;
  constexpr int kPer = kBins / kThreads;        // bins per thread: 4 or 8
  static_assert(kTile <= 65536 && kPer % 4 == 0, "");
  extern __shared__ __align__(16) uint8_t smem_raw[];
  uint32_t* s_buf = reinterpret_cast<uint32_t*>(smem_raw);              // [2][kTile + 4]
  uint32_t* s_cnt = s_buf + 2 * (kTile + 4);                            // [kBins] counts, then local bases
  uint32_t* s_delta = s_cnt + kBins;                                    // [kBins] global dst - local base
  uint16_t* s_tbl = reinterpret_cast<uint16_t*>(s_delta + kBins);       // [kBins] bin -> bucket
  __shared__ uint32_t s_w[32];
  const ScatterArr A = blockIdx.y ? a.arr[1] : a.arr[0];
  grid_dependency_wait();
  if (*A.flag) return;
  const int tid = threadIdx.x;
  for (int i = tid; i < kBins; i += kThreads) s_tbl[i] = A.bucket_of_bin[i];
  const uint32_t mis = misalign_words(A.src);   // tiles start at multiples of kTile keys: same misalignment
#pragma unroll
  for (int q = 0; q < kPer / 4; ++q) reinterpret_cast<uint4*>(s_cnt)[(kPer / 4) * tid + q] = make_uint4(0, 0, 0, 0);
  uint32_t tile = blockIdx.x;
  if (tile < a.n_tiles)
    prefetch_keys<kThreads>(s_buf + mis, A.src + (size_t)tile * kTile, min((uint32_t)kTile, a.n - tile * (uint32_t)kTile));
  for (int it = 0; tile < a.n_tiles; tile += gridDim.x, ++it) {
    uint32_t* buf = s_buf + (it & 1) * (kTile + 4) + mis;
    cp_async_wait_all();
    __syncthreads();          // this tile's keys are here; everyone is done with the other buffer
    const uint32_t next = tile + gridDim.x;
    if (next < a.n_tiles)
      prefetch_keys<kThreads>(s_buf + ((it + 1) & 1) * (kTile + 4) + mis, A.src + (size_t)next * kTile,
                              min((uint32_t)kTile, a.n - next * (uint32_t)kTile));
    const uint32_t count = min((uint32_t)kTile, a.n - tile * (uint32_t)kTile);
    const bool full = count == (uint32_t)kTile;
    uint32_t key[kScKpt], r[kScKpt];              // r = rank inside the tile's share of the bucket | bucket << 16
#pragma unroll
    for (int j = 0; j < kScKpt; ++j) {
      const uint32_t i = tid + j * kThreads;
      if (full || i < count) {
        key[j] = buf[i];
        const uint32_t b = s_tbl[key[j] >> kBinShift];
        r[j] = atomicAdd(&s_cnt[b], 1u) | (b << 16);
      }
    }
    __syncthreads();
    // exclusive scan of the bucket counts; one global reservation per non-empty (tile, bucket)
    uint32_t c[kPer], ga[kPer], lb[kPer];
    {
      uint32_t sum = 0;
#pragma unroll
      for (int q = 0; q < kPer / 4; ++q) {
        const uint4 v4 = reinterpret_cast<const uint4*>(s_cnt)[(kPer / 4) * tid + q];
        c[4 * q] = v4.x; c[4 * q + 1] = v4.y; c[4 * q + 2] = v4.z; c[4 * q + 3] = v4.w;
        sum += v4.x + v4.y + v4.z + v4.w;
      }
      uint32_t run = block_excl_scan<kThreads>(sum, s_w);
#pragma unroll
      for (int j = 0; j < kPer; ++j) {
        lb[j] = run;
        ga[j] = c[j] ? atomicAdd(&A.bucket_cursor[tid * kPer + j], c[j]) : 0u;
        run += c[j];
      }
#pragma unroll
      for (int q = 0; q < kPer / 4; ++q)
        reinterpret_cast<uint4*>(s_cnt)[(kPer / 4) * tid + q] = make_uint4(lb[4 * q], lb[4 * q + 1], lb[4 * q + 2], lb[4 * q + 3]);
    }
    __syncthreads();
    // stage in bin order, in place (every key of the tile is in a register by now)
#pragma unroll
    for (int j = 0; j < kScKpt; ++j) {
      const uint32_t i = tid + j * kThreads;
      if (full || i < count) buf[s_cnt[r[j] >> 16] + (r[j] & 0xffffu)] = key[j];
    }
#pragma unroll
    for (int q = 0; q < kPer / 4; ++q)
      reinterpret_cast<uint4*>(s_delta)[(kPer / 4) * tid + q] =
          make_uint4(ga[4 * q] - lb[4 * q], ga[4 * q + 1] - lb[4 * q + 1], ga[4 * q + 2] - lb[4 * q + 2], ga[4 * q + 3] - lb[4 * q + 3]);
    __syncthreads();
#pragma unroll
    for (int q = 0; q < kPer / 4; ++q) reinterpret_cast<uint4*>(s_cnt)[(kPer / 4) * tid + q] = make_uint4(0, 0, 0, 0);
    uint32_t* __restrict__ dst = A.dst;
#pragma unroll
    for (int j = 0; j < kScKpt; ++j) {
      const uint32_t i = tid + j * kThreads;
      if (full || i < count) { const uint32_t k = buf[i]; dst[s_delta[s_tbl[k >> kBinShift]] + i] = k; }
    }
  }
}
using ScatterCfg1x1024 = ScatterCfg<1024, 1>;
using ScatterCfg2x512 = ScatterCfg<512, 2>;

// ---------------------------------------------------------------------------------------------
// 4. per-bucket sort in shared memory.  Persistent blocks: grid = (blocks, arrays); block b takes
// buckets b, b + gridDim.x, ...; the next bucket's keys are prefetched while this one is sorted.
struct BucketArr {
  const uint32_t* src;            // scattered keys: bucket d at src + bucket_start[d], or (kSlab) at src + d * slab
  uint32_t* dst;                  // sorted keys: bucket d at dst + bucket_start[d]
  const uint32_t* bucket_start;   // [n_buckets + 1]
  const uint32_t* n_buckets;
  uint32_t* flag;                 // per-array flag word (read: kFlagBucketTooBig; or-ed: kFlagSubCrowded)
  // kSearch: the sorted queries whose rank in this array is wanted, and their range per bucket
  const uint32_t* q_sorted;       // ascending
  const uint32_t* qb;             // [n_buckets + 1]: queries qb[d] .. qb[d+1]-1 fall into bucket d's key range
};
struct BucketArgs {
  BucketArr arr[2];
  uint32_t slab;                        // kSlab: keys per slab
  uint32_t* round_flag;                 // kSearch: or-ed with kFlagSubCrowded as well (may be null)
  unsigned long long* round_total;      // kSearch: += sum of ranks (array 0, "<= q") - sum of ranks (array 1, "< q")
};

// ascending insertion sort of s[0..k), k small, by one thread
__device__ __forceinline__ void small_sort(uint32_t* s, uint32_t k) {
  for (uint32_t i = 1; i < k; ++i) {
    const uint32_t x = s[i];
    uint32_t j = i;
    while (j > 0 && s[j - 1] > x) { s[j] = s[j - 1]; --j; }
    s[j] = x;
  }
}

// kSlab: buckets are read from fixed-capacity slabs (mc_fused.cuh).  kSearch: after a bucket is
// sorted, the queries that fall into its key range are ranked against it while it is still in
// shared memory (Algorithm 1: the two BSEARCHes; the rank of q in the whole array is
// bucket_start[d] + its rank inside bucket d), and the ranks are summed.
template <bool kSlab, bool kSearch>
__global__ void __launch_bounds__(kBkThreads, 2) bucket_sort_kernel(BucketArgs a) {
  constexpr int kPer = kSub / kBkThreads;   // sub-bucket counters per thread
  static_assert(kPer % 4 == 0 && kSubLimit <= 255 && kBucketCap <= (1 << 16), "");
  extern __shared__ __align__(16) uint8_t smem_raw[];
  uint32_t* s_buf = reinterpret_cast<uint32_t*>(smem_raw);   // [2][kBucketCap + 4]
  uint32_t* s_sub = s_buf + 2 * (kBucketCap + 4);            // [kSub] counts, then bases
  uint32_t* s_wl = s_sub + kSub;                             // [kWl] pairs from the front (base), larger groups from the back (base << 8 | k)
  __shared__ uint32_t s_w[32];
  __shared__ uint32_t s_min[32], s_max[32];
  __shared__ uint32_t s_nwl;                                 // pairs | larger groups << 16
  const BucketArr A = blockIdx.y ? a.arr[1] : a.arr[0];
  grid_dependency_wait();
  if (*A.flag & kFlagBucketTooBig) return;
  const uint32_t nb = *A.n_buckets;
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const bool strict = blockIdx.y != 0;     // kSearch: array 1 (ends) wants #{keys < q}, array 0 (starts) #{keys <= q}
  uint64_t qsum = 0;                       // kSearch: this thread's sum of ranks
  {
    uint4* z = reinterpret_cast<uint4*>(s_sub);
#pragma unroll
    for (int j = 0; j < kPer / 4; ++j) z[tid + j * kBkThreads] = make_uint4(0, 0, 0, 0);
    if (tid == 0) s_nwl = 0;
  }
  uint32_t d = blockIdx.x;
  uint32_t base = 0, n = 0, nbase = 0, nn = 0;
  const uint32_t* src = A.src;
  if (d < nb) {
    base = A.bucket_start[d]; n = A.bucket_start[d + 1] - base;
    src = kSlab ? A.src + (size_t)d * a.slab : A.src + base;
    prefetch_keys<kBkThreads>(s_buf + misalign_words(src), src, n);
  }
  for (int it = 0; d < nb; d += gridDim.x, ++it, base = nbase, n = nn) {
    uint32_t* buf = s_buf + (it & 1) * (kBucketCap + 4) + misalign_words(src);
    cp_async_wait_all();
    __syncthreads();
    const uint32_t dn = d + gridDim.x;
    if (dn < nb) {
      nbase = A.bucket_start[dn]; nn = A.bucket_start[dn + 1] - nbase;
      src = kSlab ? A.src + (size_t)dn * a.slab : A.src + nbase;
      prefetch_keys<kBkThreads>(s_buf + ((it + 1) & 1) * (kBucketCap + 4) + misalign_words(src), src, nn);
    }
    uint32_t qlo = 0, qhi = 0;
    if (kSearch) { qlo = A.qb[d]; qhi = A.qb[d + 1]; }
    if (n == 0) {
      if (kSearch && tid == 0) qsum += (uint64_t)(qhi - qlo) * base;   // an empty bucket: rank = keys before it
      continue;
    }
    uint32_t key[kBkKpt], r[kBkKpt];
    uint32_t mn = 0xffffffffu, mx = 0;
#pragma unroll
    for (int j = 0; j < kBkKpt; ++j) {
      if ((uint32_t)(j * kBkThreads) >= n) break;
      const uint32_t i = tid + j * kBkThreads;
      if (i < n) { key[j] = buf[i]; mn = min(mn, key[j]); mx = max(mx, key[j]); }
    }
    mn = __reduce_min_sync(kFullMask, mn); mx = __reduce_max_sync(kFullMask, mx);
    if (lane == 0) { s_min[w] = mn; s_max[w] = mx; }
    __syncthreads();
    mn = s_min[lane < kBkThreads / 32 ? lane : 0]; mx = s_max[lane < kBkThreads / 32 ? lane : 0];
    mn = __reduce_min_sync(kFullMask, mn); mx = __reduce_max_sync(kFullMask, mx);
    const uint32_t range = mx - mn;
    uint32_t* __restrict__ dst = A.dst + base;
    if (range == 0) {   // all keys equal: already sorted (block-uniform branch)
#pragma unroll
      for (int j = 0; j < kBkKpt; ++j) { const uint32_t i = tid + j * kBkThreads; if (i < n) dst[i] = key[j]; }
      if (kSearch)
        for (uint32_t qi = qlo + tid; qi < qhi; qi += kBkThreads) {
          const uint32_t q = __ldg(A.q_sorted + qi);
          qsum += base + ((strict ? q > mn : q >= mn) ? n : 0u);
        }
      continue;
    }
    const int bits = 32 - __clz(range);
    const int shift = bits > kSubBits ? bits - kSubBits : 0;
#pragma unroll
    for (int j = 0; j < kBkKpt; ++j) {
      if ((uint32_t)(j * kBkThreads) >= n) break;
      const uint32_t i = tid + j * kBkThreads;
      if (i < n) r[j] = atomicAdd(&s_sub[(key[j] - mn) >> shift], 1u);
    }
    __syncthreads();
    // exclusive scan of the sub-bucket counts (kPer consecutive counters per thread); groups of
    // two keys and groups of three or more go on the two worklists
    {
      uint32_t c[kPer], sum = 0, n2 = 0, n3 = 0, big = 0;
      const uint4* p4 = reinterpret_cast<const uint4*>(s_sub + tid * kPer);
#pragma unroll
      for (int j = 0; j < kPer / 4; ++j) { const uint4 v = p4[j]; c[4 * j] = v.x; c[4 * j + 1] = v.y; c[4 * j + 2] = v.z; c[4 * j + 3] = v.w; }
#pragma unroll
      for (int j = 0; j < kPer; ++j) { sum += c[j]; n2 += c[j] == 2; n3 += c[j] > 2; big = max(big, c[j]); }
      if (__any_sync(kFullMask, big > (uint32_t)kSubLimit)) {
        if (lane == 0) { atomicOr(A.flag, kFlagSubCrowded); if (kSearch && a.round_flag) atomicOr(a.round_flag, kFlagSubCrowded); }
        n2 = 0; n3 = 0;
      }
      // worklist slots: warp-level scan of (n2 | n3 << 16), one shared atomic per warp
      uint32_t packed = n2 | (n3 << 16), pin = packed;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(kFullMask, pin, o); if (lane >= o) pin += t; }
      uint32_t wbase = 0;
      if (lane == 31 && pin) wbase = atomicAdd(&s_nwl, pin);
      wbase = __shfl_sync(kFullMask, wbase, 31);
      const uint32_t pex = wbase + pin - packed;
      uint32_t slot2 = pex & 0xffffu, slot3 = (uint32_t)kWl - 1u - (pex >> 16);
      uint32_t run = block_excl_scan<kBkThreads>(sum, s_w);
      uint4* o4 = reinterpret_cast<uint4*>(s_sub + tid * kPer);
#pragma unroll
      for (int j = 0; j < kPer / 4; ++j) {
        uint4 o;
        o.x = run; run += c[4 * j]; o.y = run; run += c[4 * j + 1]; o.z = run; run += c[4 * j + 2]; o.w = run; run += c[4 * j + 3];
        o4[j] = o;
      }
      if (n2 | n3) {
        run -= sum;
#pragma unroll
        for (int j = 0; j < kPer; ++j) {
          if (c[j] == 2) s_wl[slot2++] = run;
          else if (c[j] > 2) s_wl[slot3--] = (run << 8) | c[j];
          run += c[j];
        }
      }
    }
    __syncthreads();
    // stage in sub-bucket order, in place (every key of the bucket is in a register by now)
#pragma unroll
    for (int j = 0; j < kBkKpt; ++j) {
      if ((uint32_t)(j * kBkThreads) >= n) break;
      const uint32_t i = tid + j * kBkThreads;
      if (i < n) buf[s_sub[(key[j] - mn) >> shift] + r[j]] = key[j];
    }
    __syncthreads();
    {
      const uint32_t nwl = s_nwl, n2 = nwl & 0xffffu, n3 = nwl >> 16;
      for (uint32_t q = tid; q < n2; q += kBkThreads) {
        uint32_t* s = buf + s_wl[q];
        const uint32_t x = s[0], y = s[1];
        if (y < x) { s[0] = y; s[1] = x; }
      }
      for (uint32_t q = tid; q < n3; q += kBkThreads) { const uint32_t e = s_wl[kWl - 1 - q]; small_sort(buf + (e >> 8), e & 255u); }
      if (!kSearch) {
        uint4* z = reinterpret_cast<uint4*>(s_sub);
#pragma unroll
        for (int j = 0; j < kPer / 4; ++j) z[tid + j * kBkThreads] = make_uint4(0, 0, 0, 0);
      }
    }
    __syncthreads();
    if (tid == 0) s_nwl = 0;
#pragma unroll
    for (int j = 0; j < kBkKpt; ++j) {
      if ((uint32_t)(j * kBkThreads) >= n) break;
      const uint32_t i = tid + j * kBkThreads;
      if (i < n) dst[i] = buf[i];
    }
    if (kSearch) {
      // rank of q inside the bucket: all keys of earlier sub-buckets are smaller; finish inside q's own
      for (uint32_t qi = qlo + tid; qi < qhi; qi += kBkThreads) {
        const uint32_t q = __ldg(A.q_sorted + qi);
        uint32_t local;
        if (q < mn) local = 0;
        else if (q > mx) local = n;
        else {
          const uint32_t sb = (q - mn) >> shift;
          uint32_t p = s_sub[sb];
          const uint32_t hi = sb + 1 < (uint32_t)kSub ? s_sub[sb + 1] : n;
          while (p < hi && (strict ? buf[p] < q : buf[p] <= q)) ++p;
          local = p;
        }
        qsum += base + local;
      }
      __syncthreads();   // everyone is done with the sub-bucket bases
      uint4* z = reinterpret_cast<uint4*>(s_sub);
#pragma unroll
      for (int j = 0; j < kPer / 4; ++j) z[tid + j * kBkThreads] = make_uint4(0, 0, 0, 0);
    }
  }
  if (kSearch) {
    __shared__ uint64_t s_red[kBkThreads / 32];
    __syncthreads();
    qsum = warp_sum_u64(qsum);
    if (lane == 0) s_red[w] = qsum;
    __syncthreads();
    if (w == 0) {
      uint64_t t = lane < kBkThreads / 32 ? s_red[lane] : 0;
      t = warp_sum_u64(t);
      if (lane == 0 && t != 0) atomicAdd(a.round_total, (unsigned long long)(strict ? 0ull - t : t));
    }
  }
}

}  // namespace msd
}  // namespace bits
