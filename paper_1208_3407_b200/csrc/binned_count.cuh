// binned_count.cuh -- the "search" and "reduce" steps for LARGE query sets: queries binned by the
// buckets of the sorted searched set, every bucket searched out of shared memory.
//
// PAPER.md:93-99 (Algorithm 1 ICOUNT): first = #{b.start <= a.end}, last = #{b.end < a.start},
// c(a) = first - last; PAPER.md:127-131 (Sec. 2.3) runs one ICOUNT per thread over the sorted
// arrays in global memory.  With 10^7 unsorted queries against 10^7 intervals (BASELINE.json
// configs[3]) that design -- and the bucket-index form of it in search.cuh -- reads two random DRAM
// sectors per query: B_S, B_E and their indices (96 MB) do not stay in an L2 through which 120 MB
// of queries and counts stream (profiles/r2a_cfg4_launches.md: 770 MB read for 200 MB of
// algorithmic traffic).  Here the random accesses become streams:
//
//   (msd::bin_hist_kernel, msd::plan_kernel)  the queries' ends are histogrammed by bin in the sort's own
//                         histogram launch; the block that plans B_S turns that into queries per bucket
//                         (bucket = the MSD sort's bucket of B_S that holds a.end's bin), where each
//                         bucket's queries go, and work items of at most kChunk queries of one bucket.
//   query_scatter_kernel  one pass over the queries: (a.end, a.start, input index) leave in bucket
//                         order (tile-local ranks by shared-memory atomics, one global reservation
//                         per tile and bucket, staged so that a bucket's writes are contiguous).
//   bucket_search_kernel  per work item: the bucket's slice of B_S and the ends that fall into the
//                         bucket's coordinate range (a contiguous slice of B_E) are copied into
//                         shared memory, a sub-bucket index is laid over each (4,096 entries: counts by
//                         shared-memory reductions, one block scan for both), and every query of the item is
//                         answered there: rank = slice offset + index entry + a short search
//                         inside one sub-bucket.  c(a) goes back to A's input order through the
//                         carried index (reading R19); the sum is reduced per block.
//
// The arrays B_S and B_E themselves are the ones Algorithm 2 asks for (sorted in full by the
// general sort); nothing here changes a count.  A query whose start lies before its bucket's
// coordinate range (an interval longer than what is left of the bucket) takes `last` by a binary
// search over B_E in global memory; a bucket whose ends do not fit the buffer does so for all its
// queries.  When the MSD sort has fallen back to the LSD sort (its device flag), these kernels
// exit at once and the index path of search.cuh, launched behind them, does the job.
#pragma once
#include "msd_sort.cuh"
#include "search.cuh"

namespace bits {
namespace qb {

constexpr int kChunk = 16384;                      // queries per work item (one bucket's queries, or a part of them)
constexpr int kSub = 4096, kSubBits = 12;          // sub-buckets of the per-bucket index
constexpr int kCapS = msd::kBucketCap;             // starts per bucket (the MSD sort's bucket capacity)
constexpr int kCapE = 10240;                       // ends staged per bucket; more -> global search for `last`

struct Plan {                        // what the MSD sort of B left behind (device pointers)
  const uint32_t* flag;              // [2] the sort's flags: non-zero = the LSD sort redid the job, buckets are void
  const uint16_t* bucket_of_bin;     // [kBins] bucket of B_S that holds each bin (top 12 key bits)
  const uint32_t* bucket_lo;         // [n_buckets + 1] first bin of each bucket
  const uint32_t* bucket_start;      // [n_buckets + 1] where each bucket's keys start in B_S
  const uint32_t* n_buckets;         // [1]
  const uint32_t* end_prefix;        // [kBins] #{ends < bin << 20} (the exclusive prefix of the ends' bin histogram, from the plan)
};

struct Lists {                       // the queries in bucket order (workspace)
  uint32_t* q_end;                   // [n_a]
  uint32_t* q_start;                 // [n_a]
  uint32_t* q_idx;                   // [n_a] input index (used only when per-interval counts are wanted)
  uint32_t* hist;                    // [kBins] queries per BIN (zero on entry; filled by the sort's histogram launch, read and cleared by its plan)
  uint32_t* off;                     // [kBins + 1] exclusive prefix of hist
  uint32_t* cursor;                  // [kBins] reservation cursors of the scatter pass
  uint32_t* item_off;                // [kBins + 1] exclusive prefix of the work items per bucket
  uint16_t* item_bucket;             // [n_a / kChunk + kBins] the bucket of every work item
};

__device__ __forceinline__ bool sort_fell_back(const uint32_t* flag) { return (flag[0] | flag[1]) != 0u; }

// ---------------------------------------------------------------------------------------------
// Scatter of the queries into bucket order.  Persistent blocks of 1,024 threads, tiles of 16,384 queries
// staged in INPUT order in shared memory (coalesced copy in), a permutation (position in bucket order ->
// query of the tile) built from tile-local ranks, then one pass that writes the three lists.
constexpr int kScThreads = 1024, kScQpt = 16, kScTile = kScThreads * kScQpt;
constexpr size_t kScSmem = (size_t)(2 * (kScTile + 4) + msd::kBins + kScTile) * sizeof(uint32_t) + (size_t)msd::kBins * sizeof(uint16_t);

template <bool kIdx>
__global__ void __launch_bounds__(kScThreads, 1) query_scatter_kernel(const uint32_t* __restrict__ a_start,
                                                                     const uint32_t* __restrict__ a_end, uint32_t n_a, Plan p, Lists l) {
  constexpr int kPer = msd::kBins / kScThreads;
  static_assert(kPer == 4 && kScTile <= 65536, "");
  extern __shared__ __align__(16) uint8_t smem_raw[];
  uint32_t* s_as = reinterpret_cast<uint32_t*>(smem_raw);          // [kScTile + 4] starts of the tile, input order
  uint32_t* s_ae = s_as + kScTile + 4;                             // [kScTile + 4] ends
  uint32_t* s_cnt = s_ae + kScTile + 4;                            // [kBins] counts, then local bases, then global position - local base
  uint32_t* s_pp = s_cnt + msd::kBins;                             // [kScTile] position in bucket order -> query of the tile | bucket << 16
  uint16_t* s_tbl = reinterpret_cast<uint16_t*>(s_pp + kScTile);   // [kBins] bin -> bucket
  __shared__ uint32_t s_w[32];
  grid_dependency_wait();
  if (sort_fell_back(p.flag)) return;
  const int tid = threadIdx.x;
  const uint32_t mis_s = msd::misalign_words(a_start), mis_e = msd::misalign_words(a_end);   // tiles start at multiples of 16,384: same misalignment
  for (int i = tid; i < msd::kBins; i += kScThreads) s_tbl[i] = p.bucket_of_bin[i];
  const uint32_t n_tiles = (n_a + kScTile - 1) / kScTile;
  for (uint32_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    const uint32_t base = tile * (uint32_t)kScTile;
    const uint32_t count = min((uint32_t)kScTile, n_a - base);
    __syncthreads();                                   // everyone is done with the previous tile's buffers
    msd::prefetch_keys<kScThreads>(s_as + mis_s, a_start + base, count);
    msd::prefetch_keys<kScThreads>(s_ae + mis_e, a_end + base, count);
    reinterpret_cast<uint4*>(s_cnt)[tid] = make_uint4(0, 0, 0, 0);
    msd::cp_async_wait_all();
    __syncthreads();
    const uint32_t* as = s_as + mis_s;
    const uint32_t* ae = s_ae + mis_e;
    uint32_t pk[kScQpt];                               // bucket | rank << 12 of this thread's queries
#pragma unroll
    for (int j = 0; j < kScQpt; ++j) {
      const uint32_t i = tid + j * kScThreads;
      if (i < count) {
        const uint32_t b = s_tbl[ae[i] >> msd::kBinShift];
        pk[j] = b | (atomicAdd(&s_cnt[b], 1u) << 12);
      }
    }
    __syncthreads();
    uint32_t c[kPer], lb[kPer], ga[kPer];
    {
      const uint4 v4 = reinterpret_cast<const uint4*>(s_cnt)[tid];
      c[0] = v4.x; c[1] = v4.y; c[2] = v4.z; c[3] = v4.w;
      uint32_t run = msd::block_excl_scan<kScThreads>(c[0] + c[1] + c[2] + c[3], s_w);
#pragma unroll
      for (int j = 0; j < kPer; ++j) {
        lb[j] = run;
        ga[j] = c[j] ? atomicAdd(&l.cursor[tid * kPer + j], c[j]) : 0u;      // one reservation per tile and bucket
        run += c[j];
      }
      reinterpret_cast<uint4*>(s_cnt)[tid] = make_uint4(lb[0], lb[1], lb[2], lb[3]);
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < kScQpt; ++j) {
      const uint32_t i = tid + j * kScThreads;
      if (i < count) { const uint32_t b = pk[j] & 0xfffu; s_pp[s_cnt[b] + (pk[j] >> 12)] = i | (b << 16); }
    }
    __syncthreads();
    reinterpret_cast<uint4*>(s_cnt)[tid] = make_uint4(ga[0] - lb[0], ga[1] - lb[1], ga[2] - lb[2], ga[3] - lb[3]);
    __syncthreads();
#pragma unroll 4
    for (int j = 0; j < kScQpt; ++j) {
      const uint32_t pos = tid + j * kScThreads;
      if (pos < count) {
        const uint32_t pp = s_pp[pos], i = pp & 0xffffu;
        const uint32_t dst = s_cnt[pp >> 16] + pos;
        l.q_end[dst] = ae[i]; l.q_start[dst] = as[i];
        if (kIdx) l.q_idx[dst] = base + i;
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// Ranks inside a sorted slice buf[0..n) through its sub-bucket index
//   ix[s] = #{keys with sub-bucket < s} | #{keys with sub-bucket <= s} << 16,  s = 0 .. kSub - 1
// (q lies inside the slice's coordinate range; four readable words follow the slice).  The look-up is split so
// that a thread can issue the loads of all its queries before it uses any of them:
//   w = ix[(q - lo) >> sshift];  c = count4(buf, w, q);  rank = finish(buf, w, c, q).
template <bool kStrict>
__device__ __forceinline__ uint32_t count4(const uint32_t* buf, uint32_t w, uint32_t q) {
  const uint32_t l = w & 0xffffu;
  uint32_t c = 0;
#pragma unroll
  for (uint32_t t = 0; t < 4; ++t) c += (kStrict ? (buf[l + t] < q) : (buf[l + t] <= q)) ? 1u : 0u;
  return c;
}
// #{keys <= q} (kStrict: < q).  Up to four keys in the sub-bucket: whatever follows it is larger than q, except a
// padding word when q = 0xffffffff, hence the min.  A crowded sub-bucket is searched.
template <bool kStrict>
__device__ __forceinline__ uint32_t finish_rank(const uint32_t* buf, uint32_t w, uint32_t c, uint32_t q) {
  uint32_t l = w & 0xffffu, h = w >> 16;
  if (h - l <= 4u) return l + min(c, h - l);
  while (l < h) {
    const uint32_t mid = l + ((h - l) >> 1);
    const uint32_t k = buf[mid];
    if (kStrict ? (k < q) : (k <= q)) l = mid + 1; else h = mid;
  }
  return l;
}

// Sub-bucket indices of two sorted slices at once (the form rank_in_slice reads): count with shared-memory
// reductions, then one block scan that carries both arrays (starts in the low half of a word, ends in the high
// half; both totals stay below 2^16).  All threads call it; it starts and ends with a barrier.  s_w: 32 words.
template <int kThreads>
__device__ __forceinline__ void index_two_slices(const uint32_t* bs, uint32_t ns, const uint32_t* be, uint32_t ne, uint32_t lo,
                                                 uint32_t sshift, uint32_t* ixs, uint32_t* ixe, uint32_t* s_w) {
  constexpr int kPer = kSub / kThreads;                // sub-buckets per thread and array
  static_assert(kPer == 8, "two uint4 per thread and array");
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
#pragma unroll
  for (int j = 0; j < kPer / 4; ++j) {
    reinterpret_cast<uint4*>(ixs)[tid + j * kThreads] = make_uint4(0, 0, 0, 0);
    reinterpret_cast<uint4*>(ixe)[tid + j * kThreads] = make_uint4(0, 0, 0, 0);
  }
  __syncthreads();
  const uint32_t m = max(ns, ne);
#pragma unroll 4
  for (uint32_t p = tid; p < m; p += kThreads) {
    if (p < ns) atomicAdd(&ixs[(bs[p] - lo) >> sshift], 1u);
    if (p < ne) atomicAdd(&ixe[(be[p] - lo) >> sshift], 1u);
  }
  __syncthreads();
  uint32_t c[2][kPer];
#pragma unroll
  for (int j = 0; j < kPer / 4; ++j) {
    const uint4 vs = reinterpret_cast<const uint4*>(ixs)[(kPer / 4) * tid + j], ve = reinterpret_cast<const uint4*>(ixe)[(kPer / 4) * tid + j];
    c[0][4 * j] = vs.x; c[0][4 * j + 1] = vs.y; c[0][4 * j + 2] = vs.z; c[0][4 * j + 3] = vs.w;
    c[1][4 * j] = ve.x; c[1][4 * j + 1] = ve.y; c[1][4 * j + 2] = ve.z; c[1][4 * j + 3] = ve.w;
  }
  uint32_t sum[2] = {0, 0};
#pragma unroll
  for (int a = 0; a < 2; ++a)
#pragma unroll
    for (int j = 0; j < kPer; ++j) sum[a] += c[a][j];
  uint32_t incl = sum[0] | (sum[1] << 16);
  const uint32_t own = incl;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(kFullMask, incl, o); if (lane >= o) incl += t; }
  if (lane == 31) s_w[w] = incl;
  __syncthreads();
  uint32_t x = lane < kThreads / 32 ? s_w[lane] : 0u;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(kFullMask, x, o); if (lane >= o) x += t; }
  const uint32_t excl = incl - own + (w ? __shfl_sync(kFullMask, x, (w + 31) & 31) : 0u);
#pragma unroll
  for (int a = 0; a < 2; ++a) {
    uint32_t run = a ? (excl >> 16) : (excl & 0xffffu);
#pragma unroll
    for (int j = 0; j < kPer; ++j) { const uint32_t n = c[a][j]; c[a][j] = run | ((run + n) << 16); run += n; }
  }
#pragma unroll
  for (int j = 0; j < kPer / 4; ++j) {
    reinterpret_cast<uint4*>(ixs)[(kPer / 4) * tid + j] = make_uint4(c[0][4 * j], c[0][4 * j + 1], c[0][4 * j + 2], c[0][4 * j + 3]);
    reinterpret_cast<uint4*>(ixe)[(kPer / 4) * tid + j] = make_uint4(c[1][4 * j], c[1][4 * j + 1], c[1][4 * j + 2], c[1][4 * j + 3]);
  }
  __syncthreads();
}

struct SearchArgs {
  Plan p;
  Lists l;
  const uint32_t* b_s;               // B_S, B_E: sorted in full
  const uint32_t* b_e;
  uint32_t n_b;
  uint32_t* counts;                  // [n_a] in A's input order, or null
  unsigned long long* total;         // += sum of the counts, or null
};

constexpr int kSrThreads = 512;
constexpr int kSrQpt = 4;                              // queries per thread and step; an item is answered in steps of kSrThreads * kSrQpt
constexpr int kSrStep = kSrThreads * kSrQpt;
constexpr size_t kSrSmem = (size_t)(kCapS + 8 + kCapE + 8 + 2 * kSub) * sizeof(uint32_t);

struct Bucket {                      // what a block needs to know about the bucket of a work item
  uint32_t base_s, ns;               // its slice of B_S
  uint32_t e0, ne;                   // the ends inside its coordinate range: B_E[e0 .. e0 + ne)
  uint32_t lo, sshift;               // first coordinate; sub-bucket = (key - lo) >> sshift
  uint32_t q0, q1;                   // the item's queries: lists[q0 .. q1)
};

__device__ __forceinline__ Bucket load_bucket(const SearchArgs& a, uint32_t item) {
  Bucket b;
  const uint32_t d = a.l.item_bucket[item];
  const uint32_t lo_bin = a.p.bucket_lo[d], hi_bin = a.p.bucket_lo[d + 1];
  b.base_s = a.p.bucket_start[d];
  b.ns = a.p.bucket_start[d + 1] - b.base_s;           // <= kCapS (else the sort's flag is up)
  b.e0 = a.p.end_prefix[lo_bin];
  b.ne = (hi_bin < (uint32_t)msd::kBins ? a.p.end_prefix[hi_bin] : a.n_b) - b.e0;
  b.lo = lo_bin << msd::kBinShift;
  const uint32_t span_bins = hi_bin - lo_bin;          // the bucket covers span_bins << 20 coordinates
  const uint32_t bits = msd::kBinShift + (span_bins > 1u ? 32u - __clz(span_bins - 1u) : 0u);
  b.sshift = bits > (uint32_t)kSubBits ? bits - kSubBits : 0u;
  b.q0 = a.l.off[d] + (item - a.l.item_off[d]) * (uint32_t)kChunk;
  b.q1 = min(a.l.off[d + 1], b.q0 + (uint32_t)kChunk);
  return b;
}

// Persistent blocks, work items dealt round robin.  Per item: the bucket's two slices are copied in
// (cp.async) while every thread fetches its queries into registers and the NEXT item's bucket is looked
// up; the slices are indexed; the queries are answered out of shared memory.
template <bool kCounts>
__global__ void __launch_bounds__(kSrThreads, 2) bucket_search_kernel(SearchArgs a) {
  extern __shared__ __align__(16) uint8_t smem_raw[];
  uint32_t* s_bs = reinterpret_cast<uint32_t*>(smem_raw);                  // [kCapS + 8]
  uint32_t* s_be = s_bs + kCapS + 8;                                       // [kCapE + 8]
  uint32_t* s_ixs = s_be + kCapE + 8;                                      // [kSub] sub-bucket index of the starts
  uint32_t* s_ixe = s_ixs + kSub;                                          // [kSub] ... of the ends
  __shared__ uint64_t s_red[kSrThreads / 32];
  __shared__ uint32_t s_w[32];
  grid_dependency_wait();
  if (sort_fell_back(a.p.flag)) return;
  const int tid = threadIdx.x;
  const uint32_t n_items = a.l.item_off[msd::kBins];
  uint64_t sum = 0;
  uint32_t item = blockIdx.x;
  Bucket b;
  if (item < n_items) b = load_bucket(a, item);
  for (; item < n_items; item += gridDim.x) {
    const bool ends_staged = b.ne <= (uint32_t)kCapE;
    const uint32_t* src_s = a.b_s + b.base_s;
    const uint32_t* src_e = a.b_e + b.e0;
    uint32_t* bs = s_bs + msd::misalign_words(src_s);
    uint32_t* be = s_be + msd::misalign_words(src_e);
    __syncthreads();                                   // everyone is done with the previous item's slices
    msd::prefetch_keys<kSrThreads>(bs, src_s, b.ns);
    if (ends_staged) msd::prefetch_keys<kSrThreads>(be, src_e, b.ne);
    uint32_t qe[kSrQpt], qs[kSrQpt], qx[kSrQpt];       // this thread's queries of the first step: in flight during the copy and the indexing
    // (queries past the item's end read as [lo, lo]: a legal look-up whose result is dropped)
    auto fetch = [&](uint32_t from, uint32_t to, uint32_t fill, uint32_t (&e)[kSrQpt], uint32_t (&st)[kSrQpt], uint32_t (&x)[kSrQpt]) {
#pragma unroll
      for (int j = 0; j < kSrQpt; ++j) {
        const uint32_t qi = from + tid + j * kSrThreads;
        const bool ok = qi < to;
        e[j] = ok ? __ldcs(a.l.q_end + qi) : fill;
        st[j] = ok ? __ldcs(a.l.q_start + qi) : fill;
        if (kCounts) x[j] = ok ? __ldcs(a.l.q_idx + qi) : 0u;
      }
    };
    fetch(b.q0, b.q1, b.lo, qe, qs, qx);
    const Bucket cur = b;
    if (item + gridDim.x < n_items) b = load_bucket(a, item + gridDim.x);
    if (tid < 4) { bs[cur.ns + tid] = 0xffffffffu; if (ends_staged) be[cur.ne + tid] = 0xffffffffu; }   // readable words behind the slices
    msd::cp_async_wait_all();
    index_two_slices<kSrThreads>(bs, cur.ns, be, ends_staged ? cur.ne : 0u, cur.lo, cur.sshift, s_ixs, s_ixe, s_w);   // barriers inside
    for (uint32_t from = cur.q0; from < cur.q1; from += kSrStep) {
      uint32_t ne_[kSrQpt], ns_[kSrQpt], nx_[kSrQpt];  // the next step's queries are fetched before this step's are answered
      if (from + kSrStep < cur.q1) fetch(from + kSrStep, cur.q1, cur.lo, ne_, ns_, nx_);
      // index words of all look-ups, then all key loads, then the arithmetic: independent loads stay in flight together
      uint32_t ws[kSrQpt], we[kSrQpt], cs[kSrQpt], ce[kSrQpt];
#pragma unroll
      for (int j = 0; j < kSrQpt; ++j) {
        ws[j] = s_ixs[(qe[j] - cur.lo) >> cur.sshift];
        we[j] = (ends_staged && qs[j] >= cur.lo) ? s_ixe[(qs[j] - cur.lo) >> cur.sshift] : 0u;
      }
#pragma unroll
      for (int j = 0; j < kSrQpt; ++j) { cs[j] = count4<false>(bs, ws[j], qe[j]); ce[j] = count4<true>(be, we[j], qs[j]); }
#pragma unroll
      for (int j = 0; j < kSrQpt; ++j) {
        if (from + tid + j * kSrThreads < cur.q1) {
          const uint32_t first = cur.base_s + finish_rank<false>(bs, ws[j], cs[j], qe[j]);
          uint32_t last;
          if (qs[j] >= cur.lo)
            last = cur.e0 + (ends_staged ? finish_rank<true>(be, we[j], ce[j], qs[j]) : rank_plain<true>(a.b_e + cur.e0, cur.ne, qs[j]));
          else
            last = rank_plain<true>(a.b_e, cur.e0, qs[j]);   // the interval starts before this bucket's range: every end >= lo is too large
          const uint32_t c = first - last;
          if (kCounts) a.counts[qx[j]] = c;
          sum += c;
        }
      }
#pragma unroll
      for (int j = 0; j < kSrQpt; ++j) { qe[j] = ne_[j]; qs[j] = ns_[j]; if (kCounts) qx[j] = nx_[j]; }
    }
  }
  if (a.total) block_sum_atomic(sum, s_red, a.total);
}

}  // namespace qb
}  // namespace bits
