// mc_tile.cuh -- the Monte Carlo round when the SEARCHED set is re-placed (BITS_PERMUTE_B;
// "a random interval set is generated and placed into the associated data
// structure" every round), as TWO launches with no global atomics on the data path:
//
//   place_tile_kernel   place (Philox4x32-10 -> start', end') fused with the
//                       first half of the sort: every tile of up to 24,576 fresh intervals is
//                       ordered by bin (bin = start' >> shift, fixed per call) in shared memory --
//                       count pass, scan, staging pass through per-bin cursors -- and leaves as
//                       (start', end') pairs through cp.async.bulk; next to it goes the tile's row
//                       of the segment table:  off[tile][b] = #{pairs of the tile in bins < b} |
//                       #{in bin b} << 16 (written coalesced).  Fresh keys never go to HBM unsorted.
//   bin_sort_search_kernel  one bin at a time per block.  Column b of the segment table gives, per
//                       tile, where the bin's pairs sit; the sum of the starts is the number of keys in
//                       all earlier bins, i.e. where the bin starts in the sorted arrays -- no
//                       histogram pass, no scan over bins, no reservation.  The pairs are
//                       gathered (cp.async, a group of lanes per segment) into shared memory;
//                       starts and ends are each sorted there (Algorithm 2's Sort(B_S),
//                       Sort(B_E): counting sort on the next 13 bits with
//                       16-bit cursors, ties inside a sub-bucket ordered by comparison counting
//                       on the way out), written to B_S / B_E, and -- while the bin is still in
//                       shared memory -- the queries that fall into its key range are ranked
//                       against it (Algorithm 1's two BSEARCHes) and their ranks
//                       summed.
//
// An end that lies in the bin after its start's bin (span < bin width is a precondition of this
// path, checked on the host) is handed over through a small per-bin list.  A bin with more than
// kCap keys or an over-full hand-over list raises the round's flag; the host redoes flagged
// rounds with the general path (place_kernel -> sort_arrays -> sorted_query_total_kernel).
// Kernel shapes are template configurations (TileCfg, BinCfg); DESIGN.md section 5 has the
// measurements behind the defaults.
#pragma once
#include "msd_sort.cuh"
#include "philox_place.cuh"

namespace bits {
namespace mct {

constexpr int kMaxBins = 4096;
// Shape of place_tile_kernel: threads per block, intervals per thread and tile (a multiple of 4),
// resident blocks per SM.  A tile holds up to kTile intervals, staged as pairs in shared memory.
template <int kThreads_, int kIpt_, int kBlocksPerSm_>
struct TileCfg {
  static constexpr int kThreads = kThreads_, kIpt = kIpt_, kBlocksPerSm = kBlocksPerSm_;
  static constexpr int kTile = kThreads * kIpt;
  static constexpr size_t kSmem = (size_t)kTile * sizeof(uint2) + (size_t)(kMaxBins + kMaxChromSmem) * sizeof(uint32_t) +
                                  (size_t)kLutSize * sizeof(uint16_t);
};
using TileCfg2x512 = TileCfg<512, 16, 2>;        // 8192-interval tiles, two blocks per SM
using TileCfg1x1024 = TileCfg<1024, 16, 1>;      // 16384-interval tiles, one block per SM
using TileCfg1x1024L = TileCfg<1024, 24, 1>;     // 24576-interval tiles, one block per SM
constexpr int kMaxTileAny = 24576;

constexpr int kCrossCap = 512;                   // hand-over list entries per bin
constexpr int kMaxShift = 22;                    // widest bin: 2^22 coordinates
constexpr int kMaxTiles = 3072;                  // segment table of the bin sort: one word per tile
constexpr int kFront = 8;                        // halfwords in front of a cursor array (one uint4)

// Shape of the per-bin sort (bin_sort_search_kernel): threads per block, keys per thread,
// sub-bucket bits, resident blocks per SM.  kCap keys per bin and array; 2^kSubBits sub-buckets
// with 16-bit cursors, two per word.
template <int kThreads_, int kKpt_, int kSubBits_, int kBlocksPerSm_>
struct BinCfg {
  static constexpr int kThreads = kThreads_, kKpt = kKpt_, kSubBits = kSubBits_, kBlocksPerSm = kBlocksPerSm_;
  static constexpr int kCap = kThreads * kKpt;
  static constexpr int kSub = 1 << kSubBits;
  static constexpr int kCurLen = kFront + kSub + 8;      // halfwords per cursor array, a whole number of uint4s
  static constexpr size_t kSmemFixed = (size_t)(2 * kCap) * sizeof(uint32_t) + (size_t)(2 * kCurLen) * sizeof(uint16_t);
  static size_t smem_bytes(uint32_t n_tiles) { return kSmemFixed + ((size_t)n_tiles + 8) * sizeof(uint32_t); }
};
using BinCfgWide = BinCfg<512, 16, 13, 2>;       // 8192 keys per bin, two blocks per SM
using BinCfgNarrow = BinCfg<512, 8, 12, 3>;      // 4096 keys per bin, three blocks per SM
using BinCfgSmall = BinCfg<256, 16, 12, 4>;      // 4096 keys per bin, four blocks of 256 threads per SM
using BinCfgHuge = BinCfg<1024, 16, 14, 1>;      // 16384 keys per bin, one block of 1024 threads per SM

constexpr uint32_t kFlagBinTooBig = 1u, kFlagCrossFull = 4u;

// Bulk asynchronous copy shared -> global (the TMA engine moves the bytes, no LDS / STG issued).
// dst, src 16-byte aligned, bytes a multiple of 16.
// (unqualified: orders this thread's earlier generic-proxy accesses to shared AND global memory before later
// async-proxy ones -- the tile's slice of `pairs` is used as scratch through ordinary stores first)
__device__ __forceinline__ void fence_proxy_async_all() { asm volatile("fence.proxy.async;" ::: "memory"); }
__device__ __forceinline__ void bulk_store_smem_to_global(void* gdst, const void* ssrc, uint32_t bytes) {
  const uint32_t s = (uint32_t)__cvta_generic_to_shared(ssrc);
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst), "r"(s), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit_group() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_group_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }

struct PlaceTileArgs {
  const uint32_t* spans;     // dev uint32[n], padded to a multiple of 4 with zeros, 16-byte aligned
  uint32_t n;
  uint32_t tile;             // intervals per tile: a multiple of 4, <= kTile (balanced over the grid by the host)
  uint32_t n_tiles;
  uint32_t round;
  uint32_t tag;
  PhiloxKeys key;
  ChromTable chrom;
  uint32_t shift;            // bin = key >> shift, 1..31
  uint32_t n_bins;           // <= kMaxBins
  uint2* pairs;              // [n]: tile t holds its intervals [t * tile, ...) ordered by bin
  uint32_t* off;             // [n_tiles * stride]: off[t * stride + b] = #{pairs of tile t in bins < b} | #{in bin b} << 16
  uint32_t stride;           // entries per tile row: kMaxBins
  uint32_t* cross_cnt;       // [n_bins + 1] ends handed over to each bin this round (zero on entry)
  uint32_t* cross_keys;      // [n_bins * kCrossCap]
  uint32_t* flag;            // round flag
  // several rounds per launch (gridDim.y = rounds; small sets): round blockIdx.y works on its own copy of pairs /
  // off / cross_cnt / cross_keys, `slot_words` 32-bit words further on, takes flag[blockIdx.y] and round + blockIdx.y
  uint32_t slot_words;
};

// kSlots: several rounds per launch (the arguments are then moved to the round's slot; the one-round instantiation
// keeps reading them straight from the parameter bank).
template <class C, bool kSlots = false>
__global__ void __launch_bounds__(C::kThreads, C::kBlocksPerSm) place_tile_kernel(PlaceTileArgs a) {
  if (kSlots && blockIdx.y) {
    const size_t o = (size_t)blockIdx.y * a.slot_words;
    a.pairs = reinterpret_cast<uint2*>(reinterpret_cast<uint32_t*>(a.pairs) + o);
    a.off += o; a.cross_cnt += o; a.cross_keys += o; a.flag += blockIdx.y; a.round += blockIdx.y;
  }
  constexpr int kPer = kMaxBins / C::kThreads;   // bin counters per thread (4 or 8)
  static_assert(kPer % 4 == 0, "uint4 accesses");
  extern __shared__ __align__(16) uint8_t smem_raw[];
  uint2* s_stage = reinterpret_cast<uint2*>(smem_raw);                   // [C::kTile]
  uint32_t* s_cnt = reinterpret_cast<uint32_t*>(s_stage + C::kTile);        // [kMaxBins] counts, then bases
  uint32_t* s_off = s_cnt + kMaxBins;                                    // [kMaxChromSmem]
  uint16_t* s_lut = reinterpret_cast<uint16_t*>(s_off + kMaxChromSmem);  // [kLutSize]
  __shared__ uint32_t s_w[32];
  const int tid = threadIdx.x;
  for (int i = tid; i < kMaxBins; i += C::kThreads) s_cnt[i] = 0;
  const ChromView off = stage_chrom_table(a.chrom, s_off, s_lut);        // barrier inside
  const uint32_t shift = a.shift;
  grid_dependency_wait();     // the previous round's bin sort has finished reading pairs / off / hand-over lists
  bool stage_in_flight = false;   // thread 0: a bulk copy out of s_stage has been issued and not yet waited for
  for (uint32_t tile = blockIdx.x; tile < a.n_tiles; tile += gridDim.x) {
    const uint32_t base = tile * a.tile;
    const uint32_t count = min(a.tile, a.n - base);
    // the starts wait for the staging pass in the tile's own (not yet written) slice of `pairs`:
    // 24 fewer live registers in the Philox pass; the loads below hit L2
    uint32_t* const scratch = reinterpret_cast<uint32_t*>(a.pairs + base);
    uint4 dn = make_uint4(0, 0, 0, 0);                                    // spans of the next group, loaded one group ahead
    if (4u * tid < count) dn = __ldg(reinterpret_cast<const uint4*>(a.spans + base + 4u * tid));
#pragma unroll 2
    for (int g = 0; g < C::kIpt / 4; ++g) {
      const uint32_t l0 = 4u * (tid + g * C::kThreads);                   // four consecutive intervals of the tile
      const uint4 d4 = dn;
      if (g + 1 < C::kIpt / 4 && l0 + 4u * C::kThreads < count)
        dn = __ldg(reinterpret_cast<const uint4*>(a.spans + base + l0 + 4u * C::kThreads));
      if (l0 < count) {
        const uint32_t dd[4] = {d4.x, d4.y, d4.z, d4.w};
        uint32_t ss[4];
        place4(base + l0, a.round, a.tag, a.key, dd, off, a.chrom, ss);
        *reinterpret_cast<uint4*>(scratch + l0) = make_uint4(ss[0], ss[1], ss[2], ss[3]);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          if (l0 + j < count) {
            const uint32_t bin = ss[j] >> shift;
            atomicAdd(&s_cnt[bin], 1u);                             // count only: the slot is taken in the staging pass
            const uint32_t e = ss[j] + dd[j], ebin = e >> shift;
            if (ebin != bin) {                                           // rare: the end lies in the next bin
              const uint32_t slot = atomicAdd(&a.cross_cnt[ebin], 1u);
              if (slot < (uint32_t)kCrossCap) a.cross_keys[(size_t)ebin * kCrossCap + slot] = e;
              else atomicOr(a.flag, kFlagCrossFull);
            }
          }
        }
      }
    }
    __syncthreads();
    // exclusive scan of the bin counts -> bases (kept in s_cnt) and the transposed prefix row entries
    {
      uint32_t c[kPer];
#pragma unroll
      for (int j = 0; j < kPer / 4; ++j) {
        const uint4 v = reinterpret_cast<const uint4*>(s_cnt)[(kPer / 4) * tid + j];
        c[4 * j] = v.x; c[4 * j + 1] = v.y; c[4 * j + 2] = v.z; c[4 * j + 3] = v.w;
      }
      uint32_t sum = 0;
#pragma unroll
      for (int j = 0; j < kPer; ++j) sum += c[j];
      uint32_t run = msd::block_excl_scan<C::kThreads>(sum, s_w);
      uint32_t lb[kPer];
#pragma unroll
      for (int j = 0; j < kPer; ++j) { lb[j] = run; run += c[j]; }
#pragma unroll
      for (int j = 0; j < kPer / 4; ++j)
        reinterpret_cast<uint4*>(s_cnt)[(kPer / 4) * tid + j] = make_uint4(lb[4 * j], lb[4 * j + 1], lb[4 * j + 2], lb[4 * j + 3]);
      // the tile's row of the segment table, one word per bin (where the bin's pairs start in the tile | how many
      // << 16), all kMaxBins entries: coalesced
      uint32_t* o = a.off + (size_t)tile * a.stride + (size_t)tid * kPer;
#pragma unroll
      for (int j = 0; j < kPer / 4; ++j)
        reinterpret_cast<uint4*>(o)[j] = make_uint4(lb[4 * j] | (c[4 * j] << 16), lb[4 * j + 1] | (c[4 * j + 1] << 16),
                                                    lb[4 * j + 2] | (c[4 * j + 2] << 16), lb[4 * j + 3] | (c[4 * j + 3] << 16));
    }
    if (tid == 0 && stage_in_flight) { bulk_wait_group_read0(); stage_in_flight = false; }   // the previous tile has left s_stage
    __syncthreads();
    // stage the pairs in bin order: every bin's base doubles as its cursor (spans re-read: cache hits)
    // (the four slots of a group are taken first and filled afterwards, so the atomics overlap)
    {
      uint4 d4 = make_uint4(0, 0, 0, 0), s4 = d4;
      if (4u * tid < count) {
        d4 = __ldg(reinterpret_cast<const uint4*>(a.spans + base + 4u * tid));
        s4 = *reinterpret_cast<const uint4*>(scratch + 4u * tid);
      }
#pragma unroll 2
      for (int g = 0; g < C::kIpt / 4; ++g) {
        const uint32_t l0 = 4u * (tid + g * C::kThreads);
        const uint32_t dd[4] = {d4.x, d4.y, d4.z, d4.w};
        const uint32_t st[4] = {s4.x, s4.y, s4.z, s4.w};
        if (g + 1 < C::kIpt / 4) {                                       // the next group's spans and starts are on their way
          const uint32_t l1 = l0 + 4u * C::kThreads;
          if (l1 < count) {
            d4 = __ldg(reinterpret_cast<const uint4*>(a.spans + base + l1));
            s4 = *reinterpret_cast<const uint4*>(scratch + l1);
          }
        }
        if (l0 < count) {
          uint32_t slot[4];
#pragma unroll
          for (int j = 0; j < 4; ++j) slot[j] = l0 + j < count ? atomicAdd(&s_cnt[st[j] >> shift], 1u) : 0xffffffffu;
#pragma unroll
          for (int j = 0; j < 4; ++j)
            if (slot[j] != 0xffffffffu) s_stage[slot[j]] = make_uint2(st[j], st[j] + dd[j]);
        }
      }
    }
    fence_proxy_async_all();    // this thread's staged pairs are about to be read, and its scratch stores to the tile's
                                // slice of `pairs` overwritten, by the bulk-copy engine
    __syncthreads();
#pragma unroll
    for (int j = 0; j < kPer / 4; ++j) reinterpret_cast<uint4*>(s_cnt)[(kPer / 4) * tid + j] = make_uint4(0, 0, 0, 0);
    if (tid == 0) {
      // one bulk copy per 32 KB, shared -> global, no LDS / STG: the next tile's placement overlaps it
      uint2* dst = a.pairs + base;                                       // base % 4 == 0: 32-byte aligned
      const uint32_t bytes = (count & ~1u) * (uint32_t)sizeof(uint2);    // a multiple of 16
      for (uint32_t o = 0; o < bytes; o += 32768u)
        bulk_store_smem_to_global(reinterpret_cast<char*>(dst) + o, reinterpret_cast<const char*>(s_stage) + o, min(32768u, bytes - o));
      bulk_commit_group();
      if (count & 1u) dst[count - 1] = s_stage[count - 1];
      stage_in_flight = true;
    }
    __syncthreads();   // s_cnt is clear again; s_stage is free once thread 0 has waited for the bulk copies
  }
  if (tid == 0 && stage_in_flight) bulk_wait_group_read0();
}

// ---------------------------------------------------------------------------------------------
struct BinSortArgs {
  const uint2* pairs;
  const uint32_t* off;
  uint32_t stride;
  uint32_t n_tiles;
  uint32_t tile;
  uint32_t n;                           // keys per array
  uint32_t shift;
  uint32_t n_bins;
  const uint32_t* cross_cnt;            // this round's hand-over counts
  const uint32_t* cross_keys;
  uint32_t* cross_cnt_next;             // the other parity: cleared here for the next round
  uint32_t* dst[2];                     // B_S, B_E: the sorted arrays of this round
  const uint32_t* q_sorted[2];          // ascending: A's ends (ranked in B_S, "<="), A's starts (ranked in B_E, "<")
  const uint32_t* qb[2];                // [n_bins + 1]: queries qb[d] .. qb[d+1]-1 fall into bin d's key range
  uint32_t n_q;
  uint32_t group, group_log2;           // lanes that gather one (tile, bin) segment together: a power of two, 1..32
  unsigned long long* round_total;      // += sum of ranks in B_S - sum of ranks in B_E
  uint32_t* flag;
  uint32_t slot_words;                  // several rounds per launch (gridDim.y): as in PlaceTileArgs; dst, round_total and flag move too
};

// Counter arrays of one bin: uint16 cursors, two per word.  Entry kFront + sb belongs to
// sub-bucket sb; entry kFront - 1 stays 0, so after the scatter (which leaves every cursor at
// the END of its sub-bucket) the keys of sub-bucket sb sit at [cur[kFront + sb - 1], cur[kFront + sb]).

__device__ __forceinline__ uint32_t sub_of(uint32_t key, uint32_t mask, uint32_t sshift) { return (key & mask) >> sshift; }

// ++count of the key's sub-bucket (no result needed: a reduction, not an atomic with return)
__device__ __forceinline__ void count_key(uint32_t* cur32, uint32_t sb) {
  const uint32_t e = sb + kFront;
  atomicAdd(&cur32[e >> 1], 1u << ((e & 1u) << 4));
}
// position of the next key of sub-bucket sb; bumps the cursor
__device__ __forceinline__ uint32_t take_slot(uint32_t* cur32, uint32_t sb) {
  const uint32_t e = sb + kFront, sh = (e & 1u) << 4;
  return (atomicAdd(&cur32[e >> 1], 1u << sh) >> sh) & 0xffffu;
}

// Counts -> exclusive prefixes, in place, for both cursor arrays (starts, ends) with one pair of
// barriers.  total[0], total[1] = keys counted per array.  s_w: 64 words of scratch.
template <class C>
__device__ __forceinline__ void scan_cursors(uint16_t* cur_s, uint16_t* cur_e, uint32_t* s_w, uint32_t total[2]) {
  constexpr int kWords = C::kSub / 2 / C::kThreads;   // cursor words per thread and array
  static_assert(kWords % 4 == 0, "uint4 accesses");
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  uint32_t c[2][kWords], sum[2] = {0, 0};
#pragma unroll
  for (int a = 0; a < 2; ++a) {
    const uint4* src = reinterpret_cast<const uint4*>((a ? cur_e : cur_s) + kFront) + (kWords / 4) * tid;
#pragma unroll
    for (int j = 0; j < kWords / 4; ++j) {
      const uint4 v = src[j];
      c[a][4 * j] = v.x; c[a][4 * j + 1] = v.y; c[a][4 * j + 2] = v.z; c[a][4 * j + 3] = v.w;
    }
#pragma unroll
    for (int j = 0; j < kWords; ++j) sum[a] += (c[a][j] & 0xffffu) + (c[a][j] >> 16);
  }
  // both sums travel through one scan: starts in the low half, ends in the high half (each <= C::kCap)
  uint32_t incl = sum[0] | (sum[1] << 16);
  const uint32_t own = incl;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(kFullMask, incl, o); if (lane >= o) incl += t; }
  if (lane == 31) s_w[w] = incl;
  __syncthreads();
  uint32_t x = lane < C::kThreads / 32 ? s_w[lane] : 0u;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(kFullMask, x, o); if (lane >= o) x += t; }
  const uint32_t before = w ? __shfl_sync(kFullMask, x, (w + 31) & 31) : 0u;
  const uint32_t tot = __shfl_sync(kFullMask, x, 31);
  total[0] = tot & 0xffffu; total[1] = tot >> 16;
  const uint32_t excl = incl - own + before;
#pragma unroll
  for (int a = 0; a < 2; ++a) {
    uint32_t run = a ? (excl >> 16) : (excl & 0xffffu);
#pragma unroll
    for (int j = 0; j < kWords; ++j) {
      const uint32_t lo = c[a][j] & 0xffffu, hi = c[a][j] >> 16;
      c[a][j] = run | ((run + lo) << 16);
      run += lo + hi;
    }
    uint4* dst = reinterpret_cast<uint4*>((a ? cur_e : cur_s) + kFront) + (kWords / 4) * tid;
#pragma unroll
    for (int j = 0; j < kWords / 4; ++j) dst[j] = make_uint4(c[a][4 * j], c[a][4 * j + 1], c[a][4 * j + 2], c[a][4 * j + 3]);
  }
  __syncthreads();
}

// Counting-sort scatter of buf[0..m) in place: every key is read into a register, then (after a
// barrier) stored at the slot its sub-bucket's cursor hands out.  With kCheckBin, entries whose
// bin is not d are dropped.  Ends with a barrier; afterwards buf[0..mv) (mv = the keys that stay) is ordered
// by sub-bucket, buf[mv..mv+3) holds 0xffffffff and cur[kFront + sb] is the END of sub-bucket sb.
template <class C, bool kCheckBin, bool kTrailingBarrier = true>
__device__ __forceinline__ void scatter_in_place(uint32_t* buf, uint32_t m, uint32_t d, uint32_t shift, uint32_t mask,
                                                 uint32_t sshift, uint16_t* cur, uint32_t mv) {
  const int tid = threadIdx.x;
  uint32_t* cur32 = reinterpret_cast<uint32_t*>(cur);
  uint32_t key[C::kKpt];
#pragma unroll
  for (int j = 0; j < C::kKpt; ++j) {
    const uint32_t i = tid + j * C::kThreads;
    key[j] = i < m ? buf[i] : 0u;
  }
  __syncthreads();
  if (tid < 3) buf[mv + tid] = 0xffffffffu;           // sentinels behind the mv keys that stay (no slot lies there)
#pragma unroll
  for (int j0 = 0; j0 < C::kKpt; j0 += 4) {           // four slots are taken, then filled: the atomics overlap
    if ((uint32_t)(j0 * C::kThreads) >= m) break;
    uint32_t slot[4];
#pragma unroll
    for (int j = j0; j < j0 + 4; ++j) {
      const uint32_t k = key[j];
      const bool ok = tid + j * C::kThreads < m && (!kCheckBin || (k >> shift) == d);
      slot[j - j0] = ok ? take_slot(cur32, sub_of(k, mask, sshift)) : 0xffffffffu;
    }
#pragma unroll
    for (int j = j0; j < j0 + 4; ++j)
      if (slot[j - j0] != 0xffffffffu) buf[slot[j - j0]] = key[j];
  }
  if (kTrailingBarrier) __syncthreads();
}

// Write buf[0..mv) (ordered by sub-bucket) to dst[gbase ..] in ascending order: the keys that
// share a sub-bucket are ordered by comparison counting (ties by position), the first three
// candidates without a loop.  Then rank the sorted queries q_sorted[qlo..qhi), all of which fall
// into this bin's key range: every key of an earlier sub-bucket is smaller, the count is finished
// inside the query's own sub-bucket.  Returns this thread's sum of query ranks.
template <class C, bool kStrict>
__device__ __forceinline__ uint64_t write_and_rank(const uint32_t* buf, uint32_t mv, uint32_t mask, uint32_t sshift,
                                                   const uint16_t* cur, uint32_t gbase, uint32_t* __restrict__ dst,
                                                   const uint32_t* __restrict__ q_sorted, uint32_t qlo, uint32_t qhi,
                                                   uint32_t q_first) {
  const int tid = threadIdx.x;
#pragma unroll 2
  for (uint32_t p = tid; p < mv; p += C::kThreads) {
    const uint32_t k = buf[p];
    const uint32_t sb = sub_of(k, mask, sshift);
    const uint32_t lo = cur[kFront - 1 + sb], hi = cur[kFront + sb];
    uint32_t rank = 0;
#pragma unroll
    for (uint32_t i = 0; i < 3; ++i) {
      const uint32_t t = lo + i;
      const uint32_t kk = buf[t];                    // t < mv + 3: beyond the sub-bucket lie larger keys, beyond mv sentinels
      rank += kk < k + (t < p ? 1u : 0u);            // (k + 1 cannot wrap: coordinates are < 2^32 - 1)
    }
    if (hi - lo > 3) {
#pragma unroll 1
      for (uint32_t t = lo + 3; t < hi; ++t) rank += buf[t] < k + (t < p ? 1u : 0u);
    }
    dst[gbase + lo + rank] = k;
  }
  uint64_t qsum = 0;
  for (uint32_t qi = qlo + tid; qi < qhi; qi += C::kThreads) {
    const uint32_t q = qi == qlo + tid ? q_first : __ldg(q_sorted + qi);   // (the thread's first query was fetched before the sort)
    const uint32_t sb = sub_of(q, mask, sshift);
    const uint32_t lo = cur[kFront - 1 + sb], hi = cur[kFront + sb];
    uint32_t c = 0;
#pragma unroll 1
    for (uint32_t t = lo; t < hi; ++t) c += kStrict ? (buf[t] < q) : (buf[t] <= q);
    qsum += (uint64_t)gbase + lo + c;
  }
  return qsum;
}

template <class C, bool kSlots = false>
__global__ void __launch_bounds__(C::kThreads, C::kBlocksPerSm) bin_sort_search_kernel(BinSortArgs a) {
  if (kSlots && blockIdx.y) {
    const size_t o = (size_t)blockIdx.y * a.slot_words;
    a.pairs = reinterpret_cast<const uint2*>(reinterpret_cast<const uint32_t*>(a.pairs) + o);
    a.off += o; a.cross_cnt += o; a.cross_keys += o; a.cross_cnt_next += o; a.dst[0] += o; a.dst[1] += o;
    a.round_total += blockIdx.y; a.flag += blockIdx.y;
  }
  extern __shared__ __align__(16) uint8_t smem_raw[];
  uint32_t* s_ks = reinterpret_cast<uint32_t*>(smem_raw);          // [C::kCap] starts
  uint32_t* s_ke = s_ks + C::kCap;                                    // [C::kCap] ends (own + handed over)
  uint16_t* s_cur_s = reinterpret_cast<uint16_t*>(s_ke + C::kCap);    // [C::kCurLen] cursors of the starts
  uint16_t* s_cur_e = s_cur_s + C::kCurLen;                           // [C::kCurLen] cursors of the ends
  __shared__ uint32_t s_w[32], s_w2[32];
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const uint32_t shift = a.shift, mask = (1u << shift) - 1u;
  const uint32_t sshift = shift > (uint32_t)C::kSubBits ? shift - C::kSubBits : 0u;
  uint32_t* s_seg = reinterpret_cast<uint32_t*>(s_cur_e + C::kCurLen);   // [n_tiles + 1] per tile: lo | pos << 16
  const uint32_t runs = (a.n_tiles + C::kThreads - 1) / C::kThreads;    // tiles per thread (contiguous)
  const uint32_t t0 = min(a.n_tiles, (uint32_t)tid * runs), t1 = min(a.n_tiles, t0 + runs);
  const uint32_t gl = (uint32_t)tid & (a.group - 1u), gid = (uint32_t)tid >> a.group_log2;   // gather groups of a.group lanes
  const uint32_t n_groups = (uint32_t)C::kThreads >> a.group_log2;
  uint64_t qsum = 0;    // two's-complement: + ranks in B_S, - ranks in B_E
  // bins are handed out dynamically: the first one is the block's index, the rest come from a ticket
  // counter (spare word kMaxBins + 1 of this round's hand-over counts; zero on entry, reset for the
  // round after next by block 0 through the other parity's array)
  __shared__ uint32_t s_next;
  grid_dependency_wait();     // this round's placement has written pairs / off / hand-over lists
  if (blockIdx.x == 0 && tid == 0) a.cross_cnt_next[kMaxBins + 1] = 0;
  uint32_t d = blockIdx.x;
  while (d < a.n_bins) {
    if (tid == 0) s_next = gridDim.x + atomicAdd(const_cast<uint32_t*>(a.cross_cnt) + kMaxBins + 1, 1u);
    a.cross_cnt_next[d] = 0;   // (every thread writes the same zero: harmless, and no divergence)
    // column d (and d + 1) of the per-tile prefix table: one scattered read per tile here instead of one
    // scattered write per (tile, bin) in the placement kernel
    const uint32_t* __restrict__ col = a.off + d;
    // (loaded here, used after the scan: the latency overlaps the segment words')
    const uint32_t n_in = min(__ldg(a.cross_cnt + d), (uint32_t)kCrossCap);
    const uint32_t qlo0 = __ldg(a.qb[0] + d), qhi0 = __ldg(a.qb[0] + d + 1);
    const uint32_t qlo1 = __ldg(a.qb[1] + d), qhi1 = __ldg(a.qb[1] + d + 1);
    uint32_t len_sum = 0, lo_sum = 0;
    uint32_t seg0 = 0, seg1 = 0;                     // lo | len << 16 of this thread's first two tiles (usually all it has)
    for (uint32_t t = t0; t < t1; ++t) {
      const uint32_t sg = __ldg(col + (size_t)t * a.stride);
      len_sum += sg >> 16; lo_sum += sg & 0xffffu;
      if (t == t0) seg0 = sg; else if (t == t0 + 1u) seg1 = sg;
    }
    // each thread's first query of either kind (usually its only one): in flight during the gather and the sort
    const uint32_t qf0 = qlo0 + tid < qhi0 ? __ldg(a.q_sorted[0] + qlo0 + tid) : 0u;
    const uint32_t qf1 = qlo1 + tid < qhi1 ? __ldg(a.q_sorted[1] + qlo1 + tid) : 0u;
    // exclusive scan of len_sum (where this thread's pairs go) and block sum of lo_sum (keys in earlier bins)
    uint32_t incl = len_sum, ls = lo_sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(kFullMask, incl, o); if (lane >= o) incl += t; }
    ls = __reduce_add_sync(kFullMask, ls);
    __syncthreads();           // everyone is done with the previous bin's buffers, cursors, s_seg and s_w / s_w2
    if (lane == 31) { s_w[w] = incl; s_w2[w] = ls; }
    // clear both cursor arrays (they are adjacent)
    for (int i = tid; i < 2 * C::kCurLen / 8; i += C::kThreads) reinterpret_cast<uint4*>(s_cur_s)[i] = make_uint4(0, 0, 0, 0);
    __syncthreads();
    uint32_t x = lane < C::kThreads / 32 ? s_w[lane] : 0u;
    const uint32_t gbase = __reduce_add_sync(kFullMask, lane < C::kThreads / 32 ? s_w2[lane] : 0u);
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(kFullMask, x, o); if (lane >= o) x += t; }
    const uint32_t np = __shfl_sync(kFullMask, x, 31);                  // pairs in this bin
    uint32_t pos = incl - len_sum + (w ? __shfl_sync(kFullMask, x, (w + 31) & 31) : 0u);
    const uint32_t d_next = s_next;
    if (np + n_in + 4u > (uint32_t)C::kCap) {                              // block-uniform (4: room for the sentinels)
      if (tid == 0) atomicOr(a.flag, kFlagBinTooBig);
      d = d_next;
      __syncthreads();       // every thread has read s_next before thread 0 takes the next ticket at the loop top
      continue;
    }
    // where each tile's segment of this bin sits in the tile (lo) and goes in the bin's buffers (pos)
    for (uint32_t t = t0; t < t1; ++t) {
      const uint32_t sg = t == t0 ? seg0 : (t == t0 + 1u ? seg1 : __ldg(col + (size_t)t * a.stride));
      const uint32_t lo = sg & 0xffffu, len = sg >> 16;
      s_seg[t] = lo | (pos << 16);
      pos += len;
    }
    if (tid == 0) s_seg[a.n_tiles] = np << 16;
    __syncthreads();
    // gather: a group of lanes per segment, so that one instruction touches few cache lines
    // (a scattered access costs the L1 one cycle per line); starts and ends go to separate arrays
    for (uint32_t t = gid; t < a.n_tiles; t += n_groups) {
      const uint32_t seg = s_seg[t], p0 = seg >> 16, len = (s_seg[t + 1] >> 16) - p0;
      const uint2* src = a.pairs + (size_t)t * a.tile + (seg & 0xffffu);
      for (uint32_t j = gl; j < len; j += a.group) {
        msd::cp_async4(s_ks + p0 + j, &src[j].x);
        msd::cp_async4(s_ke + p0 + j, &src[j].y);
      }
    }
    if ((uint32_t)tid < n_in) msd::cp_async4(s_ke + np + tid, a.cross_keys + (size_t)d * kCrossCap + tid);
    msd::cp_async_wait_all();
    __syncthreads();
    // Algorithm 2's Sort(B_S), Sort(B_E) for this bin: count, scan, scatter
    const uint32_t me = np + n_in;    // ends held: own ones (some belong to the next bin) + handed over
    {
      uint32_t* cs = reinterpret_cast<uint32_t*>(s_cur_s);
      uint32_t* ce = reinterpret_cast<uint32_t*>(s_cur_e);
#pragma unroll 2
      for (uint32_t i = tid; i < me; i += C::kThreads) {
        if (i < np) count_key(cs, sub_of(s_ks[i], mask, sshift));
        const uint32_t e = s_ke[i];
        if ((e >> shift) == d) count_key(ce, sub_of(e, mask, sshift));
      }
    }
    __syncthreads();
    uint32_t total[2];
    scan_cursors<C>(s_cur_s, s_cur_e, s_w, total);                         // barriers inside
    // starts: all np keys belong to bin d; the bin begins at gbase in B_S
    // (both scatters first: the two long write-out phases then follow each other with no barrier between them)
    scatter_in_place<C, false, false>(s_ks, np, d, shift, mask, sshift, s_cur_s, np);   // (the barriers of the next call cover it)
    scatter_in_place<C, true>(s_ke, me, d, shift, mask, sshift, s_cur_e, total[1]);
    qsum += write_and_rank<C, false>(s_ks, np, mask, sshift, s_cur_s, gbase, a.dst[0], a.q_sorted[0], qlo0, qhi0, qf0);
    // ends: n_in ends of earlier pairs lie in this bin, so it begins at gbase - n_in in B_E
    qsum -= write_and_rank<C, true>(s_ke, total[1], mask, sshift, s_cur_e, gbase - n_in, a.dst[1], a.q_sorted[1], qlo1, qhi1, qf1);
    d = d_next;
  }
  if (blockIdx.x == 0 && tid == 0) {
    // queries beyond the last bin count every key
    qsum += (uint64_t)(a.n_q - __ldg(a.qb[0] + a.n_bins)) * a.n;
    qsum -= (uint64_t)(a.n_q - __ldg(a.qb[1] + a.n_bins)) * a.n;
  }
  __shared__ uint64_t s_red[C::kThreads / 32];
  __syncthreads();
  qsum = warp_sum_u64(qsum);
  if (lane == 0) s_red[w] = qsum;
  __syncthreads();
  if (w == 0) {
    uint64_t t = lane < C::kThreads / 32 ? s_red[lane] : 0;
    t = warp_sum_u64(t);
    if (lane == 0 && t != 0) atomicAdd(a.round_total, (unsigned long long)t);
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

}  // namespace mct
}  // namespace bits
