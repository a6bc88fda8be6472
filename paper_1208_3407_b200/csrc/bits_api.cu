// bits_api.cu -- the C ABI of libbits_b200 (include/bits.h): argument checks, workspace carving
// and kernel launches.  Every step of the path (place, sort, search, reduce) runs in the kernels
// of this directory; there is no CPU fallback.
#include <math.h>
#include <string.h>

#include <algorithm>
#include <vector>

#include "common.cuh"
#include "philox_place.cuh"
#include "place_kernels.cuh"
#include "radix_sort.cuh"
#include "msd_sort.cuh"
#include "mc_tile.cuh"
#include "mc_small.cuh"
#include "search.cuh"
#include "enumerate.cuh"
#include "screen.cuh"
#include "binned_count.cuh"

namespace bits {

std::atomic<unsigned long long> g_launches{0};

struct Options {
  int64_t sort_msd = 1;            // 1 = MSD bucket sort with the LSD sort as device-side fallback, 0 = LSD sort only
  int64_t mc_fused = 1;            // PERMUTE_B rounds: 1 = place+tile sort / bin sort+search (mc_tile.cuh)
  int64_t mc_sorted_queries = 1;   // PERMUTE_B rounds: 1 = search with A's keys sorted once, 0 = bucket index per round
  int64_t place_fused_hist = 1;    // PERMUTE_B rounds: 1 = histogram inside the placement kernel
  int64_t search_variant = 0;      // count kernel: 0 bucket index, 1 plain binary search (the paper's), 2 top 11 levels in shared memory
  int64_t mc_symmetric = 0;        // PERMUTE_B rounds: 1 = sort-free variant (fresh B intervals counted against the once-sorted A)
  int64_t mc_pdl = 1;              // PERMUTE_B fused rounds: launch the two kernels with programmatic stream serialization
  int64_t mc_force_redo = 0;       // PERMUTE_B fused rounds: n > 0 redoes every n-th round by the general path as if its flag were raised (tests)
  int64_t mc_tile_variant = 2;     // PERMUTE_B fused rounds: shape of place_tile_kernel (0: 2 x 512 threads, 1: 1 x 1024, 2: 1 x 1024 with longer tiles)
  int64_t mc_bin_variant = 0;      // PERMUTE_B fused rounds: shape of the per-bin sort (0 wide, 1 narrow, 2 small blocks)
  int64_t mc_gather_group = -1;    // PERMUTE_B fused rounds: log2 of the lanes per gathered segment (-1 = from the mean segment length)
  int64_t msd_pack = 7168;         // MSD sort plan: 0 = buckets by the prefix / target rule, n = consecutive bins packed greedily up to n keys (measured on config 4: 0 -> 146 us, 8192 -> 134, 7168 -> 124 for the bucket sort)
  int64_t msd_scatter_shape = 0;   // MSD scatter pass: 0 = one 1,024-thread block per SM and 16,384-key tiles, 1 = two 512-thread blocks and 8,192-key tiles
  int64_t count_binned = -1;       // count path: 1 = queries binned by B's buckets and searched out of shared memory (binned_count.cuh), 0 = bucket index + count_kernel, -1 = by size
  int64_t mc_a_rounds_per_block = 4;   // PERMUTE_A rounds (and the sort-free variant): rounds a block serves for its query tile
  int64_t mc_batch = 1;            // PERMUTE_B fused rounds of small sets: 1 = several rounds per launch pair (gridDim.y), 0 = one
  int64_t mc_small = 1;            // PERMUTE_B rounds of a set that fits one block's shared memory: 1 = one block per round (mc_small.cuh) when the rounds fill the GPU, 2 = always, 0 = never
  int64_t mc_shift_bias = 0;       // PERMUTE_B fused rounds: added to the bin width (log2) the host picked; > 0 overflows bins on purpose (tests)
  int64_t grid_mult = 8;           // grid-stride kernels launch min(needed, 148 * grid_mult) blocks
};
// Options and the per-kernel event timers belong to the calling host thread (bits.h, "Threads"): two threads
// driving the library do not see each other's knobs.
static thread_local Options g_opt;

constexpr int kSMs = 148;
// Largest interval set an entry point accepts (bits.h, "Sizes").  Element indices inside the kernels are 32-bit, and some
// are scaled before use (four positions per thread: t << 2; tile index x tile size; counts padded by kPad): below 2^28
// every such product stays under 2^31.  The largest sets the GPU tests run are 2.5e7 intervals.
constexpr uint64_t kMaxIntervals = 1ull << 28;
constexpr size_t kMaxSmemPerBlock = 232448 - 2048;   // 227 KB opt-in limit of shared memory per block on sm_100, less room for static shared memory

// ---------------------------------------------------------------------------------------------
// Optional per-kernel-class timing with CUDA events on the launching stream (bits_set_option
// "profile" = 1; read with bits_profile_read).  Used by bench.py for the roofline figures.
enum { kClsPlace = 0, kClsHist, kClsSortPass, kClsIndex, kClsCount, kClsSortedQuery, kClsMcA, kClsOther,
       kClsPlan, kClsScatter, kClsBucketSort, kClsPlaceScatter, kClsBucketSortSearch, kClsQueryScatter, kClsBucketSearch, kNumCls };
struct Profiler {
  bool on = false;
  std::vector<cudaEvent_t> ev;     // pairs: 2k = start, 2k+1 = stop
  std::vector<int> cls;            // class of pair k
  size_t used = 0;                 // pairs in flight
  double ms[kNumCls] = {0};
  uint64_t launches[kNumCls] = {0};
  void collect() {
    for (size_t k = 0; k < used; ++k) {
      float t = 0.f;
      if (cudaEventSynchronize(ev[2 * k + 1]) == cudaSuccess &&
          cudaEventElapsedTime(&t, ev[2 * k], ev[2 * k + 1]) == cudaSuccess) {
        ms[cls[k]] += t;
        ++launches[cls[k]];
      }
    }
    (void)cudaGetLastError();
    used = 0;
  }
  void reset() { collect(); for (int i = 0; i < kNumCls; ++i) { ms[i] = 0; launches[i] = 0; } }
};
static thread_local Profiler g_prof;

struct ProfScope {
  cudaStream_t st;
  long k = -1;
  ProfScope(int c, cudaStream_t s) : st(s) {
    if (!g_prof.on) return;
    if (g_prof.used >= (1u << 16)) g_prof.collect();
    if (g_prof.ev.size() < 2 * (g_prof.used + 1)) {
      cudaEvent_t a, b;
      if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) { (void)cudaGetLastError(); return; }
      g_prof.ev.push_back(a); g_prof.ev.push_back(b); g_prof.cls.push_back(c);
    }
    k = (long)g_prof.used++;
    g_prof.cls[k] = c;
    cudaEventRecord(g_prof.ev[2 * k], st);
  }
  ~ProfScope() { if (k >= 0) cudaEventRecord(g_prof.ev[2 * k + 1], st); }
};

// Kernels that follow another kernel of the same call are launched with programmatic stream serialization
// (unless the per-kernel event timers are on, or option mc_pdl = 0): each may be scheduled while its predecessor
// drains, and waits on the device (griddepcontrol.wait, its first statement) before it touches global memory.
// Only kernels that carry that wait may be launched through here.
template <typename... KArgs, typename... Args>
static void launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = (g_opt.mc_pdl != 0 && !g_prof.on) ? 1 : 0;
  cfg.attrs = attr; cfg.numAttrs = 1;
  (void)cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}


// ---------------------------------------------------------------------------------------------
// Workspace: a bump allocator that is run twice -- once with base == nullptr to size, once to carve.
struct Carver {
  char* base;
  size_t used = 0;
  explicit Carver(void* b) : base(static_cast<char*>(b)) {}
  template <typename T>
  T* take(uint64_t count) {
    used = align_up(used, 256);
    T* p = base ? reinterpret_cast<T*>(base + used) : nullptr;
    used += count * sizeof(T);
    return p;
  }
};

// Buffers for sorting a pair of equally long arrays (starts and ends), plus their bucket indices.
struct SortCtx {
  uint32_t n = 0, n_tiles = 0;
  uint32_t* buf[2][2] = {{nullptr, nullptr}, {nullptr, nullptr}};   // [array][0 = result "Y", 1 = temp "X"]
  uint32_t* hist[2][2] = {{nullptr, nullptr}, {nullptr, nullptr}};  // [parity][array] -> uint32[4][256]
  uint64_t* status[2] = {nullptr, nullptr};
  uint32_t* ticket = nullptr;                                       // uint32[2]
  uint32_t* idx[2] = {nullptr, nullptr};
  uint32_t shift = 31;
  // MSD bucket sort (msd_sort.cuh)
  uint32_t* bin_hist[2] = {nullptr, nullptr};       // uint32[kBins]
  uint32_t* bin_cursor[2] = {nullptr, nullptr};     // uint32[kBins]
  uint32_t* bucket_start[2] = {nullptr, nullptr};   // uint32[kBins + 1]
  uint32_t* n_buckets = nullptr;                    // uint32[2]
  uint32_t* msd_flag = nullptr;                     // uint32[2]
  uint16_t* bucket_of_bin[2] = {nullptr, nullptr};  // uint16[kBins] the bucket that holds each bin
  uint32_t* bucket_cursor[2] = {nullptr, nullptr};  // uint32[kBins] reservation cursors of the scatter pass
  uint32_t* bucket_lo = nullptr;                    // uint32[kBins + 1] first bin of each bucket of array 0
  size_t zero_bytes = 0;                            // from hist[0][0]: digit histograms, tickets, bin histograms, bucket counts, flags, status words
  void carve(Carver& c, uint64_t n_keys, bool with_index) {
    n = (uint32_t)n_keys;
    n_tiles = rs::num_tiles(n_keys);
    const uint64_t padded = align_up(n_keys + kPad, 64);
    for (int a = 0; a < 2; ++a)
      for (int b = 0; b < 2; ++b) buf[a][b] = c.take<uint32_t>(padded);
    // everything a call clears before its first sort sits in one stretch, so that one memset does it
    const size_t z0 = align_up(c.used, 256);
    for (int p = 0; p < 2; ++p)
      for (int a = 0; a < 2; ++a) hist[p][a] = c.take<uint32_t>(rs::kPasses * rs::kRadix);
    ticket = c.take<uint32_t>(64);
    for (int a = 0; a < 2; ++a) bin_hist[a] = c.take<uint32_t>(msd::kBins);
    n_buckets = c.take<uint32_t>(64);
    msd_flag = n_buckets ? n_buckets + 8 : nullptr;
    for (int a = 0; a < 2; ++a) status[a] = c.take<uint64_t>((uint64_t)n_tiles * rs::kRadix);
    zero_bytes = c.used - z0;
    for (int a = 0; a < 2; ++a) {
      bin_cursor[a] = c.take<uint32_t>(msd::kBins);
      bucket_start[a] = c.take<uint32_t>(msd::kBins + 4);
    }
    for (int a = 0; a < 2; ++a) {
      bucket_of_bin[a] = c.take<uint16_t>(msd::kBins);
      bucket_cursor[a] = c.take<uint32_t>(msd::kBins);
    }
    bucket_lo = c.take<uint32_t>(msd::kBins + 4);
    shift = index_shift_for(n_keys);
    if (with_index)
      for (int a = 0; a < 2; ++a) idx[a] = c.take<uint32_t>(index_entries(shift));
  }
};

struct Small {            // small device scalars
  uint32_t* max_span;     // [1]
  uint32_t* bad;          // [1]
  unsigned long long* span_sum;   // [1]
  uint32_t* chrom;        // [n_chrom + 1]
  uint16_t* lut;          // [kLutSize] position -> chromosome look-up table
  void carve(Carver& c, uint32_t n_chrom) {
    max_span = c.take<uint32_t>(64);
    bad = max_span ? max_span + 1 : nullptr;
    span_sum = max_span ? reinterpret_cast<unsigned long long*>(max_span + 2) : nullptr;
    chrom = c.take<uint32_t>((uint64_t)n_chrom + 1);
    lut = c.take<uint16_t>(kLutSize);
  }
};

struct Layout {
  Small small;
  SortCtx b;              // the searched set
  SortCtx q;              // PERMUTE_B: A's ends (array 0) and starts (array 1), sorted once
  uint32_t* spans = nullptr;
  // PERMUTE_B fused rounds (mc_tile.cuh); null when the set is too large for that path
  uint2* pairs = nullptr;                // [n_b] tile-sorted (start, end) pairs
  uint32_t* tile_off = nullptr;          // [n_tiles * tile_stride] per tile and bin: start of the bin's pairs in the tile | count << 16
  uint32_t tile_stride = 0;
  uint32_t* cross_cnt[2] = {nullptr, nullptr};   // [kMaxBins + 1] by round parity
  uint32_t* cross_keys = nullptr;        // [kMaxBins * kCrossCap]
  uint32_t* qb[2] = {nullptr, nullptr};
  uint32_t* round_flags = nullptr;       // uint32[kFlagChunk]
  // several fused rounds per launch pair (small re-placed sets): `batch_slots` copies of the per-round buffers,
  // slot_words 32-bit words apart; null when the set is too large for that to pay
  uint32_t batch_slots = 1, batch_rows = 0;
  size_t slot_words = 0;
  uint2* bt_pairs = nullptr;
  uint32_t* bt_off = nullptr;
  uint32_t* bt_cross_cnt[2] = {nullptr, nullptr};
  uint32_t* bt_cross_keys = nullptr;
  uint32_t* bt_dst[2] = {nullptr, nullptr};
  // count path with binned queries (binned_count.cuh)
  qb::Lists ql = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};   // (eight pointers)
  // enumeration (enumerate.cuh)
  uint32_t* e_counts = nullptr;                  // [n_a]
  unsigned long long* e_offsets = nullptr;       // [n_a]
  unsigned long long* e_tile_sums = nullptr;     // [ceil(n_a / kScanTile) + 1]
  uint32_t* e_tie = nullptr;                     // [n_b + 1]
  uint32_t* e_end_by_start = nullptr;            // [n_b]
  uint32_t* e_idx_by_start = nullptr;            // [n_b]
  uint32_t* e_max[3] = {nullptr, nullptr, nullptr};   // largest end per run of 32 / 1,024 / 32,768 positions of e_end_by_start
  size_t bytes = 0;
};
constexpr uint32_t kFlagChunk = 4096;    // fused rounds are checked for raised flags in chunks of this many
constexpr uint64_t kFusedMaxKeys = 24u << 20;   // beyond this the bins of the fused path cannot hold the set
constexpr uint64_t kBatchMaxKeys = 4u << 20;    // re-placed sets up to this size run several rounds per launch pair
constexpr uint32_t kBatchMaxSlots = 32, kBatchBins = 512;
static inline uint32_t batch_slots_for(uint64_t n) {
  if (n <= (uint64_t)mcs::kMaxKeys || n > kBatchMaxKeys) return 1;     // (smaller sets: one block per round, mc_small.cuh)
  const uint64_t s = (16ull << 20) / n;
  return (uint32_t)(s < 2 ? 2 : (s > kBatchMaxSlots ? kBatchMaxSlots : s));
}
// Tiles are balanced: every block of place_tile_kernel gets the same number of equally sized tiles.
static inline uint32_t tile_size_for(uint64_t n, uint32_t blocks, uint32_t max_tile) {
  const uint64_t per_block = ceil_div(n, (uint64_t)blocks * max_tile);
  uint64_t tile = align_up(ceil_div(n, (uint64_t)blocks * (per_block ? per_block : 1)), 4);
  if (tile > (uint64_t)max_tile) tile = max_tile;
  if (tile < 4) tile = 4;
  return (uint32_t)tile;
}
template <class C>
static inline uint32_t tile_size_cfg(uint64_t n) { return tile_size_for(n, (uint32_t)C::kBlocksPerSm * 148u, (uint32_t)C::kTile); }
// the workspace is sized for the shape with the most tiles, whatever shape a call ends up using
static inline uint32_t max_tiles_for(uint64_t n) { return (uint32_t)ceil_div(n, tile_size_cfg<mct::TileCfg2x512>(n)); }

// The count path bins the queries by B's buckets (binned_count.cuh) when both sets are large, B is not already sorted
// and the MSD sort is in use; knob count_binned forces it on (> 0) or off (0).  The same rule sizes the workspace: the
// query lists (8-12 bytes per query) are carved only for calls that can take that path.
static inline bool count_can_bin(uint32_t flags) { return g_opt.sort_msd != 0 && !(flags & BITS_B_SORTED); }
static inline bool count_bins_queries(uint64_t n_a, uint64_t n_b, uint32_t flags) {
  return count_can_bin(flags) && (g_opt.count_binned > 0 || (g_opt.count_binned < 0 && n_a >= (1u << 20) && n_b >= (3u << 20)));
}

static Layout make_layout(void* ws, int fn, uint64_t n_a, uint64_t n_b, uint32_t n_chrom, int which, uint32_t flags = 0) {
  Layout L;
  Carver c(ws);
  L.small.carve(c, n_chrom);
  switch (fn) {
    case BITS_FN_COUNT:
    case BITS_FN_COUNT_PER_INTERVAL:
      L.b.carve(c, n_b, true);
      if (!count_bins_queries(n_a, n_b, flags)) break;     // (L.ql stays null: the index path needs no query lists)
      L.ql.q_end = c.take<uint32_t>(n_a + 4);
      L.ql.q_start = c.take<uint32_t>(n_a + 4);
      L.ql.q_idx = c.take<uint32_t>(fn == BITS_FN_COUNT_PER_INTERVAL ? n_a + 4 : 4);
      L.ql.hist = c.take<uint32_t>(msd::kBins + 64);
      L.ql.item_bucket = c.take<uint16_t>(ceil_div(n_a, (uint64_t)qb::kChunk) + msd::kBins + 8);
      L.ql.off = c.take<uint32_t>(msd::kBins + 4);
      L.ql.cursor = c.take<uint32_t>(msd::kBins + 4);
      L.ql.item_off = c.take<uint32_t>(msd::kBins + 4);
      break;
    case BITS_FN_MC_ROUNDS:
      L.b.carve(c, n_b, true);
      if (which == BITS_PERMUTE_A) {
        L.spans = c.take<uint32_t>(align_up(n_a, 4) + 4);
      } else {
        L.spans = c.take<uint32_t>(align_up(n_b, 4) + 4);
        L.q.carve(c, n_a, true);
        if (n_b <= kFusedMaxKeys) {
          const uint32_t n_tiles = max_tiles_for(n_b);
          L.tile_stride = (uint32_t)mct::kMaxBins;       // entries per tile row
          L.pairs = c.take<uint2>(align_up(n_b, 4) + 4);
          L.tile_off = c.take<uint32_t>((uint64_t)(n_tiles + 1) * L.tile_stride);
          for (int a = 0; a < 2; ++a) {
            L.cross_cnt[a] = c.take<uint32_t>(mct::kMaxBins + 4);
            L.qb[a] = c.take<uint32_t>(mct::kMaxBins + 4);
          }
          L.cross_keys = c.take<uint32_t>((uint64_t)mct::kMaxBins * mct::kCrossCap);
          L.round_flags = c.take<uint32_t>(kFlagChunk);
          L.batch_slots = batch_slots_for(n_b);
          if (L.batch_slots > 1) {
            // one slot, carved relative to its own start; every slot has the same shape
            L.batch_rows = (uint32_t)ceil_div(n_b, 4096) + 2;
            size_t used = 0;
            auto place = [&](uint64_t bytes) { used = align_up(used, 256); const size_t o = used; used += bytes; return o; };
            const size_t o_pairs = place(sizeof(uint2) * (align_up(n_b, 4) + 4));
            const size_t o_off = place(sizeof(uint32_t) * (uint64_t)L.batch_rows * L.tile_stride);
            size_t o_cc[2], o_dst[2];
            for (int a = 0; a < 2; ++a) o_cc[a] = place(sizeof(uint32_t) * (mct::kMaxBins + 4));
            const size_t o_ck = place(sizeof(uint32_t) * (uint64_t)kBatchBins * mct::kCrossCap);
            for (int a = 0; a < 2; ++a) o_dst[a] = place(sizeof(uint32_t) * align_up(n_b + kPad, 64));
            const size_t slot_bytes = align_up(used, 256);
            L.slot_words = slot_bytes / sizeof(uint32_t);
            char* base = c.take<char>((uint64_t)slot_bytes * L.batch_slots);
            if (base) {
              L.bt_pairs = reinterpret_cast<uint2*>(base + o_pairs);
              L.bt_off = reinterpret_cast<uint32_t*>(base + o_off);
              for (int a = 0; a < 2; ++a) {
                L.bt_cross_cnt[a] = reinterpret_cast<uint32_t*>(base + o_cc[a]);
                L.bt_dst[a] = reinterpret_cast<uint32_t*>(base + o_dst[a]);
              }
              L.bt_cross_keys = reinterpret_cast<uint32_t*>(base + o_ck);
            }
          }
        }
      }
      break;
    case BITS_FN_ENUMERATE:
      L.b.carve(c, n_b, true);
      L.e_counts = c.take<uint32_t>(n_a + 4);
      L.e_offsets = c.take<unsigned long long>(n_a + 4);
      L.e_tile_sums = c.take<unsigned long long>(ceil_div(n_a, (uint64_t)enu::kScanTile) + 4);
      L.e_tie = c.take<uint32_t>(n_b + 4);
      L.e_end_by_start = c.take<uint32_t>(n_b + 4);
      L.e_idx_by_start = c.take<uint32_t>(n_b + 4);
      L.e_max[0] = c.take<uint32_t>((n_b >> enu::kSkip1) + 4);
      L.e_max[1] = c.take<uint32_t>((n_b >> enu::kSkip2) + 4);
      L.e_max[2] = c.take<uint32_t>((n_b >> enu::kSkip3) + 4);
      break;
    case BITS_FN_PLACE:
      break;
    case BITS_FN_SORT:
      L.b.carve(c, n_b, false);
      break;
    default:
      break;
  }
  L.bytes = align_up(c.used, 256);
  return L;
}

static inline bool ws_ok(const void* ws, size_t have, size_t need) {
  return ws != nullptr && ((uintptr_t)ws & 255) == 0 && have >= need;
}

static inline int grid_for(uint64_t threads_needed, int block) {
  const uint64_t blocks = ceil_div(threads_needed, block);
  const uint64_t cap = (uint64_t)kSMs * (uint64_t)g_opt.grid_mult;
  return (int)(blocks < cap ? (blocks ? blocks : 1) : cap);
}

// ---------------------------------------------------------------------------------------------
// Sort of a pair of arrays: src -> X -> Y -> X -> Y, so the result lands in Y.  `hist` must
// already hold the four digit histograms of both arrays.  `epoch` is advanced per pass.
struct SortPlan {
  const uint32_t* src[2];
  uint32_t* x[2];
  uint32_t* y[2];
  const uint32_t* hist[2];
  uint64_t* status[2];
  uint32_t* ticket;
  uint32_t n, n_tiles;
  int n_arrays;
  const uint32_t* run_if = nullptr;   // device uint32[2]: passes run only if one of them is non-zero (null: always)
};

static int launch_sort_passes(const SortPlan& p, uint32_t* epoch, cudaStream_t st) {
  for (int pass = 0; pass < rs::kPasses; ++pass) {
    rs::SortPassArgs a;
    for (int k = 0; k < 2; ++k) {
      const int kk = k < p.n_arrays ? k : 0;
      a.arr[k].src = pass == 0 ? p.src[kk] : ((pass & 1) ? p.x[kk] : p.y[kk]);
      a.arr[k].dst = (pass & 1) ? p.y[kk] : p.x[kk];
      a.arr[k].hist = p.hist[kk] + pass * rs::kRadix;
      a.arr[k].status = p.status[kk];
      a.arr[k].ticket = p.ticket + 4 * k + pass;
    }
    a.n = p.n; a.n_tiles = p.n_tiles; a.shift = 8 * pass; a.epoch = (*epoch)++;
    a.run_if[0] = p.run_if; a.run_if[1] = p.run_if ? p.run_if + (p.n_arrays > 1 ? 1 : 0) : nullptr;
    ProfScope prof(kClsSortPass, st);
    launch_pdl(rs::onesweep_pass_kernel, dim3(p.n_tiles < 2u * kSMs ? p.n_tiles : 2u * kSMs, p.n_arrays), rs::kThreads, 0, st, a);
    BITS_LAUNCH_CHECK();
  }
  return BITS_OK;
}

static int launch_histogram(const uint32_t* k0, const uint32_t* k1, uint32_t* h0, uint32_t* h1, uint32_t n,
                            int n_arrays, cudaStream_t st, const uint32_t* run_if = nullptr) {
  rs::HistArgs h;
  h.keys[0] = k0; h.keys[1] = n_arrays > 1 ? k1 : k0;
  h.hist[0] = h0; h.hist[1] = n_arrays > 1 ? h1 : h0;
  h.n = n;
  h.run_if[0] = run_if; h.run_if[1] = run_if ? run_if + (n_arrays > 1 ? 1 : 0) : nullptr;
  ProfScope prof(kClsHist, st);
  // (a gated launch gets the same grid as an ungated one: when the gate opens -- the MSD sort fell back on a
  // clustered set -- this is the whole job, and retiring the blocks of a closed gate costs well under a microsecond)
  const int grid = grid_for(ceil_div(n, 4), 512);
  launch_pdl(rs::histogram_kernel, dim3(grid, n_arrays), 512, 0, st, h);
  BITS_LAUNCH_CHECK();
  return BITS_OK;
}

// Clear the sort bookkeeping of a context (once per library call); epochs restart at 1.
static int reset_sort_ctx(const SortCtx& c, cudaStream_t st) {
  BITS_CUDA_TRY(cudaMemsetAsync(c.hist[0][0], 0, c.zero_bytes, st));   // one stretch of the workspace (SortCtx::carve)
  return BITS_OK;
}

static SortPlan plan_for(const SortCtx& c, const uint32_t* src0, const uint32_t* src1, int parity) {
  SortPlan p;
  p.src[0] = src0; p.src[1] = src1;
  for (int a = 0; a < 2; ++a) {
    p.x[a] = c.buf[a][1]; p.y[a] = c.buf[a][0];
    p.hist[a] = c.hist[parity][a];
    p.status[a] = c.status[a];
  }
  p.ticket = c.ticket;
  p.n = c.n; p.n_tiles = c.n_tiles; p.n_arrays = 2;
  return p;
}

// Attribute setup for the kernels that use more than 48 KB of shared memory: once per DEVICE
// (cudaFuncSetAttribute applies to the current device only).
static int msd_configure() {
  constexpr int kMaxDevices = 64;
  static std::atomic<int> done_on[kMaxDevices];      // zero-initialised
  int device = 0;
  BITS_CUDA_TRY(cudaGetDevice(&device));
  const bool tracked = device >= 0 && device < kMaxDevices;
  if (!tracked || done_on[device].load(std::memory_order_acquire) == 0) {
    cudaError_t e1 = cudaFuncSetAttribute(msd::scatter_kernel<msd::ScatterCfg1x1024>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)msd::ScatterCfg1x1024::kSmem);
    if (e1 == cudaSuccess)
      e1 = cudaFuncSetAttribute(msd::scatter_kernel<msd::ScatterCfg2x512>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)msd::ScatterCfg2x512::kSmem);
    const cudaError_t e2 = cudaFuncSetAttribute(msd::bucket_sort_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)msd::kBkSmem);
    cudaError_t e3 = cudaFuncSetAttribute(mct::bin_sort_search_kernel<mct::BinCfgWide>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)mct::BinCfgWide::smem_bytes(mct::kMaxTiles));
    // (the several-rounds-per-launch instantiations)
    if (e3 == cudaSuccess) e3 = cudaFuncSetAttribute(mct::bin_sort_search_kernel<mct::BinCfgWide, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)mct::BinCfgWide::smem_bytes(mct::kMaxTiles));
    if (e3 == cudaSuccess) e3 = cudaFuncSetAttribute(mct::bin_sort_search_kernel<mct::BinCfgNarrow, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)mct::BinCfgNarrow::smem_bytes(mct::kMaxTiles));
    if (e3 == cudaSuccess) e3 = cudaFuncSetAttribute(mct::bin_sort_search_kernel<mct::BinCfgSmall, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)mct::BinCfgSmall::smem_bytes(mct::kMaxTiles));
    if (e3 == cudaSuccess) e3 = cudaFuncSetAttribute(mct::bin_sort_search_kernel<mct::BinCfgHuge, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                     (int)(mct::BinCfgHuge::smem_bytes(mct::kMaxTiles) < kMaxSmemPerBlock ? mct::BinCfgHuge::smem_bytes(mct::kMaxTiles) : kMaxSmemPerBlock));
    if (e3 == cudaSuccess)
      e3 = cudaFuncSetAttribute(mct::bin_sort_search_kernel<mct::BinCfgNarrow>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)mct::BinCfgNarrow::smem_bytes(mct::kMaxTiles));
    if (e3 == cudaSuccess)
      e3 = cudaFuncSetAttribute(mct::bin_sort_search_kernel<mct::BinCfgHuge>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)(mct::BinCfgHuge::smem_bytes(mct::kMaxTiles) < kMaxSmemPerBlock ? mct::BinCfgHuge::smem_bytes(mct::kMaxTiles) : kMaxSmemPerBlock));
    if (e3 == cudaSuccess)
      e3 = cudaFuncSetAttribute(mct::bin_sort_search_kernel<mct::BinCfgSmall>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)mct::BinCfgSmall::smem_bytes(mct::kMaxTiles));
    cudaError_t e4 = cudaFuncSetAttribute(mct::place_tile_kernel<mct::TileCfg2x512>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)mct::TileCfg2x512::kSmem);
    if (e4 == cudaSuccess) e4 = cudaFuncSetAttribute(mct::place_tile_kernel<mct::TileCfg2x512, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)mct::TileCfg2x512::kSmem);
    if (e4 == cudaSuccess) e4 = cudaFuncSetAttribute(mct::place_tile_kernel<mct::TileCfg1x1024, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)mct::TileCfg1x1024::kSmem);
    if (e4 == cudaSuccess) e4 = cudaFuncSetAttribute(mct::place_tile_kernel<mct::TileCfg1x1024L, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)mct::TileCfg1x1024L::kSmem);
    if (e4 == cudaSuccess)
      e4 = cudaFuncSetAttribute(mct::place_tile_kernel<mct::TileCfg1x1024>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)mct::TileCfg1x1024::kSmem);
    if (e4 == cudaSuccess)
      e4 = cudaFuncSetAttribute(mct::place_tile_kernel<mct::TileCfg1x1024L>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)mct::TileCfg1x1024L::kSmem);
    if (e4 == cudaSuccess)
      e4 = cudaFuncSetAttribute(mcs::mc_small_b_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)mcs::kSmem);
    if (e1 != cudaSuccess || e2 != cudaSuccess || e3 != cudaSuccess || e4 != cudaSuccess) { (void)cudaGetLastError(); return BITS_ERR_CUDA; }
    if (tracked) done_on[device].store(1, std::memory_order_release);
  }
  return BITS_OK;
}

// Sort n_arrays (1 or 2) arrays of c.n keys: src -> ... -> y (c.buf[a][0] unless y_override).
// MSD bucket sort (plan -> scatter -> bucket sort) with the LSD sort as device-side fallback.
// bin_hist_ready: c.bin_hist already holds the top-bits histogram of the sources (made by the
// placement kernel).  The stage is complete once the stream reaches the end of what is enqueued.
// `queries` (optional): a query set to be planned into the order of array 0's buckets in the same launches
// (binned_count.cuh): its ends are histogrammed beside the keys, its plan is made by the block that plans array 0.
struct QueryBinning {
  const uint32_t* a_end;
  uint32_t n_a;
  msd::QueryPlan plan;
};
static int sort_arrays(const SortCtx& c, const uint32_t* src0, const uint32_t* src1, int n_arrays, uint32_t* y_override,
                       bool bin_hist_ready, uint32_t* epoch, cudaStream_t st, const QueryBinning* queries = nullptr) {
  SortPlan p = plan_for(c, src0, n_arrays > 1 ? src1 : src0, 0);
  p.n_arrays = n_arrays;
  if (y_override) p.y[0] = y_override;
  if (!g_opt.sort_msd) {
    BITS_CUDA_TRY(cudaMemsetAsync(c.hist[0][0], 0, sizeof(uint32_t) * rs::kPasses * rs::kRadix, st));
    if (n_arrays > 1) BITS_CUDA_TRY(cudaMemsetAsync(c.hist[0][1], 0, sizeof(uint32_t) * rs::kPasses * rs::kRadix, st));
    BITS_CUDA_TRY(cudaMemsetAsync(c.ticket, 0, sizeof(uint32_t) * 8, st));
    BITS_TRY(launch_histogram(src0, src1, c.hist[0][0], c.hist[0][1], c.n, n_arrays, st));
    return launch_sort_passes(p, epoch, st);
  }
  BITS_TRY(msd_configure());
  if (!bin_hist_ready) {
    msd::BinHistArgs h;
    h.keys[0] = src0; h.keys[1] = n_arrays > 1 ? src1 : src0;
    h.hist[0] = c.bin_hist[0]; h.hist[1] = c.bin_hist[1];
    h.n[0] = h.n[1] = c.n;
    h.keys[2] = queries ? queries->a_end : src0; h.hist[2] = queries ? queries->plan.bin_hist : c.bin_hist[0]; h.n[2] = queries ? queries->n_a : 0u;
    ProfScope prof(kClsHist, st);
    // (every block ends with up to 4,096 global reductions: a few resident blocks per SM, not one per 2,048 keys)
    const uint32_t n_big = queries && queries->n_a > c.n ? queries->n_a : c.n;
    const int hb = grid_for(ceil_div(n_big, 4), 512);
    launch_pdl(msd::bin_hist_kernel, dim3(hb < 2 * kSMs ? hb : 2 * kSMs, queries && n_arrays == 2 ? 3 : n_arrays), 512, 0, st, h);
    BITS_LAUNCH_CHECK();
  }
  {
    msd::PlanArgs pa;
    if (queries && n_arrays == 2 && !bin_hist_ready) pa.q = queries->plan; else pa.q.bin_hist = nullptr;
    for (int a = 0; a < 2; ++a) {
      pa.p[a].hist = c.bin_hist[a]; pa.p[a].bin_cursor = c.bin_cursor[a]; pa.p[a].bucket_start = c.bucket_start[a];
      pa.p[a].n_buckets = c.n_buckets + a; pa.p[a].flag = c.msd_flag + a; pa.p[a].lsd_hist = c.hist[0][a]; pa.p[a].lsd_ticket = c.ticket + 4 * a;
      pa.p[a].bucket_of_bin = c.bucket_of_bin[a]; pa.p[a].bucket_cursor = c.bucket_cursor[a]; pa.p[a].bucket_lo = a == 0 ? c.bucket_lo : nullptr;
    }
    // fuller buckets pay once there are enough of them to fill the GPU either way (config 2, 10^6 keys: 0.089 ms per
    // call with the prefix rule, 0.103 ms packed; config 4, 10^7 keys: bucket sort 146 us against 124 us)
    pa.pack_cap = c.n >= (4u << 20) ? (uint32_t)g_opt.msd_pack : 0u;
    ProfScope prof(kClsPlan, st);
    launch_pdl(msd::plan_kernel, n_arrays, 1024, 0, st, pa);
    BITS_LAUNCH_CHECK();
  }
  {
    msd::ScatterArgs sa;
    for (int a = 0; a < 2; ++a) {
      const int aa = a < n_arrays ? a : 0;
      sa.arr[a].src = p.src[aa]; sa.arr[a].dst = p.x[aa]; sa.arr[a].bucket_of_bin = c.bucket_of_bin[aa]; sa.arr[a].bucket_cursor = c.bucket_cursor[aa]; sa.arr[a].flag = c.msd_flag + aa;
    }
    sa.n = c.n;
    ProfScope prof(kClsScatter, st);
    if (g_opt.msd_scatter_shape == 0) {
      using C = msd::ScatterCfg1x1024;
      sa.n_tiles = (uint32_t)ceil_div(c.n, C::kTile);
      const uint32_t per = (uint32_t)kSMs / (uint32_t)n_arrays;
      launch_pdl(msd::scatter_kernel<C>, dim3(sa.n_tiles < per ? sa.n_tiles : per, n_arrays), C::kThreads, C::kSmem, st, sa);
    } else {
      using C = msd::ScatterCfg2x512;
      sa.n_tiles = (uint32_t)ceil_div(c.n, C::kTile);
      const uint32_t per = 2u * (uint32_t)kSMs / (uint32_t)n_arrays;
      launch_pdl(msd::scatter_kernel<C>, dim3(sa.n_tiles < per ? sa.n_tiles : per, n_arrays), C::kThreads, C::kSmem, st, sa);
    }
    BITS_LAUNCH_CHECK();
  }
  {
    msd::BucketArgs ba;
    for (int a = 0; a < 2; ++a) {
      const int aa = a < n_arrays ? a : 0;
      ba.arr[a].src = p.x[aa]; ba.arr[a].dst = p.y[aa]; ba.arr[a].bucket_start = c.bucket_start[aa];
      ba.arr[a].n_buckets = c.n_buckets + aa; ba.arr[a].flag = c.msd_flag + aa;
    }
    const uint32_t want = (uint32_t)ceil_div((uint64_t)c.n * 2, msd::kBucketCap) + 1;   // about the number of buckets
    const uint32_t per = 2u * (uint32_t)kSMs / (uint32_t)n_arrays;
    ProfScope prof(kClsBucketSort, st);
    ba.slab = 0; ba.round_flag = nullptr; ba.round_total = nullptr;
    for (int a = 0; a < 2; ++a) { ba.arr[a].q_sorted = nullptr; ba.arr[a].qb = nullptr; }
    launch_pdl(msd::bucket_sort_kernel<false, false>, dim3(want < per ? want : per, n_arrays), msd::kBkThreads, msd::kBkSmem, st, ba);
    BITS_LAUNCH_CHECK();
  }
  // fallback: the stable LSD sort redoes everything if a flag was raised, else these launches exit at once
  p.run_if = c.msd_flag;
  BITS_TRY(launch_histogram(src0, src1, c.hist[0][0], c.hist[0][1], c.n, n_arrays, st, c.msd_flag));
  return launch_sort_passes(p, epoch, st);
}

static int launch_build_index(const SortCtx& c, cudaStream_t st, const uint32_t* run_if = nullptr) {
  IndexArgs ia;
  ia.run_if = run_if;
  ia.keys[0] = c.buf[0][0]; ia.keys[1] = c.buf[1][0];
  ia.idx[0] = c.idx[0]; ia.idx[1] = c.idx[1];
  ia.n = c.n; ia.shift = c.shift;
  const uint64_t need = ceil_div((uint64_t)c.n, 4) + 1;   // four positions per thread
  const uint64_t threads = need > (uint64_t)kPad ? need : (uint64_t)kPad;
  const uint64_t blocks = ceil_div(threads, 256);
  ia.total = blocks * 256;
  ProfScope prof(kClsIndex, st);
  // (a gated launch is almost always skipped, so it is capped like the grid-stride kernels -- 148 * grid_mult blocks,
  // which fill the GPU when the gate does open -- rather than given one block per 1,024 keys)
  const uint64_t gate_cap = (uint64_t)kSMs * (uint64_t)g_opt.grid_mult;
  launch_pdl(build_index_kernel, dim3((unsigned)(run_if && blocks > gate_cap ? gate_cap : blocks), 2), 256, 0, st, ia);
  BITS_LAUNCH_CHECK();
  return BITS_OK;
}

// B_S, B_E (+ indices) from the caller's b_start / b_end.  Result: c.buf[0][0], c.buf[1][0].
static int setup_searched_set(const SortCtx& c, const uint32_t* b_start, const uint32_t* b_end, uint32_t flags,
                              uint32_t* epoch, cudaStream_t st) {
  if (flags & BITS_B_SORTED) {
    BITS_CUDA_TRY(cudaMemcpyAsync(c.buf[0][0], b_start, sizeof(uint32_t) * (size_t)c.n, cudaMemcpyDeviceToDevice, st));
    BITS_CUDA_TRY(cudaMemcpyAsync(c.buf[1][0], b_end, sizeof(uint32_t) * (size_t)c.n, cudaMemcpyDeviceToDevice, st));
  } else {
    BITS_TRY(sort_arrays(c, b_start, b_end, 2, nullptr, false, epoch, st));
  }
  return launch_build_index(c, st);
}

static inline SortedSet sorted_set(const SortCtx& c, int a) {
  SortedSet s;
  s.keys = c.buf[a][0]; s.idx = c.idx[a]; s.n = c.n; s.shift = c.shift;
  return s;
}

static int launch_count(const uint32_t* a_start, const uint32_t* a_end, uint32_t n_a, const SortCtx& b,
                        uint32_t* counts, uint64_t* total, cudaStream_t st, const uint32_t* run_if = nullptr) {
  const bool vec = (((uintptr_t)a_start | (uintptr_t)a_end | (uintptr_t)counts) & 15) == 0;
  const int grid = grid_for(ceil_div(n_a, 4), 256);
  ProfScope prof(kClsCount, st);
  const SortedSet s0 = sorted_set(b, 0), s1 = sorted_set(b, 1);
  unsigned long long* tot = reinterpret_cast<unsigned long long*>(total);
  const int sv = (int)g_opt.search_variant;
#define BITS_COUNT_LAUNCH(V, S) launch_pdl(count_kernel<V, S>, grid, 256, 0, st, a_start, a_end, n_a, s0, s1, counts, tot, run_if)
  if (vec) {
    if (sv == kSearchPlain) BITS_COUNT_LAUNCH(true, kSearchPlain);
    else if (sv == kSearchStaged) BITS_COUNT_LAUNCH(true, kSearchStaged);
    else BITS_COUNT_LAUNCH(true, kSearchIndex);
  } else {
    if (sv == kSearchPlain) BITS_COUNT_LAUNCH(false, kSearchPlain);
    else if (sv == kSearchStaged) BITS_COUNT_LAUNCH(false, kSearchStaged);
    else BITS_COUNT_LAUNCH(false, kSearchIndex);
  }
#undef BITS_COUNT_LAUNCH
  BITS_LAUNCH_CHECK();
  return BITS_OK;
}

static int validate_inputs(const uint32_t* a_start, const uint32_t* a_end, uint32_t n_a, const uint32_t* b_start,
                           const uint32_t* b_end, uint32_t n_b, uint32_t* bad, cudaStream_t st) {
  BITS_CUDA_TRY(cudaMemsetAsync(bad, 0, sizeof(uint32_t), st));
  if (n_a) { validate_kernel<<<grid_for(n_a, 256), 256, 0, st>>>(a_start, a_end, n_a, bad); BITS_LAUNCH_CHECK(); }
  if (n_b) { validate_kernel<<<grid_for(n_b, 256), 256, 0, st>>>(b_start, b_end, n_b, bad); BITS_LAUNCH_CHECK(); }
  uint32_t h = 0;
  BITS_CUDA_TRY(cudaMemcpyAsync(&h, bad, sizeof(uint32_t), cudaMemcpyDeviceToHost, st));
  BITS_CUDA_TRY(cudaStreamSynchronize(st));
  return h ? BITS_ERR_MALFORMED : BITS_OK;
}

static int check_common(const void* a_start, const void* a_end, uint64_t n_a, const void* b_start, const void* b_end,
                        uint64_t n_b, uint32_t flags) {
  if (n_a >= kMaxIntervals || n_b >= kMaxIntervals) return BITS_ERR_SIZE;
  if (flags & ~(uint32_t)(BITS_B_SORTED | BITS_VALIDATE)) return BITS_ERR_FLAGS;
  if (n_a && (!a_start || !a_end)) return BITS_ERR_NULL;
  if (n_b && (!b_start || !b_end)) return BITS_ERR_NULL;
  return BITS_OK;
}

// Search + reduce with the queries binned by B's buckets (binned_count.cuh).  L.b has just been sorted by the MSD sort.
static int launch_binned_count(const uint32_t* a_start, const uint32_t* a_end, uint32_t n_a, const Layout& L,
                               uint32_t* counts, uint64_t* total, cudaStream_t st) {
  static std::atomic<int> configured[64];
  int device = 0;
  BITS_CUDA_TRY(cudaGetDevice(&device));
  if (device < 0 || device >= 64 || configured[device].load(std::memory_order_acquire) == 0) {
    BITS_CUDA_TRY(cudaFuncSetAttribute(qb::query_scatter_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)qb::kScSmem));
    BITS_CUDA_TRY(cudaFuncSetAttribute(qb::query_scatter_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)qb::kScSmem));
    BITS_CUDA_TRY(cudaFuncSetAttribute(qb::bucket_search_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)qb::kSrSmem));
    BITS_CUDA_TRY(cudaFuncSetAttribute(qb::bucket_search_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)qb::kSrSmem));
    if (device >= 0 && device < 64) configured[device].store(1, std::memory_order_release);
  }
  qb::Plan p;
  p.flag = L.b.msd_flag; p.bucket_of_bin = L.b.bucket_of_bin[0]; p.bucket_lo = L.b.bucket_lo; p.bucket_start = L.b.bucket_start[0];
  p.n_buckets = L.b.n_buckets; p.end_prefix = L.b.bin_cursor[1];
  const uint32_t n_tiles = (uint32_t)ceil_div(n_a, (uint64_t)qb::kScTile);
  {
    ProfScope prof(kClsQueryScatter, st);
    const uint32_t blocks = n_tiles < (uint32_t)kSMs ? n_tiles : (uint32_t)kSMs;
    if (counts) launch_pdl(qb::query_scatter_kernel<true>, blocks, qb::kScThreads, qb::kScSmem, st, a_start, a_end, n_a, p, L.ql);
    else launch_pdl(qb::query_scatter_kernel<false>, blocks, qb::kScThreads, qb::kScSmem, st, a_start, a_end, n_a, p, L.ql);
    BITS_LAUNCH_CHECK();
  }
  {
    qb::SearchArgs sa;
    sa.p = p; sa.l = L.ql; sa.b_s = L.b.buf[0][0]; sa.b_e = L.b.buf[1][0]; sa.n_b = L.b.n; sa.counts = counts;
    sa.total = reinterpret_cast<unsigned long long*>(total);
    ProfScope prof(kClsBucketSearch, st);
    const uint32_t want = (uint32_t)ceil_div(n_a, (uint64_t)qb::kChunk) + 1u;
    const uint32_t blocks = want < 2u * kSMs ? want : 2u * (uint32_t)kSMs;
    if (counts) launch_pdl(qb::bucket_search_kernel<true>, blocks, qb::kSrThreads, qb::kSrSmem, st, sa);
    else launch_pdl(qb::bucket_search_kernel<false>, blocks, qb::kSrThreads, qb::kSrSmem, st, sa);
    BITS_LAUNCH_CHECK();
  }
  return BITS_OK;
}

static int count_impl(const uint32_t* a_start, const uint32_t* a_end, uint64_t n_a, const uint32_t* b_start,
                      const uint32_t* b_end, uint64_t n_b, uint32_t flags, void* ws, size_t ws_bytes, int fn,
                      uint32_t* counts_out, uint64_t* total_out, cudaStream_t st) {
  BITS_TRY(check_common(a_start, a_end, n_a, b_start, b_end, n_b, flags));
  if (fn == BITS_FN_COUNT && !total_out) return BITS_ERR_NULL;
  if (fn == BITS_FN_COUNT_PER_INTERVAL && n_a && !counts_out) return BITS_ERR_NULL;
  const Layout L = make_layout(ws, fn, n_a, n_b, 0, 0, flags);
  if (!ws_ok(ws, ws_bytes, L.bytes)) return BITS_ERR_WORKSPACE;
  if (flags & BITS_VALIDATE)
    BITS_TRY(validate_inputs(a_start, a_end, (uint32_t)n_a, b_start, b_end, (uint32_t)n_b, L.small.bad, st));
  if (total_out) BITS_CUDA_TRY(cudaMemsetAsync(total_out, 0, sizeof(uint64_t), st));
  if (n_a == 0) return BITS_OK;
  if (n_b == 0) {
    if (counts_out) BITS_CUDA_TRY(cudaMemsetAsync(counts_out, 0, sizeof(uint32_t) * (size_t)n_a, st));
    return BITS_OK;
  }
  uint32_t epoch = 1;
  BITS_TRY(reset_sort_ctx(L.b, st));
  // Large query sets against a large B: queries binned by B's buckets, every bucket searched out of shared
  // memory (binned_count.cuh); needs the MSD sort's plan.  The index path behind it runs only if the sort fell back.
  const bool binned = count_bins_queries(n_a, n_b, flags);   // (the rule that carved L.ql)
  if (!binned) {
    BITS_TRY(setup_searched_set(L.b, b_start, b_end, flags, &epoch, st));
    return launch_count(a_start, a_end, (uint32_t)n_a, L.b, counts_out, total_out, st);
  }
  BITS_CUDA_TRY(cudaMemsetAsync(L.ql.hist, 0, sizeof(uint32_t) * (msd::kBins + 64), st));
  // (the queries' bin histogram and their plan ride in the sort's own histogram and plan launches)
  QueryBinning qbin;
  qbin.a_end = a_end; qbin.n_a = (uint32_t)n_a;
  qbin.plan.bin_hist = L.ql.hist; qbin.plan.off = L.ql.off; qbin.plan.cursor = L.ql.cursor; qbin.plan.item_off = L.ql.item_off;
  qbin.plan.item_bucket = L.ql.item_bucket; qbin.plan.chunk = (uint32_t)qb::kChunk;
  BITS_TRY(sort_arrays(L.b, b_start, b_end, 2, nullptr, false, &epoch, st, &qbin));
  BITS_TRY(launch_binned_count(a_start, a_end, (uint32_t)n_a, L, counts_out, total_out, st));
  BITS_TRY(launch_build_index(L.b, st, L.b.msd_flag));
  return launch_count(a_start, a_end, (uint32_t)n_a, L.b, counts_out, total_out, st, L.b.msd_flag);
}

// ---------------------------------------------------------------------------------------------
static int check_genome(const uint32_t* off, uint32_t n_chrom, ChromTable* t, uint32_t* l_max) {
  if (!off) return BITS_ERR_NULL;
  if (n_chrom == 0 || off[0] != 0) return BITS_ERR_GENOME;
  uint32_t lmin = 0xffffffffu, lmax = 0;
  for (uint32_t c = 0; c < n_chrom; ++c) {
    if (off[c + 1] <= off[c]) return BITS_ERR_GENOME;
    const uint32_t L = off[c + 1] - off[c];
    lmin = L < lmin ? L : lmin;
    lmax = L > lmax ? L : lmax;
  }
  t->n_chrom = n_chrom;
  t->l_min = lmin;
  t->genome = off[n_chrom];
  uint32_t s = 0;
  if (n_chrom > 1) { s = 1; while ((uint64_t)s * 2 <= n_chrom - 1) s *= 2; }
  t->step0 = s;
  *l_max = lmax;
  return BITS_OK;
}

// Copy the offset table and its look-up table into the workspace and point `t` at them.
static int upload_genome(const uint32_t* off, uint32_t n_chrom, const Small& sm, ChromTable* t, cudaStream_t st) {
  t->off = sm.chrom;
  t->lut = nullptr;
  t->lut_shift = 0;
  BITS_CUDA_TRY(cudaMemcpyAsync(sm.chrom, off, sizeof(uint32_t) * ((size_t)n_chrom + 1), cudaMemcpyHostToDevice, st));
  if (n_chrom + 2 <= (uint32_t)kMaxChromSmem && n_chrom < 65536u) {
    uint16_t lut[kLutSize];
    t->lut_shift = make_chrom_lut(off, n_chrom, lut);
    BITS_CUDA_TRY(cudaMemcpyAsync(sm.lut, lut, sizeof(lut), cudaMemcpyHostToDevice, st));   // pageable: staged before return
    t->lut = sm.lut;
  }
  return BITS_OK;
}

static int launch_place(const uint32_t* spans, uint32_t* start_out, uint32_t* end_out, uint32_t n, uint32_t round,
                        uint32_t tag, const PhiloxKeys& key, const ChromTable& chrom, bool vec, int hist_mode,
                        uint32_t* hist_s, uint32_t* hist_e, uint32_t* zero_s, uint32_t* zero_e, cudaStream_t st) {
  PlaceArgs a;
  a.spans = spans; a.start_out = start_out; a.end_out = end_out; a.n = n; a.round = round; a.tag = tag;
  a.key = key; a.chrom = chrom; a.hist_start = hist_s; a.hist_end = hist_e; a.zero_a = zero_s; a.zero_b = zero_e;
  const int grid = grid_for(ceil_div(n, 4), 256);
  ProfScope prof(kClsPlace, st);
  if (hist_mode == kHistBins) {
    if (vec) place_kernel<true, kHistBins><<<grid, 256, 0, st>>>(a); else place_kernel<false, kHistBins><<<grid, 256, 0, st>>>(a);
  } else if (hist_mode == kHistDigits) {
    if (vec) place_kernel<true, kHistDigits><<<grid, 256, 0, st>>>(a); else place_kernel<false, kHistDigits><<<grid, 256, 0, st>>>(a);
  } else {
    if (vec) place_kernel<true, kHistNone><<<grid, 256, 0, st>>>(a); else place_kernel<false, kHistNone><<<grid, 256, 0, st>>>(a);
  }
  BITS_LAUNCH_CHECK();
  return BITS_OK;
}

template <class C>
static void launch_place_tile(const mct::PlaceTileArgs& pt, uint32_t rounds, cudaStream_t st) {
  const uint32_t blocks = (uint32_t)C::kBlocksPerSm * (uint32_t)kSMs;
  if (pt.slot_words) launch_pdl(mct::place_tile_kernel<C, true>, dim3(pt.n_tiles < blocks ? pt.n_tiles : blocks, rounds), C::kThreads, C::kSmem, st, pt);
  else launch_pdl(mct::place_tile_kernel<C, false>, dim3(pt.n_tiles < blocks ? pt.n_tiles : blocks, 1), C::kThreads, C::kSmem, st, pt);
}

template <class C>
static void launch_bin_sort(const mct::BinSortArgs& bs, uint32_t rounds, cudaStream_t st) {
  const uint32_t blocks = (uint32_t)C::kBlocksPerSm * (uint32_t)kSMs;
  if (bs.slot_words) launch_pdl(mct::bin_sort_search_kernel<C, true>, dim3(bs.n_bins < blocks ? bs.n_bins : blocks, rounds), C::kThreads, C::smem_bytes(bs.n_tiles), st, bs);
  else launch_pdl(mct::bin_sort_search_kernel<C, false>, dim3(bs.n_bins < blocks ? bs.n_bins : blocks, 1), C::kThreads, C::smem_bytes(bs.n_tiles), st, bs);
}

// Rounds a block of the PERMUTE_A / screen kernels serves for its query tile: the option's value, fewer when the
// launch would otherwise not fill the GPU (eight 256-thread blocks per SM).
static inline uint32_t rounds_per_block(uint64_t tile_rounds) {
  const uint64_t fill = tile_rounds / ((uint64_t)kSMs * 8u);
  const uint64_t want = (uint64_t)g_opt.mc_a_rounds_per_block;
  return (uint32_t)(fill < 1 ? 1 : (fill < want ? fill : want));
}

static int mc_impl(const uint32_t* a_start, const uint32_t* a_end, uint64_t n_a, const uint32_t* b_start,
                   const uint32_t* b_end, uint64_t n_b, const uint32_t* off, uint32_t n_chrom, int which, uint64_t seed,
                   uint32_t round_begin, uint32_t n_rounds, uint32_t flags, void* ws, size_t ws_bytes,
                   uint64_t* observed_out, uint64_t* round_counts_out, cudaStream_t st) {
  BITS_TRY(check_common(a_start, a_end, n_a, b_start, b_end, n_b, flags));
  if (which != BITS_PERMUTE_A && which != BITS_PERMUTE_B) return BITS_ERR_FLAGS;
  // independently sorted arrays no longer pair starts with ends: the lengths that re-placement must keep
  // are gone
  if (which == BITS_PERMUTE_B && (flags & BITS_B_SORTED)) return BITS_ERR_FLAGS;
  if (!observed_out || (n_rounds && !round_counts_out)) return BITS_ERR_NULL;
  if ((uint64_t)round_begin + n_rounds > (1ull << 32)) return BITS_ERR_SIZE;
  ChromTable chrom;
  uint32_t l_max = 0;
  BITS_TRY(check_genome(off, n_chrom, &chrom, &l_max));
  const Layout L = make_layout(ws, BITS_FN_MC_ROUNDS, n_a, n_b, n_chrom, which);
  if (!ws_ok(ws, ws_bytes, L.bytes)) return BITS_ERR_WORKSPACE;
  if (flags & BITS_VALIDATE)
    BITS_TRY(validate_inputs(a_start, a_end, (uint32_t)n_a, b_start, b_end, (uint32_t)n_b, L.small.bad, st));
  BITS_TRY(upload_genome(off, n_chrom, L.small, &chrom, st));
  BITS_CUDA_TRY(cudaMemsetAsync(observed_out, 0, sizeof(uint64_t), st));
  if (n_rounds) BITS_CUDA_TRY(cudaMemsetAsync(round_counts_out, 0, sizeof(uint64_t) * (size_t)n_rounds, st));

  // spans of the permuted set + the NO_PLACEMENT check (one synchronisation)
  const uint32_t n_p = (uint32_t)(which == BITS_PERMUTE_A ? n_a : n_b);
  uint32_t h_max_span = 0;
  double h_mean_span = 0.0;
  if (n_p) {
    BITS_CUDA_TRY(cudaMemsetAsync(L.small.max_span, 0, 4 * sizeof(uint32_t), st));
    spans_kernel<<<grid_for(n_p, 256), 256, 0, st>>>(which == BITS_PERMUTE_A ? a_start : b_start,
                                                     which == BITS_PERMUTE_A ? a_end : b_end, n_p, L.spans,
                                                     L.small.max_span, L.small.span_sum);
    BITS_LAUNCH_CHECK();
    uint32_t h_small[4] = {0, 0, 0, 0};
    BITS_CUDA_TRY(cudaMemcpyAsync(h_small, L.small.max_span, sizeof(h_small), cudaMemcpyDeviceToHost, st));
    BITS_CUDA_TRY(cudaStreamSynchronize(st));
    h_max_span = h_small[0];
    h_mean_span = (double)(((uint64_t)h_small[3] << 32) | h_small[2]) / (double)n_p;
    if (h_max_span >= l_max) return BITS_ERR_NO_PLACEMENT;
  }
  if (n_a == 0 || n_b == 0) return BITS_OK;   // every count is 0 (already written)

  // observed = total(A, B)
  uint32_t epoch = 1;
  BITS_TRY(reset_sort_ctx(L.b, st));
  BITS_TRY(setup_searched_set(L.b, b_start, b_end, flags, &epoch, st));
  BITS_TRY(launch_count(a_start, a_end, (uint32_t)n_a, L.b, nullptr, observed_out, st));
  if (n_rounds == 0) return BITS_OK;

  const PhiloxKeys key = make_philox_keys(seed);
  if (which == BITS_PERMUTE_A) {
    McAArgs m;
    m.spans = L.spans; m.n_a = (uint32_t)n_a; m.tag = 0u; m.key = key; m.chrom = chrom;
    m.bs = sorted_set(L.b, 0); m.be = sorted_set(L.b, 1);
    m.round_counts = reinterpret_cast<unsigned long long*>(round_counts_out);
    const unsigned gx = (unsigned)ceil_div(ceil_div(n_a, 4), 256);
    for (uint32_t done = 0; done < n_rounds;) {
      const uint32_t chunk = n_rounds - done < 32768u ? n_rounds - done : 32768u;
      m.round0 = round_begin + done; m.out0 = done; m.n_launch = chunk;
      m.rpb = rounds_per_block((uint64_t)gx * chunk);
      ProfScope prof(kClsMcA, st);
      if (m.rpb > 1) mc_permute_a_rounds_kernel<<<dim3(gx, (unsigned)ceil_div(chunk, m.rpb)), 256, 0, st>>>(m);
      else mc_permute_a_kernel<<<dim3(gx, chunk), 256, 0, st>>>(m);
      BITS_LAUNCH_CHECK();
      done += chunk;
    }
    return BITS_OK;
  }

  // PERMUTE_B: A's ends and starts sorted once; every round place -> sort x2 -> search -> reduce.
  uint32_t q_epoch = 1;
  BITS_TRY(reset_sort_ctx(L.q, st));
  BITS_TRY(sort_arrays(L.q, a_end, a_start, 2, nullptr, false, &q_epoch, st));
  const uint32_t* q_end_sorted = L.q.buf[0][0];
  const uint32_t* q_start_sorted = L.q.buf[1][0];
  if (g_opt.mc_symmetric) {
    // SURVEY 8(f).1, the sort-free variant: count(A, B') = count(B', A), so every fresh interval of B is
    // counted against the once-sorted A (first = #{A.start <= b'.end}, last = #{A.end < b'.start}) and
    // nothing is sorted per round.  Same integers; B_S / B_E of the round are NOT produced.
    BITS_TRY(launch_build_index(L.q, st));
    McAArgs m;
    m.spans = L.spans; m.n_a = (uint32_t)n_b; m.tag = 1u; m.key = key; m.chrom = chrom;
    m.bs = sorted_set(L.q, 1); m.be = sorted_set(L.q, 0);
    m.round_counts = reinterpret_cast<unsigned long long*>(round_counts_out);
    const unsigned gx = (unsigned)ceil_div(ceil_div(n_b, 4), 256);
    for (uint32_t done = 0; done < n_rounds;) {
      const uint32_t chunk = n_rounds - done < 4096u ? n_rounds - done : 4096u;
      m.round0 = round_begin + done; m.out0 = done; m.n_launch = chunk;
      m.rpb = rounds_per_block((uint64_t)gx * chunk);
      ProfScope prof(kClsMcA, st);
      if (m.rpb > 1) mc_permute_a_rounds_kernel<<<dim3(gx, (unsigned)ceil_div(chunk, m.rpb)), 256, 0, st>>>(m);
      else mc_permute_a_kernel<<<dim3(gx, chunk), 256, 0, st>>>(m);
      BITS_LAUNCH_CHECK();
      done += chunk;
    }
    return BITS_OK;
  }
  // (each block ranks all n_a sorted queries on its own: with fewer rounds than the GPU has SMs and a large A -- round
  // slicing, warm-up calls -- a launch would run on a handful of SMs for milliseconds; such calls take the two-launch
  // path below, which spreads the queries of ONE round over all blocks.  Knob mc_small = 2 takes the path regardless.)
  const bool small_fills_gpu = n_rounds >= (uint32_t)kSMs || n_a * (uint64_t)n_rounds <= (1ull << 22) || g_opt.mc_small == 2;
  if (g_opt.mc_small != 0 && small_fills_gpu && n_b <= (uint64_t)mcs::kMaxKeys && g_opt.mc_fused != 0 && g_opt.mc_sorted_queries != 0) {
    // a set that fits one block's shared memory: one block per round, the grid strides over the rounds (mc_small.cuh)
    BITS_TRY(msd_configure());
    mcs::SmallArgs m;
    m.spans = L.spans; m.n = (uint32_t)n_b; m.tag = 1u; m.round0 = round_begin; m.n_rounds = n_rounds;
    const uint32_t g_bits = 32u - (uint32_t)__builtin_clz((off[n_chrom] - 1u) | 1u);      // bits of the largest coordinate
    m.sshift = g_bits > (uint32_t)mcs::Cfg::kSubBits ? g_bits - (uint32_t)mcs::Cfg::kSubBits : 0u;
    m.key = key; m.chrom = chrom; m.q_sorted[0] = q_end_sorted; m.q_sorted[1] = q_start_sorted; m.n_q = (uint32_t)n_a;
    m.dst[0] = L.b.buf[0][0]; m.dst[1] = L.b.buf[1][0];
    m.round_counts = reinterpret_cast<unsigned long long*>(round_counts_out);
    const uint32_t blocks = (uint32_t)mcs::Cfg::kBlocksPerSm * (uint32_t)kSMs;
    ProfScope prof(kClsBucketSortSearch, st);
    mcs::mc_small_b_kernel<<<n_rounds < blocks ? n_rounds : blocks, mcs::Cfg::kThreads, mcs::kSmem, st>>>(m);
    BITS_LAUNCH_CHECK();
    return BITS_OK;
  }
  const bool msd_on = g_opt.sort_msd != 0;
  const bool hist_in_place = g_opt.place_fused_hist != 0;
  // histograms the placement kernel accumulates into: the MSD sort's bins (left zero by plan_kernel)
  // or, with the LSD sort only, the four digit histograms (parity double-buffered, cleared by the
  // placement kernel of the previous round)
  if (!msd_on) {
    BITS_CUDA_TRY(cudaMemsetAsync(L.b.hist[0][0], 0, sizeof(uint32_t) * rs::kPasses * rs::kRadix, st));
    BITS_CUDA_TRY(cudaMemsetAsync(L.b.hist[0][1], 0, sizeof(uint32_t) * rs::kPasses * rs::kRadix, st));
    BITS_CUDA_TRY(cudaMemsetAsync(L.b.hist[1][0], 0, sizeof(uint32_t) * rs::kPasses * rs::kRadix, st));
    BITS_CUDA_TRY(cudaMemsetAsync(L.b.hist[1][1], 0, sizeof(uint32_t) * rs::kPasses * rs::kRadix, st));
  }
  uint32_t n_general = 0;   // rounds done by the general path so far (parity of the LSD histograms)
  // One round by the general path: place -> sort both arrays -> search with the sorted queries.
  auto general_round = [&](uint32_t k) -> int {
    const int par = (int)(n_general++ & 1);
    // epochs (30 bits) must not wrap
    if (epoch > (1u << 30) - 16u) {
      BITS_CUDA_TRY(cudaMemsetAsync(L.b.status[0], 0, sizeof(uint64_t) * (uint64_t)L.b.n_tiles * rs::kRadix, st));
      BITS_CUDA_TRY(cudaMemsetAsync(L.b.status[1], 0, sizeof(uint64_t) * (uint64_t)L.b.n_tiles * rs::kRadix, st));
      epoch = 1;
    }
    // placed keys go to the "result" buffers; the sort reads them, works through the temp buffers
    // and lands back in the result buffers
    if (msd_on) {
      BITS_TRY(launch_place(L.spans, L.b.buf[0][0], L.b.buf[1][0], (uint32_t)n_b, round_begin + k, 1u, key, chrom, true,
                            hist_in_place ? kHistBins : kHistNone, hist_in_place ? L.b.bin_hist[0] : nullptr,
                            hist_in_place ? L.b.bin_hist[1] : nullptr, nullptr, nullptr, st));
      BITS_TRY(sort_arrays(L.b, L.b.buf[0][0], L.b.buf[1][0], 2, nullptr, hist_in_place, &epoch, st));
    } else {
      if (hist_in_place) {
        BITS_TRY(launch_place(L.spans, L.b.buf[0][0], L.b.buf[1][0], (uint32_t)n_b, round_begin + k, 1u, key, chrom, true,
                              kHistDigits, L.b.hist[par][0], L.b.hist[par][1], L.b.hist[par ^ 1][0], L.b.hist[par ^ 1][1], st));
      } else {
        BITS_TRY(launch_place(L.spans, L.b.buf[0][0], L.b.buf[1][0], (uint32_t)n_b, round_begin + k, 1u, key, chrom, true,
                              kHistNone, nullptr, nullptr, nullptr, nullptr, st));
        BITS_CUDA_TRY(cudaMemsetAsync(L.b.hist[par][0], 0, sizeof(uint32_t) * rs::kPasses * rs::kRadix, st));
        BITS_CUDA_TRY(cudaMemsetAsync(L.b.hist[par][1], 0, sizeof(uint32_t) * rs::kPasses * rs::kRadix, st));
        BITS_TRY(launch_histogram(L.b.buf[0][0], L.b.buf[1][0], L.b.hist[par][0], L.b.hist[par][1], (uint32_t)n_b, 2, st));
      }
      BITS_CUDA_TRY(cudaMemsetAsync(L.b.ticket, 0, sizeof(uint32_t) * 8, st));
      BITS_TRY(launch_sort_passes(plan_for(L.b, L.b.buf[0][0], L.b.buf[1][0], par), &epoch, st));
    }
    unsigned long long* out = reinterpret_cast<unsigned long long*>(round_counts_out + k);
    if (g_opt.mc_sorted_queries) {
      ProfScope prof(kClsSortedQuery, st);
      sorted_query_total_kernel<<<grid_for(n_a, 256), 256, 0, st>>>(q_end_sorted, q_start_sorted, (uint32_t)n_a,
                                                                    L.b.buf[0][0], L.b.buf[1][0], (uint32_t)n_b, out);
      BITS_LAUNCH_CHECK();
    } else {
      BITS_TRY(launch_build_index(L.b, st));
      BITS_TRY(launch_count(a_start, a_end, (uint32_t)n_a, L.b, nullptr, reinterpret_cast<uint64_t*>(out), st));
    }
    return BITS_OK;
  };

  // Fused rounds (mc_tile.cuh): possible when fixed bins (key >> shift) hold the re-placed keys with a
  // wide margin (expected keys per bin <= n_b * 2^shift / V(d_max), V(d) = number of valid starts for
  // span d), every span is shorter than a bin, and few ends fall into the bin after their start's.
  mct::PlaceTileArgs pt;
  mct::BinSortArgs bs;
  uint32_t rounds_per_launch = 1, batch_tile = 0;
  bool fused_ok = msd_on && g_opt.mc_fused != 0 && g_opt.mc_sorted_queries != 0 && L.pairs != nullptr;
  const int variant = (int)g_opt.mc_bin_variant;
  const int tile_variant = (int)g_opt.mc_tile_variant;
  const double bin_cap = variant == 0 ? (double)mct::BinCfgWide::kCap
                       : (variant == 1 ? (double)mct::BinCfgNarrow::kCap : (variant == 2 ? (double)mct::BinCfgSmall::kCap : (double)mct::BinCfgHuge::kCap));
  if (fused_ok) {
    uint64_t v_min = 0;
    for (uint32_t c = 0; c < n_chrom; ++c) { const uint32_t Lc = off[c + 1] - off[c]; v_min += Lc > h_max_span ? Lc - h_max_span : 0; }
    const uint64_t G = off[n_chrom];
    // does a bin of 2^sh coordinates hold its keys, its hand-over list and every span with a wide margin?
    auto fits = [&](int sh) -> bool {
      const uint64_t nbins = (G + (1ull << sh) - 1) >> sh;
      if (nbins >= (uint64_t)mct::kMaxBins) return false;
      if ((uint64_t)h_max_span >= (1ull << sh)) return false;   // an end may lie at most one bin after its start
      const double avg = (double)n_b * (double)(1ull << sh) / (double)v_min;
      if (avg * 1.125 + 8.0 * sqrt(avg) + 32.0 > bin_cap) return false;
      const double cross = avg * h_mean_span / (double)(1ull << sh);   // ends handed over per bin
      return cross * 2.0 + 8.0 * sqrt(cross) + 32.0 <= (double)mct::kCrossCap;
    };
    int best = -1;
    for (int sh = mct::kMaxShift; sh >= 1 && v_min > 0; --sh)
      if (fits(sh)) { best = sh; break; }
    // a small set: narrower bins (finer sub-buckets, more blocks) as long as there are no more bins than blocks
    while (best > 1 && fits(best - 1) && ((G + (1ull << (best - 1)) - 1) >> (best - 1)) <= 2ull * kSMs) --best;
    fused_ok = best >= 0;
    // A small set does not fill the GPU with one round: several rounds per launch pair (gridDim.y), each in its own
    // slot of the workspace, and the WIDEST bins that fit (few, full bins per round instead of many nearly empty ones).
    if (fused_ok && L.batch_slots > 1 && L.bt_pairs && g_opt.mc_batch != 0 && g_opt.mc_shift_bias == 0) {
      int wide = -1;
      for (int sh = 31; sh >= 1; --sh)
        if (fits(sh)) { wide = sh; break; }
      if (wide >= 0) {
        const uint64_t nb = (G + (1ull << wide) - 1) >> wide;
        const uint32_t per = (uint32_t)(nb < 2ull * kSMs ? nb : 2ull * kSMs);
        uint32_t r = 8u * (uint32_t)kSMs / (per ? per : 1u);           // about four waves of bin blocks per launch
        if (r > L.batch_slots) r = L.batch_slots;
        const uint32_t max_tile = tile_variant == 0 ? (uint32_t)mct::TileCfg2x512::kTile
                                : (tile_variant == 1 ? (uint32_t)mct::TileCfg1x1024::kTile : (uint32_t)mct::TileCfg1x1024L::kTile);
        const uint32_t blocks_per_round = r ? ((uint32_t)kSMs / r ? (uint32_t)kSMs / r : 1u) : 1u;
        uint32_t tile = tile_size_for(n_b, blocks_per_round, max_tile);
        if (tile < 4096u) tile = (uint32_t)(align_up(n_b, 4) < 4096u ? align_up(n_b, 4) : 4096u);
        if (r >= 2 && nb <= (uint64_t)kBatchBins && ceil_div(n_b, tile) + 1 <= (uint64_t)L.batch_rows) {
          rounds_per_launch = r; best = wide; batch_tile = tile;
        }
      }
    }
    if (fused_ok && g_opt.mc_shift_bias > 0) {     // tests: wider bins than the margin allows, so that bins overflow on the device
      best += (int)g_opt.mc_shift_bias;
      if (best > mct::kMaxShift) best = mct::kMaxShift;
    }
    if (fused_ok) {
      pt.spans = L.spans; pt.n = (uint32_t)n_b; pt.tag = 1u; pt.key = key; pt.chrom = chrom;
      pt.shift = (uint32_t)best; pt.n_bins = (uint32_t)((G + (1ull << best) - 1) >> best);
      pt.tile = tile_variant == 0 ? tile_size_cfg<mct::TileCfg2x512>(n_b)
                                  : (tile_variant == 1 ? tile_size_cfg<mct::TileCfg1x1024>(n_b) : tile_size_cfg<mct::TileCfg1x1024L>(n_b));
      const bool batched = rounds_per_launch > 1;
      if (batched) pt.tile = batch_tile;
      pt.n_tiles = (uint32_t)ceil_div(n_b, pt.tile);
      pt.pairs = batched ? L.bt_pairs : L.pairs; pt.off = batched ? L.bt_off : L.tile_off; pt.stride = L.tile_stride;
      pt.cross_keys = batched ? L.bt_cross_keys : L.cross_keys;
      pt.slot_words = bs.slot_words = batched ? (uint32_t)L.slot_words : 0u;
      bs.pairs = pt.pairs; bs.off = pt.off; bs.stride = L.tile_stride; bs.n_tiles = pt.n_tiles; bs.tile = pt.tile;
      bs.n = (uint32_t)n_b; bs.shift = pt.shift; bs.n_bins = pt.n_bins; bs.cross_keys = pt.cross_keys;
      bs.dst[0] = batched ? L.bt_dst[0] : L.b.buf[0][0]; bs.dst[1] = batched ? L.bt_dst[1] : L.b.buf[1][0];
      bs.q_sorted[0] = q_end_sorted; bs.q_sorted[1] = q_start_sorted; bs.qb[0] = L.qb[0]; bs.qb[1] = L.qb[1];
      bs.n_q = (uint32_t)n_a;
      // lanes per gathered segment: the power of two at or above the mean segment length
      const double seg = (double)n_b / ((double)pt.n_tiles * (double)pt.n_bins);
      bs.group_log2 = 0;
      while (bs.group_log2 < 5 && (double)(1u << bs.group_log2) < seg) ++bs.group_log2;
      if (g_opt.mc_gather_group >= 0) bs.group_log2 = (uint32_t)g_opt.mc_gather_group;
      bs.group = 1u << bs.group_log2;
      if (pt.n_tiles > (uint32_t)mct::kMaxTiles) fused_ok = false;
      if (variant == 3 && mct::BinCfgHuge::smem_bytes(pt.n_tiles) > kMaxSmemPerBlock) fused_ok = false;
    }
  }
  if (!fused_ok) {
    for (uint32_t k = 0; k < n_rounds; ++k) BITS_TRY(general_round(k));
    return BITS_OK;
  }
  BITS_TRY(msd_configure());
  const bool batched = rounds_per_launch > 1;
  uint32_t* const cc[2] = {batched ? L.bt_cross_cnt[0] : L.cross_cnt[0], batched ? L.bt_cross_cnt[1] : L.cross_cnt[1]};
  if (batched) {     // both hand-over count arrays of every slot (they are neighbours inside a slot)
    const size_t width = (size_t)(reinterpret_cast<char*>(cc[1]) - reinterpret_cast<char*>(cc[0])) + sizeof(uint32_t) * (mct::kMaxBins + 4);
    BITS_CUDA_TRY(cudaMemset2DAsync(cc[0], L.slot_words * sizeof(uint32_t), 0, width, L.batch_slots, st));
  } else {
    BITS_CUDA_TRY(cudaMemsetAsync(cc[0], 0, sizeof(uint32_t) * (mct::kMaxBins + 4), st));
    BITS_CUDA_TRY(cudaMemsetAsync(cc[1], 0, sizeof(uint32_t) * (mct::kMaxBins + 4), st));
  }
  {
    mct::QueryBinsArgs qa;
    qa.q_sorted[0] = q_end_sorted; qa.q_sorted[1] = q_start_sorted; qa.qb[0] = L.qb[0]; qa.qb[1] = L.qb[1];
    qa.n_q = (uint32_t)n_a; qa.n_bins = pt.n_bins; qa.shift = pt.shift;
    mct::query_bins_kernel<<<dim3((unsigned)ceil_div(pt.n_bins + 1, 256), 2), 256, 0, st>>>(qa);
    BITS_LAUNCH_CHECK();
  }
  std::vector<uint32_t> h_flags;
  uint32_t n_fused = 0;     // launch pairs so far (parity of the hand-over counters)
  // flags are read back per chunk of rounds; a chunk is a whole number of launch pairs, so that only the call's last
  // launch pair can be a partial one (a slot that sat out a pair would miss the clearing of its hand-over counts)
  const uint32_t flag_chunk = kFlagChunk / rounds_per_launch * rounds_per_launch;
  for (uint32_t done = 0; done < n_rounds;) {
    const uint32_t chunk = n_rounds - done < flag_chunk ? n_rounds - done : flag_chunk;
    BITS_CUDA_TRY(cudaMemsetAsync(L.round_flags, 0, sizeof(uint32_t) * chunk, st));
    for (uint32_t j = 0; j < chunk; ++n_fused) {
      const uint32_t k = done + j;
      const uint32_t nr = chunk - j < rounds_per_launch ? chunk - j : rounds_per_launch;
      const int par = (int)(n_fused & 1u);
      pt.round = round_begin + k; pt.flag = L.round_flags + j; pt.cross_cnt = cc[par];
      {
        ProfScope prof(kClsPlaceScatter, st);
        if (tile_variant == 0) launch_place_tile<mct::TileCfg2x512>(pt, nr, st);
        else if (tile_variant == 1) launch_place_tile<mct::TileCfg1x1024>(pt, nr, st);
        else launch_place_tile<mct::TileCfg1x1024L>(pt, nr, st);
        BITS_LAUNCH_CHECK();
      }
      bs.cross_cnt = cc[par]; bs.cross_cnt_next = cc[par ^ 1]; bs.flag = pt.flag;
      bs.round_total = reinterpret_cast<unsigned long long*>(round_counts_out + k);
      {
        ProfScope prof(kClsBucketSortSearch, st);
        if (variant == 0) launch_bin_sort<mct::BinCfgWide>(bs, nr, st);
        else if (variant == 1) launch_bin_sort<mct::BinCfgNarrow>(bs, nr, st);
        else if (variant == 2) launch_bin_sort<mct::BinCfgSmall>(bs, nr, st);
        else launch_bin_sort<mct::BinCfgHuge>(bs, nr, st);
        BITS_LAUNCH_CHECK();
      }
      j += nr;
    }
    if (batched && done + chunk == n_rounds) {
      // B_S and B_E of the call's last round go from their slot to where bits_workspace_sorted_offset points
      const size_t slot = (size_t)((chunk - 1) % rounds_per_launch) * L.slot_words;
      for (int a = 0; a < 2; ++a)
        BITS_CUDA_TRY(cudaMemcpyAsync(L.b.buf[a][0], L.bt_dst[a] + slot, sizeof(uint32_t) * (size_t)n_b, cudaMemcpyDeviceToDevice, st));
    }
    // rounds whose flag was raised are redone by the general path (one synchronisation per chunk)
    h_flags.assign(chunk, 0);
    BITS_CUDA_TRY(cudaMemcpyAsync(h_flags.data(), L.round_flags, sizeof(uint32_t) * chunk, cudaMemcpyDeviceToHost, st));
    BITS_CUDA_TRY(cudaStreamSynchronize(st));
    uint32_t last_redone = 0xffffffffu;
    for (uint32_t j = 0; j < chunk; ++j) {
      const bool forced = g_opt.mc_force_redo > 0 && (done + j) % (uint32_t)g_opt.mc_force_redo == 0;
      if (!h_flags[j] && !forced) continue;
      BITS_CUDA_TRY(cudaMemsetAsync(round_counts_out + done + j, 0, sizeof(uint64_t), st));
      BITS_TRY(general_round(done + j));
      last_redone = done + j;
    }
    // general_round sorts into the buffers bits_workspace_sorted_offset points to.  If a redo in the call's final
    // chunk left another round's arrays there, the last round is done once more by the general path (same count,
    // bit for bit), so that the workspace holds B_S and B_E of the LAST round whatever the overflow flags were.
    if (done + chunk == n_rounds && last_redone != 0xffffffffu && last_redone != n_rounds - 1) {
      BITS_CUDA_TRY(cudaMemsetAsync(round_counts_out + (n_rounds - 1), 0, sizeof(uint64_t), st));
      BITS_TRY(general_round(n_rounds - 1));
    }
    done += chunk;
  }
  return BITS_OK;
}


// ---------------------------------------------------------------------------------------------
// The many-pair screen (screen.cuh).
struct ScreenLayout {
  Small small;
  SortCtx scratch;                    // sort bookkeeping and the temp buffers, sized for the largest track
  std::vector<uint32_t*> keys[2];     // per track: B_S, B_E
  std::vector<uint32_t*> idx[2];      // per track: their bucket indices
  std::vector<uint32_t*> spans;       // per track
  scr::Track* tracks = nullptr;       // dev [K]
  uint32_t* tile_track = nullptr;     // dev [n_tiles]
  uint32_t* tile_first = nullptr;     // dev [K]
  uint64_t n_tiles = 0;
  size_t bytes = 0;
};

static ScreenLayout make_screen_layout(void* ws, const uint64_t* toff, uint32_t K, uint32_t n_chrom) {
  ScreenLayout L;
  Carver c(ws);
  L.small.carve(c, n_chrom);
  uint64_t n_max = 0;
  for (uint32_t t = 0; t < K; ++t) {
    const uint64_t n = toff[t + 1] - toff[t];
    n_max = n > n_max ? n : n_max;
    L.n_tiles += ceil_div(n, (uint64_t)scr::kTile);
  }
  L.scratch.carve(c, n_max, false);
  for (int a = 0; a < 2; ++a) { L.keys[a].resize(K); L.idx[a].resize(K); }
  L.spans.resize(K);
  for (uint32_t t = 0; t < K; ++t) {
    const uint64_t n = toff[t + 1] - toff[t];
    const uint32_t shift = index_shift_for(n);
    for (int a = 0; a < 2; ++a) L.keys[a][t] = c.take<uint32_t>(align_up(n + kPad, 64));
    for (int a = 0; a < 2; ++a) L.idx[a][t] = c.take<uint32_t>(index_entries(shift));
    L.spans[t] = c.take<uint32_t>(align_up(n, 4) + 4);
  }
  L.tracks = c.take<scr::Track>(K);
  L.tile_track = c.take<uint32_t>(L.n_tiles + 1);
  L.tile_first = c.take<uint32_t>((uint64_t)K + 1);
  L.bytes = align_up(c.used, 256);
  return L;
}

static int check_tracks(const uint64_t* toff, uint32_t K) {
  if (!toff) return BITS_ERR_NULL;
  if (K == 0 || K > 65535u) return BITS_ERR_SIZE;             // pair ids i * K + j are 32-bit Philox counter words
  if (toff[0] != 0) return BITS_ERR_SIZE;
  for (uint32_t t = 0; t < K; ++t)
    if (toff[t + 1] < toff[t]) return BITS_ERR_SIZE;
  if (toff[K] >= kMaxIntervals) return BITS_ERR_SIZE;
  return BITS_OK;
}

static int screen_impl(const uint32_t* starts, const uint32_t* ends, const uint64_t* toff, uint32_t K, const uint32_t* off,
                       uint32_t n_chrom, uint64_t seed, uint32_t round_begin, uint32_t n_rounds, uint32_t flags, void* ws,
                       size_t ws_bytes, uint64_t* observed_out, uint64_t* round_counts_out, cudaStream_t st) {
  BITS_TRY(check_tracks(toff, K));
  if (flags & ~(uint32_t)BITS_VALIDATE) return BITS_ERR_FLAGS;
  const uint64_t n_total = toff[K];
  if (n_total && (!starts || !ends)) return BITS_ERR_NULL;
  if (!observed_out || (n_rounds && !round_counts_out)) return BITS_ERR_NULL;
  if ((uint64_t)round_begin + n_rounds > (1ull << 32)) return BITS_ERR_SIZE;
  ChromTable chrom;
  uint32_t l_max = 0;
  BITS_TRY(check_genome(off, n_chrom, &chrom, &l_max));
  const ScreenLayout L = make_screen_layout(ws, toff, K, n_chrom);
  if (!ws_ok(ws, ws_bytes, L.bytes)) return BITS_ERR_WORKSPACE;
  if ((flags & BITS_VALIDATE) && n_total)
    BITS_TRY(validate_inputs(starts, ends, (uint32_t)n_total, nullptr, nullptr, 0, L.small.bad, st));
  BITS_TRY(upload_genome(off, n_chrom, L.small, &chrom, st));
  const uint64_t n_pairs = (uint64_t)K * K;
  BITS_CUDA_TRY(cudaMemsetAsync(observed_out, 0, sizeof(uint64_t) * n_pairs, st));
  if (n_rounds) BITS_CUDA_TRY(cudaMemsetAsync(round_counts_out, 0, sizeof(uint64_t) * n_pairs * n_rounds, st));
  if (n_total == 0) return BITS_OK;

  // spans of every track + the NO_PLACEMENT check over all of them (the call's one synchronisation)
  BITS_CUDA_TRY(cudaMemsetAsync(L.small.max_span, 0, 4 * sizeof(uint32_t), st));
  for (uint32_t t = 0; t < K; ++t) {
    const uint32_t n = (uint32_t)(toff[t + 1] - toff[t]);
    if (!n) continue;
    spans_kernel<<<grid_for(n, 256), 256, 0, st>>>(starts + toff[t], ends + toff[t], n, L.spans[t], L.small.max_span, L.small.span_sum);
    BITS_LAUNCH_CHECK();
  }
  uint32_t h_small[4] = {0, 0, 0, 0};
  BITS_CUDA_TRY(cudaMemcpyAsync(h_small, L.small.max_span, sizeof(h_small), cudaMemcpyDeviceToHost, st));
  BITS_CUDA_TRY(cudaStreamSynchronize(st));
  if (n_rounds && h_small[0] >= l_max) return BITS_ERR_NO_PLACEMENT;

  // every track sorted and indexed once
  std::vector<scr::Track> h_tracks(K);
  std::vector<uint32_t> h_tile_track((size_t)L.n_tiles + 1, 0u), h_tile_first((size_t)K + 1, 0u);
  uint32_t epoch = 1, tile = 0;
  BITS_TRY(reset_sort_ctx(L.scratch, st));
  for (uint32_t t = 0; t < K; ++t) {
    const uint64_t n = toff[t + 1] - toff[t];
    SortCtx c = L.scratch;
    c.n = (uint32_t)n; c.n_tiles = rs::num_tiles(n); c.shift = index_shift_for(n);
    for (int a = 0; a < 2; ++a) { c.buf[a][0] = L.keys[a][t]; c.idx[a] = L.idx[a][t]; }
    scr::Track& T = h_tracks[t];
    T.start = starts + toff[t]; T.end = ends + toff[t]; T.spans = L.spans[t];
    for (int a = 0; a < 2; ++a) { T.keys[a] = L.keys[a][t]; T.idx[a] = L.idx[a][t]; }
    T.n = (uint32_t)n; T.shift = c.shift;
    h_tile_first[t] = tile;
    for (uint64_t k = 0; k < ceil_div(n, (uint64_t)scr::kTile); ++k) h_tile_track[tile++] = t;
    if (!n) continue;
    if (epoch > (1u << 30) - 16u) {       // epochs (30 bits) must not wrap
      BITS_CUDA_TRY(cudaMemsetAsync(L.scratch.status[0], 0, sizeof(uint64_t) * (uint64_t)L.scratch.n_tiles * rs::kRadix, st));
      BITS_CUDA_TRY(cudaMemsetAsync(L.scratch.status[1], 0, sizeof(uint64_t) * (uint64_t)L.scratch.n_tiles * rs::kRadix, st));
      epoch = 1;
    }
    BITS_TRY(sort_arrays(c, T.start, T.end, 2, nullptr, false, &epoch, st));
    BITS_TRY(launch_build_index(c, st));
  }
  BITS_CUDA_TRY(cudaMemcpyAsync(L.tracks, h_tracks.data(), sizeof(scr::Track) * K, cudaMemcpyHostToDevice, st));   // pageable: staged before return
  BITS_CUDA_TRY(cudaMemcpyAsync(L.tile_track, h_tile_track.data(), sizeof(uint32_t) * (L.n_tiles + 1), cudaMemcpyHostToDevice, st));
  BITS_CUDA_TRY(cudaMemcpyAsync(L.tile_first, h_tile_first.data(), sizeof(uint32_t) * ((size_t)K + 1), cudaMemcpyHostToDevice, st));

  scr::ScreenArgs a;
  a.tracks = L.tracks; a.tile_track = L.tile_track; a.tile_first = L.tile_first; a.n_tracks = K;
  a.round0 = round_begin; a.out0 = 0; a.n_rounds = n_rounds; a.key = make_philox_keys(seed); a.chrom = chrom;
  a.rpb = 1; a.n_launch = 1;
  a.observed = reinterpret_cast<unsigned long long*>(observed_out);
  a.round_counts = reinterpret_cast<unsigned long long*>(round_counts_out);
  {
    ProfScope prof(kClsCount, st);
    scr::screen_kernel<true><<<dim3((unsigned)L.n_tiles, K, 1), scr::kThreads, 0, st>>>(a);
    BITS_LAUNCH_CHECK();
  }
  for (uint32_t done = 0; done < n_rounds;) {
    const uint32_t chunk = n_rounds - done < 4096u ? n_rounds - done : 4096u;
    a.round0 = round_begin + done; a.out0 = done; a.n_launch = chunk; a.rpb = rounds_per_block((uint64_t)L.n_tiles * K * chunk);
    ProfScope prof(kClsMcA, st);
    if (a.rpb > 1) scr::screen_kernel<false><<<dim3((unsigned)L.n_tiles, K, (unsigned)ceil_div(chunk, a.rpb)), scr::kThreads, 0, st>>>(a);
    else scr::screen_round_kernel<<<dim3((unsigned)L.n_tiles, K, chunk), scr::kThreads, 0, st>>>(a);
    BITS_LAUNCH_CHECK();
    done += chunk;
  }
  return BITS_OK;
}


// ---------------------------------------------------------------------------------------------
struct HostStage {
  uint32_t *a_s, *a_e, *b_s, *b_e, *counts;
  uint64_t *total, *rounds;
  size_t bytes;
};
static HostStage make_stage(void* base, uint64_t n_a, uint64_t n_b, uint32_t n_rounds, bool with_counts) {
  Carver c(base);
  HostStage h;
  h.a_s = c.take<uint32_t>(align_up(n_a, 4) + 4);
  h.a_e = c.take<uint32_t>(align_up(n_a, 4) + 4);
  h.b_s = c.take<uint32_t>(align_up(n_b, 4) + 4);
  h.b_e = c.take<uint32_t>(align_up(n_b, 4) + 4);
  h.counts = with_counts ? c.take<uint32_t>(align_up(n_a, 4) + 4) : nullptr;
  h.total = c.take<uint64_t>(32);
  h.rounds = c.take<uint64_t>((uint64_t)n_rounds + 1);
  h.bytes = align_up(c.used, 256);
  return h;
}

static int stage_in(const HostStage& h, const uint32_t* a_start, const uint32_t* a_end, uint64_t n_a,
                    const uint32_t* b_start, const uint32_t* b_end, uint64_t n_b, cudaStream_t st) {
  if (n_a) {
    BITS_CUDA_TRY(cudaMemcpyAsync(h.a_s, a_start, 4 * (size_t)n_a, cudaMemcpyHostToDevice, st));
    BITS_CUDA_TRY(cudaMemcpyAsync(h.a_e, a_end, 4 * (size_t)n_a, cudaMemcpyHostToDevice, st));
  }
  if (n_b) {
    BITS_CUDA_TRY(cudaMemcpyAsync(h.b_s, b_start, 4 * (size_t)n_b, cudaMemcpyHostToDevice, st));
    BITS_CUDA_TRY(cudaMemcpyAsync(h.b_e, b_end, 4 * (size_t)n_b, cudaMemcpyHostToDevice, st));
  }
  return BITS_OK;
}

// ---------------------------------------------------------------------------------------------
// Built-in scratch for bits_count_static (bits.h): one fixed array that lives in the library's own device image,
// so the counting path can run for a caller that has no way to hand over a workspace.  Every CUDA context that
// loads this library carries these BITS_STATIC_SCRATCH_BYTES until the process (or the context) ends.
//
// In host code the name `g_static_scratch` is only the host-side handle of the symbol -- it is NOT a device
// address and must never be given to a kernel or a cudaMemsetAsync.  The address the device sees comes from
// cudaGetSymbolAddress, asked once per device while that device is current, and kept.
static __device__ __align__(256) unsigned char g_static_scratch[BITS_STATIC_SCRATCH_BYTES];

static int static_scratch_address(void** out) {
  constexpr int kMaxDevices = 64;
  static std::atomic<void*> addr_on[kMaxDevices];     // zero-initialised; one slot per device ordinal
  int device = 0;
  BITS_CUDA_TRY(cudaGetDevice(&device));
  const bool tracked = device >= 0 && device < kMaxDevices;
  void* p = tracked ? addr_on[device].load(std::memory_order_acquire) : nullptr;
  if (!p) {
    // first call on this device (or a device ordinal past the table: asked every time, which is cheap)
    const cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
    if (e != cudaSuccess || p == nullptr) { (void)cudaGetLastError(); return BITS_ERR_CUDA; }
    if (tracked) addr_on[device].store(p, std::memory_order_release);
  }
  *out = p;
  return BITS_OK;
}

// The per-kernel event timers create CUDA events on demand (ProfScope); a call that promises to allocate nothing
// runs with them switched off and puts the caller's setting back afterwards.
struct ProfilerPause {
  bool was;
  ProfilerPause() : was(g_prof.on) { g_prof.on = false; }
  ~ProfilerPause() { g_prof.on = was; }
};

}  // namespace bits

using namespace bits;

extern "C" {

size_t bits_workspace_bytes(int fn, uint64_t n_a, uint64_t n_b, uint32_t n_chrom, int which, uint32_t flags) {
  (void)flags;
  if (fn < BITS_FN_COUNT || fn > BITS_FN_ENUMERATE) return 0;
  if (n_a >= kMaxIntervals || n_b >= kMaxIntervals) return 0;
  return make_layout(nullptr, fn, n_a, n_b, n_chrom, which, flags).bytes;
}

int bits_workspace_sorted_offset(int fn, uint64_t n_a, uint64_t n_b, uint32_t n_chrom, int which, int array,
                                 size_t* offset_out) {
  if (!offset_out) return BITS_ERR_NULL;
  if (fn < BITS_FN_COUNT || fn > BITS_FN_MC_ROUNDS || (array != 0 && array != 1)) return BITS_ERR_FLAGS;
  if (n_a >= kMaxIntervals || n_b >= kMaxIntervals) return BITS_ERR_SIZE;
  char* const base = reinterpret_cast<char*>(uintptr_t(1) << 20);   // any non-null base: only differences are used
  const Layout L = make_layout(base, fn, n_a, n_b, n_chrom, which);
  *offset_out = (size_t)(reinterpret_cast<char*>(L.b.buf[array][0]) - base);
  return BITS_OK;
}

size_t bits_host_staging_bytes(int fn, uint64_t n_a, uint64_t n_b, uint32_t n_rounds) {
  if (fn < BITS_FN_COUNT || fn > BITS_FN_MC_ROUNDS) return 0;
  return make_stage(nullptr, n_a, n_b, n_rounds, fn == BITS_FN_COUNT_PER_INTERVAL).bytes;
}

int bits_count(const uint32_t* a_start, const uint32_t* a_end, uint64_t n_a, const uint32_t* b_start,
               const uint32_t* b_end, uint64_t n_b, uint32_t flags, void* workspace, size_t workspace_bytes,
               uint64_t* total_out, void* stream) {
  return count_impl(a_start, a_end, n_a, b_start, b_end, n_b, flags, workspace, workspace_bytes, BITS_FN_COUNT,
                    nullptr, total_out, static_cast<cudaStream_t>(stream));
}

int bits_count_static(const uint32_t* a_start, const uint32_t* a_end, uint64_t n_a, const uint32_t* b_start,
                      const uint32_t* b_end, uint64_t n_b, uint32_t flags, uint64_t* total_out, void* stream) {
  // argument errors first, exactly as bits_count reports them (no CUDA call yet)
  BITS_TRY(check_common(a_start, a_end, n_a, b_start, b_end, n_b, flags));
  if (!total_out) return BITS_ERR_NULL;
  // the limit: the scratch this problem needs must fit the built-in array
  if (make_layout(nullptr, BITS_FN_COUNT, n_a, n_b, 0, 0, flags).bytes > (size_t)BITS_STATIC_SCRATCH_BYTES) return BITS_ERR_STATIC_LIMIT;
  void* scratch = nullptr;
  BITS_TRY(static_scratch_address(&scratch));   // device address of the array on the current device (set up on first use)
  ProfilerPause no_event_creation;
  // Same kernels, same order as bits_count; only the scratch pointer differs.  count_impl clears every word of the
  // scratch that must start at zero (sort bookkeeping, query histogram, validation flag) on `stream` before the first
  // kernel reads it, so whatever the previous call left in the array does not matter.
  return count_impl(a_start, a_end, n_a, b_start, b_end, n_b, flags, scratch, (size_t)BITS_STATIC_SCRATCH_BYTES,
                    BITS_FN_COUNT, nullptr, total_out, static_cast<cudaStream_t>(stream));
}

int bits_decide(const uint32_t* a_start, const uint32_t* a_end, uint64_t n_a, const uint32_t* b_start,
                const uint32_t* b_end, uint64_t n_b, uint32_t flags, void* workspace, size_t workspace_bytes,
                uint32_t* any_out, void* stream) {
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  BITS_TRY(check_common(a_start, a_end, n_a, b_start, b_end, n_b, flags));
  if (!any_out) return BITS_ERR_NULL;
  const Layout L = make_layout(workspace, BITS_FN_COUNT, n_a, n_b, 0, 0, flags);
  if (!ws_ok(workspace, workspace_bytes, L.bytes)) return BITS_ERR_WORKSPACE;
  if (flags & BITS_VALIDATE)
    BITS_TRY(validate_inputs(a_start, a_end, (uint32_t)n_a, b_start, b_end, (uint32_t)n_b, L.small.bad, st));
  BITS_CUDA_TRY(cudaMemsetAsync(any_out, 0, sizeof(uint32_t), st));
  if (n_a == 0 || n_b == 0) return BITS_OK;
  uint32_t epoch = 1;
  BITS_TRY(reset_sort_ctx(L.b, st));
  BITS_TRY(setup_searched_set(L.b, b_start, b_end, flags, &epoch, st));
  ProfScope prof(kClsCount, st);
  launch_pdl(decide_kernel, grid_for(n_a, 256), 256, 0, st, a_start, a_end, (uint32_t)n_a, sorted_set(L.b, 0), sorted_set(L.b, 1), any_out);
  BITS_LAUNCH_CHECK();
  return BITS_OK;
}

int bits_enumerate(const uint32_t* a_start, const uint32_t* a_end, uint64_t n_a, const uint32_t* b_start,
                   const uint32_t* b_end, uint64_t n_b, uint32_t flags, void* workspace, size_t workspace_bytes,
                   uint32_t* pair_a_out, uint32_t* pair_b_out, uint64_t capacity, uint64_t* total_out, void* stream) {
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  BITS_TRY(check_common(a_start, a_end, n_a, b_start, b_end, n_b, flags));
  if (!total_out || (capacity && (!pair_a_out || !pair_b_out))) return BITS_ERR_NULL;
  if (flags & BITS_B_SORTED) return BITS_ERR_FLAGS;   // independently sorted arrays have lost which end belongs to which start
  const Layout L = make_layout(workspace, BITS_FN_ENUMERATE, n_a, n_b, 0, 0);
  if (!ws_ok(workspace, workspace_bytes, L.bytes)) return BITS_ERR_WORKSPACE;
  if (flags & BITS_VALIDATE)
    BITS_TRY(validate_inputs(a_start, a_end, (uint32_t)n_a, b_start, b_end, (uint32_t)n_b, L.small.bad, st));
  BITS_CUDA_TRY(cudaMemsetAsync(total_out, 0, sizeof(uint64_t), st));
  if (n_a == 0 || n_b == 0) return BITS_OK;
  uint32_t epoch = 1;
  BITS_TRY(reset_sort_ctx(L.b, st));
  BITS_TRY(setup_searched_set(L.b, b_start, b_end, flags, &epoch, st));
  // per-interval counts (the termination condition), their exclusive scan, B's ends and indices in start order
  BITS_TRY(launch_count(a_start, a_end, (uint32_t)n_a, L.b, L.e_counts, nullptr, st));
  const uint32_t n_tiles = (uint32_t)ceil_div(n_a, (uint64_t)enu::kScanTile);
  ProfScope prof(kClsOther, st);
  launch_pdl(enu::scan_tile_sums_kernel, n_tiles, enu::kScanThreads, 0, st, L.e_counts, (uint32_t)n_a, L.e_tile_sums);
  BITS_LAUNCH_CHECK();
  launch_pdl(enu::scan_tile_prefix_kernel, 1, 1024, 0, st, L.e_tile_sums, n_tiles, reinterpret_cast<unsigned long long*>(total_out));
  BITS_LAUNCH_CHECK();
  launch_pdl(enu::scan_apply_kernel, n_tiles, enu::kScanThreads, 0, st, L.e_counts, (uint32_t)n_a, L.e_tile_sums, L.e_offsets);
  BITS_LAUNCH_CHECK();
  if (capacity == 0) return BITS_OK;
  BITS_CUDA_TRY(cudaMemsetAsync(L.e_tie, 0, sizeof(uint32_t) * ((size_t)n_b + 1), st));
  launch_pdl(enu::start_order_kernel, grid_for(n_b, 256), 256, 0, st, b_start, b_end, (uint32_t)n_b, sorted_set(L.b, 0), L.e_tie,
             L.e_end_by_start, L.e_idx_by_start);
  BITS_LAUNCH_CHECK();
  BITS_CUDA_TRY(cudaMemsetAsync(L.e_max[2], 0, sizeof(uint32_t) * (((size_t)n_b >> enu::kSkip3) + 4), st));
  launch_pdl(enu::end_maxima_kernel, (unsigned)ceil_div(n_b, 1024), 1024, 0, st, L.e_end_by_start, (uint32_t)n_b, L.e_max[0], L.e_max[1], L.e_max[2]);
  BITS_LAUNCH_CHECK();
  launch_pdl(enu::emit_pairs_kernel, grid_for(n_a, 256), 256, 0, st, a_start, a_end, (uint32_t)n_a, sorted_set(L.b, 0), L.e_counts, L.e_offsets,
             L.e_end_by_start, L.e_idx_by_start, L.e_max[0], L.e_max[1], L.e_max[2], pair_a_out, pair_b_out, capacity);
  BITS_LAUNCH_CHECK();
  return BITS_OK;
}

int bits_count_per_interval(const uint32_t* a_start, const uint32_t* a_end, uint64_t n_a, const uint32_t* b_start,
                            const uint32_t* b_end, uint64_t n_b, uint32_t flags, void* workspace,
                            size_t workspace_bytes, uint32_t* counts_out, uint64_t* total_out, void* stream) {
  return count_impl(a_start, a_end, n_a, b_start, b_end, n_b, flags, workspace, workspace_bytes,
                    BITS_FN_COUNT_PER_INTERVAL, counts_out, total_out, static_cast<cudaStream_t>(stream));
}

int bits_mc_rounds(const uint32_t* a_start, const uint32_t* a_end, uint64_t n_a, const uint32_t* b_start,
                   const uint32_t* b_end, uint64_t n_b, const uint32_t* chrom_offsets, uint32_t n_chrom, int which,
                   uint64_t seed, uint32_t round_begin, uint32_t n_rounds, uint32_t flags, void* workspace,
                   size_t workspace_bytes, uint64_t* observed_out, uint64_t* round_counts_out, void* stream) {
  return mc_impl(a_start, a_end, n_a, b_start, b_end, n_b, chrom_offsets, n_chrom, which, seed, round_begin, n_rounds,
                 flags, workspace, workspace_bytes, observed_out, round_counts_out, static_cast<cudaStream_t>(stream));
}

int bits_place(const uint32_t* spans, uint64_t n, const uint32_t* chrom_offsets, uint32_t n_chrom, uint64_t seed,
               uint32_t round, uint32_t tag, void* workspace, size_t workspace_bytes, uint32_t* start_out,
               uint32_t* end_out, void* stream) {
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  if (n >= kMaxIntervals) return BITS_ERR_SIZE;
  if (n && (!spans || !start_out || !end_out)) return BITS_ERR_NULL;
  ChromTable chrom;
  uint32_t l_max = 0;
  BITS_TRY(check_genome(chrom_offsets, n_chrom, &chrom, &l_max));
  const Layout L = make_layout(workspace, BITS_FN_PLACE, 0, 0, n_chrom, 0);
  if (!ws_ok(workspace, workspace_bytes, L.bytes)) return BITS_ERR_WORKSPACE;
  if (n == 0) return BITS_OK;
  BITS_TRY(upload_genome(chrom_offsets, n_chrom, L.small, &chrom, st));
  const bool vec = (n & 3) == 0 && (((uintptr_t)spans | (uintptr_t)start_out | (uintptr_t)end_out) & 15) == 0;
  return launch_place(spans, start_out, end_out, (uint32_t)n, round, tag, make_philox_keys(seed), chrom, vec, kHistNone,
                      nullptr, nullptr, nullptr, nullptr, st);
}

int bits_sort_u32(const uint32_t* keys_in, uint32_t* keys_out, uint64_t n, void* workspace, size_t workspace_bytes,
                  void* stream) {
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  if (n >= kMaxIntervals) return BITS_ERR_SIZE;
  if (n && (!keys_in || !keys_out)) return BITS_ERR_NULL;
  const Layout L = make_layout(workspace, BITS_FN_SORT, 0, n, 0, 0);
  if (!ws_ok(workspace, workspace_bytes, L.bytes)) return BITS_ERR_WORKSPACE;
  if (n == 0) return BITS_OK;
  BITS_TRY(reset_sort_ctx(L.b, st));
  uint32_t epoch = 1;
  return sort_arrays(L.b, keys_in, keys_in, 1, keys_out, false, &epoch, st);
}

int bits_count_host(const uint32_t* a_start, const uint32_t* a_end, uint64_t n_a, const uint32_t* b_start,
                    const uint32_t* b_end, uint64_t n_b, uint32_t flags, void* workspace, size_t workspace_bytes,
                    uint64_t* total_out, void* stream) {
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  BITS_TRY(check_common(a_start, a_end, n_a, b_start, b_end, n_b, flags));
  if (!total_out) return BITS_ERR_NULL;
  const size_t main_bytes = bits_workspace_bytes(BITS_FN_COUNT, n_a, n_b, 0, 0, flags);
  const HostStage h = make_stage(workspace ? static_cast<char*>(workspace) + main_bytes : nullptr, n_a, n_b, 0, false);
  if (!ws_ok(workspace, workspace_bytes, main_bytes + h.bytes)) return BITS_ERR_WORKSPACE;
  BITS_TRY(stage_in(h, a_start, a_end, n_a, b_start, b_end, n_b, st));
  BITS_TRY(count_impl(h.a_s, h.a_e, n_a, h.b_s, h.b_e, n_b, flags, workspace, main_bytes, BITS_FN_COUNT, nullptr,
                      h.total, st));
  BITS_CUDA_TRY(cudaMemcpyAsync(total_out, h.total, sizeof(uint64_t), cudaMemcpyDeviceToHost, st));
  BITS_CUDA_TRY(cudaStreamSynchronize(st));
  return BITS_OK;
}

int bits_count_per_interval_host(const uint32_t* a_start, const uint32_t* a_end, uint64_t n_a,
                                 const uint32_t* b_start, const uint32_t* b_end, uint64_t n_b, uint32_t flags,
                                 void* workspace, size_t workspace_bytes, uint32_t* counts_out, uint64_t* total_out,
                                 void* stream) {
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  BITS_TRY(check_common(a_start, a_end, n_a, b_start, b_end, n_b, flags));
  if (n_a && !counts_out) return BITS_ERR_NULL;
  const size_t main_bytes = bits_workspace_bytes(BITS_FN_COUNT_PER_INTERVAL, n_a, n_b, 0, 0, flags);
  const HostStage h = make_stage(workspace ? static_cast<char*>(workspace) + main_bytes : nullptr, n_a, n_b, 0, true);
  if (!ws_ok(workspace, workspace_bytes, main_bytes + h.bytes)) return BITS_ERR_WORKSPACE;
  BITS_TRY(stage_in(h, a_start, a_end, n_a, b_start, b_end, n_b, st));
  BITS_TRY(count_impl(h.a_s, h.a_e, n_a, h.b_s, h.b_e, n_b, flags, workspace, main_bytes, BITS_FN_COUNT_PER_INTERVAL,
                      h.counts, h.total, st));
  if (n_a) BITS_CUDA_TRY(cudaMemcpyAsync(counts_out, h.counts, 4 * (size_t)n_a, cudaMemcpyDeviceToHost, st));
  if (total_out) BITS_CUDA_TRY(cudaMemcpyAsync(total_out, h.total, sizeof(uint64_t), cudaMemcpyDeviceToHost, st));
  BITS_CUDA_TRY(cudaStreamSynchronize(st));
  return BITS_OK;
}

int bits_mc_rounds_host(const uint32_t* a_start, const uint32_t* a_end, uint64_t n_a, const uint32_t* b_start,
                        const uint32_t* b_end, uint64_t n_b, const uint32_t* chrom_offsets, uint32_t n_chrom,
                        int which, uint64_t seed, uint32_t round_begin, uint32_t n_rounds, uint32_t flags,
                        void* workspace, size_t workspace_bytes, uint64_t* observed_out, uint64_t* round_counts_out,
                        void* stream) {
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  BITS_TRY(check_common(a_start, a_end, n_a, b_start, b_end, n_b, flags));
  if (!observed_out || (n_rounds && !round_counts_out)) return BITS_ERR_NULL;
  const size_t main_bytes = bits_workspace_bytes(BITS_FN_MC_ROUNDS, n_a, n_b, n_chrom, which, flags);
  const HostStage h =
      make_stage(workspace ? static_cast<char*>(workspace) + main_bytes : nullptr, n_a, n_b, n_rounds, false);
  if (!ws_ok(workspace, workspace_bytes, main_bytes + h.bytes)) return BITS_ERR_WORKSPACE;
  BITS_TRY(stage_in(h, a_start, a_end, n_a, b_start, b_end, n_b, st));
  BITS_TRY(mc_impl(h.a_s, h.a_e, n_a, h.b_s, h.b_e, n_b, chrom_offsets, n_chrom, which, seed, round_begin, n_rounds,
                   flags, workspace, main_bytes, h.total, h.rounds, st));
  BITS_CUDA_TRY(cudaMemcpyAsync(observed_out, h.total, sizeof(uint64_t), cudaMemcpyDeviceToHost, st));
  if (n_rounds)
    BITS_CUDA_TRY(cudaMemcpyAsync(round_counts_out, h.rounds, sizeof(uint64_t) * (size_t)n_rounds,
                                  cudaMemcpyDeviceToHost, st));
  BITS_CUDA_TRY(cudaStreamSynchronize(st));
  return BITS_OK;
}

double bits_pvalue(uint64_t observed, const uint64_t* round_counts, uint32_t n_rounds, int tail) {
  if ((tail != 0 && tail != 1) || (n_rounds && !round_counts)) return NAN;
  uint64_t k = 0;
  for (uint32_t r = 0; r < n_rounds; ++r)
    k += tail == 0 ? (round_counts[r] >= observed) : (round_counts[r] <= observed);
  return (double)(k + 1) / (double)((uint64_t)n_rounds + 1);
}

double bits_enrichment(uint64_t observed, const uint64_t* round_counts, uint32_t n_rounds) {
  if (n_rounds == 0 || !round_counts) return NAN;
  std::vector<uint64_t> v(round_counts, round_counts + n_rounds);
  const size_t m = n_rounds / 2;
  std::nth_element(v.begin(), v.begin() + m, v.end());
  double median = (double)v[m];
  if ((n_rounds & 1u) == 0) {
    const uint64_t lower = *std::max_element(v.begin(), v.begin() + m);   // the order statistic just below
    median = ((double)lower + (double)v[m]) / 2.0;
  }
  if (median == 0.0) return observed ? INFINITY : NAN;
  return log2((double)observed / median);
}

size_t bits_screen_workspace_bytes(const uint64_t* track_offsets, uint32_t n_tracks, uint32_t n_chrom) {
  if (check_tracks(track_offsets, n_tracks) != BITS_OK) return 0;
  return make_screen_layout(nullptr, track_offsets, n_tracks, n_chrom).bytes;
}

int bits_screen(const uint32_t* starts, const uint32_t* ends, const uint64_t* track_offsets, uint32_t n_tracks,
                const uint32_t* chrom_offsets, uint32_t n_chrom, uint64_t seed, uint32_t round_begin, uint32_t n_rounds,
                uint32_t flags, void* workspace, size_t workspace_bytes, uint64_t* observed_out,
                uint64_t* round_counts_out, void* stream) {
  return screen_impl(starts, ends, track_offsets, n_tracks, chrom_offsets, n_chrom, seed, round_begin, n_rounds, flags,
                     workspace, workspace_bytes, observed_out, round_counts_out, static_cast<cudaStream_t>(stream));
}

int bits_screen_enrichment(const uint64_t* observed, const uint64_t* round_counts, uint64_t n_pairs, uint32_t n_rounds,
                           double* enrichment_out) {
  if (n_pairs && (!observed || !enrichment_out || (n_rounds && !round_counts))) return BITS_ERR_NULL;
  for (uint64_t p = 0; p < n_pairs; ++p)
    enrichment_out[p] = bits_enrichment(observed[p], n_rounds ? round_counts + p * n_rounds : nullptr, n_rounds);
  return BITS_OK;
}

uint64_t bits_launch_count(void) { return g_launches.load(); }

int bits_profile_read(int cls, double* ms_out, uint64_t* launches_out) {
  if (cls < 0 || cls >= kNumCls) return BITS_ERR_FLAGS;
  g_prof.collect();
  if (ms_out) *ms_out = g_prof.ms[cls];
  if (launches_out) *launches_out = g_prof.launches[cls];
  return BITS_OK;
}

int bits_set_option(const char* name, int64_t value) {
  if (!name) return BITS_ERR_NULL;
  if (!strcmp(name, "mc_fused")) { g_opt.mc_fused = value; return BITS_OK; }
  if (!strcmp(name, "search_variant")) { if (value < 0 || value > 2) return BITS_ERR_FLAGS; g_opt.search_variant = value; return BITS_OK; }
  if (!strcmp(name, "mc_symmetric")) { g_opt.mc_symmetric = value != 0; return BITS_OK; }
  if (!strcmp(name, "mc_pdl")) { g_opt.mc_pdl = value != 0; return BITS_OK; }
  if (!strcmp(name, "mc_force_redo")) { if (value < 0) return BITS_ERR_FLAGS; g_opt.mc_force_redo = value; return BITS_OK; }
  if (!strcmp(name, "mc_tile_variant")) { if (value < 0 || value > 2) return BITS_ERR_FLAGS; g_opt.mc_tile_variant = value; return BITS_OK; }
  if (!strcmp(name, "mc_bin_variant")) { if (value < 0 || value > 3) return BITS_ERR_FLAGS; g_opt.mc_bin_variant = value; return BITS_OK; }
  if (!strcmp(name, "mc_gather_group")) { if (value < -1 || value > 5) return BITS_ERR_FLAGS; g_opt.mc_gather_group = value; return BITS_OK; }
  if (!strcmp(name, "msd_pack")) { if (value < 0 || value > msd::kBucketCap) return BITS_ERR_FLAGS; g_opt.msd_pack = value; return BITS_OK; }
  if (!strcmp(name, "msd_scatter_shape")) { if (value < 0 || value > 1) return BITS_ERR_FLAGS; g_opt.msd_scatter_shape = value; return BITS_OK; }
  if (!strcmp(name, "count_binned")) { if (value < -1 || value > 1) return BITS_ERR_FLAGS; g_opt.count_binned = value; return BITS_OK; }
  if (!strcmp(name, "mc_a_rounds_per_block")) { if (value < 1 || value > 64) return BITS_ERR_FLAGS; g_opt.mc_a_rounds_per_block = value; return BITS_OK; }
  if (!strcmp(name, "mc_batch")) { g_opt.mc_batch = value != 0; return BITS_OK; }
  if (!strcmp(name, "mc_small")) { if (value < 0 || value > 2) return BITS_ERR_FLAGS; g_opt.mc_small = value; return BITS_OK; }
  if (!strcmp(name, "mc_shift_bias")) { if (value < 0 || value > 8) return BITS_ERR_FLAGS; g_opt.mc_shift_bias = value; return BITS_OK; }
  if (!strcmp(name, "sort_msd")) { g_opt.sort_msd = value; return BITS_OK; }
  if (!strcmp(name, "mc_sorted_queries")) { g_opt.mc_sorted_queries = value; return BITS_OK; }
  if (!strcmp(name, "place_fused_hist")) { g_opt.place_fused_hist = value; return BITS_OK; }
  if (!strcmp(name, "profile")) {   // 0 = off, 1 = on, 2 = reset the accumulated times
    if (value == 2) g_prof.reset(); else g_prof.on = value != 0;
    return BITS_OK;
  }
  if (!strcmp(name, "grid_mult")) { if (value < 1 || value > 64) return BITS_ERR_FLAGS; g_opt.grid_mult = value; return BITS_OK; }
  return BITS_ERR_FLAGS;
}

const char* bits_strerror(int status) {
  switch (status) {
    case BITS_OK: return "ok";
    case BITS_ERR_NULL: return "a required pointer is NULL";
    case BITS_ERR_SIZE: return "size out of range (n_a, n_b < 2^28; round_begin + n_rounds <= 2^32)";
    case BITS_ERR_GENOME: return "bad chromosome offset table";
    case BITS_ERR_NO_PLACEMENT: return "an interval of the permuted set is as long as every chromosome";
    case BITS_ERR_WORKSPACE: return "workspace NULL, misaligned or too small";
    case BITS_ERR_FLAGS: return "unknown flag, option, fn, which or tail";
    case BITS_ERR_MALFORMED: return "malformed interval (start > end)";
    case BITS_ERR_CUDA: return "CUDA error (or no CUDA device)";
    case BITS_ERR_STATIC_LIMIT: return "problem too large for the built-in scratch of bits_count_static (BITS_STATIC_SCRATCH_BYTES); use bits_count with a workspace";
    default: return "unknown status";
  }
}

const char* bits_version(void) { return "bits_b200 0.1 (sm_100a)"; }

}  // extern "C"
