// radix_sort.cuh -- the "sort" step: onesweep-style LSD radix sort of uint32 keys.
//
// PAPER.md:117-125 (Algorithm 2): Sort(B_S), Sort(B_E) -- B's starts and ends are sorted
// ascending, each on its own.  Keys only, so any correct sort gives the same
// array.  The paper points at GPU radix sorts of its day; this is a
// single-pass-per-digit design: 8-bit digits, 4 passes, one up-front histogram (fused into the
// placement kernel inside the Monte Carlo loop), per-tile ranks by warp match, and a chained
// scan with decoupled look-back between tiles.  Two arrays (starts, ends) per launch.
#pragma once
#include "common.cuh"

namespace bits {
namespace rs {

constexpr int kRadixBits = 8;
constexpr int kRadix = 1 << kRadixBits;
constexpr int kPasses = 32 / kRadixBits;
constexpr int kThreads = 512;
constexpr int kWarps = kThreads / 32;
constexpr int kKeysPerThread = 16;
constexpr int kTile = kThreads * kKeysPerThread;   // 8192 keys

// Tile status word: [epoch:30 | flag:2 | value:32].  A word whose epoch is not the current pass's
// epoch is "not written yet", so the status array is cleared once per library call, not per pass.
constexpr uint64_t kFlagLocal = 1, kFlagIncl = 2;
__host__ __device__ inline uint64_t pack_status(uint32_t epoch, uint64_t flag, uint32_t value) {
  return ((uint64_t)epoch << 34) | (flag << 32) | value;
}

struct SortArray {
  const uint32_t* src;
  uint32_t* dst;
  const uint32_t* hist;   // global histogram of THIS pass's digit: uint32[256]
  uint64_t* status;       // uint64[n_tiles * 256]
  uint32_t* ticket;       // tile ticket counter of THIS pass and array: zero when the pass starts
};

struct SortPassArgs {
  SortArray arr[2];
  uint32_t n;
  uint32_t n_tiles;
  uint32_t shift;
  uint32_t epoch;         // 1 .. 2^30-1, unique per pass since the status array was cleared
  const uint32_t* run_if[2];   // both null: always run; else run only if *run_if[0] | *run_if[1] (fallback of msd_sort.cuh)
};



__device__ __forceinline__ bool skip_launch(const uint32_t* const run_if[2]) {
  return run_if[0] != nullptr && ((*run_if[0]) | (*run_if[1])) == 0u;
}

inline uint32_t num_tiles(uint64_t n) { return (uint32_t)ceil_div(n, kTile); }

__device__ __forceinline__ uint64_t ld_relaxed_u64(const uint64_t* p) {
  uint64_t v;
  asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_relaxed_u64(uint64_t* p, uint64_t v) {
  asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// Exclusive scan of one value per thread over the first 256 threads (8 warps).  Must be called
// by ALL threads of the block (two barriers inside); threads >= 256 pass 0 and ignore the result.
__device__ __forceinline__ uint32_t block_excl_scan_256(uint32_t v, uint32_t* s_wsum) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  uint32_t incl = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t t = __shfl_up_sync(kFullMask, incl, o);
    if (lane >= o) incl += t;
  }
  if (lane == 31 && w < 8) s_wsum[w] = incl;
  __syncthreads();
  uint32_t before = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) before += (i < w) ? s_wsum[i] : 0u;
  __syncthreads();
  return before + incl - v;
}

// ---------------------------------------------------------------------------------------------
// Up-front histogram of all four digits (stand-alone version, used when the keys are not made
// by the placement kernel).  hist layout per array: uint32[kPasses][256].  gridDim.y = arrays.
struct HistArgs {
  const uint32_t* keys[2];
  uint32_t* hist[2];
  uint32_t n;
  const uint32_t* run_if[2];
};

__global__ void __launch_bounds__(512) histogram_kernel(HistArgs a) {
  __shared__ uint32_t s_h[kPasses * kRadix];
  grid_dependency_wait();
  if (skip_launch(a.run_if)) return;
  for (int i = threadIdx.x; i < kPasses * kRadix; i += blockDim.x) s_h[i] = 0;
  __syncthreads();
  const uint32_t* __restrict__ keys = blockIdx.y ? a.keys[1] : a.keys[0];
  const uint32_t n = a.n;
  const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
  const bool vec = ((uintptr_t)keys & 15) == 0;
  if (vec) {
    const uint32_t n4 = n >> 2;
    const uint4* __restrict__ k4 = reinterpret_cast<const uint4*>(keys);
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += stride) {
      const uint4 k = __ldg(k4 + i);
      const uint32_t kk[4] = {k.x, k.y, k.z, k.w};
#pragma unroll
      for (int j = 0; j < 4; ++j)
#pragma unroll
        for (int p = 0; p < kPasses; ++p) atomicAdd(&s_h[p * kRadix + ((kk[j] >> (8 * p)) & 255u)], 1u);
    }
    if (blockIdx.x == 0 && threadIdx.x < (n & 3u)) {
      const uint32_t k = keys[(n & ~3u) + threadIdx.x];
#pragma unroll
      for (int p = 0; p < kPasses; ++p) atomicAdd(&s_h[p * kRadix + ((k >> (8 * p)) & 255u)], 1u);
    }
  } else {
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
      const uint32_t k = keys[i];
#pragma unroll
      for (int p = 0; p < kPasses; ++p) atomicAdd(&s_h[p * kRadix + ((k >> (8 * p)) & 255u)], 1u);
    }
  }
  __syncthreads();
  uint32_t* __restrict__ g = blockIdx.y ? a.hist[1] : a.hist[0];
  for (int i = threadIdx.x; i < kPasses * kRadix; i += blockDim.x)
    if (s_h[i]) atomicAdd(&g[i], s_h[i]);
}

// ---------------------------------------------------------------------------------------------
// One digit pass over both arrays.  grid = (n_tiles, n_arrays), block = kThreads.
__global__ void __launch_bounds__(kThreads, 2) onesweep_pass_kernel(SortPassArgs a) {
  __shared__ uint32_t s_keys[kTile];
  __shared__ uint16_t s_whist[kWarps][kRadix];   // per-warp digit counts, then prefixes (<= 8192)
  __shared__ uint32_t s_tileoff[kRadix];
  __shared__ uint32_t s_dstbase[kRadix];
  __shared__ uint32_t s_wsum[8];
  __shared__ uint32_t s_tile;

  grid_dependency_wait();
  if (skip_launch(a.run_if)) return;
  const SortArray A = blockIdx.y ? a.arr[1] : a.arr[0];   // (no dynamic indexing of the parameter block)
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t shift = a.shift;
  // Persistent blocks: tiles are handed out in ticket order, so a block only ever waits (look-back) for
  // tiles whose owners are already running.  A skipped launch (the fallback that is not needed) costs
  // a few hundred blocks that exit at once instead of one block per tile.
  for (;;) {
  __syncthreads();                                         // the previous tile of this block is done with shared memory
  if (tid == 0) s_tile = atomicAdd(A.ticket, 1u);
  for (int i = tid; i < kWarps * kRadix / 2; i += kThreads) reinterpret_cast<uint32_t*>(&s_whist[0][0])[i] = 0;
  __syncthreads();

  const uint32_t tile = s_tile;
  if (tile >= a.n_tiles) break;                            // block-uniform
  const uint32_t base = tile * (uint32_t)kTile;
  const uint32_t count = min((uint32_t)kTile, a.n - base);

  // ---- load: warp-striped, key order inside the tile = warp*512 + j*32 + lane ----
  uint32_t key[kKeysPerThread];
  {
    const uint32_t* __restrict__ src = A.src + base;
    const uint32_t w0 = warp * (32 * kKeysPerThread) + lane;
    if (count == (uint32_t)kTile) {
#pragma unroll
      for (int j = 0; j < kKeysPerThread; ++j) key[j] = src[w0 + j * 32];
    } else {
#pragma unroll
      for (int j = 0; j < kKeysPerThread; ++j) {
        const uint32_t i = w0 + j * 32;
        key[j] = i < count ? src[i] : 0xffffffffu;   // padding: digit 255, last in tile order
      }
    }
  }

  // ---- rank inside the warp: stable, via match on the digit ----
  uint16_t rank[kKeysPerThread];
  const uint32_t lt_mask = (1u << lane) - 1u;
  uint16_t* wh = s_whist[warp];
#pragma unroll
  for (int j = 0; j < kKeysPerThread; ++j) {
    const uint32_t d = (key[j] >> shift) & 255u;
    const uint32_t m = __match_any_sync(kFullMask, d);
    const uint32_t below = __popc(m & lt_mask);
    const uint32_t prev = wh[d];
    __syncwarp();
    if (below == 0) wh[d] = (uint16_t)(prev + __popc(m));
    __syncwarp();
    rank[j] = (uint16_t)(prev + below);
  }
  __syncthreads();

  // ---- per digit: exclusive prefix over warps, tile count, tile offsets ----
  uint32_t cnt = 0;
  if (tid < kRadix) {
#pragma unroll
    for (int w = 0; w < kWarps; ++w) {
      const uint32_t c = s_whist[w][tid];
      s_whist[w][tid] = (uint16_t)cnt;
      cnt += c;
    }
  }
  const uint32_t tile_off = block_excl_scan_256(cnt, s_wsum);   // includes padding in digit 255
  if (tid < kRadix) s_tileoff[tid] = tile_off;
  if (tid == kRadix - 1) cnt -= (uint32_t)kTile - count;        // padding is not published

  // ---- chained scan with decoupled look-back, one digit per thread ----
  uint32_t digit_base = 0;
  if (tile == 0) {   // tile 0 folds the global digit base (exclusive scan of the histogram) in
    const uint32_t h = tid < kRadix ? A.hist[tid] : 0u;
    digit_base = block_excl_scan_256(h, s_wsum);
  }
  if (tid < kRadix) {
    uint64_t* st = A.status + (size_t)tile * kRadix + tid;
    uint32_t excl;
    if (tile == 0) {
      excl = digit_base;
      st_relaxed_u64(st, pack_status(a.epoch, kFlagIncl, excl + cnt));
    } else {
      st_relaxed_u64(st, pack_status(a.epoch, kFlagLocal, cnt));
      excl = 0;
      const uint64_t* p = st - kRadix;
      while (true) {
        const uint64_t v = ld_relaxed_u64(p);
        if ((uint32_t)(v >> 34) != a.epoch) continue;          // predecessor not published yet
        excl += (uint32_t)v;
        if ((v >> 32) & kFlagIncl) break;
        p -= kRadix;
      }
      st_relaxed_u64(st, pack_status(a.epoch, kFlagIncl, excl + cnt));
    }
    s_dstbase[tid] = excl - tile_off;   // final index = s_dstbase[d] + position in the sorted tile
  }
  __syncthreads();   // s_tileoff ready (s_dstbase too)

  // ---- scatter to shared memory in tile-sorted order ----
#pragma unroll
  for (int j = 0; j < kKeysPerThread; ++j) {
    const uint32_t d = (key[j] >> shift) & 255u;
    s_keys[s_tileoff[d] + wh[d] + rank[j]] = key[j];
  }
  __syncthreads();

  // ---- write out: runs of equal digits land contiguously ----
  uint32_t* __restrict__ dst = A.dst;
  if (count == (uint32_t)kTile) {
#pragma unroll
    for (int j = 0; j < kKeysPerThread; ++j) {
      const uint32_t i = tid + j * kThreads;
      const uint32_t k = s_keys[i];
      dst[s_dstbase[(k >> shift) & 255u] + i] = k;
    }
  } else {
    for (uint32_t i = tid; i < count; i += kThreads) {
      const uint32_t k = s_keys[i];
      dst[s_dstbase[(k >> shift) & 255u] + i] = k;
    }
  }
  }   // tile loop
}

}  // namespace rs
}  // namespace bits
