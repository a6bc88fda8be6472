// screen.cuh -- the many-pair co-localisation screen as ONE device job.
//
// PAPER.md:165-171 (Sec. 3.3): every pairwise comparison of K interval sets (159 tracks, 25,281 pairs)
// by the Monte Carlo simulation of Sec. 3.2 with 10,000 iterations; Fig. 3 caption (:224): the score
// of a pair is log2(observed / median of the simulated counts).
//
// Every track is sorted and indexed ONCE (B_S, B_E and their bucket indices stay in the workspace);
// then one grid covers (query tile of track i) x (partner track j) x (round): each block re-places
// 1,024 intervals of track i for its round (Philox4x32-10, counter (interval >> 1, round, 0, pair id
// i * K + j) -- every ordered pair has its own null draws, reading R24), counts them against
// track j (Algorithm 1's two rank look-ups) and adds its sum to the pair's round
// count.  Nothing is stored in between.  The observed counts come from the
// same grid with the tracks' own coordinates instead of placed ones.
#pragma once
#include "search.cuh"

namespace bits {
namespace scr {

constexpr int kThreads = 256;
constexpr int kTile = 4 * kThreads;      // query intervals per block

struct Track {
  const uint32_t* start;     // the caller's arrays (input order), n each
  const uint32_t* end;
  const uint32_t* spans;     // workspace: uint32[align_up(n, 4)], zero padded, 16-byte aligned
  const uint32_t* keys[2];   // workspace: B_S, B_E (padded with kPad sentinels)
  const uint32_t* idx[2];    // workspace: their bucket indices
  uint32_t n;
  uint32_t shift;
};

struct ScreenArgs {
  const Track* tracks;            // dev [n_tracks]
  const uint32_t* tile_track;     // dev [n_tiles]: the track each query tile belongs to
  const uint32_t* tile_first;     // dev [n_tracks]: first tile of each track
  uint32_t n_tracks;
  uint32_t round0;                // round of blockIdx.z == 0
  uint32_t out0;                  // its position in a pair's row of round_counts
  uint32_t n_rounds;              // row length of round_counts
  uint32_t rpb;                   // rounds a block serves for its (query tile, partner): gridDim.z = ceil(n_launch / rpb)
  uint32_t n_launch;              // rounds of this launch
  PhiloxKeys key;
  ChromTable chrom;
  unsigned long long* observed;       // dev [n_tracks * n_tracks]
  unsigned long long* round_counts;   // dev [n_tracks * n_tracks * n_rounds]
};

// grid = (query tiles of all tracks, partner track j, rounds of this launch)
template <bool kObserved>
__global__ void __launch_bounds__(kThreads) screen_kernel(ScreenArgs a) {
  __shared__ uint32_t s_off[kObserved ? 1 : kMaxChromSmem];
  __shared__ __align__(16) uint16_t s_lut[kObserved ? 8 : kLutSize];
  __shared__ uint64_t s_red[kThreads / 32];
  const uint32_t i = __ldg(a.tile_track + blockIdx.x), j = blockIdx.y;
  const Track ti = a.tracks[i], tj = a.tracks[j];
  if (tj.n == 0) return;                                  // nothing to intersect: the counts stay 0
  ChromView off;
  if (!kObserved) off = stage_chrom_table(a.chrom, s_off, s_lut);
  SortedSet bs, be;
  bs.keys = tj.keys[0]; bs.idx = tj.idx[0]; bs.n = tj.n; bs.shift = tj.shift;
  be.keys = tj.keys[1]; be.idx = tj.idx[1]; be.n = tj.n; be.shift = tj.shift;
  const uint32_t t = (blockIdx.x - __ldg(a.tile_first + i)) * kThreads + threadIdx.x;
  const uint32_t i0 = t << 2;
  const uint32_t pair = i * a.n_tracks + j;
  const bool active = i0 < ti.n;
  if (kObserved) {
    uint64_t sum = 0;
    if (active) {
#pragma unroll
      for (int q = 0; q < 4; ++q)
        if (i0 + q < ti.n) sum += icount(bs, be, __ldg(ti.start + i0 + q), __ldg(ti.end + i0 + q));
    }
    block_sum_atomic(sum, s_red, a.observed + pair);
    return;
  }
  // the staged chromosome table and the spans are paid once for a.rpb consecutive rounds; one atomicAdd per warp and round
  const uint4 d4 = active ? __ldg(reinterpret_cast<const uint4*>(ti.spans) + t) : make_uint4(0, 0, 0, 0);
  const uint32_t d[4] = {d4.x, d4.y, d4.z, d4.w};
  const uint32_t r_first = blockIdx.z * a.rpb, r_end = min(r_first + a.rpb, a.n_launch);
  unsigned long long* row = a.round_counts + (size_t)pair * a.n_rounds + a.out0;
  for (uint32_t r = r_first; r < r_end; ++r) {
    uint64_t sum = 0;
    if (active) {
      uint32_t st[4];
      place4(i0, a.round0 + r, 0u, a.key, d, off, a.chrom, st, pair);
#pragma unroll
      for (int q = 0; q < 4; ++q)
        if (i0 + q < ti.n) sum += icount(bs, be, st[q], st[q] + d[q]);
    }
    sum = warp_sum_u64(sum);
    if ((threadIdx.x & 31) == 0 && sum) atomicAdd(row + r, (unsigned long long)sum);
  }
}

// One round per block (grid = (query tiles of all tracks, partner track j, rounds of this launch)): for launches too
// small to give every block several rounds.
__global__ void __launch_bounds__(kThreads) screen_round_kernel(ScreenArgs a) {
  constexpr bool kObserved = false;
  __shared__ uint32_t s_off[kObserved ? 1 : kMaxChromSmem];
  __shared__ __align__(16) uint16_t s_lut[kObserved ? 8 : kLutSize];
  __shared__ uint64_t s_red[kThreads / 32];
  const uint32_t i = __ldg(a.tile_track + blockIdx.x), j = blockIdx.y;
  const Track ti = a.tracks[i], tj = a.tracks[j];
  if (tj.n == 0) return;                                  // nothing to intersect: the counts stay 0
  ChromView off;
  if (!kObserved) off = stage_chrom_table(a.chrom, s_off, s_lut);
  SortedSet bs, be;
  bs.keys = tj.keys[0]; bs.idx = tj.idx[0]; bs.n = tj.n; bs.shift = tj.shift;
  be.keys = tj.keys[1]; be.idx = tj.idx[1]; be.n = tj.n; be.shift = tj.shift;
  const uint32_t t = (blockIdx.x - __ldg(a.tile_first + i)) * kThreads + threadIdx.x;
  const uint32_t i0 = t << 2;
  const uint32_t pair = i * a.n_tracks + j;
  uint64_t sum = 0;
  if (i0 < ti.n) {
    if (kObserved) {
#pragma unroll
      for (int q = 0; q < 4; ++q)
        if (i0 + q < ti.n) sum += icount(bs, be, __ldg(ti.start + i0 + q), __ldg(ti.end + i0 + q));
    } else {
      const uint4 d4 = __ldg(reinterpret_cast<const uint4*>(ti.spans) + t);
      const uint32_t d[4] = {d4.x, d4.y, d4.z, d4.w};
      uint32_t st[4];
      place4(i0, a.round0 + blockIdx.z, 0u, a.key, d, off, a.chrom, st, pair);
#pragma unroll
      for (int q = 0; q < 4; ++q)
        if (i0 + q < ti.n) sum += icount(bs, be, st[q], st[q] + d[q]);
    }
  }
  unsigned long long* out = kObserved ? a.observed + pair
                                      : a.round_counts + (size_t)pair * a.n_rounds + a.out0 + blockIdx.z;
  block_sum_atomic(sum, s_red, out);
}



}  // namespace scr
}  // namespace bits
