// mc_small.cuh -- the Monte Carlo round with the SEARCHED set re-placed (BITS_PERMUTE_B) for SMALL sets:
// one block per round, everything in shared memory, many rounds per launch.
//
// every round "a random interval set is generated and placed into the associated data
// structure" (place -> Sort(B_S), Sort(B_E) -> one ICOUNT per query -> sum).  With a few thousand intervals the
// two launches per round of mc_tile.cuh are bound by launch latency (BASELINE.json configs[0]: 1,000 intervals);
// here a block of 512 threads does a whole round -- Philox placement into shared memory, a counting sort of the
// starts and of the ends on their top 13 significant bits (the cursor machinery of mc_tile.cuh), the rank of every
// (once sorted) query key against them, the sum -- and the grid strides over the rounds of the call.  The sorted
// arrays B_S and B_E are written out for the LAST round of the call only (bits_workspace_sorted_offset).
#pragma once
#include "mc_tile.cuh"

namespace bits {
namespace mcs {

using Cfg = mct::BinCfgWide;                       // 512 threads, 8,192 keys, 2^13 sub-buckets, two blocks per SM
constexpr uint32_t kMaxKeys = Cfg::kCap - 4;        // room for the sentinels behind the keys
constexpr size_t kSmem = Cfg::kSmemFixed + (size_t)(kMaxChromSmem) * sizeof(uint32_t) + (size_t)kLutSize * sizeof(uint16_t);

struct SmallArgs {
  const uint32_t* spans;           // dev uint32[align_up(n, 4)], zero padded
  uint32_t n;                      // intervals of the re-placed set, <= kMaxKeys
  uint32_t tag;
  uint32_t round0;                 // round of output position 0
  uint32_t n_rounds;
  uint32_t sshift;                 // sub-bucket = key >> sshift < 2^13 for every coordinate of the genome
  PhiloxKeys key;
  ChromTable chrom;
  const uint32_t* q_sorted[2];     // ascending: A's ends (ranked in B_S, "<="), A's starts (ranked in B_E, "<")
  uint32_t n_q;
  uint32_t* dst[2];                // B_S, B_E of the call's last round
  unsigned long long* round_counts;   // [n_rounds], zero on entry
};

// sum over the sorted queries of #{keys <= q} (kStrict: < q); buf is grouped by sub-bucket, cur holds the groups' ends
template <bool kStrict>
__device__ __forceinline__ uint64_t rank_sum(const uint32_t* buf, const uint16_t* cur, uint32_t sshift,
                                             const uint32_t* __restrict__ q_sorted, uint32_t n_q) {
  uint64_t sum = 0;
  for (uint32_t qi = threadIdx.x; qi < n_q; qi += Cfg::kThreads) {
    const uint32_t q = __ldg(q_sorted + qi);
    const uint32_t sb = min(q >> sshift, (uint32_t)Cfg::kSub - 1u);     // (a query beyond the genome's end: past every key)
    const uint32_t lo = cur[mct::kFront - 1 + sb], hi = cur[mct::kFront + sb];
    uint32_t c = lo;
    for (uint32_t t = lo; t < hi; ++t) c += kStrict ? (buf[t] < q) : (buf[t] <= q);
    sum += c;
  }
  return sum;
}

__global__ void __launch_bounds__(Cfg::kThreads, Cfg::kBlocksPerSm) mc_small_b_kernel(SmallArgs a) {
  extern __shared__ __align__(16) uint8_t smem_raw[];
  uint32_t* s_ks = reinterpret_cast<uint32_t*>(smem_raw);                // [kCap] starts
  uint32_t* s_ke = s_ks + Cfg::kCap;                                      // [kCap] ends
  uint16_t* s_cur_s = reinterpret_cast<uint16_t*>(s_ke + Cfg::kCap);      // [kCurLen]
  uint16_t* s_cur_e = s_cur_s + Cfg::kCurLen;                             // [kCurLen]
  uint32_t* s_off = reinterpret_cast<uint32_t*>(s_cur_e + Cfg::kCurLen);  // [kMaxChromSmem]
  uint16_t* s_lut = reinterpret_cast<uint16_t*>(s_off + kMaxChromSmem);   // [kLutSize]
  __shared__ uint32_t s_w[32];
  __shared__ uint64_t s_red[Cfg::kThreads / 32];
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const ChromView off = stage_chrom_table(a.chrom, s_off, s_lut);        // barrier inside
  const uint32_t mask = 0xffffffffu, sshift = a.sshift, n = a.n;
  for (uint32_t k = blockIdx.x; k < a.n_rounds; k += gridDim.x) {
    __syncthreads();                                                     // everyone is done with the previous round's buffers
    for (int i = tid; i < 2 * Cfg::kCurLen / 8; i += Cfg::kThreads) reinterpret_cast<uint4*>(s_cur_s)[i] = make_uint4(0, 0, 0, 0);
    // place: four intervals per step, two Philox calls
    for (uint32_t i0 = 4u * tid; i0 < n; i0 += 4u * Cfg::kThreads) {
      const uint4 d4 = __ldg(reinterpret_cast<const uint4*>(a.spans + i0));
      const uint32_t d[4] = {d4.x, d4.y, d4.z, d4.w};
      uint32_t st[4];
      place4(i0, a.round0 + k, a.tag, a.key, d, off, a.chrom, st);
#pragma unroll
      for (int j = 0; j < 4; ++j)
        if (i0 + j < n) { s_ks[i0 + j] = st[j]; s_ke[i0 + j] = st[j] + d[j]; }
    }
    __syncthreads();
    // Sort(B_S), Sort(B_E): count, scan, scatter through the cursors
    {
      uint32_t* cs = reinterpret_cast<uint32_t*>(s_cur_s);
      uint32_t* ce = reinterpret_cast<uint32_t*>(s_cur_e);
      for (uint32_t i = tid; i < n; i += Cfg::kThreads) {
        mct::count_key(cs, s_ks[i] >> sshift);
        mct::count_key(ce, s_ke[i] >> sshift);
      }
    }
    __syncthreads();
    uint32_t total[2];
    mct::scan_cursors<Cfg>(s_cur_s, s_cur_e, s_w, total);                 // barriers inside
    mct::scatter_in_place<Cfg, false, false>(s_ks, n, 0u, 0u, mask, sshift, s_cur_s, n);
    mct::scatter_in_place<Cfg, false>(s_ke, n, 0u, 0u, mask, sshift, s_cur_e, n);
    if (k + 1 == a.n_rounds) {            // (block-uniform) the last round leaves B_S and B_E behind, in order (no queries in these calls)
      mct::write_and_rank<Cfg, false>(s_ks, n, mask, sshift, s_cur_s, 0u, a.dst[0], a.q_sorted[0], 0u, 0u, 0u);
      mct::write_and_rank<Cfg, true>(s_ke, n, mask, sshift, s_cur_e, 0u, a.dst[1], a.q_sorted[1], 0u, 0u, 0u);
    }
    uint64_t qsum = rank_sum<false>(s_ks, s_cur_s, sshift, a.q_sorted[0], a.n_q);
    qsum -= rank_sum<true>(s_ke, s_cur_e, sshift, a.q_sorted[1], a.n_q);
    // reduce: two's-complement partial sums, the block's total is non-negative
    qsum = warp_sum_u64(qsum);
    __syncthreads();
    if (lane == 0) s_red[w] = qsum;
    __syncthreads();
    if (w == 0) {
      uint64_t t = lane < Cfg::kThreads / 32 ? s_red[lane] : 0;
      t = warp_sum_u64(t);
      if (lane == 0) a.round_counts[k] = t;
    }
  }
}

}  // namespace mcs
}  // namespace bits
