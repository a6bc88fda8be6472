// place_kernels.cuh -- array-producing placement kernels (the "place" row when the SEARCHED set
// is re-placed: "a random interval set is generated and placed into the
// associated data structure" every round).  Optionally fused with the radix sort's up-front
// digit histograms of the freshly made start and end keys, which saves one read of both arrays.
#pragma once
#include "philox_place.cuh"
#include "radix_sort.cuh"
#include "msd_sort.cuh"

namespace bits {

// spans[i] = end[i] - start[i]; also the maximum span (for the NO_PLACEMENT check) and the sum of
// the spans (their mean sizes the fused Monte Carlo path).  Output padded to a multiple of 4 with zeros.
__global__ void __launch_bounds__(256) spans_kernel(const uint32_t* __restrict__ start, const uint32_t* __restrict__ end,
                                                    uint32_t n, uint32_t* __restrict__ spans, uint32_t* max_span,
                                                    unsigned long long* span_sum) {
  uint32_t m = 0;
  uint64_t sum = 0;
  const uint64_t n_pad = align_up(n, 4);
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_pad; i += (uint64_t)gridDim.x * blockDim.x) {
    const uint32_t d = i < n ? end[i] - start[i] : 0u;
    spans[i] = d;
    m = max(m, d);
    sum += d;
  }
  m = __reduce_max_sync(kFullMask, m);
  sum = warp_sum_u64(sum);
  if ((threadIdx.x & 31) == 0 && m) { atomicMax(max_span, m); atomicAdd(span_sum, (unsigned long long)sum); }
}

// flag |= 1 if any start > end
__global__ void __launch_bounds__(256) validate_kernel(const uint32_t* __restrict__ start, const uint32_t* __restrict__ end,
                                                       uint32_t n, uint32_t* flag) {
  bool bad = false;
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x)
    bad |= start[i] > end[i];
  if (__any_sync(kFullMask, bad) && (threadIdx.x & 31) == 0) atomicOr(flag, 1u);
}

struct PlaceArgs {
  const uint32_t* spans;   // dev uint32[n], readable up to align_up(n,4) when kVec
  uint32_t* start_out;
  uint32_t* end_out;
  uint32_t n;
  uint32_t round;
  uint32_t tag;
  PhiloxKeys key;
  ChromTable chrom;
  uint32_t* hist_start;    // kHistDigits: uint32[4][256], kHistBins: uint32[msd::kBins] -- global histograms to add into
  uint32_t* hist_end;
  uint32_t* zero_a;        // kHistDigits: 2 x uint32[4][256] to clear for the NEXT round (block 0), or null
  uint32_t* zero_b;
};

// which histogram of the freshly made keys the placement kernel accumulates
enum { kHistNone = 0, kHistDigits = 1, kHistBins = 2 };

// Four intervals per thread.  kVec: all three arrays 16-byte aligned and padded to a multiple
// of four elements (the library's own workspace buffers); otherwise scalar accesses.
// kHist: kHistDigits = the LSD sort's four 8-bit digit histograms, kHistBins = the MSD sort's
// histogram of the top msd::kBinBits bits (one shared-memory atomic per key).
template <bool kVec, int kHist>
__global__ void __launch_bounds__(256) place_kernel(PlaceArgs a) {
  constexpr int kHalf = kHist == kHistDigits ? rs::kPasses * rs::kRadix : (kHist == kHistBins ? msd::kBins : 1);
  __shared__ uint32_t s_off[kMaxChromSmem];
  __shared__ __align__(16) uint16_t s_lut[kLutSize];
  __shared__ uint32_t s_h[kHist != kHistNone ? 2 * kHalf : 1];
  if (kHist != kHistNone) {
    for (int i = threadIdx.x; i < 2 * kHalf; i += blockDim.x) s_h[i] = 0;
    if (kHist == kHistDigits && blockIdx.x == 0 && a.zero_a)
      for (int i = threadIdx.x; i < kHalf; i += blockDim.x) { a.zero_a[i] = 0; a.zero_b[i] = 0; }
  }
  const ChromView off = stage_chrom_table(a.chrom, s_off, s_lut);   // barrier inside
  const uint32_t n = a.n;
  const uint32_t n4 = (uint32_t)(((uint64_t)n + 3) >> 2);
  for (uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; t < n4; t += (uint64_t)gridDim.x * blockDim.x) {
    const uint64_t i0 = t << 2;
    uint32_t d[4], st[4];
    if (kVec) {
      const uint4 d4 = __ldg(reinterpret_cast<const uint4*>(a.spans) + t);
      d[0] = d4.x; d[1] = d4.y; d[2] = d4.z; d[3] = d4.w;
    } else {
#pragma unroll
      for (int j = 0; j < 4; ++j) d[j] = i0 + j < n ? a.spans[i0 + j] : 0u;
    }
    place4((uint32_t)i0, a.round, a.tag, a.key, d, off, a.chrom, st);
    uint32_t en[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) en[j] = st[j] + d[j];
    if (kVec) {
      reinterpret_cast<uint4*>(a.start_out)[t] = make_uint4(st[0], st[1], st[2], st[3]);
      reinterpret_cast<uint4*>(a.end_out)[t] = make_uint4(en[0], en[1], en[2], en[3]);
    } else {
#pragma unroll
      for (int j = 0; j < 4; ++j)
        if (i0 + j < n) { a.start_out[i0 + j] = st[j]; a.end_out[i0 + j] = en[j]; }
    }
    if (kHist != kHistNone) {
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        if (i0 + j < n) {
          if (kHist == kHistDigits) {
#pragma unroll
            for (int p = 0; p < rs::kPasses; ++p) {
              atomicAdd(&s_h[p * rs::kRadix + ((st[j] >> (8 * p)) & 255u)], 1u);
              atomicAdd(&s_h[kHalf + p * rs::kRadix + ((en[j] >> (8 * p)) & 255u)], 1u);
            }
          } else {
            atomicAdd(&s_h[st[j] >> msd::kBinShift], 1u);
            atomicAdd(&s_h[kHalf + (en[j] >> msd::kBinShift)], 1u);
          }
        }
      }
    }
  }
  if (kHist != kHistNone) {
    __syncthreads();
    for (int i = threadIdx.x; i < kHalf; i += blockDim.x) {
      if (s_h[i]) atomicAdd(&a.hist_start[i], s_h[i]);
      if (s_h[kHalf + i]) atomicAdd(&a.hist_end[i], s_h[kHalf + i]);
    }
  }
}

}  // namespace bits
