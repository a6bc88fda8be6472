// philox_place.cuh -- the "place" step: counter-based Philox4x32-10 + exact uniform placement.
//
// PAPER.md:155-157 (Sec. 3.2): per Monte Carlo round "only an array of random starts must be
// generated", lengths kept.  The paper's own RNG (a hash-based generator for its
// GPU) is unspecified; this build uses Philox4x32-10 (Salmon et al., SC'11) addressed by
// (seed, round, interval) -- DESIGN.md readings R10-R12.  Written for this library only; the CPU
// oracle has its own, separate implementation.
#pragma once
#include "common.cuh"

namespace bits {

constexpr int kMaxChromSmem = 1024;   // offset tables up to this many entries are staged in shared memory
constexpr int kLutSize = 1024;        // entries of the position -> chromosome look-up table

struct ChromTable {
  const uint32_t* off;   // dev uint32[n_chrom + 1]
  const uint16_t* lut;   // dev uint16[kLutSize]: lut[e] = chromosome that holds position e << lut_shift
  uint32_t n_chrom;
  uint32_t l_min;        // shortest chromosome: spans below it fit every chromosome (fast path)
  uint32_t genome;       // G = off[n_chrom]
  uint32_t step0;        // largest power of two <= max(n_chrom - 1, 1); 0 if n_chrom == 1
  uint32_t lut_shift;    // (G >> lut_shift) < kLutSize
};

// The offset table as a kernel searches it: in shared memory (with the look-up table) when it fits.
struct ChromView {
  const uint32_t* off;
  const uint16_t* lut;   // null: binary search
};

// lut[e] = #{c >= 1 : off[c] <= e << shift}, e = 0 .. G >> shift (host side, once per call).
inline uint32_t make_chrom_lut(const uint32_t* off, uint32_t n_chrom, uint16_t* lut) {
  const uint64_t G = off[n_chrom];
  uint32_t shift = 0;
  while ((G >> shift) >= (uint64_t)kLutSize) ++shift;
  uint32_t c = 0;
  for (uint32_t e = 0; e < (uint32_t)kLutSize; ++e) {
    const uint64_t pos = (uint64_t)e << shift;
    while (c + 1 < n_chrom && (uint64_t)off[c + 1] <= pos) ++c;
    lut[e] = (uint16_t)c;
  }
  return shift;
}

// The ten round keys (k0 + r*0x9E3779B9, k1 + r*0xBB67AE85), computed once on the host.
struct PhiloxKeys {
  uint32_t k0[10], k1[10];
};

inline PhiloxKeys make_philox_keys(uint64_t seed) {
  PhiloxKeys k;
  uint32_t a = (uint32_t)(seed & 0xffffffffu), b = (uint32_t)(seed >> 32);
  for (int r = 0; r < 10; ++r) {
    k.k0[r] = a; k.k1[r] = b;
    a += 0x9E3779B9u; b += 0xBB67AE85u;
  }
  return k;
}

// Philox4x32-10: ten rounds of two 32x32->64 multiplies and a word permutation.
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               const PhiloxKeys& key) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
    const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ key.k0[r];
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ key.k1[r];
    c1 = (uint32_t)p1; c3 = (uint32_t)p0; c0 = n0; c2 = n2;
  }
  return make_uint4(c0, c1, c2, c3);
}

// start' for 64 random bits (xl, xh) and span d.  `off` may point to shared or global memory.
// Fast path (d < l_min, every chromosome can hold the span): V = G - C*d < 2^32, the running
// count of valid starts before chromosome c is off[c] - c*d, so the chromosome is found by a
// fixed-trip binary search and start' = u + c*d.  General path: the literal walk in 64 bits.
__device__ __forceinline__ uint32_t place_start(uint32_t xl, uint32_t xh, uint32_t d, const ChromView& cv,
                                                const ChromTable& t) {
  const uint32_t* __restrict__ off = cv.off;
  if (d < t.l_min) {
    const uint32_t V = t.genome - t.n_chrom * d;
    // u = (x * V) >> 64 with x = xh:xl (64 bits) and V < 2^32
    const uint32_t carry = __umulhi(xl, V);
    const uint32_t u = (uint32_t)(((uint64_t)xh * V + carry) >> 32);
    uint32_t c = 0;
    if (cv.lut) {
      // the thresholds off[c] - c*d only move down as d grows, so the chromosome of u for d = 0
      // (read from the table at the start of u's block) is a lower bound: step up from there
      // (two steps without a loop -- almost always enough -- then the general loop)
      c = cv.lut[u >> t.lut_shift];
      const uint32_t o1 = off[c + 1], o2 = off[c + 2];                 // staged table: >= n_chrom + 2 words
      const bool s1 = c + 1 < t.n_chrom && o1 - (c + 1) * d <= u;
      const bool s2 = s1 && c + 2 < t.n_chrom && o2 - (c + 2) * d <= u;
      c += (uint32_t)s1 + (uint32_t)s2;
      if (s2)
        while (c + 1 < t.n_chrom && off[c + 1] - (c + 1) * d <= u) ++c;
    } else {
      for (uint32_t s = t.step0; s > 0; s >>= 1) {
        const uint32_t m = c + s;
        if (m < t.n_chrom && off[m] - m * d <= u) c = m;
      }
    }
    return u + c * d;
  }
  uint64_t V = 0;
  for (uint32_t c = 0; c < t.n_chrom; ++c) {
    const uint32_t L = off[c + 1] - off[c];
    V += L > d ? (uint64_t)(L - d) : 0ull;
  }
  const uint64_t x = ((uint64_t)xh << 32) | xl;
  uint64_t u = __umul64hi(x, V);
  uint32_t start = 0;
  for (uint32_t c = 0; c < t.n_chrom; ++c) {
    const uint32_t L = off[c + 1] - off[c];
    const uint64_t v = L > d ? (uint64_t)(L - d) : 0ull;
    if (u < v) { start = off[c] + (uint32_t)u; break; }
    u -= v;
  }
  return start;
}

// Stage the offset table (and the look-up table, s_lut = kLutSize entries) in shared memory when
// it fits; returns the view to search through.  Ends with __syncthreads().
__device__ __forceinline__ ChromView stage_chrom_table(const ChromTable& t, uint32_t* s_off, uint16_t* s_lut) {
  const bool fits = t.n_chrom + 2 <= (uint32_t)kMaxChromSmem;
  const bool with_lut = fits && t.lut != nullptr && s_lut != nullptr;
  if (fits)
    for (uint32_t i = threadIdx.x; i <= t.n_chrom; i += blockDim.x) s_off[i] = t.off[i];
  if (with_lut)
    for (uint32_t i = threadIdx.x; i < (uint32_t)kLutSize / 2; i += blockDim.x)
      reinterpret_cast<uint32_t*>(s_lut)[i] = reinterpret_cast<const uint32_t*>(t.lut)[i];
  __syncthreads();
  ChromView v;
  v.off = fits ? s_off : t.off;
  v.lut = with_lut ? s_lut : nullptr;
  return v;
}

// Four consecutive intervals i0..i0+3 (i0 % 4 == 0) of round `round`: two Philox calls.
// Interval i uses counter (i >> 1, round, tag, stream) and output words 2h, 2h+1 with h = i & 1;
// stream = 0 for a single Monte Carlo job, the pair id inside the many-pair screen (R11, R24).
__device__ __forceinline__ void place4(uint32_t i0, uint32_t round, uint32_t tag, const PhiloxKeys& key,
                                       const uint32_t d[4], const ChromView& off, const ChromTable& t,
                                       uint32_t start[4], uint32_t stream = 0u) {
  const uint4 r0 = philox4x32_10(i0 >> 1, round, tag, stream, key);
  const uint4 r1 = philox4x32_10((i0 >> 1) + 1u, round, tag, stream, key);
  start[0] = place_start(r0.x, r0.y, d[0], off, t);
  start[1] = place_start(r0.z, r0.w, d[1], off, t);
  start[2] = place_start(r1.x, r1.y, d[2], off, t);
  start[3] = place_start(r1.z, r1.w, d[3], off, t);
}

}  // namespace bits
