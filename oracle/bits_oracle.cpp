// bits_oracle.cpp — CPU ORACLE for the BITS hot path (arXiv 1208.3407).
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
// header, table or constant generator with paper_1208_3407_b200/csrc (the CUDA path).
//
// Plain, single-threaded C++17: std::sort + std::upper_bound / std::lower_bound and its
// own Philox4x32-10.  No blocking, fusion or reordering beyond what the paper states, so
// each function can be checked against PAPER.md by eye.
//
// What each function follows
//   oracle_count_per_interval  Algorithm 1 ICOUNT inside Algorithm 2
//                              COUNTER; ranks as fixed by the set
//                              definitions L, R:
//                                first = #{b.start <= a.end} = upper_bound(B_S, a.end)
//                                last  = #{b.end   <  a.start} = lower_bound(B_E, a.start)
//                                c = first - last.
//   oracle_sort_u32            Sort(B_S), Sort(B_E) of Algorithm 2.
//   oracle_philox4x32_10       the counter-based generator that stands in for the paper's
//                              unspecified parallel RNG; Salmon et al. SC'11.
//   oracle_place_from_bits,    the Monte Carlo re-placement of PAPER.md:155-157 §3.2
//   oracle_place_round         ("uniformly distributed random interval set", "only an
//                              array of random starts must be generated"), with lengths
//                              kept and chromosome ends respected (DESIGN.md readings
//                              R10-R12).
//   oracle_mc_rounds           the Monte Carlo loop of PAPER.md:157-159.
//   oracle_mc_rounds_stream    the same with the fourth Philox counter word given (the pair id of
//                              the many-pair screen; the screen itself is the
//                              loop over ordered pairs in oracle/__init__.py).
//   oracle_pvalue              add-one empirical p (reading R13; the paper gives
//                              no formula).
//
// Pins (tests/test_oracle_pins.py, -m "not gpu"): O(N*M) brute force from the closed
// predicate, shared-endpoint cases, closed forms, the exclusion identity,
// invariants, Philox known-answer vectors + cuRAND's header routine, Python big-integer
// multiply-high, placement structure and the closed-form hit probability.
// PARITY UNPINNED BY THE PAPER: per-round Monte Carlo counts (the paper prints no counts
// and does not specify its RNG); pinned only by the procedure + brute force on config 1.
#include <algorithm>
#include <cmath>
#include <limits>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

// ---- Philox4x32-10 (own implementation; ten rounds, two 32x32->64 products per round) ----
constexpr uint32_t kM0 = 0xD2511F53u, kM1 = 0xCD9E8D57u;
constexpr uint32_t kW0 = 0x9E3779B9u, kW1 = 0xBB67AE85u;

inline void philox_round(uint32_t c[4], const uint32_t k[2]) {
  const uint64_t p0 = static_cast<uint64_t>(kM0) * c[0];
  const uint64_t p1 = static_cast<uint64_t>(kM1) * c[2];
  const uint32_t n0 = static_cast<uint32_t>(p1 >> 32) ^ c[1] ^ k[0];
  const uint32_t n1 = static_cast<uint32_t>(p1);
  const uint32_t n2 = static_cast<uint32_t>(p0 >> 32) ^ c[3] ^ k[1];
  const uint32_t n3 = static_cast<uint32_t>(p0);
  c[0] = n0; c[1] = n1; c[2] = n2; c[3] = n3;
}

inline void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c[4] = {ctr[0], ctr[1], ctr[2], ctr[3]};
  uint32_t k[2] = {key[0], key[1]};
  for (int r = 0; r < 10; ++r) {
    if (r > 0) { k[0] += kW0; k[1] += kW1; }
    philox_round(c, k);
  }
  out[0] = c[0]; out[1] = c[1]; out[2] = c[2]; out[3] = c[3];
}

// ---- placement: x (64 random bits), span d -> start; SURVEY §8c step 3 ----
// returns 0 on success, 1 if no chromosome can hold the span.
inline int place_from_bits(uint64_t x, uint32_t d, const uint32_t* off, uint32_t n_chrom,
                           uint32_t* start_out) {
  uint64_t V = 0;
  for (uint32_t c = 0; c < n_chrom; ++c) {
    const uint64_t L = static_cast<uint64_t>(off[c + 1]) - off[c];
    V += (L > d) ? (L - d) : 0;
  }
  if (V == 0) return 1;
  uint64_t u = static_cast<uint64_t>((static_cast<unsigned __int128>(x) * V) >> 64);
  for (uint32_t c = 0; c < n_chrom; ++c) {
    const uint64_t L = static_cast<uint64_t>(off[c + 1]) - off[c];
    const uint64_t v = (L > d) ? (L - d) : 0;
    if (u < v) { *start_out = static_cast<uint32_t>(off[c] + u); return 0; }
    u -= v;
  }
  return 1;  // unreachable: u < V
}

// `stream` is the fourth counter word: 0 for a single Monte Carlo job, the pair id inside the many-pair
// screen (SURVEY.md section 8(f).3 reserves it; readings R11, R24).
inline int place_round(const uint32_t* spans, uint64_t n, const uint32_t* off, uint32_t n_chrom,
                       uint64_t seed, uint32_t round, uint32_t tag, uint32_t stream,
                       uint32_t* start_out, uint32_t* end_out) {
  const uint32_t key[2] = {static_cast<uint32_t>(seed & 0xffffffffu), static_cast<uint32_t>(seed >> 32)};
  for (uint64_t i = 0; i < n; ++i) {
    const uint32_t ctr[4] = {static_cast<uint32_t>(i >> 1), round, tag, stream};
    uint32_t o[4];
    philox4x32_10(ctr, key, o);
    const uint32_t h = static_cast<uint32_t>(i & 1);
    const uint64_t x = static_cast<uint64_t>(o[2 * h]) | (static_cast<uint64_t>(o[2 * h + 1]) << 32);
    uint32_t s;
    if (place_from_bits(x, spans[i], off, n_chrom, &s)) return 1;
    start_out[i] = s;
    end_out[i] = s + spans[i];
  }
  return 0;
}

// ---- counting: Algorithm 1 + 2 on already sorted B_S, B_E ----
inline uint64_t count_sorted(const uint32_t* a_start, const uint32_t* a_end, uint64_t n_a,
                             const std::vector<uint32_t>& BS, const std::vector<uint32_t>& BE,
                             uint32_t* counts_out) {
  uint64_t total = 0;
  for (uint64_t i = 0; i < n_a; ++i) {
    const uint64_t first = std::upper_bound(BS.begin(), BS.end(), a_end[i]) - BS.begin();
    const uint64_t last = std::lower_bound(BE.begin(), BE.end(), a_start[i]) - BE.begin();
    const uint32_t c = static_cast<uint32_t>(first - last);
    if (counts_out) counts_out[i] = c;
    total += c;
  }
  return total;
}

inline bool well_formed(const uint32_t* s, const uint32_t* e, uint64_t n) {
  for (uint64_t i = 0; i < n; ++i) if (s[i] > e[i]) return false;
  return true;
}

}  // namespace

extern "C" {

enum { ORACLE_OK = 0, ORACLE_ERR_MALFORMED = 1, ORACLE_ERR_NO_PLACEMENT = 2, ORACLE_ERR_ARG = 3 };

int oracle_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) {
  philox4x32_10(ctr, key, out);
  return ORACLE_OK;
}

int oracle_sort_u32(uint32_t* keys, uint64_t n) {
  std::sort(keys, keys + n);
  return ORACLE_OK;
}

// counts_out may be NULL.  Per-interval counts are in A's input order.
int oracle_count_per_interval(const uint32_t* a_start, const uint32_t* a_end, uint64_t n_a,
                              const uint32_t* b_start, const uint32_t* b_end, uint64_t n_b,
                              uint32_t* counts_out, uint64_t* total_out) {
  if (!well_formed(a_start, a_end, n_a) || !well_formed(b_start, b_end, n_b)) return ORACLE_ERR_MALFORMED;
  std::vector<uint32_t> BS(b_start, b_start + n_b), BE(b_end, b_end + n_b);
  std::sort(BS.begin(), BS.end());
  std::sort(BE.begin(), BE.end());
  *total_out = count_sorted(a_start, a_end, n_a, BS, BE, counts_out);
  return ORACLE_OK;
}

int oracle_place_from_bits(uint64_t x, uint32_t d, const uint32_t* off, uint32_t n_chrom,
                           uint32_t* start_out) {
  return place_from_bits(x, d, off, n_chrom, start_out) ? ORACLE_ERR_NO_PLACEMENT : ORACLE_OK;
}

int oracle_place_round_stream(const uint32_t* spans, uint64_t n, const uint32_t* off, uint32_t n_chrom,
                              uint64_t seed, uint32_t round, uint32_t tag, uint32_t stream,
                              uint32_t* start_out, uint32_t* end_out) {
  return place_round(spans, n, off, n_chrom, seed, round, tag, stream, start_out, end_out)
             ? ORACLE_ERR_NO_PLACEMENT : ORACLE_OK;
}

int oracle_place_round(const uint32_t* spans, uint64_t n, const uint32_t* off, uint32_t n_chrom,
                       uint64_t seed, uint32_t round, uint32_t tag,
                       uint32_t* start_out, uint32_t* end_out) {
  return oracle_place_round_stream(spans, n, off, n_chrom, seed, round, tag, 0u, start_out, end_out);
}

// which: 0 = re-place A (queries; B sorted once), 1 = re-place B (searched set; re-sorted every round).
// stream: the fourth Philox counter word of every draw (0 = a single job; pair id in the screen).
int oracle_mc_rounds_stream(const uint32_t* a_start, const uint32_t* a_end, uint64_t n_a,
                            const uint32_t* b_start, const uint32_t* b_end, uint64_t n_b,
                            const uint32_t* off, uint32_t n_chrom, int which, uint64_t seed, uint32_t stream,
                            uint32_t round_begin, uint32_t n_rounds,
                            uint64_t* observed_out, uint64_t* round_counts_out) {
  if (which != 0 && which != 1) return ORACLE_ERR_ARG;
  if (!well_formed(a_start, a_end, n_a) || !well_formed(b_start, b_end, n_b)) return ORACLE_ERR_MALFORMED;
  // 1. observed = total(A, B)
  std::vector<uint32_t> BS(b_start, b_start + n_b), BE(b_end, b_end + n_b);
  std::sort(BS.begin(), BS.end());
  std::sort(BE.begin(), BE.end());
  *observed_out = count_sorted(a_start, a_end, n_a, BS, BE, nullptr);
  // 2. spans of the permuted set
  const uint64_t n_p = which == 0 ? n_a : n_b;
  const uint32_t* ps = which == 0 ? a_start : b_start;
  const uint32_t* pe = which == 0 ? a_end : b_end;
  std::vector<uint32_t> spans(n_p), s2(n_p), e2(n_p);
  for (uint64_t i = 0; i < n_p; ++i) spans[i] = pe[i] - ps[i];
  // 3-4. rounds
  for (uint32_t k = 0; k < n_rounds; ++k) {
    const uint32_t r = round_begin + k;
    if (n_p && place_round(spans.data(), n_p, off, n_chrom, seed, r, static_cast<uint32_t>(which), stream,
                           s2.data(), e2.data()))
      return ORACLE_ERR_NO_PLACEMENT;
    if (which == 0) {
      round_counts_out[k] = count_sorted(s2.data(), e2.data(), n_p, BS, BE, nullptr);
    } else {
      std::vector<uint32_t> PS(s2), PE(e2);
      std::sort(PS.begin(), PS.end());
      std::sort(PE.begin(), PE.end());
      round_counts_out[k] = count_sorted(a_start, a_end, n_a, PS, PE, nullptr);
    }
  }
  return ORACLE_OK;
}

int oracle_mc_rounds(const uint32_t* a_start, const uint32_t* a_end, uint64_t n_a,
                     const uint32_t* b_start, const uint32_t* b_end, uint64_t n_b,
                     const uint32_t* off, uint32_t n_chrom, int which, uint64_t seed,
                     uint32_t round_begin, uint32_t n_rounds,
                     uint64_t* observed_out, uint64_t* round_counts_out) {
  return oracle_mc_rounds_stream(a_start, a_end, n_a, b_start, b_end, n_b, off, n_chrom, which, seed, 0u,
                                 round_begin, n_rounds, observed_out, round_counts_out);
}

// tail 0: p_enrich = (#{count_r >= observed} + 1) / (R + 1); tail 1: p_deplete with <=.
double oracle_pvalue(uint64_t observed, const uint64_t* round_counts, uint32_t n_rounds, int tail) {
  uint64_t k = 0;
  for (uint32_t r = 0; r < n_rounds; ++r)
    k += (tail == 0) ? (round_counts[r] >= observed) : (round_counts[r] <= observed);
  return static_cast<double>(k + 1) / static_cast<double>(static_cast<uint64_t>(n_rounds) + 1);
}

// Enrichment score of the screen (Fig. 3 caption :224): log2(observed / median of the
// round counts); median of an even number of rounds = mean of the two middle order statistics
// (reading R13).  Median 0: +inf if observed > 0, else NaN.
double oracle_enrichment(uint64_t observed, const uint64_t* round_counts, uint32_t n_rounds) {
  if (n_rounds == 0) return std::nan("");
  std::vector<uint64_t> v(round_counts, round_counts + n_rounds);
  std::sort(v.begin(), v.end());
  const double median = (n_rounds % 2) ? static_cast<double>(v[n_rounds / 2])
                                       : (static_cast<double>(v[n_rounds / 2 - 1]) + static_cast<double>(v[n_rounds / 2])) / 2.0;
  if (median == 0.0) return observed ? std::numeric_limits<double>::infinity() : std::nan("");
  return std::log2(static_cast<double>(observed) / median);
}

}  // extern "C"
