/* bits.h -- C ABI of libbits_b200: the data-parallel hot path of the BITS method
 * (Binary Interval Search, arXiv 1208.3407) on one NVIDIA B200 (sm_100a).
 *
 * The path (PAPER.md = /root/reference/PAPER.md; see DESIGN.md for the readings taken):
 *   place   PAPER.md:155-157 (Sec. 3.2)  random re-placement of one interval set per Monte Carlo
 *           round: uniform random starts, lengths kept, chromosome ends respected.
 *   sort    PAPER.md:117-125 (Algorithm 2 COUNTER, "Sort(B_S); Sort(B_E)"), :101 (Sec. 2.1):
 *           B's starts and B's ends sorted ascending, each on its own.
 *   search  PAPER.md:93-99 (Algorithm 1 ICOUNT), :103-107: per query interval a,
 *           first = #{b in B : b.start <= a.end}, last = #{b in B : b.end < a.start},
 *           c(a) = first - last  (closed intervals).
 *   reduce  PAPER.md:111, :115, Algorithm 2: total = sum over a in A of c(a).
 *
 * Conventions
 *   - Coordinates are 0-based CLOSED intervals [start, end], start <= end, already projected to
 *     the 1-D genome: chromosome c occupies [off[c], off[c+1]-1].
 *   - "dev" pointers are CUDA device pointers owned by the caller; "host" pointers are ordinary
 *     host memory.  The library never allocates or frees device memory, and never writes to
 *     its inputs: all scratch lives in the caller's workspace (size from bits_workspace_bytes,
 *     256-byte aligned).  Workspace contents are undefined on entry and on return.
 *   - `stream` is a cudaStream_t (NULL = the legacy default stream).  The device-pointer entry
 *     points validate on the host, enqueue on `stream` and return; outputs are valid once the
 *     caller has synchronised the stream.  The *_host entry points copy in, run, copy out and
 *     synchronise `stream` before they return.
 *   - Every function returns a bits_status (0 = BITS_OK); no exceptions, no printing, no exit.
 *     On error no output is defined.  There is no CPU fallback: without a usable CUDA device
 *     the compute entry points return BITS_ERR_CUDA.
 *   - Sizes: n_a, n_b < 2^28 (268,435,456 intervals per set; larger sets are refused with BITS_ERR_SIZE -- element
 *     indices inside the kernels are 32-bit and some are scaled by up to 8 before use; the GPU tests go up to 2.5e7
 *     intervals).  Coordinates use the full uint32 range.  Degenerate sizes are legal: n_a == 0 or n_b == 0 gives total 0,
 *     all per-interval counts 0 and all round counts 0.
 *   - All results are integers: per-interval counts uint32, totals and round counts uint64.
 *   - Threads: the library keeps no state between calls except (a) the tuning knobs of
 *     bits_set_option and the event timers of bits_profile_read, which are THREAD-LOCAL (a host
 *     thread sees only the knobs it set itself), (b) the launch counter of bits_launch_count
 *     (atomic, process-wide) and (c) a per-device "kernel attributes are set" flag (atomic).
 *     Calls from different host threads are independent as long as their workspaces and streams are.
 *   - Devices: every call runs on the CUDA device that is current in the calling thread; pointers
 *     and stream must belong to it.  Any number of devices may be used from one process.
 */
#ifndef BITS_B200_H_
#define BITS_B200_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  BITS_OK = 0,
  BITS_ERR_NULL = 1,          /* a required pointer is NULL */
  BITS_ERR_SIZE = 2,          /* n_a or n_b >= 2^28, or n_rounds / round_begin overflow uint32 */
  BITS_ERR_GENOME = 3,        /* offset table: off[0] != 0, not strictly ascending, or n_chrom == 0 */
  BITS_ERR_NO_PLACEMENT = 4,  /* an interval of the permuted set is as long as every chromosome */
  BITS_ERR_WORKSPACE = 5,     /* workspace NULL, misaligned (256 B) or smaller than required */
  BITS_ERR_FLAGS = 6,         /* unknown flag bit, bad `which`, bad `fn`, bad `tail` */
  BITS_ERR_MALFORMED = 7,     /* BITS_VALIDATE: some start > end */
  BITS_ERR_CUDA = 8,          /* a CUDA call failed (including: no device) */
  BITS_ERR_STATIC_LIMIT = 9   /* bits_count_static only: the problem needs more scratch than the built-in array holds */
} bits_status;

/* flags */
enum {
  BITS_B_SORTED = 1u,   /* b_start / b_end already are B_S / B_E: each ascending on its own.  The
                           sort step is skipped (the arrays are read in place). */
  BITS_VALIDATE = 2u    /* check start <= end for every interval of A and B first; synchronises
                           the stream once.  Without it malformed input gives undefined counts. */
};

/* `which` of bits_mc_rounds: the set that is re-placed each round */
enum {
  BITS_PERMUTE_A = 0,   /* queries re-placed; B sorted once (BASELINE.json configs[2]) */
  BITS_PERMUTE_B = 1    /* the searched set re-placed and re-sorted every round
                           (BASELINE.json configs[4]) */
};

/* `fn` of bits_workspace_bytes */
enum {
  BITS_FN_COUNT = 0,
  BITS_FN_COUNT_PER_INTERVAL = 1,
  BITS_FN_MC_ROUNDS = 2,
  BITS_FN_PLACE = 3,
  BITS_FN_SORT = 4,
  BITS_FN_ENUMERATE = 5
};

/* Bytes of device workspace `fn` needs for these sizes (device-pointer entry points).
 * `which` matters only for BITS_FN_MC_ROUNDS; n_chrom only for MC_ROUNDS and PLACE; for
 * BITS_FN_SORT n_b is the key count (n_a ignored).  Add bits_host_staging_bytes for *_host.
 * The size is NOT monotone in the set sizes (a small re-placed set gets room for several rounds per
 * launch): size a workspace that is shared between calls by the maximum over the calls.
 * BITS_FN_COUNT / COUNT_PER_INTERVAL: four key buffers of n_b plus sort bookkeeping (about 19 bytes per interval
 * of B); only where the call can bin the queries by B's buckets -- n_a >= 2^20 and n_b >= 3 * 2^20, `flags` without
 * BITS_B_SORTED -- another 8 (COUNT) or 12 (COUNT_PER_INTERVAL) bytes per query.  Pass the flags the call will get;
 * the study knobs count_binned / sort_msd (bits_set_option) change this rule, so size after setting them.
 * Returns 0 for an unknown fn. */
size_t bits_workspace_bytes(int fn, uint64_t n_a, uint64_t n_b, uint32_t n_chrom, int which,
                            uint32_t flags);

/* Where, inside a workspace of bits_workspace_bytes(fn, ...) bytes, the call leaves the sorted
 * arrays it searched (Algorithm 2's B_S and B_E): array 0 = B_S (ascending
 * starts), 1 = B_E (ascending ends), n_b keys each, valid once the stream has drained.  After
 * bits_mc_rounds with BITS_PERMUTE_B they are those of the LAST round.  For inspection and for
 * the parity tests of the sort step inside the Monte Carlo loop.  *offset_out: host, bytes.
 * Returns BITS_ERR_FLAGS for an fn that sorts no interval set or a bad array. */
int bits_workspace_sorted_offset(int fn, uint64_t n_a, uint64_t n_b, uint32_t n_chrom, int which,
                                 int array, size_t* offset_out);

/* Extra device bytes the *_host variant of `fn` needs to stage its inputs and outputs. */
size_t bits_host_staging_bytes(int fn, uint64_t n_a, uint64_t n_b, uint32_t n_rounds);

/* Counting problem (Algorithm 2):
 *   *total_out = |{(a,b) in A x B : a.start <= b.end and a.end >= b.start}|.
 * a_start, a_end: dev uint32[n_a]; b_start, b_end: dev uint32[n_b]; total_out: dev uint64[1]. */
int bits_count(const uint32_t* a_start, const uint32_t* a_end, uint64_t n_a,
               const uint32_t* b_start, const uint32_t* b_end, uint64_t n_b,
               uint32_t flags, void* workspace, size_t workspace_bytes,
               uint64_t* total_out, void* stream);

/* The counting problem for a caller that cannot supply a workspace.
 *
 * Every other compute entry point takes its scratch from a caller-allocated device workspace.  Some callers
 * have no way to make one: they are handed their input and output buffers by somebody else and may not, or
 * cannot, create device memory themselves.  Typical cases: a processing stage plugged into a host application
 * that owns the whole device-memory pool and gives a stage nothing but its buffers; code on a latency-critical
 * path where cudaMalloc / cudaFree are banned because they synchronise the whole device; a process on a GPU whose
 * memory another framework's caching allocator has already claimed, so that a fresh cudaMalloc would fail.
 * bits_count_static serves them: same result as bits_count (Algorithm 2), same kernels in the
 * same order, but the scratch is an array of BITS_STATIC_SCRATCH_BYTES that is part of the library's device image.
 * The call makes no cudaMalloc / cudaFree and no CUDA call that allocates (it also runs with the "profile" event
 * timers paused, because those create events); the caller passes inputs and the output only.
 *
 * Cost and limit: every GPU on which the library is used holds those BITS_STATIC_SCRATCH_BYTES (32 MiB) from the
 * moment the library's device code is loaded there until the process ends, whether or not this function is ever
 * called.  The problem must fit: bits_workspace_bytes(BITS_FN_COUNT, n_a, n_b, 0, 0, flags) <=
 * BITS_STATIC_SCRATCH_BYTES -- about 19 bytes per interval of B, so up to about 1.75 million intervals in B with any
 * number of queries (10^6 x 10^6 intervals take 17.9 MiB; n_b = 2*10^6 does not fit).  A larger problem is refused
 * with BITS_ERR_STATIC_LIMIT before anything is enqueued; nothing is truncated.
 *
 * Set-up: the first call on each device asks the CUDA runtime for the array's device address
 * (cudaGetSymbolAddress, with that device current) and keeps it; the return code is checked (BITS_ERR_CUDA).
 * Make that first call per device outside any stream capture.
 *
 * Sharing: there is ONE array per device and every call uses it, from whichever host thread or stream.  Two calls
 * whose GPU work overlaps in time (different streams, or different threads without ordering between them) race
 * on it and give undefined counts; calls enqueued one after the other on the same stream are safe.  The array
 * keeps what the last call left there; each call clears on `stream` whatever it needs zeroed before use.
 *
 * Arguments, flags, errors and synchronisation otherwise as bits_count. */
#define BITS_STATIC_SCRATCH_BYTES (32u << 20)
int bits_count_static(const uint32_t* a_start, const uint32_t* a_end, uint64_t n_a,
                      const uint32_t* b_start, const uint32_t* b_end, uint64_t n_b,
                      uint32_t flags, uint64_t* total_out, void* stream);

/* Decision problem (PAPER.md:47, sub-problem 1; :91): *any_out = 1 if at least one interval of A
 * intersects an interval of B, else 0 (dev uint32[1]).  Same inputs, workspace (BITS_FN_COUNT) and
 * flags as bits_count; the search stops early once an intersection is found. */
int bits_decide(const uint32_t* a_start, const uint32_t* a_end, uint64_t n_a,
                const uint32_t* b_start, const uint32_t* b_end, uint64_t n_b,
                uint32_t flags, void* workspace, size_t workspace_bytes,
                uint32_t* any_out, void* stream);

/* Enumeration (PAPER.md:47, sub-problem 4; :91: the count |I(B, a_i)| is the termination condition of the
 * walk): every pair <a_i, b_j> with a_i.start <= b_j.end and a_i.end >= b_j.start, as indices into the
 * caller's arrays.  The pairs of a_i occupy positions [offset_i, offset_i + c(a_i)) of pair_a_out /
 * pair_b_out (offset = exclusive prefix of the per-interval counts in A's input order; pair_a_out holds
 * i there); inside one a_i the order of the b_j is unspecified.  capacity = elements of each output
 * array (dev uint32[capacity]); pairs at positions >= capacity are not written, *total_out (dev
 * uint64[1]) is the full count either way, so a first call with capacity 0 sizes the arrays.
 * BITS_B_SORTED is rejected (BITS_ERR_FLAGS): independently sorted arrays no longer pair starts with ends.
 * Workspace: bits_workspace_bytes(BITS_FN_ENUMERATE, n_a, n_b, 0, 0, flags). */
int bits_enumerate(const uint32_t* a_start, const uint32_t* a_end, uint64_t n_a,
                   const uint32_t* b_start, const uint32_t* b_end, uint64_t n_b,
                   uint32_t flags, void* workspace, size_t workspace_bytes,
                   uint32_t* pair_a_out, uint32_t* pair_b_out, uint64_t capacity,
                   uint64_t* total_out, void* stream);

/* Per-interval counting (Algorithm 1):
 *   counts_out[i] = c(a_i), in A's input order (dev uint32[n_a]);
 *   *total_out = sum_i c(a_i) (dev uint64[1]; may be NULL). */
int bits_count_per_interval(const uint32_t* a_start, const uint32_t* a_end, uint64_t n_a,
                            const uint32_t* b_start, const uint32_t* b_end, uint64_t n_b,
                            uint32_t flags, void* workspace, size_t workspace_bytes,
                            uint32_t* counts_out, uint64_t* total_out, void* stream);

/* Monte Carlo rounds (Sec. 3.2; procedure in DESIGN.md "Monte Carlo"):
 *   *observed_out = total(A, B);
 *   for k in [0, n_rounds): r = round_begin + k; the permuted set P (A or B, by `which`) is
 *   re-placed with Philox4x32-10: interval i draws counter (i >> 1, r, which, 0) under key
 *   (seed lo32, seed hi32), takes the 64 bits x = out[2h] | out[2h+1] << 32 with h = i & 1,
 *   u = (x * V) >> 64 where V = sum_c max(L_c - d_i, 0) counts the valid starts for its span
 *   d_i = end_i - start_i, and start' = the u-th valid start in chromosome-table order,
 *   end' = start' + d_i.  round_counts_out[k] = total(A', B) or total(A, B'), B' re-sorted.
 * Results depend only on (seed, r, i): any split of the rounds over calls is bit-identical.
 * chrom_offsets: HOST uint32[n_chrom + 1], off[0] = 0, strictly ascending, off[n_chrom] = G <= 2^32-1
 * (read before the call returns).  Every interval of the permuted set must satisfy end < G.
 * observed_out: dev uint64[1]; round_counts_out: dev uint64[n_rounds].
 * BITS_B_SORTED together with BITS_PERMUTE_B is rejected (BITS_ERR_FLAGS): arrays sorted each on its
 * own no longer pair a start with its end, so the lengths the re-placement must keep are lost.
 * Synchronisation: `stream` is synchronised once before the first round (the longest span of the
 * permuted set is checked against the longest chromosome: BITS_ERR_NO_PLACEMENT) and, with
 * BITS_PERMUTE_B and more than 8,188 re-placed intervals, once more per (at most) 4,096 rounds: the
 * overflow flags of the fused rounds are read back; a flagged round is redone by the general path.  The "sorted
 * arrays of the last round" (bits_workspace_sorted_offset) are those of round round_begin + n_rounds - 1 either way:
 * if a redo overwrote them, the last round is done once more by the general path. */
int bits_mc_rounds(const uint32_t* a_start, const uint32_t* a_end, uint64_t n_a,
                   const uint32_t* b_start, const uint32_t* b_end, uint64_t n_b,
                   const uint32_t* chrom_offsets, uint32_t n_chrom, int which, uint64_t seed,
                   uint32_t round_begin, uint32_t n_rounds,
                   uint32_t flags, void* workspace, size_t workspace_bytes,
                   uint64_t* observed_out, uint64_t* round_counts_out, void* stream);

/* One placement step on its own (the "place" row of the path; same arithmetic as inside
 * bits_mc_rounds): spans dev uint32[n] -> start_out, end_out dev uint32[n] for round `round`,
 * stream tag `tag` (0 for A, 1 for B).  Spans must be shorter than the longest chromosome. */
int bits_place(const uint32_t* spans, uint64_t n, const uint32_t* chrom_offsets, uint32_t n_chrom,
               uint64_t seed, uint32_t round, uint32_t tag,
               void* workspace, size_t workspace_bytes,
               uint32_t* start_out, uint32_t* end_out, void* stream);

/* One sort step on its own (the "sort" row: Algorithm 2's Sort(B_S)):
 * keys_out = keys_in ascending (dev uint32[n] each, must not overlap). */
int bits_sort_u32(const uint32_t* keys_in, uint32_t* keys_out, uint64_t n,
                  void* workspace, size_t workspace_bytes, void* stream);

/* Host-buffer variants: same semantics, every array argument is a HOST pointer (pinned memory
 * makes the copies asynchronous).  workspace is still a device pointer and must hold
 * bits_workspace_bytes(fn, ...) + bits_host_staging_bytes(fn, ...) bytes.  They copy the inputs
 * to the device, run the path, copy the outputs back and synchronise `stream`. */
int bits_count_host(const uint32_t* a_start, const uint32_t* a_end, uint64_t n_a,
                    const uint32_t* b_start, const uint32_t* b_end, uint64_t n_b,
                    uint32_t flags, void* workspace, size_t workspace_bytes,
                    uint64_t* total_out, void* stream);
int bits_count_per_interval_host(const uint32_t* a_start, const uint32_t* a_end, uint64_t n_a,
                                 const uint32_t* b_start, const uint32_t* b_end, uint64_t n_b,
                                 uint32_t flags, void* workspace, size_t workspace_bytes,
                                 uint32_t* counts_out, uint64_t* total_out, void* stream);
int bits_mc_rounds_host(const uint32_t* a_start, const uint32_t* a_end, uint64_t n_a,
                        const uint32_t* b_start, const uint32_t* b_end, uint64_t n_b,
                        const uint32_t* chrom_offsets, uint32_t n_chrom, int which, uint64_t seed,
                        uint32_t round_begin, uint32_t n_rounds,
                        uint32_t flags, void* workspace, size_t workspace_bytes,
                        uint64_t* observed_out, uint64_t* round_counts_out, void* stream);

/* Empirical p-value from the integer outputs (host pointers; reading R13 -- the paper
 * prints only log2(observed/median)):
 *   tail 0: (#{r : count_r >= observed} + 1) / (n_rounds + 1)      (enrichment)
 *   tail 1: (#{r : count_r <= observed} + 1) / (n_rounds + 1)      (depletion)
 * Returns NaN for a bad tail or a NULL array with n_rounds > 0. */
double bits_pvalue(uint64_t observed, const uint64_t* round_counts, uint32_t n_rounds, int tail);

/* Enrichment score of the paper's screen (Fig. 3 caption :224): log2 of the observed
 * count over the MEDIAN count of the Monte Carlo rounds (host pointers).  Median of an even number of
 * rounds = mean of the two middle order statistics.  Median 0: +inf if observed > 0, else NaN;
 * observed 0 with a positive median: -inf.  NaN for n_rounds == 0 or a NULL array. */
double bits_enrichment(uint64_t observed, const uint64_t* round_counts, uint32_t n_rounds);

/* The many-pair screen as one device job (Sec. 3.3: every pairwise comparison of K interval
 * sets by the Monte Carlo simulation; Fig. 3 caption :224: score = log2(observed / median of the simulated counts)).
 * The K tracks are passed concatenated: track t = starts/ends[track_offsets[t] .. track_offsets[t+1]) (dev uint32;
 * track_offsets: HOST uint64[n_tracks + 1], [0] = 0, non-decreasing, last < 2^28; n_tracks <= 65535).
 * For every ORDERED pair (i, j), p = i * n_tracks + j:
 *   observed_out[p] = |I(T_i, T_j)|                                            (dev uint64[n_tracks^2])
 *   round_counts_out[p * n_rounds + k] = total(T_i', T_j), k in [0, n_rounds)     (dev uint64[n_tracks^2 * n_rounds])
 * where T_i' is track i re-placed for round r = round_begin + k exactly as in bits_mc_rounds with
 * BITS_PERMUTE_A, except that the fourth Philox counter word is the pair id p: interval q of track i draws
 * counter (q >> 1, r, 0, p).  Every pair therefore has its own null draws, and pair (0, 0) reproduces
 * bits_mc_rounds(T_0, T_0, BITS_PERMUTE_A) (reading R24).
 * Every track is sorted and indexed once; all (pair, round) work runs in gridded launches with no host
 * round trip in between.  flags: BITS_VALIDATE only.  Synchronises `stream` once (longest span of any track
 * against the longest chromosome: BITS_ERR_NO_PLACEMENT, only if n_rounds > 0).  Empty tracks are legal (counts 0).
 * Workspace: bits_screen_workspace_bytes(track_offsets, n_tracks, n_chrom) (0 for a bad offset table). */
size_t bits_screen_workspace_bytes(const uint64_t* track_offsets, uint32_t n_tracks, uint32_t n_chrom);
int bits_screen(const uint32_t* starts, const uint32_t* ends, const uint64_t* track_offsets, uint32_t n_tracks,
                const uint32_t* chrom_offsets, uint32_t n_chrom, uint64_t seed,
                uint32_t round_begin, uint32_t n_rounds, uint32_t flags,
                void* workspace, size_t workspace_bytes,
                uint64_t* observed_out, uint64_t* round_counts_out, void* stream);

/* bits_enrichment for every pair of a screen (all HOST pointers): enrichment_out[p] =
 * bits_enrichment(observed[p], round_counts + p * n_rounds, n_rounds), p in [0, n_pairs). */
int bits_screen_enrichment(const uint64_t* observed, const uint64_t* round_counts, uint64_t n_pairs,
                           uint32_t n_rounds, double* enrichment_out);

/* Kernels launched by this library in this process since load (for bench.py's gpu_launches). */
uint64_t bits_launch_count(void);

/* Per-kernel-class device time, measured with CUDA events on the launching stream while
 * bits_set_option("profile", 1) is on (2 resets the totals).  cls: 0 place, 1 histogram,
 * 2 LSD sort pass, 3 index build, 4 count (search + reduce), 5 sorted-query search + reduce,
 * 6 fused Monte Carlo kernel (place + search + reduce), 7 other, 8 MSD sort plan, 9 MSD sort
 * scatter, 10 MSD per-bucket sort, 11 fused place + scatter, 12 fused per-bucket sort + search + reduce,
 * 13 scatter of the queries into bucket order, 14 per-bucket search + reduce out of shared memory.
 * Synchronises the recorded
 * events.  ms_out / launches_out: host pointers, may be NULL. */
int bits_profile_read(int cls, double* ms_out, uint64_t* launches_out);

/* Tuning knobs for design studies (bench.py --opt NAME=VALUE); returns BITS_ERR_FLAGS for an unknown
 * name or a value out of range.  They never change results.  Thread-local (see "Threads" above).
 * Names, values, defaults and measured effects are tabulated in DESIGN.md section 10 ("Knobs").
 * Two names are TEST HOOKS, not tuning knobs -- "mc_force_redo" (every n-th fused Monte Carlo round is redone by
 * the general path as if its overflow flag had been raised) and "mc_shift_bias" (bins widened until they overflow on
 * the device): they let the parity tests reach the overflow branches through this ABI and have no use in production. */
int bits_set_option(const char* name, int64_t value);

const char* bits_strerror(int status);
const char* bits_version(void);

#ifdef __cplusplus
}
#endif
#endif /* BITS_B200_H_ */
