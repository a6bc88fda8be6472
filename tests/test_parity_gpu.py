"""Parity of the CUDA path (through the C ABI, via the thin binding) against the CPU oracle.

All comparisons are BIT-EXACT: the path is integer-only (uint32 coordinates and ranks, uint64
sums), so there is no tolerance anywhere.  Run on the B200 box with  pytest -m gpu.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_1208_3407_b200 import bits
from paper_1208_3407_b200 import workloads as W

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def dev(a):
    a = np.ascontiguousarray(a, dtype=np.uint32)
    return torch.from_numpy(a.view(np.int32)).to(DEV)


def host_u32(t):
    return t.cpu().numpy().view(np.uint32)


def host_u64(t):
    return t.cpu().numpy().view(np.uint64)


def sync():
    torch.cuda.synchronize()


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    bits.lib()


# ------------------------------------------------------------------------------------- sort
@pytest.mark.parametrize("n", [0, 1, 2, 31, 33, 8191, 8192, 8193, 16384, 100_003, 1_000_000, 3_000_017])
def test_sort_random_full_range(n):
    rng = np.random.default_rng(n + 1)
    k = rng.integers(0, 2**32, n, dtype=np.uint64).astype(np.uint32)
    got = host_u32(bits.sort_u32(dev(k)))
    assert np.array_equal(got, oracle.sort_u32(k))


@pytest.mark.parametrize("kind", ["equal", "sorted", "reverse", "low_bits", "high_bits", "two_values", "max"])
def test_sort_structured(kind):
    n = 70_001
    rng = np.random.default_rng(5)
    k = {
        "equal": np.full(n, 0xDEADBEEF, dtype=np.uint64),
        "sorted": np.sort(rng.integers(0, 2**32, n, dtype=np.uint64)),
        "reverse": np.sort(rng.integers(0, 2**32, n, dtype=np.uint64))[::-1],
        "low_bits": rng.integers(0, 1000, n, dtype=np.uint64),
        "high_bits": rng.integers(0, 200, n, dtype=np.uint64) << np.uint64(24),
        "two_values": rng.integers(0, 2, n, dtype=np.uint64) * np.uint64(0xFFFFFFFF),
        "max": np.full(n, 0xFFFFFFFF, dtype=np.uint64),
    }[kind].astype(np.uint32)
    assert np.array_equal(host_u32(bits.sort_u32(dev(k))), oracle.sort_u32(k))


@pytest.mark.parametrize("n", [1, 8191, 8193, 300_007, 5_000_011])
def test_sort_lsd_only(n):
    """The stable LSD onesweep sort on its own (sort_msd = 0): persistent blocks, tiles by ticket, look-back."""
    rng = np.random.default_rng(n)
    k = rng.integers(0, 2**32, n, dtype=np.uint64).astype(np.uint32)
    bits.set_option("sort_msd", 0)
    try:
        ws = torch.empty(bits.workspace_bytes(bits.FN_SORT, 0, n), dtype=torch.uint8, device=DEV)
        for _ in range(2):                               # twice on one workspace: tickets and epochs restart per call
            assert np.array_equal(host_u32(bits.sort_u32(dev(k), workspace=ws)), oracle.sort_u32(k))
        w = W.make_config(5, scale=0.01)                 # and inside the Monte Carlo loop (general path, LSD per round)
        obs, rc = run_mc(w, 1, 4, 0, 3)
        o_obs, o_rc = oracle.mc_rounds(w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets, 1, 4, 0, 3)
        assert obs == o_obs and np.array_equal(rc, o_rc)
    finally:
        bits.set_option("sort_msd", 1)


@pytest.mark.parametrize("pack", [7168, 8192, 3000, 0])
def test_sort_large_sets_with_packed_buckets(pack):
    """Sorts of at least 4M keys pack consecutive bins greedily into buckets (msd_pack): uniform keys over the genome's
    range, and keys in clusters (uneven bins: some buckets hold one bin, some dozens, some bins overflow a bucket)."""
    rng = np.random.default_rng(pack + 3)
    G = 3_564_000_011
    uniform = rng.integers(0, G, 4_500_001, dtype=np.uint64)
    centres = rng.integers(0, G, 3000, dtype=np.uint64)
    clustered = (centres[rng.integers(0, 3000, 5_000_003)] + rng.integers(0, 400_000, 5_000_003, dtype=np.uint64)) % np.uint64(2**32)
    bits.set_option("msd_pack", pack)
    try:
        for k in (uniform, clustered, np.concatenate([uniform[:2_500_000], clustered[:2_500_000]])):
            k = k.astype(np.uint32)
            assert np.array_equal(host_u32(bits.sort_u32(dev(k))), oracle.sort_u32(k))
    finally:
        bits.set_option("msd_pack", 7168)


def test_sort_repeated_calls_share_workspace():
    rng = np.random.default_rng(17)
    n = 50_000
    ws = torch.empty(bits.workspace_bytes(bits.FN_SORT, 0, n), dtype=torch.uint8, device=DEV)
    ws.fill_(0xAB)                         # garbage workspace must not matter
    for _ in range(5):
        k = rng.integers(0, 2**32, n, dtype=np.uint64).astype(np.uint32)
        assert np.array_equal(host_u32(bits.sort_u32(dev(k), workspace=ws)), np.sort(k))


# ------------------------------------------------------------------------------------- place
GEN = W.genome_offsets(W.GENOME24_LENGTHS)
SMALL = np.array([0, 10, 25, 1000, 1003, 5000], dtype=np.uint32)


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 1023, 1024, 1025, 250_001])
def test_place_genome(n):
    rng = np.random.default_rng(n)
    spans = np.clip(np.rint(1000 * np.exp(rng.standard_normal(n))), 20, 100_000).astype(np.uint32) - 1
    for seed, rnd, tag in ((1, 0, 0), (0xFEDCBA9876543210, 4_000_000_000, 1)):
        s, e = bits.place(dev(spans), GEN, seed, rnd, tag)
        os_, oe = oracle.place_round(spans, GEN, seed, rnd, tag)
        assert np.array_equal(host_u32(s), os_) and np.array_equal(host_u32(e), oe)


def test_place_general_path_some_chromosomes_too_short():
    rng = np.random.default_rng(2)
    spans = rng.integers(0, 900, 10_000).astype(np.uint32)     # many spans exceed chromosomes 0, 1, 3
    s, e = bits.place(dev(spans), SMALL, 7, 3, 0)
    os_, oe = oracle.place_round(spans, SMALL, 7, 3, 0)
    assert np.array_equal(host_u32(s), os_) and np.array_equal(host_u32(e), oe)


def test_place_many_chromosomes_and_unaligned_pointers():
    rng = np.random.default_rng(3)
    lens = rng.integers(1000, 5000, 1500)                      # table too large for shared memory
    off = W.genome_offsets(lens)
    spans = rng.integers(0, 999, 4099).astype(np.uint32)
    d = dev(np.concatenate([[0], spans]))[1:]                  # 4-byte aligned only
    s, e = bits.place(d, off, 11, 5, 1)
    os_, oe = oracle.place_round(spans, off, 11, 5, 1)
    assert np.array_equal(host_u32(s), os_) and np.array_equal(host_u32(e), oe)


# ------------------------------------------------------------------------------------- count
def check_counts(a_s, a_e, b_s, b_e, flags=0, b_for_gpu=None):
    """Per-interval counts and totals against the oracle, by both designs of the search step: queries binned by B's
    buckets and searched out of shared memory (count_binned = 1, the default for large sets) and the bucket index
    (count_binned = 0); -1 = the library's own choice by size."""
    want_total, want_counts = oracle.count_per_interval(a_s, a_e, b_s, b_e)
    gb_s, gb_e = b_for_gpu if b_for_gpu is not None else (b_s, b_e)
    d = [dev(x) for x in (a_s, a_e, gb_s, gb_e)]
    try:
        for binned in (1, 0, -1):
            bits.set_option("count_binned", binned)
            counts, total = bits.count_per_interval(*d, flags=flags)
            total_only = bits.count(*d, flags=flags)
            sync()
            bad = np.nonzero(host_u32(counts) != want_counts)[0]
            assert bad.size == 0, (binned, bad.size, bad[:5])
            assert int(host_u64(total)[0]) == want_total, binned
            assert int(host_u64(total_only)[0]) == want_total, binned
    finally:
        bits.set_option("count_binned", -1)
    return want_total


def test_count_binned_queries_special_cases():
    """binned_count.cuh: queries longer than a bucket (their start lies before the bucket's coordinate range: `last`
    by a global search), a bucket range holding more ends than the staging buffer, buckets with several work items
    (more than 4,096 queries), and a searched set whose MSD sort falls back to the LSD sort (the binned kernels
    exit, the index path behind them answers)."""
    rng = np.random.default_rng(90)
    G = 3_000_000_000
    b_s = rng.integers(0, G, 400_000)
    b_e = b_s + rng.integers(0, 5000, 400_000)
    # (1) long queries: spans up to 2^23, far beyond the 2^20-wide bins
    a_s = rng.integers(0, G, 60_000)
    a_e = a_s + rng.integers(0, 2**23, 60_000)
    check_counts(a_s, a_e, b_s, b_e)
    # (2) 30,000 long intervals of B end inside one 2^20-wide bin: more ends in that bucket's range than kCapE
    ls = rng.integers(0, 2_000_000_000, 30_000)
    le = 2_500_000_000 + rng.integers(0, 900_000, 30_000)
    b2_s, b2_e = np.concatenate([b_s, ls]), np.concatenate([b_e, le])
    qs = 2_500_000_000 + rng.integers(-500_000, 1_200_000, 50_000)
    check_counts(np.concatenate([a_s, qs]), np.concatenate([a_e, qs + rng.integers(0, 3000, 50_000)]), b2_s, b2_e)
    # (3) 40,000 queries inside one bucket (ten work items), the rest spread out
    qs = 1_000_000_000 + rng.integers(0, 500_000, 40_000)
    check_counts(np.concatenate([qs, a_s[:5000]]), np.concatenate([qs + rng.integers(0, 300, 40_000), a_e[:5000]]), b_s, b_e)
    # (5) at a size where the library itself picks the binned design and packs buckets: 4.2M intervals, half of them in
    # clusters, against 1.5M queries of which a million sit in a few dozen buckets (work items of 16,384 queries, several
    # per bucket, answered in steps) and 20,000 are longer than a bucket
    n_b5 = 4_200_000
    u = rng.integers(0, G, n_b5 // 2)
    c5 = rng.integers(0, G, 2000)[rng.integers(0, 2000, n_b5 - n_b5 // 2)] + rng.integers(0, 300_000, n_b5 - n_b5 // 2)
    b5_s = np.concatenate([u, c5]); b5_e = b5_s + rng.integers(0, 20_000, n_b5)
    q5 = np.concatenate([rng.integers(0, G, 480_000), 1_700_000_000 + rng.integers(0, 40_000_000, 1_000_000), rng.integers(0, G, 20_000)])
    q5_e = q5 + np.concatenate([rng.integers(0, 3000, 1_480_000), rng.integers(2**20, 2**24, 20_000)])
    check_counts(q5, q5_e, b5_s, b5_e)
    # (4) 60,000 starts inside one bin: the MSD sort raises its flag, the LSD sort and the index path take over
    cs = 123_456_789 + rng.integers(0, 200_000, 60_000)
    b4_s, b4_e = np.concatenate([b_s[:50_000], cs]), np.concatenate([b_e[:50_000], cs + rng.integers(0, 100, 60_000)])
    bits.set_option("count_binned", 1)
    try:
        check_counts(a_s[:20_000], a_e[:20_000], b4_s, b4_e)
    finally:
        bits.set_option("count_binned", -1)
    # (6) the same fallback at a size where the library picks the binned design itself and the gated launches behind it
    # (histogram, sort passes, index, count) are the whole job: 3.3M intervals of which 60,000 start inside one bin, 1.3M queries
    b6_s = np.concatenate([rng.integers(0, G, 3_240_000), cs]); b6_e = b6_s + rng.integers(0, 2000, b6_s.size)
    q6 = rng.integers(0, G, 1_300_000)
    check_counts(q6, q6 + rng.integers(0, 4000, q6.size), b6_s, b6_e)



def test_count_config1_tiny():
    w = W.make_config(1)
    check_counts(w.a_start, w.a_end, w.b_start, w.b_end)


@pytest.mark.parametrize("n_a,n_b", [(1, 1), (5, 3), (3, 5), (1000, 7), (7, 1000), (4097, 8193), (10_001, 70_001)])
def test_count_random_ragged(n_a, n_b):
    rng = np.random.default_rng(n_a * 31 + n_b)
    a_s = rng.integers(0, 2**31, n_a, dtype=np.int64)
    a_e = a_s + rng.integers(0, 2**22, n_a)
    b_s = rng.integers(0, 2**31, n_b, dtype=np.int64)
    b_e = b_s + rng.integers(0, 2**22, n_b)
    check_counts(a_s, a_e, b_s, b_e)


def test_count_dense_small_coordinates_with_ties():
    rng = np.random.default_rng(12)
    a_s = rng.integers(0, 300, 5000)
    a_e = a_s + rng.integers(0, 40, 5000)
    b_s = rng.integers(0, 300, 20_000)                         # thousands of duplicates per key
    b_e = b_s + rng.integers(0, 40, 20_000)
    check_counts(a_s, a_e, b_s, b_e)


def test_count_edge_cases():
    top = 2**32 - 2
    check_counts([0, top - 5, 0, top, 5], [0, top, top, top, 5], [0, top, 7, top - 1], [0, top, 9, top])
    K = 3000                                                   # nested B: the containment trap
    k = np.arange(K)
    check_counts(np.arange(0, K, 7), np.arange(0, K, 7), k, 2 * K - k)
    check_counts([10, 10, 10, 10], [20, 20, 20, 20], [20, 21, 0, 0], [30, 30, 10, 9])   # shared endpoints
    check_counts(np.arange(100), np.arange(100) + 3, np.full(5000, 50), np.full(5000, 60))  # one huge bucket
    # keys equal to 0xffffffff (no genome table on the counting calls, so the full range is legal)
    check_counts([0, 2**32 - 1], [2**32 - 1, 2**32 - 1], [2**32 - 1, 5, 2**32 - 1], [2**32 - 1, 2**32 - 1, 2**32 - 1])


def test_count_empty_sets():
    a = dev([1, 5]), dev([3, 9])
    e = dev([]), dev([])
    counts, total = bits.count_per_interval(*a, *e)
    sync()
    assert host_u32(counts).tolist() == [0, 0] and int(host_u64(total)[0]) == 0
    counts, total = bits.count_per_interval(*e, *a)
    sync()
    assert counts.numel() == 0 and int(host_u64(total)[0]) == 0
    assert int(host_u64(bits.count(*e, *e))[0]) == 0


def test_count_flags_sorted_and_validate():
    w = W.make_config(2, scale=0.02)
    bs, be = np.sort(w.b_start), np.sort(w.b_end)
    check_counts(w.a_start, w.a_end, w.b_start, w.b_end, flags=bits.B_SORTED, b_for_gpu=(bs, be))
    check_counts(w.a_start, w.a_end, w.b_start, w.b_end, flags=bits.VALIDATE)
    bad_e = w.a_end.copy()
    bad_e[123] = w.a_start[123] - 1
    with pytest.raises(bits.BitsError) as ei:
        bits.count(dev(w.a_start), dev(bad_e), dev(w.b_start), dev(w.b_end), flags=bits.VALIDATE)
    assert ei.value.status == 7


def test_count_unaligned_query_pointers():
    w = W.make_config(2, scale=0.01)
    a_s = dev(np.concatenate([[0], w.a_start]))[1:]
    a_e = dev(np.concatenate([[0], w.a_end]))[1:]
    want_total, want_counts = oracle.count_per_interval(w.a_start, w.a_end, w.b_start, w.b_end)
    counts, total = bits.count_per_interval(a_s, a_e, dev(w.b_start), dev(w.b_end))
    sync()
    assert np.array_equal(host_u32(counts), want_counts) and int(host_u64(total)[0]) == want_total


def test_count_config2_full_size():
    w = W.make_config(2)
    total = check_counts(w.a_start, w.a_end, w.b_start, w.b_end)
    assert 0.5e6 < total < 1.5e6
    # count(A, B) = count(B, A), and self-comparison >= N, at full size on the GPU path
    t_ba = bits.count(dev(w.b_start), dev(w.b_end), dev(w.a_start), dev(w.a_end))
    t_aa = bits.count(dev(w.a_start), dev(w.a_end), dev(w.a_start), dev(w.a_end))
    sync()
    assert int(host_u64(t_ba)[0]) == total and int(host_u64(t_aa)[0]) >= w.n_a


@pytest.mark.parametrize("variant", [1, 2])
def test_count_search_design_variants(variant):
    """The other search designs of the study (plain binary search, top levels in shared memory) give the same counts."""
    rng = np.random.default_rng(40 + variant)
    bits.set_option("search_variant", variant)
    try:
        w = W.make_config(2, scale=0.05)
        check_counts(w.a_start, w.a_end, w.b_start, w.b_end)
        for n_b in (1, 2, 7, 2047, 2048, 2049, 5000):
            b_s = rng.integers(0, 100_000, n_b).astype(np.uint32)
            b_e = b_s + rng.integers(0, 300, n_b).astype(np.uint32)
            a_s = rng.integers(0, 100_000, 777).astype(np.uint32)
            a_e = a_s + rng.integers(0, 500, 777).astype(np.uint32)
            a_s[0] = 0; a_e[0] = 0
            check_counts(a_s, a_e, b_s, b_e)
    finally:
        bits.set_option("search_variant", 0)


def test_decide_matches_oracle():
    """bits_decide (PAPER.md:47 sub-problem 1): 1 iff some interval of A meets one of B."""
    rng = np.random.default_rng(3)
    cases = [([10], [20], [20], [30]), ([10], [20], [21], [30]), ([], [], [1], [2]), ([5], [6], [], [])]
    for _ in range(6):                                   # sparse sets: some meet, some do not
        n_a, n_b = int(rng.integers(1, 2000)), int(rng.integers(1, 2000))
        a_s = rng.integers(0, 2**31, n_a); b_s = rng.integers(0, 2**31, n_b)
        cases.append((a_s, a_s + rng.integers(0, 40000, n_a), b_s, b_s + rng.integers(0, 40000, n_b)))
    w = W.make_config(2, scale=0.05)
    cases.append((w.a_start, w.a_end, w.b_start, w.b_end))
    seen = set()
    for a_s, a_e, b_s, b_e in cases:
        got = bits.decide(dev(a_s), dev(a_e), dev(b_s), dev(b_e))
        sync()
        want = oracle.decide(a_s, a_e, b_s, b_e)
        assert bool(got.cpu().numpy()[0]) == want
        seen.add(want)
    assert seen == {True, False}


def _enumerated(a_s, a_e, b_s, b_e):
    pa, pb, n = bits.enumerate_pairs(dev(a_s), dev(a_e), dev(b_s), dev(b_e))
    sync()
    got = np.stack([host_u32(pa).astype(np.int64), host_u32(pb).astype(np.int64)], axis=1) if n else np.zeros((0, 2), dtype=np.int64)
    return got[np.lexsort((got[:, 1], got[:, 0]))]


def test_enumerate_small_sets_equal_the_definition():
    """bits_enumerate (PAPER.md:47 sub-problem 4): the emitted set of pairs is exactly I(A, B)."""
    rng = np.random.default_rng(21)
    w = W.make_config(1)
    cases = [(w.a_start, w.a_end, w.b_start, w.b_end), ([10], [20], [20, 21, 0, 0], [30, 30, 10, 9]), ([], [], [1], [2]), ([1], [2], [], [])]
    for n_a, n_b, span in ((700, 3000, 3000), (2500, 900, 50), (300, 5000, 200_000)):
        a_s = rng.integers(0, 1_000_000, n_a); b_s = rng.integers(0, 1_000_000, n_b)
        cases.append((a_s, a_s + rng.integers(0, span, n_a), b_s, b_s + rng.integers(0, span, n_b)))
    b_s = rng.integers(0, 50, 4000)                       # many equal starts, long and short intervals mixed (containment)
    cases.append((rng.integers(0, 60, 500), rng.integers(60, 90, 500), b_s, b_s + rng.integers(0, 40, 4000)))
    for a_s, a_e, b_s, b_e in cases:
        want = oracle.enumerate_pairs(a_s, a_e, b_s, b_e)
        got = _enumerated(a_s, a_e, b_s, b_e)
        assert got.shape == want.shape and np.array_equal(got, want)


def test_enumerate_config2_is_valid_and_complete():
    """At a size the definition is too slow for: every emitted pair intersects, no pair twice, and every
    a_i has exactly c(a_i) pairs in its own slice of the output -- together that is the set I(A, B)."""
    w = W.make_config(2, scale=0.3)
    pa, pb, n = bits.enumerate_pairs(dev(w.a_start), dev(w.a_end), dev(w.b_start), dev(w.b_end))
    sync()
    pa, pb = host_u32(pa).astype(np.int64), host_u32(pb).astype(np.int64)
    o_total, o_counts = oracle.count_per_interval(w.a_start, w.a_end, w.b_start, w.b_end)
    assert n == o_total
    a_s, a_e = w.a_start.astype(np.int64), w.a_end.astype(np.int64)
    b_s, b_e = w.b_start.astype(np.int64), w.b_end.astype(np.int64)
    assert np.all((a_s[pa] <= b_e[pb]) & (a_e[pa] >= b_s[pb]))
    assert np.array_equal(np.bincount(pa, minlength=w.n_a), o_counts)
    assert np.all(np.diff(pa) >= 0)                        # A-major order: slices by exclusive prefix of the counts
    assert np.unique(pa * (1 << 32) + pb).size == n
    # one call with a known capacity (no sizing call): the same pairs in the same slices
    qa, qb, n2 = bits.enumerate_pairs(dev(w.a_start), dev(w.a_end), dev(w.b_start), dev(w.b_end), capacity=n + 7)
    sync()
    assert n2 == n and np.array_equal(host_u32(qa)[:n].astype(np.int64), pa)
    assert np.array_equal(np.sort(pa * (1 << 32) + host_u32(qb)[:n].astype(np.int64)), np.sort(pa * (1 << 32) + pb))


def test_enumerate_walk_is_bounded_when_one_interval_spans_everything():
    """a scan back from the binary-search position is what BITS replaces.  With one genome-wide
    interval in B (a tiny start, the largest end) every query must reach position 0 of the start order; the
    walk steps over runs of 32 / 1,024 / 32,768 positions whose largest end lies before a.start, so that case
    costs about what the uniform one does instead of O(|B|) per query.  Set equality on a sample + validity and
    completeness on the whole + a timing bound against the same sets without the long interval."""
    w = W.make_config(2, scale=0.4)
    G = int(w.chrom_offsets[-1])
    b_s = np.concatenate([w.b_start, [0, 5]]).astype(np.uint32)
    b_e = np.concatenate([w.b_end, [G - 1, 4_000_000]]).astype(np.uint32)     # one genome-wide, one long interval
    d_long = [dev(x) for x in (w.a_start, w.a_end, b_s, b_e)]
    d_base = [dev(x) for x in (w.a_start, w.a_end, w.b_start, w.b_end)]
    pa, pb, n = bits.enumerate_pairs(*d_long)
    sync()
    pa, pb = host_u32(pa).astype(np.int64), host_u32(pb).astype(np.int64)
    o_total, o_counts = oracle.count_per_interval(w.a_start, w.a_end, b_s, b_e)
    assert n == o_total and o_counts.min() >= 1
    assert np.all((w.a_start.astype(np.int64)[pa] <= b_e.astype(np.int64)[pb]) & (w.a_end.astype(np.int64)[pa] >= b_s.astype(np.int64)[pb]))
    assert np.array_equal(np.bincount(pa, minlength=w.n_a), o_counts)
    assert np.unique(pa * (1 << 32) + pb).size == n
    assert int(np.bincount(pb, minlength=b_s.size)[-2]) == w.n_a                 # the genome-wide interval meets every query
    sample = np.arange(0, w.n_a, 997)[:300]                                   # set equality with the definition on a sample of A
    want = oracle.enumerate_pairs(w.a_start[sample], w.a_end[sample], b_s, b_e)
    sel = np.isin(pa, sample)
    got = np.stack([np.searchsorted(sample, pa[sel]), pb[sel]], 1)
    assert np.array_equal(got[np.lexsort((got[:, 1], got[:, 0]))], want)
    def timed(d):
        ws = torch.empty(bits.workspace_bytes(bits.FN_ENUMERATE, d[0].numel(), d[2].numel()), dtype=torch.uint8, device=DEV)
        bits.enumerate_pairs(*d, workspace=ws); sync()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(3):
            bits.enumerate_pairs(*d, workspace=ws)
        e1.record(); sync()
        return e0.elapsed_time(e1) / 3
    t_long, t_base = timed(d_long), timed(d_base)
    assert t_long < 5.0 * t_base + 1.0, (t_long, t_base)      # (an unbounded walk takes seconds here: 4e5 queries x 4e5 steps)


def test_enumerate_with_too_small_a_capacity_writes_a_prefix_only():
    """include/bits.h: pairs at positions >= capacity are not written, *total_out is the full count either way."""
    w = W.make_config(2, scale=0.05)
    d = [dev(x) for x in (w.a_start, w.a_end, w.b_start, w.b_end)]
    pa, pb, n = bits.enumerate_pairs(*d)
    sync()
    assert n > 1000
    cap = n // 3
    guard = 0x7fffffff
    qa = torch.full((n,), guard, dtype=torch.int32, device=DEV)
    qb = torch.full((n,), guard, dtype=torch.int32, device=DEV)
    total = torch.zeros(1, dtype=torch.int64, device=DEV)
    ws = torch.empty(bits.workspace_bytes(bits.FN_ENUMERATE, w.n_a, w.n_b), dtype=torch.uint8, device=DEV)
    st = bits.lib().bits_enumerate(d[0].data_ptr(), d[1].data_ptr(), w.n_a, d[2].data_ptr(), d[3].data_ptr(), w.n_b, 0,
                                   ws.data_ptr(), ws.numel(), qa.data_ptr(), qb.data_ptr(), cap, total.data_ptr(),
                                   torch.cuda.current_stream().cuda_stream)
    sync()
    assert st == 0 and int(total.item()) == n
    assert torch.equal(qa[:cap], pa[:cap])                 # A-major slices: the same positions hold the same a_i
    got = torch.stack([qa[:cap], qb[:cap]], 1).cpu().numpy().astype(np.int64)
    full = torch.stack([pa, pb], 1).cpu().numpy().astype(np.int64)
    # inside one a_i the order of the b_j is unspecified: compare as sets per a_i over the a_i that fit entirely
    last_a = int(got[-1, 0])
    keep_g, keep_f = got[got[:, 0] < last_a], full[full[:, 0] < last_a]
    assert np.array_equal(keep_g[np.lexsort((keep_g[:, 1], keep_g[:, 0]))], keep_f[np.lexsort((keep_f[:, 1], keep_f[:, 0]))])
    assert bool((qa[cap:] == guard).all()) and bool((qb[cap:] == guard).all())


def test_results_do_not_depend_on_programmatic_launch():
    """The kernels of a call are chained by programmatic dependent launch (option mc_pdl, on by default):
    with it off every launch is fully serialised.  Counts, pairs, decisions and Monte Carlo rounds must be
    the same integers either way, call after call on one workspace (a kernel that touched memory before its
    griddepcontrol.wait would show up as a difference or as a mismatch with the oracle)."""
    w = W.make_config(2, scale=0.2)
    g = W.make_config(5, scale=0.02)
    o_total, o_counts = oracle.count_per_interval(w.a_start, w.a_end, w.b_start, w.b_end)
    o_obs, o_rc = oracle.mc_rounds(g.a_start, g.a_end, g.b_start, g.b_end, g.chrom_offsets, bits.PERMUTE_B, 7, 0, 3)
    d = [dev(x) for x in (w.a_start, w.a_end, w.b_start, w.b_end)]
    dg = [dev(x) for x in (g.a_start, g.a_end, g.b_start, g.b_end)]
    try:
        for pdl in (1, 0, 1):
            bits.set_option("mc_pdl", pdl)
            for _ in range(3):
                counts, total = bits.count_per_interval(*d)
                pa, pb, n = bits.enumerate_pairs(*d)
                any_ = bits.decide(*d)
                obs, rc = bits.mc_rounds(*dg, g.chrom_offsets, bits.PERMUTE_B, 7, 0, 3)
                sync()
                assert int(host_u64(total)[0]) == o_total and np.array_equal(host_u32(counts), o_counts)
                assert n == o_total and np.array_equal(np.bincount(host_u32(pa).astype(np.int64), minlength=w.n_a), o_counts)
                assert bool(any_.cpu().numpy()[0]) == (o_total > 0)
                assert int(host_u64(obs)[0]) == o_obs and np.array_equal(host_u64(rc), o_rc)
    finally:
        bits.set_option("mc_pdl", 1)


def test_count_config4_full_size():
    w = W.make_config(4)
    total = check_counts(w.a_start, w.a_end, w.b_start, w.b_end)
    assert total > 5e7


# ------------------------------------------------------------------------------------- Monte Carlo
def run_mc(w, which, seed, r0, n, flags=0):
    obs, rc = bits.mc_rounds(dev(w.a_start), dev(w.a_end), dev(w.b_start), dev(w.b_end), w.chrom_offsets, which,
                             seed, r0, n, flags=flags)
    sync()
    return int(host_u64(obs)[0]), host_u64(rc)


@pytest.mark.parametrize("which", [0, 1])
def test_mc_config1_all_rounds(which):
    w = W.make_config(1)
    obs, rc = run_mc(w, which, w.mc_seed, 0, 100)
    o_obs, o_rc = oracle.mc_rounds(w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets, which, w.mc_seed, 0, 100)
    assert obs == o_obs and np.array_equal(rc, o_rc)
    assert bits.pvalue(obs, rc, 0) == oracle.pvalue(o_obs, o_rc, 0)
    assert bits.pvalue(obs, rc, 1) == oracle.pvalue(o_obs, o_rc, 1)


@pytest.mark.parametrize("which", [0, 1])
def test_mc_round_slicing_and_big_round_numbers(which):
    w = W.make_config(1)
    seed = 0xA5A5_5A5A_1234_5678
    _, full = run_mc(w, which, seed, 4_294_967_000, 40)
    _, lo = run_mc(w, which, seed, 4_294_967_000, 13)
    _, hi = run_mc(w, which, seed, 4_294_967_013, 27)
    assert np.array_equal(full, np.concatenate([lo, hi]))
    _, o_rc = oracle.mc_rounds(w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets, which, seed, 4_294_967_000, 40)
    assert np.array_equal(full, o_rc)


@pytest.mark.parametrize("k,which,scale,rounds", [(3, 0, 0.1, 60), (5, 1, 0.01, 12), (3, 1, 0.05, 6), (5, 0, 0.01, 9)])
def test_mc_scaled_configs(k, which, scale, rounds):
    w = W.make_config(k, scale=scale)
    obs, rc = run_mc(w, which, 1, 0, rounds)
    o_obs, o_rc = oracle.mc_rounds(w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets, which, 1, 0, rounds)
    assert obs == o_obs and np.array_equal(rc, o_rc)


def test_mc_small_genome_general_placement_path():
    rng = np.random.default_rng(6)
    off = np.array([0, 40_000, 41_000, 90_000, 100_000], dtype=np.uint32)
    lo = np.array([0, 41_000, 90_000])
    a_s = lo[rng.integers(0, 3, 3000)] + rng.integers(0, 3000, 3000)
    a_e = a_s + rng.integers(0, 2500, 3000)                    # spans above the 1,000 bp chromosome
    b_s = lo[rng.integers(0, 3, 5000)] + rng.integers(0, 3000, 5000)
    b_e = b_s + rng.integers(0, 2500, 5000)
    for which in (0, 1):
        obs, rc = bits.mc_rounds(dev(a_s), dev(a_e), dev(b_s), dev(b_e), off, which, 9, 0, 15)
        sync()
        o_obs, o_rc = oracle.mc_rounds(a_s, a_e, b_s, b_e, off, which, 9, 0, 15)
        assert int(host_u64(obs)[0]) == o_obs and np.array_equal(host_u64(rc), o_rc)


def test_mc_errors_and_degenerate():
    off = np.array([0, 1000, 3000], dtype=np.uint32)
    a = dev([1, 5]), dev([3, 9])
    e = dev([]), dev([])
    for which in (0, 1):
        obs, rc = bits.mc_rounds(*a, *e, off, which, 1, 0, 4)
        sync()
        assert int(host_u64(obs)[0]) == 0 and not host_u64(rc).any()
        obs, rc = bits.mc_rounds(*e, *a, off, which, 1, 0, 4)
        sync()
        assert int(host_u64(obs)[0]) == 0 and not host_u64(rc).any()
        obs, rc = bits.mc_rounds(*a, *a, off, which, 1, 0, 0)
        sync()
        assert int(host_u64(obs)[0]) == oracle.count([1, 5], [3, 9], [1, 5], [3, 9]) and rc.numel() == 0
    long_ = dev([0]), dev([2000])                              # span 2000 >= longest chromosome (2000)
    with pytest.raises(bits.BitsError) as ei:
        bits.mc_rounds(*long_, *a, off, 0, 1, 0, 4)
    assert ei.value.status == 4
    obs, rc = bits.mc_rounds(*a, *long_, off, 0, 1, 0, 4)       # the long interval is not permuted: fine
    sync()


def test_mc_config3_full_size_sampled_rounds():
    w = W.make_config(3)
    obs, rc = run_mc(w, 0, 1, 0, 10_000)
    o_obs, o_lo = oracle.mc_rounds(w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets, 0, 1, 0, 150)
    _, o_hi = oracle.mc_rounds(w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets, 0, 1, 9_900, 100)
    assert obs == o_obs
    assert np.array_equal(rc[:150], o_lo) and np.array_equal(rc[9_900:], o_hi)
    assert rc.min() > 0 and 0.5 < rc.mean() / 1.3e4 < 2.0       # every round ran; E[count] ~ 1.3e4


def test_mc_config5_full_size_sampled_rounds():
    w = W.make_config(5)
    obs, rc = run_mc(w, 1, 1, 0, 40)
    o_obs, o_lo = oracle.mc_rounds(w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets, 1, 1, 0, 2)
    _, o_hi = oracle.mc_rounds(w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets, 1, 1, 39, 1)
    assert obs == o_obs
    assert np.array_equal(rc[:2], o_lo) and rc[39] == o_hi[0]
    assert rc.min() > 0 and np.unique(rc).size > 30
    # the other search design (bucket index rebuilt per round) must give the same integers
    bits.set_option("mc_sorted_queries", 0)
    bits.set_option("place_fused_hist", 0)
    try:
        _, rc2 = run_mc(w, 1, 1, 0, 3)
    finally:
        bits.set_option("mc_sorted_queries", 1)
        bits.set_option("place_fused_hist", 1)
    assert np.array_equal(rc2, rc[:3])


def _mc_b_case(a_s, a_e, b_s, b_e, off, seed, r0, n, expect_fused=None):
    bits.set_option("profile", 2)
    bits.set_option("profile", 1)
    try:
        obs, rc = bits.mc_rounds(dev(a_s), dev(a_e), dev(b_s), dev(b_e), off, 1, seed, r0, n)
        sync()
        fused_launches = bits.profile_read()["place_scatter"][1]
    finally:
        bits.set_option("profile", 0)
    if expect_fused is not None:                              # which path ran: the fused launch pairs (one per round, or one per
        assert (0 < fused_launches <= n) if expect_fused else fused_launches == 0   # batch of rounds for small sets), or not
    o_obs, o_rc = oracle.mc_rounds(a_s, a_e, b_s, b_e, off, 1, seed, r0, n)
    assert int(host_u64(obs)[0]) == o_obs
    assert np.array_equal(host_u64(rc), o_rc)


def _golden(config):
    import importlib.util
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "make_golden.py")
    spec = importlib.util.spec_from_file_location("make_golden", path)
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod.load(config)


@pytest.mark.parametrize("config,split", [(3, 3333), (5, 437)])
def test_mc_full_length_golden(config, split):
    """EVERY per-round count of the full-size Monte Carlo configs (10,000 rounds of config 3, 1,000 rounds of
    config 5, in the launch configuration bench.py times) against the oracle's golden counts
    (tests/golden/cfg{3,5}_seed1_rounds.txt, written by tests/golden/make_golden.py from the oracle alone), the
    p-values derived from them, and the same rounds by two calls split at an odd round_begin."""
    header, golden = _golden(config)
    w = W.make_config(config)
    assert header["checksums"] == w.checksums()
    R = w.n_rounds
    obs, rc = run_mc(w, w.which, w.mc_seed, 0, R)
    assert obs == header["observed"]
    bad = np.nonzero(rc != golden)[0]
    assert bad.size == 0, f"{bad.size} rounds differ, first {bad[:5]}"
    assert bits.pvalue(obs, rc, 0) == header["p_enrich"] and bits.pvalue(obs, rc, 1) == header["p_deplete"]
    _, lo = run_mc(w, w.which, w.mc_seed, 0, split)
    _, hi = run_mc(w, w.which, w.mc_seed, split, R - split)
    assert np.array_equal(np.concatenate([lo, hi]), golden)
    if config == 5:                                  # and through the host-buffer entry point bench.py's e2e leg times
        r = bits.mc_rounds_host(w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets, w.which, w.mc_seed, 900, 100)
        assert r.observed == header["observed"] and np.array_equal(r.round_counts, golden[900:])


def test_mc_permute_b_bins_overflow_on_the_device():
    """Bins wider than the host's margin allows (mc_shift_bias): about half of the bins of every round hold more
    than kCap keys, so bin_sort_search_kernel takes its overflow branch on the device, raises the round's flag and
    moves on to its next ticket; the flagged rounds are redone by the general path.  The kernel must terminate
    cleanly and every count must be the oracle's."""
    off = W.genome_offsets(W.GENOME24_LENGTHS)
    G = int(off[-1])
    n_b = int(4090 * G / 2**21)                      # ~4,090 keys per 2^21-wide bin: the host picks shift 21; bias + 1 -> ~8,180
    rng = np.random.default_rng(77)
    def draw(n, max_len):
        c = rng.integers(0, 24, n)
        ln = rng.integers(1, max_len, n)
        lo, hi = off[:-1][c].astype(np.int64), off[1:][c].astype(np.int64)
        s = lo + (rng.random(n) * (hi - lo - ln)).astype(np.int64)
        return s.astype(np.uint32), (s + ln - 1).astype(np.uint32)
    b_s, b_e = draw(n_b, 500)
    a_s, a_e = draw(100_000, 2000)
    bits.set_option("mc_shift_bias", 1)
    try:
        # (programmatic dependent launch is on here; the event timers of _mc_b_case switch it off)
        obs, rc = bits.mc_rounds(dev(a_s), dev(a_e), dev(b_s), dev(b_e), off, 1, 21, 5, 3)
        sync()
        o_obs, o_rc = oracle.mc_rounds(a_s, a_e, b_s, b_e, off, 1, 21, 5, 3)
        assert int(host_u64(obs)[0]) == o_obs and np.array_equal(host_u64(rc), o_rc)
        for _ in range(2):                           # twice: tickets, flags and hand-over counters restart correctly
            _mc_b_case(a_s, a_e, b_s, b_e, off, 21, 5, 3, expect_fused=True)
            assert bits.profile_read()["sorted_query"][1] == 3          # every round was flagged and redone
    finally:
        bits.set_option("mc_shift_bias", 0)
    _mc_b_case(a_s, a_e, b_s, b_e, off, 21, 5, 3, expect_fused=True)
    assert bits.profile_read()["sorted_query"][1] == 0                  # without the bias nothing overflows


@pytest.mark.parametrize("tile_variant", [0, 1, 2])
@pytest.mark.parametrize("bin_variant", [0, 1, 2, 3])
def test_mc_permute_b_kernel_shapes(tile_variant, bin_variant):
    """Every shape of the two fused kernels gives the oracle's integers (config 5 at 3 % and config 1)."""
    bits.set_option("mc_tile_variant", tile_variant)
    bits.set_option("mc_bin_variant", bin_variant)
    bits.set_option("mc_small", 0)                   # (config 1 would otherwise take the one-block-per-round kernel)
    try:
        for k, scale, rounds in ((5, 0.03, 3), (1, 1.0, 4)):
            w = W.make_config(k, scale=scale)
            _mc_b_case(w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets, 3, 7, rounds, expect_fused=True)
    finally:
        bits.set_option("mc_tile_variant", 2)
        bits.set_option("mc_bin_variant", 0)
        bits.set_option("mc_small", 1)


def test_mc_permute_b_several_rounds_per_launch():
    """Re-placed sets between 8,189 and 2M intervals run several rounds per launch pair (gridDim.y, one workspace slot
    per round, the widest bins that fit): more rounds than one flag chunk holds, a partial last launch pair, forced
    redo of some rounds, the sorted arrays of the last round out of their slot, and the one-round-per-launch path."""
    rng = np.random.default_rng(66)
    off = W.genome_offsets(W.GENOME24_LENGTHS)
    def draw(n, max_len):
        c = rng.integers(0, 24, n); ln = rng.integers(1, max_len, n)
        lo, hi = off[:-1][c].astype(np.int64), off[1:][c].astype(np.int64)
        st = lo + (rng.random(n) * (hi - lo - ln)).astype(np.int64)
        return st.astype(np.uint32), (st + ln - 1).astype(np.uint32)
    b_s, b_e = draw(20_000, 3000)
    a_s, a_e = draw(5_000, 20_000)
    R = 4_321                                                   # > 4,096: two flag chunks, the last launch pair partial
    obs, rc = bits.mc_rounds(dev(a_s), dev(a_e), dev(b_s), dev(b_e), off, 1, 5, 10, R)
    sync()
    o_obs, o_rc = oracle.mc_rounds(a_s, a_e, b_s, b_e, off, 1, 5, 10, R)
    assert int(host_u64(obs)[0]) == o_obs
    bad = np.nonzero(host_u64(rc) != o_rc)[0]
    assert bad.size == 0, (bad.size, bad[:8])
    bits.set_option("mc_force_redo", 7)
    try:
        _mc_b_case(a_s, a_e, b_s, b_e, off, 5, 10, 45, expect_fused=True)
    finally:
        bits.set_option("mc_force_redo", 0)
    for rounds in (1, 2, 30, 31):                               # the last round sits in different slots
        ws = torch.empty(bits.workspace_bytes(bits.FN_MC_ROUNDS, 5_000, 20_000, 24, 1), dtype=torch.uint8, device=DEV)
        bits.mc_rounds(dev(a_s), dev(a_e), dev(b_s), dev(b_e), off, 1, 5, 3, rounds, workspace=ws)
        sync()
        g_s, g_e = bits.sorted_arrays_in_workspace(ws, bits.FN_MC_ROUNDS, 5_000, 20_000, 24, 1)
        p_s, p_e = oracle.place_round((b_e - b_s).astype(np.uint32), off, 5, 3 + rounds - 1, 1)
        assert np.array_equal(host_u32(g_s), oracle.sort_u32(p_s)) and np.array_equal(host_u32(g_e), oracle.sort_u32(p_e))
    bits.set_option("mc_batch", 0)
    try:
        _, rc1 = bits.mc_rounds(dev(a_s), dev(a_e), dev(b_s), dev(b_e), off, 1, 5, 10, 40)
        sync()
    finally:
        bits.set_option("mc_batch", 1)
    assert np.array_equal(host_u64(rc1), o_rc[:40])


def test_mc_permute_b_small_sets_one_block_per_round():
    """Sets of at most 8,188 intervals: one block does a whole round in shared memory and the grid strides over the
    rounds (mc_small.cuh).  Sizes around the limit, more rounds than blocks, tiny genomes with heavy ties, a query
    beyond the genome's end, and the same rounds by the two-launch path."""
    rng = np.random.default_rng(55)
    w = W.make_config(1)
    _mc_b_case(w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets, 1, 0, 100, expect_fused=False)
    _mc_b_case(w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets, 7, 4_294_960_000, 700, expect_fused=False)   # 700 rounds > 296 blocks
    off = W.genome_offsets(W.GENOME24_LENGTHS)
    def draw(n, max_len):
        c = rng.integers(0, 24, n); ln = rng.integers(1, max_len, n)
        lo, hi = off[:-1][c].astype(np.int64), off[1:][c].astype(np.int64)
        st = lo + (rng.random(n) * (hi - lo - ln)).astype(np.int64)
        return st.astype(np.uint32), (st + ln - 1).astype(np.uint32)
    a_s, a_e = draw(30_000, 5000)
    for n_b, fused in ((1, False), (3, False), (8187, False), (8188, False), (8189, True)):
        b_s, b_e = draw(n_b, 100_000)
        _mc_b_case(a_s, a_e, b_s, b_e, off, 3, 2, 5, expect_fused=fused if n_b > 8188 else False)
    off2 = np.array([0, 300, 500], dtype=np.uint32)             # every coordinate hit dozens of times: long tie runs
    b_s2 = rng.integers(0, 250, 6000).astype(np.uint32); b_e2 = np.minimum(b_s2 + rng.integers(0, 40, 6000), 299).astype(np.uint32)
    a_s2 = np.array([0, 5, 100, 299, 450, 600_000], dtype=np.uint32); a_e2 = np.array([0, 50, 100, 400, 499, 700_000], dtype=np.uint32)
    _mc_b_case(a_s2, a_e2, b_s2, b_e2, off2, 9, 0, 6, expect_fused=False)
    bits.set_option("mc_small", 0)                                # the two-launch path gives the same integers
    try:
        obs0, rc0 = bits.mc_rounds(dev(w.a_start), dev(w.a_end), dev(w.b_start), dev(w.b_end), w.chrom_offsets, 1, 1, 0, 30)
    finally:
        bits.set_option("mc_small", 1)
    obs1, rc1 = bits.mc_rounds(dev(w.a_start), dev(w.a_end), dev(w.b_start), dev(w.b_end), w.chrom_offsets, 1, 1, 0, 30)
    sync()
    assert torch.equal(rc0, rc1) and torch.equal(obs0, obs1)


def test_mc_permute_b_small_set_few_rounds_large_query_set():
    """A re-placed set that fits one block, a large A and fewer rounds than SMs (round slicing, warm-up calls): the
    one-block-per-round kernel would rank all of A on a handful of SMs, so the call takes the two-launch path; with
    knob mc_small = 2 it takes the one-block path.  Both must give the oracle's integers."""
    rng = np.random.default_rng(77)
    off = W.genome_offsets(W.GENOME24_LENGTHS)
    def draw(n, max_len):
        c = rng.integers(0, 24, n); ln = rng.integers(1, max_len, n)
        lo, hi = off[:-1][c].astype(np.int64), off[1:][c].astype(np.int64)
        st = lo + (rng.random(n) * (hi - lo - ln)).astype(np.int64)
        return st.astype(np.uint32), (st + ln - 1).astype(np.uint32)
    a_s, a_e = draw(1_500_000, 3000)
    b_s, b_e = draw(6_000, 200_000)
    _mc_b_case(a_s, a_e, b_s, b_e, off, 4, 7, 3, expect_fused=True)          # 3 rounds x 1.5M queries: two-launch path
    bits.set_option("mc_small", 2)
    try:
        _mc_b_case(a_s, a_e, b_s, b_e, off, 4, 7, 3, expect_fused=False)     # forced: one block per round
    finally:
        bits.set_option("mc_small", 1)
    _mc_b_case(a_s, a_e, b_s, b_e, off, 4, 7, 150, expect_fused=False)       # 150 rounds fill the GPU: one block per round


def test_mc_permute_b_redo_leaves_the_last_rounds_arrays():
    """A redo of an EARLIER round of the final chunk (forced here for rounds 0 and 2 of 4) sorts into the buffers that
    hold 'the sorted arrays of the last round'; the library then puts the last round's arrays back.  With one round per
    launch pair and with several rounds per launch pair."""
    for k, scale in ((5, 0.02), (5, 0.6)):                       # 2e5 intervals: round batches; 6e6: one round per launch pair
        w = W.make_config(k, scale=scale)
        n_chrom = int(w.chrom_offsets.size - 1)
        ws = torch.empty(bits.workspace_bytes(bits.FN_MC_ROUNDS, w.n_a, w.n_b, n_chrom, 1), dtype=torch.uint8, device=DEV)
        bits.set_option("mc_force_redo", 2)
        try:
            _, rc = bits.mc_rounds(dev(w.a_start), dev(w.a_end), dev(w.b_start), dev(w.b_end), w.chrom_offsets, 1, w.mc_seed, 0, 4,
                                   workspace=ws)
            sync()
        finally:
            bits.set_option("mc_force_redo", 0)
        _, o_rc = oracle.mc_rounds(w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets, 1, w.mc_seed, 0, 4)
        assert np.array_equal(host_u64(rc), o_rc)
        b_s, b_e = bits.sorted_arrays_in_workspace(ws, bits.FN_MC_ROUNDS, w.n_a, w.n_b, n_chrom, 1)
        spans = (w.b_end - w.b_start).astype(np.uint32)
        o_s, o_e = oracle.place_round(spans, w.chrom_offsets, w.mc_seed, 3, 1)
        assert np.array_equal(host_u32(b_s), oracle.sort_u32(o_s))
        assert np.array_equal(host_u32(b_e), oracle.sort_u32(o_e))


def test_mc_permute_b_redo_path_gives_the_same_counts():
    """Rounds whose flag is raised are redone by the general path: force that for every 2nd round."""
    w = W.make_config(5, scale=0.02)
    bits.set_option("mc_force_redo", 2)
    try:
        _mc_b_case(w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets, 1, 0, 5, expect_fused=True)
    finally:
        bits.set_option("mc_force_redo", 0)
    bits.set_option("mc_fused", 0)                            # and the general path for every round
    try:
        _mc_b_case(w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets, 1, 0, 3, expect_fused=False)
    finally:
        bits.set_option("mc_fused", 1)


@pytest.mark.parametrize("n_b,n_chrom,max_len", [(3_300_001, 1, 700), (17_000_003, 24, 400), (1_234_567, 900, 50), (4_000_003, 2, 300)])
def test_mc_permute_b_other_shapes(n_b, n_chrom, max_len):
    """Fused rounds on set sizes, tile counts and chromosome tables other than config 5's."""
    rng = np.random.default_rng(n_chrom)
    if n_chrom == 24:
        lens = np.array(W.GENOME24_LENGTHS)
    elif n_chrom == 1:
        lens = np.array([1_500_000_000])
    elif n_chrom == 2:
        lens = np.array([2**32 - 1 - 3_000_000, 3_000_000])      # the largest genome the coordinate space holds: keys up to 2^32 - 2
    else:
        lens = rng.integers(200_000, 4_000_000, n_chrom)
    off = W.genome_offsets(lens)
    def draw(n):
        c = rng.integers(0, n_chrom, n)
        ln = rng.integers(1, max_len, n)
        lo, hi = off[:-1][c].astype(np.int64), off[1:][c].astype(np.int64)
        s = lo + (rng.random(n) * (hi - lo - ln)).astype(np.int64)
        return s.astype(np.uint32), (s + ln - 1).astype(np.uint32)
    b_s, b_e = draw(n_b)
    a_s, a_e = draw(50_000)
    _mc_b_case(a_s, a_e, b_s, b_e, off, 12, 3, 2, expect_fused=True)


def test_mc_permute_b_many_rounds_back_to_back():
    """120 fused rounds in one call (programmatic dependent launches, buffers reused by parity): every round's count."""
    w = W.make_config(5, scale=0.03)
    _mc_b_case(w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets, 17, 1000, 120, expect_fused=True)


def test_mc_workspace_contents_do_not_matter():
    """A workspace full of garbage, reused by calls of different sizes and kinds, gives the same integers."""
    big = W.make_config(5, scale=0.03)
    small = W.make_config(5, scale=0.01)
    n_chrom = int(big.chrom_offsets.size - 1)
    # (the smaller set takes more round slots per launch pair: its workspace is not the smaller one)
    ws = torch.empty(max(bits.workspace_bytes(bits.FN_MC_ROUNDS, x.n_a, x.n_b, n_chrom, 1) for x in (big, small)), dtype=torch.uint8, device=DEV)
    for fill, w, which, rounds in ((0xFF, big, 1, 3), (0xAB, small, 1, 4), (0x01, big, 0, 3), (0x80, small, 1, 2), (0x00, big, 1, 2)):
        ws.fill_(fill)
        obs, rc = bits.mc_rounds(dev(w.a_start), dev(w.a_end), dev(w.b_start), dev(w.b_end), w.chrom_offsets, which, 9, 2, rounds,
                                 workspace=ws)
        sync()
        o_obs, o_rc = oracle.mc_rounds(w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets, which, 9, 2, rounds)
        assert int(host_u64(obs)[0]) == o_obs and np.array_equal(host_u64(rc), o_rc)
    # back-to-back calls on one workspace without a fill in between
    for _ in range(2):
        obs, rc = bits.mc_rounds(dev(small.a_start), dev(small.a_end), dev(small.b_start), dev(small.b_end), small.chrom_offsets, 1,
                                 9, 2, 3, workspace=ws)
        sync()
        _, o_rc = oracle.mc_rounds(small.a_start, small.a_end, small.b_start, small.b_end, small.chrom_offsets, 1, 9, 2, 3)
        assert np.array_equal(host_u64(rc), o_rc)


def test_mc_permute_b_symmetric_sort_free_variant():
    """count(A, B') = count(B', A) -- the fresh B intervals searched against the sorted A."""
    bits.set_option("mc_symmetric", 1)
    try:
        for k, scale, rounds in ((1, 1.0, 6), (5, 0.02, 3)):
            w = W.make_config(k, scale=scale)
            _mc_b_case(w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets, 2, 11, rounds, expect_fused=False)
    finally:
        bits.set_option("mc_symmetric", 0)


def test_mc_permute_b_hand_over_lists_and_crowded_sub_buckets():
    rng = np.random.default_rng(8)
    # (1) long spans against narrow bins: many ends fall into the bin after their start's
    off = W.genome_offsets([x // 1000 for x in W.GENOME24_LENGTHS])
    G = int(off[-1])
    n_b, n_a = 200_000, 5_000
    def draw(n, max_len):
        ln = rng.integers(1, max_len, n)
        c = rng.integers(0, 24, n)
        lo, hi = off[:-1][c].astype(np.int64), off[1:][c].astype(np.int64)
        ln = np.minimum(ln, hi - lo - 1)
        s = lo + (rng.random(n) * (hi - lo - ln)).astype(np.int64)
        return s.astype(np.uint32), (s + ln - 1).astype(np.uint32)
    b_s, b_e = draw(n_b, 4000)
    a_s, a_e = draw(n_a, 3000)
    _mc_b_case(a_s, a_e, b_s, b_e, off, 5, 0, 4, expect_fused=True)
    # (2) a tiny genome: every coordinate is hit many times, so runs of equal keys go far beyond the
    # 4-wide tie window; short spans keep it on the fused path, long ones send it to the general path
    off2 = np.array([0, 3000, 5000], dtype=np.uint32)
    a_s2 = rng.integers(0, 2500, 700).astype(np.uint32); a_e2 = np.minimum(a_s2 + rng.integers(0, 300, 700), 2999).astype(np.uint32)
    for max_span, fused in ((40, True), (400, False)):
        b_s2 = rng.integers(0, 2500, 12_000).astype(np.uint32)
        b_e2 = np.minimum(b_s2 + rng.integers(0, max_span, 12_000), 2999).astype(np.uint32)
        _mc_b_case(a_s2, a_e2, b_s2, b_e2, off2, 6, 1, 4, expect_fused=fused)
    # (3) very small sets
    for n in (1, 2, 5, 33):
        _mc_b_case(a_s2[:7], a_e2[:7], b_s2[:n], b_e2[:n], off2, 7, 0, 3)
        _mc_b_case(a_s2[:n], a_e2[:n], b_s2[:100], b_e2[:100], off2, 7, 0, 3)


@pytest.mark.parametrize("k,scale,rounds", [(1, 1.0, 3), (5, 0.02, 2), (5, 1.0, 2)])
def test_mc_permute_b_leaves_sorted_arrays_of_last_round(k, scale, rounds):
    """The sort step inside the Monte Carlo loop: after R rounds the workspace holds B_S and B_E of round
    R-1, which must equal std::sort of the oracle's placement of that round, element for element."""
    w = W.make_config(k, scale=scale)
    n_chrom = int(w.chrom_offsets.size - 1)
    ws = torch.empty(bits.workspace_bytes(bits.FN_MC_ROUNDS, w.n_a, w.n_b, n_chrom, 1), dtype=torch.uint8, device=DEV)
    bits.mc_rounds(dev(w.a_start), dev(w.a_end), dev(w.b_start), dev(w.b_end), w.chrom_offsets, 1, w.mc_seed, 5, rounds,
                   workspace=ws)
    sync()
    b_s, b_e = bits.sorted_arrays_in_workspace(ws, bits.FN_MC_ROUNDS, w.n_a, w.n_b, n_chrom, 1)
    spans = (w.b_end - w.b_start).astype(np.uint32)
    o_s, o_e = oracle.place_round(spans, w.chrom_offsets, w.mc_seed, 5 + rounds - 1, 1)
    assert np.array_equal(host_u32(b_s), oracle.sort_u32(o_s))
    assert np.array_equal(host_u32(b_e), oracle.sort_u32(o_e))


def _screen_tracks(rng, off, shapes):
    n_chrom = off.size - 1
    tracks = []
    for n, max_len in shapes:
        c = rng.integers(0, n_chrom, n)
        ln = rng.integers(1, max_len, n)
        lo, hi = off[:-1][c].astype(np.int64), off[1:][c].astype(np.int64)
        s = lo + (rng.random(n) * (hi - lo - ln)).astype(np.int64)
        tracks.append((s.astype(np.uint32), (s + ln - 1).astype(np.uint32)))
    return tracks


def test_screen_of_tracks_matches_oracle():
    """bits_screen: K x K observed counts, every round count (pair id in the Philox counter) and
    log2(observed / median), against oracle.screen; tracks of very different sizes, one of them empty; round slicing."""
    rng = np.random.default_rng(31)
    off = W.genome_offsets([3_000_000, 2_000_000, 1_200_000])
    tracks = _screen_tracks(rng, off, ((4000, 400), (2500, 2000), (0, 10), (6000, 120), (1, 50), (1025, 300)))
    K, R, seed = len(tracks), 21, 4
    dtracks = [(dev(s), dev(e)) for s, e in tracks]
    before = bits.launch_count()
    obs, enr, rc = bits.screen(dtracks, off, seed, R)
    n_launches = bits.launch_count() - before
    o_obs, o_rc, o_enr = oracle.screen(tracks, off, seed, 0, R)
    assert np.array_equal(obs, o_obs) and np.array_equal(rc, o_rc)
    assert np.array_equal(enr, o_enr, equal_nan=True)
    assert n_launches < 40 * K                                # setup per track + two gridded launches, not per pair
    # pair (0, 0) is the plain Monte Carlo job (stream 0); other pairs draw from their own stream
    _, plain = run_mc(W.Workload("t", *tracks[0], *tracks[0], off), 0, seed, 0, R)
    assert np.array_equal(rc[0, 0], plain)
    _, plain01 = run_mc(W.Workload("t", *tracks[0], *tracks[1], off), 0, seed, 0, R)
    assert not np.array_equal(rc[0, 1], plain01)
    # rounds are addressed by (seed, round, pair): slices of the round range are bit-identical
    _, _, hi = bits.screen(dtracks, off, seed, R - 8, round_begin=8)
    assert np.array_equal(hi, o_rc[:, :, 8:])
    # a single track, and no rounds
    obs1, _, rc1 = bits.screen(dtracks[:1], off, seed, 0)
    assert obs1.shape == (1, 1) and int(obs1[0, 0]) == int(o_obs[0, 0]) and rc1.shape == (1, 1, 0)


def test_screen_genome_scale_tracks():
    """A screen on the 24-chromosome genome with tracks large enough for several query tiles and the MSD sort."""
    rng = np.random.default_rng(32)
    off = W.genome_offsets(W.GENOME24_LENGTHS)
    tracks = _screen_tracks(rng, off, ((30_000, 3000), (70_001, 800), (12_345, 20_000)))
    obs, enr, rc = bits.screen([(dev(s), dev(e)) for s, e in tracks], off, 9, 5, round_begin=4_000_000_000)
    o_obs, o_rc, o_enr = oracle.screen(tracks, off, 9, 4_000_000_000, 5)
    assert np.array_equal(obs, o_obs) and np.array_equal(rc, o_rc) and np.array_equal(enr, o_enr, equal_nan=True)


def test_screen_errors():
    off = np.array([0, 1000, 3000], dtype=np.uint32)
    s, e = dev([1, 5, 0]), dev([3, 9, 2000])                  # the third interval is as long as the longest chromosome
    with pytest.raises(bits.BitsError) as ei:
        bits.screen_concat(s, e, [0, 2, 3], off, 1, 4)
    assert ei.value.status == 4
    obs, rc = bits.screen_concat(s, e, [0, 2, 3], off, 1, 0)  # no rounds: nothing is placed, the observed counts are fine
    sync()
    assert host_u64(obs).reshape(2, 2)[0, 1] == 2
    with pytest.raises(bits.BitsError):
        bits.screen_concat(s, e, [0, 3, 2], off, 1, 4)        # offsets must not decrease


def test_cli_on_bed_files(tmp_path, capsys):
    """The command line end to end on small BED files: counts, per-interval counts, pairs and Monte Carlo summary."""
    from paper_1208_3407_b200 import cli, frontend as F
    rng = np.random.default_rng(12)
    (tmp_path / "g.txt").write_text("chr1 50000\nchr2 30000\nchr3 20000\n")
    names, lens = ["chr1", "chr2", "chr3"], [50000, 30000, 20000]
    def bed(n, max_len):
        out = []
        for _ in range(n):
            c = int(rng.integers(0, 3)); ln = int(rng.integers(1, max_len)); s = int(rng.integers(0, lens[c] - ln))
            out.append(f"{names[c]}\t{s}\t{s + ln}\n")
        return "".join(out)
    (tmp_path / "a.bed").write_text(bed(400, 300))
    (tmp_path / "b.bed").write_text("track x\n" + bed(900, 600))
    base = ["-a", str(tmp_path / "a.bed"), "-b", str(tmp_path / "b.bed"), "-g", str(tmp_path / "g.txt")]
    g = F.read_genome(str(tmp_path / "g.txt"))
    a_s, a_e = F.read_bed(str(tmp_path / "a.bed"), g)
    b_s, b_e = F.read_bed(str(tmp_path / "b.bed"), g)
    total, counts = oracle.count_per_interval(a_s, a_e, b_s, b_e)
    assert cli.main(["count"] + base) == 0 and int(capsys.readouterr().out) == total
    assert cli.main(["per-interval"] + base) == 0 and list(map(int, capsys.readouterr().out.split())) == counts.tolist()
    assert cli.main(["decide"] + base) == 0 and int(capsys.readouterr().out) == int(total > 0)
    assert cli.main(["enumerate"] + base) == 0
    pairs = sorted(tuple(map(int, l.split())) for l in capsys.readouterr().out.splitlines())
    assert pairs == [tuple(p) for p in oracle.enumerate_pairs(a_s, a_e, b_s, b_e).tolist()]
    for permute, which in (("a", 0), ("b", 1)):
        assert cli.main(["mc"] + base + ["-n", "25", "--permute", permute, "--seed", "3"]) == 0
        out = dict(l.split("\t") for l in capsys.readouterr().out.splitlines())
        o_obs, o_rc = oracle.mc_rounds(a_s, a_e, b_s, b_e, g.offsets, which, 3, 0, 25)
        assert int(out["observed"]) == o_obs and float(out["p_enrichment"]) == oracle.pvalue(o_obs, o_rc, 0)
        assert float(out["log2_observed_over_median"]) == oracle.enrichment(o_obs, o_rc)
    assert cli.main(["count", "-a", str(tmp_path / "nope.bed"), "-b", str(tmp_path / "b.bed"), "-g", str(tmp_path / "g.txt")]) == 2


# ------------------------------------------------------------------------------------- input checking, large sizes
def test_validate_flag_through_every_entry_point():
    """BITS_VALIDATE through bits_mc_rounds (both kinds), bits_enumerate and bits_screen: a set with one start > end is
    refused with status 7 (BITS_ERR_MALFORMED), well-formed sets give the oracle's integers with the flag on."""
    rng = np.random.default_rng(41)
    off = W.genome_offsets([3_000_000, 2_000_000, 1_200_000])
    tracks = _screen_tracks(rng, off, ((3000, 400), (20_000, 900)))
    (a_s, a_e), (b_s, b_e) = tracks
    i_a = int(np.argmax(a_s > 0))
    bad_e = a_e.copy(); bad_e[i_a] = a_s[i_a] - 1                        # a malformed interval in A
    assert b_s[-1] > 0
    bad_be = b_e.copy(); bad_be[-1] = b_s[-1] - 1                        # ... and one in B (the last element)
    for which in (0, 1):
        obs, rc = bits.mc_rounds(dev(a_s), dev(a_e), dev(b_s), dev(b_e), off, which, 3, 0, 7, flags=bits.VALIDATE)
        sync()
        o_obs, o_rc = oracle.mc_rounds(a_s, a_e, b_s, b_e, off, which, 3, 0, 7)
        assert int(host_u64(obs)[0]) == o_obs and np.array_equal(host_u64(rc), o_rc)
        for args in ((a_s, bad_e, b_s, b_e), (a_s, a_e, b_s, bad_be)):
            with pytest.raises(bits.BitsError) as e:
                bits.mc_rounds(*[dev(x) for x in args], off, which, 3, 0, 7, flags=bits.VALIDATE)
            assert e.value.status == 7
    pa, pb, n = bits.enumerate_pairs(dev(a_s), dev(a_e), dev(b_s), dev(b_e), flags=bits.VALIDATE)
    sync()
    want = oracle.enumerate_pairs(a_s, a_e, b_s, b_e)
    got = np.stack([host_u32(pa), host_u32(pb)], axis=1)
    assert n == len(want) and np.array_equal(got[np.lexsort((got[:, 1], got[:, 0]))], want)
    for args in ((a_s, bad_e, b_s, b_e), (a_s, a_e, b_s, bad_be)):
        with pytest.raises(bits.BitsError) as e:
            bits.enumerate_pairs(*[dev(x) for x in args], flags=bits.VALIDATE)
        assert e.value.status == 7
    toff = np.array([0, a_s.size, a_s.size + b_s.size], dtype=np.uint64)
    cat = lambda x, y: dev(np.concatenate([x, y]))
    obs, rc = bits.screen_concat(cat(a_s, b_s), cat(a_e, b_e), toff, off, 5, 4, flags=bits.VALIDATE)
    sync()
    o_obs, o_rc, _ = oracle.screen(tracks, off, 5, 0, 4)
    assert np.array_equal(obs.cpu().numpy().view(np.uint64), o_obs) and np.array_equal(rc.cpu().numpy().view(np.uint64), o_rc)
    with pytest.raises(bits.BitsError) as e:
        bits.screen_concat(cat(a_s, b_s), cat(a_e, bad_be), toff, off, 5, 4, flags=bits.VALIDATE)
    assert e.value.status == 7


def test_count_per_interval_host_config4_full_size():
    """The host-buffer entry point at a size where the staging matters (160 MB in, 40 MB out): every one of the 10^7
    per-interval counts and the total against the oracle."""
    w = W.make_config(4)
    o_total, o_counts = oracle.count_per_interval(w.a_start, w.a_end, w.b_start, w.b_end)
    counts, total = bits.count_per_interval_host(w.a_start, w.a_end, w.b_start, w.b_end)
    assert total == o_total
    bad = np.nonzero(counts != o_counts)[0]
    assert bad.size == 0, (bad.size, bad[:5])
    assert bits.count_host(w.a_start, w.a_end, w.b_start, w.b_end) == o_total


def test_mc_permute_b_above_the_fused_limit():
    """A re-placed set of 25M intervals (above the 24M the fused bins hold): every round goes through the general path
    (placement kernel, MSD sort of both arrays, search with the sorted queries).  Two rounds against the oracle, and the
    sorted arrays of the last round."""
    rng = np.random.default_rng(43)
    off = W.genome_offsets(W.GENOME24_LENGTHS)
    n_b, n_a = 25_000_000, 200_000
    def draw(n, max_len):
        c = rng.integers(0, 24, n); ln = rng.integers(1, max_len, n)
        lo, hi = off[:-1][c].astype(np.int64), off[1:][c].astype(np.int64)
        st = lo + (rng.random(n) * (hi - lo - ln)).astype(np.int64)
        return st.astype(np.uint32), (st + ln - 1).astype(np.uint32)
    b_s, b_e = draw(n_b, 500)
    a_s, a_e = draw(n_a, 3000)
    ws = torch.empty(bits.workspace_bytes(bits.FN_MC_ROUNDS, n_a, n_b, 24, 1), dtype=torch.uint8, device=DEV)
    bits.set_option("profile", 2); bits.set_option("profile", 1)
    try:
        obs, rc = bits.mc_rounds(dev(a_s), dev(a_e), dev(b_s), dev(b_e), off, 1, 9, 3, 2, workspace=ws)
        sync()
        prof = bits.profile_read()
    finally:
        bits.set_option("profile", 0)
    assert prof["place_scatter"][1] == 0 and prof["place"][1] == 2          # the general path ran, twice
    o_obs, o_rc = oracle.mc_rounds(a_s, a_e, b_s, b_e, off, 1, 9, 3, 2)
    assert int(host_u64(obs)[0]) == o_obs and np.array_equal(host_u64(rc), o_rc)
    g_s, g_e = bits.sorted_arrays_in_workspace(ws, bits.FN_MC_ROUNDS, n_a, n_b, 24, 1)
    p_s, p_e = oracle.place_round((b_e - b_s).astype(np.uint32), off, 9, 4, 1)
    assert np.array_equal(host_u32(g_s), oracle.sort_u32(p_s)) and np.array_equal(host_u32(g_e), oracle.sort_u32(p_e))


# ------------------------------------------------------------------------------------- host-buffer entry points
def test_host_variants_config1():
    w = W.make_config(1)
    o_total, o_counts = oracle.count_per_interval(w.a_start, w.a_end, w.b_start, w.b_end)
    assert bits.count_host(w.a_start, w.a_end, w.b_start, w.b_end) == o_total
    counts, total = bits.count_per_interval_host(w.a_start, w.a_end, w.b_start, w.b_end)
    assert total == o_total and np.array_equal(counts, o_counts)
    for which in (0, 1):
        r = bits.mc_rounds_host(w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets, which, 1, 0, 25)
        o_obs, o_rc = oracle.mc_rounds(w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets, which, 1, 0, 25)
        assert r.observed == o_obs and np.array_equal(r.round_counts, o_rc)
        assert r.p_enrich == oracle.pvalue(o_obs, o_rc, 0) and r.p_deplete == oracle.pvalue(o_obs, o_rc, 1)


def test_launches_are_counted():
    before = bits.launch_count()
    w = W.make_config(1)
    bits.count(dev(w.a_start), dev(w.a_end), dev(w.b_start), dev(w.b_end))
    sync()
    assert bits.launch_count() >= before + 7     # histogram + 4 passes + index + count


@pytest.mark.skipif(torch.cuda.device_count() < 2, reason="needs two CUDA devices")
def test_second_device_gets_its_own_kernel_attributes():
    """cudaFuncSetAttribute applies per device: the kernels that need more than 48 KB of shared memory must be
    configured on every device the library is used on (round 1 cached the opt-in process-wide)."""
    w = W.make_config(5, scale=0.02)
    want = None
    for d in (0, 1):
        with torch.cuda.device(d):
            t = [torch.from_numpy(np.ascontiguousarray(x, dtype=np.uint32).view(np.int32)).to(f"cuda:{d}")
                 for x in (w.a_start, w.a_end, w.b_start, w.b_end)]
            obs, rc = bits.mc_rounds(*t, w.chrom_offsets, 1, 3, 0, 4)
            counts, total = bits.count_per_interval(*t)
            torch.cuda.synchronize(d)
            got = (int(host_u64(obs)[0]), host_u64(rc).tolist(), int(host_u64(total)[0]))
        if want is None:
            o_obs, o_rc = oracle.mc_rounds(w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets, 1, 3, 0, 4)
            want = (o_obs, o_rc.tolist(), o_obs)
        assert got == want


# ------------------------------------------------------------------------------------- randomised sweep
@pytest.mark.parametrize("seed,cases,big", [(1, 400, False), (2, 400, False), (3, 30, True), (4, 30, True)])
def test_randomised_cases_against_the_oracle(seed, cases, big):
    """Seeded random genomes (1-39 chromosomes of 10^3..2*10^8 bp), set sizes over all size classes of every path
    (one block per round, several rounds per launch pair, one round per launch pair; bucket index and binned search),
    uniform and clustered placement, spans up to the chromosome length: Monte Carlo rounds of both kinds, counts by
    both search designs, screens -- every integer against the oracle."""
    rng = np.random.default_rng(seed)
    def genome():
        k = int(rng.integers(1, 40))
        scale = int(10 ** (rng.uniform(6.5, 8.3) if big else rng.uniform(3, 8.3)))
        lens = rng.integers(max(2, scale // 10), scale + 2, k)
        while lens.sum() >= 2**32 - 1:
            lens = lens // 2 + 1
        return W.genome_offsets(lens)
    def draw(off, n, max_len):
        c = rng.integers(0, off.size - 1, n)
        lo, hi = off[:-1][c].astype(np.int64), off[1:][c].astype(np.int64)
        ln = np.minimum(rng.integers(1, max_len + 1, n), hi - lo)
        frac = rng.beta(0.3, 0.3, n) if rng.random() < 0.3 else rng.random(n)     # clustered at the chromosome ends, or uniform
        st = np.minimum(lo + ((hi - lo - ln + 1) * frac).astype(np.int64), hi - ln)
        return st.astype(np.uint32), (st + ln - 1).astype(np.uint32)
    done = 0
    while done < cases:
        off = genome()
        lmax = int(np.diff(off.astype(np.int64)).max())
        kind = int(rng.integers(0, 3))
        if kind == 0:
            n_b = int(10 ** (rng.uniform(3.9, 6.5) if big else rng.uniform(0, 4.9)))
            n_a = int(10 ** (rng.uniform(2, 5.3) if big else rng.uniform(0, 4.3)))
            max_len = max(1, int(min(lmax - 1, 10 ** rng.uniform(0, 5))))
            b_s, b_e = draw(off, n_b, max_len); a_s, a_e = draw(off, n_a, max_len)
            which = 1 if big else int(rng.integers(0, 2))
            R = int(rng.integers(1, 10 if big else 70)); r0 = int(rng.integers(0, 2**32 - 100)); mc_seed = int(rng.integers(0, 2**63))
            if int(((b_e - b_s) if which else (a_e - a_s)).max()) >= lmax:
                continue
            obs, rc = bits.mc_rounds(dev(a_s), dev(a_e), dev(b_s), dev(b_e), off, which, mc_seed, r0, R)
            sync()
            o_obs, o_rc = oracle.mc_rounds(a_s, a_e, b_s, b_e, off, which, mc_seed, r0, R)
            assert int(host_u64(obs)[0]) == o_obs and np.array_equal(host_u64(rc), o_rc), ("mc", n_a, n_b, off.size - 1, which, R, r0, mc_seed)
        elif kind == 1:
            n_b = int(10 ** (rng.uniform(5, 6.7) if big else rng.uniform(0, 5.5)))
            n_a = int(10 ** (rng.uniform(5, 6.4) if big else rng.uniform(0, 5.3)))
            b_s, b_e = draw(off, n_b, int(10 ** rng.uniform(0, 7))); a_s, a_e = draw(off, n_a, int(10 ** rng.uniform(0, 7)))
            check_counts(a_s, a_e, b_s, b_e)
        else:
            K = int(rng.integers(1, 6)); R = int(rng.integers(0, 8))
            tracks = [draw(off, int(10 ** rng.uniform(0, 4)), max(1, int(min(lmax - 1, 10 ** rng.uniform(0, 4))))) for _ in range(K)]
            if max(int((e - st).max()) for st, e in tracks) >= lmax:
                continue
            obs, enr, rc = bits.screen([(dev(st), dev(e)) for st, e in tracks], off, 7, R, round_begin=3)
            o_obs, o_rc, o_enr = oracle.screen(tracks, off, 7, 3, R)
            assert np.array_equal(obs, o_obs) and np.array_equal(rc, o_rc) and np.array_equal(enr, o_enr, equal_nan=True), ("screen", K, R)
        done += 1
