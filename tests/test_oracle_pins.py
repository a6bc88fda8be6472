"""Pins for the CPU oracle (oracle/bits_oracle.cpp) -- run with -m "not gpu".

Nothing here touches the CUDA path.  Every check ties the oracle to something other than
itself: the paper's closed-interval predicate evaluated by O(N*M) brute force
(PAPER.md:31, :43-45), the exclusion sets L and R counted directly,
closed forms, invariants named in BASELINE.json's north_star, the Philox4x32-10 known-answer
vectors (tests/golden/philox4x32_10_kat.txt) and cuRAND's own header routine, Python
big-integer arithmetic for the multiply-high, and the exact hit probability of a uniformly
placed interval.
"""
import ctypes as C
import os
import subprocess

import numpy as np
import pytest

import oracle
from paper_1208_3407_b200 import workloads as W

HERE = os.path.dirname(os.path.abspath(__file__))


# ----------------------------------------------------------------------------- helpers
def brute_counts(a_s, a_e, b_s, b_e):
    """c(a) = #{b : a.start <= b.end and a.end >= b.start}  (closed intervals)."""
    a_s = np.asarray(a_s, dtype=np.int64)[:, None]
    a_e = np.asarray(a_e, dtype=np.int64)[:, None]
    b_s = np.asarray(b_s, dtype=np.int64)[None, :]
    b_e = np.asarray(b_e, dtype=np.int64)[None, :]
    return ((a_s <= b_e) & (a_e >= b_s)).sum(axis=1).astype(np.uint32)


def rand_sets(rng, n_a, n_b, span=2000, max_len=60):
    a_s = rng.integers(0, span, n_a)
    a_e = a_s + rng.integers(0, max_len, n_a)
    b_s = rng.integers(0, span, n_b)
    b_e = b_s + rng.integers(0, max_len, n_b)
    return a_s, a_e, b_s, b_e


@pytest.fixture(scope="module")
def curand_philox(tmp_path_factory):
    """cuRAND's curand_Philox4x32_10 compiled for the host: an independent library Philox."""
    d = tmp_path_factory.mktemp("curand")
    so = str(d / "curand_philox_host.so")
    subprocess.check_call(["g++", "-O2", "-fPIC", "-shared", "-I/usr/local/cuda/include",
                           "-o", so, os.path.join(HERE, "golden", "curand_philox_host.cpp")])
    lib = C.CDLL(so)
    u32p = C.POINTER(C.c_uint32)
    lib.curand_philox_host.argtypes = [u32p, u32p, u32p]

    def call(ctr, key):
        c = np.asarray(ctr, dtype=np.uint32)
        k = np.asarray(key, dtype=np.uint32)
        o = np.zeros(4, dtype=np.uint32)
        lib.curand_philox_host(c.ctypes.data_as(u32p), k.ctypes.data_as(u32p), o.ctypes.data_as(u32p))
        return o
    return call


# ----------------------------------------------------------------------------- Philox
def test_philox_known_answers():
    rows = 0
    with open(os.path.join(HERE, "golden", "philox4x32_10_kat.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            v = [int(x, 16) for x in line.split()]
            out = oracle.philox4x32_10(v[0:4], v[4:6])
            assert [int(x) for x in out] == v[6:10], line
            rows += 1
    assert rows == 5


def test_philox_matches_curand_header(curand_philox):
    rng = np.random.default_rng(7)
    for _ in range(300):
        ctr = rng.integers(0, 2**32, 4, dtype=np.uint64).astype(np.uint32)
        key = rng.integers(0, 2**32, 2, dtype=np.uint64).astype(np.uint32)
        assert np.array_equal(oracle.philox4x32_10(ctr, key), curand_philox(ctr, key))
    # structured counters of the kind the placement uses: (i>>1, round, tag, 0)
    for i in (0, 1, 2, 12345, 2**31, 2**32 - 1):
        for r in (0, 1, 999, 2**32 - 1):
            for tag in (0, 1):
                ctr = [i, r, tag, 0]
                assert np.array_equal(oracle.philox4x32_10(ctr, [1, 0]), curand_philox(ctr, [1, 0]))


# ----------------------------------------------------------------------------- counting
@pytest.mark.parametrize("seed", range(6))
def test_count_equals_brute_force(seed):
    rng = np.random.default_rng(seed)
    n_a, n_b = int(rng.integers(1, 200)), int(rng.integers(1, 300))
    a_s, a_e, b_s, b_e = rand_sets(rng, n_a, n_b, span=int(rng.integers(5, 3000)))
    total, counts = oracle.count_per_interval(a_s, a_e, b_s, b_e)
    bc = brute_counts(a_s, a_e, b_s, b_e)
    assert np.array_equal(counts, bc)
    assert total == int(bc.sum())
    assert oracle.count(a_s, a_e, b_s, b_e) == total


def test_shared_endpoints_closed_rule():
    # PAPER.md:31 closed intervals: touching endpoints intersect.
    one = lambda a, b: oracle.count([a[0]], [a[1]], [b[0]], [b[1]])
    assert one((10, 20), (20, 30)) == 1
    assert one((10, 20), (21, 30)) == 0
    assert one((10, 20), (0, 10)) == 1
    assert one((10, 20), (0, 9)) == 0
    assert one((10, 20), (12, 13)) == 1      # contained
    assert one((12, 13), (10, 20)) == 1      # containing
    assert one((5, 5), (5, 5)) == 1          # point intervals
    assert one((5, 5), (6, 6)) == 0


def test_exclusion_identity():
    # |I| = |B| - |L| - |R| with L = {b.end < a.start}, R = {b.start > a.end}.
    rng = np.random.default_rng(11)
    a_s, a_e, b_s, b_e = rand_sets(rng, 150, 400)
    _, counts = oracle.count_per_interval(a_s, a_e, b_s, b_e)
    for i in range(a_s.size):
        L = int((b_e < a_s[i]).sum())
        R = int((b_s > a_e[i]).sum())
        assert int(counts[i]) == b_s.size - L - R


def test_closed_form_points():
    M = 500
    k = np.arange(M)
    xs = np.array([0, 3, 100, 499, 250, 499])
    ys = np.array([0, 10, 100, 499, 900, 10_000])
    _, c = oracle.count_per_interval(xs, ys, k, k)
    assert np.array_equal(c, np.minimum(ys, M - 1) - xs + 1)
    # queries entirely to the right of every point
    assert oracle.count([600], [700], k, k) == 0


def test_closed_form_copies_ties():
    M, p, q = 257, 1000, 2000
    b_s, b_e = np.full(M, p), np.full(M, q)
    qs = [(0, 999), (0, 1000), (1500, 1600), (2000, 2500), (2001, 2500), (0, 5000)]
    want = [0, M, M, M, 0, M]
    _, c = oracle.count_per_interval([x for x, _ in qs], [y for _, y in qs], b_s, b_e)
    assert list(c) == want


def test_closed_form_nested_containment_trap():
    # B nested [k, 2K-k]; a point query x < K meets exactly the x+1 outermost intervals.
    # The naive "one search then scan back" method misses these (Fig. 1A/B).
    K = 300
    k = np.arange(K)
    xs = np.arange(0, K, 7)
    _, c = oracle.count_per_interval(xs, xs, k, 2 * K - k)
    assert np.array_equal(c, xs + 1)


def test_closed_form_tiles():
    s, w, n = 100, 40, 64          # tiles [k*s, k*s+w-1]
    b_s = np.arange(n) * s
    b_e = b_s + w - 1
    rng = np.random.default_rng(3)
    x = rng.integers(0, n * s, 200)
    y = x + rng.integers(0, 1000, 200)
    # tile k meets [x,y] iff k*s <= y and k*s+w-1 >= x  <=>  ceil((x-w+1)/s) <= k <= floor(y/s)
    lo = np.maximum(0, -((-(x - w + 1)) // s))
    hi = np.minimum(n - 1, y // s)
    want = np.maximum(0, hi - lo + 1)
    _, c = oracle.count_per_interval(x, y, b_s, b_e)
    assert np.array_equal(c, want)


def test_invariants():
    rng = np.random.default_rng(5)
    a_s, a_e, b_s, b_e = rand_sets(rng, 300, 500, span=5000)
    total, counts = oracle.count_per_interval(a_s, a_e, b_s, b_e)
    assert int(counts.astype(np.uint64).sum()) == total                      # sum of per-interval
    assert oracle.count(b_s, b_e, a_s, a_e) == total                         # symmetry
    assert oracle.count(a_s, a_e, [], []) == 0 and oracle.count([], [], b_s, b_e) == 0
    assert oracle.count(a_s, a_e, a_s, a_e) >= a_s.size                      # self-comparison
    assert oracle.count(a_s + 12345, a_e + 12345, b_s + 12345, b_e + 12345) == total   # translation
    p = rng.permutation(b_s.size)
    t2, c2 = oracle.count_per_interval(a_s, a_e, b_s[p], b_e[p])             # shuffling B
    assert t2 == total and np.array_equal(c2, counts)
    q = rng.permutation(a_s.size)
    _, c3 = oracle.count_per_interval(a_s[q], a_e[q], b_s, b_e)              # shuffling A permutes
    assert np.array_equal(c3, counts[q])
    _, c4 = oracle.count_per_interval(a_s, a_e, np.tile(b_s, 2), np.tile(b_e, 2))      # duplicating B
    assert np.array_equal(c4, 2 * counts)
    h = b_s.size // 3                                                        # additivity
    assert oracle.count(a_s, a_e, b_s[:h], b_e[:h]) + oracle.count(a_s, a_e, b_s[h:], b_e[h:]) == total
    _, c5 = oracle.count_per_interval(np.maximum(a_s - 5, 0), a_e + 9, b_s, b_e)       # widening
    assert np.all(c5 >= counts)
    assert counts.max() <= b_s.size


def test_uint32_extremes():
    top = 2**32 - 2
    assert oracle.count([top - 5], [top], [top], [top]) == 1
    assert oracle.count([0], [top], [0, top, 7], [0, top, 9]) == 3
    assert oracle.count([0], [0], [1], [top]) == 0


def test_malformed_rejected():
    with pytest.raises(oracle.OracleError):
        oracle.count([5], [4], [1], [2])
    with pytest.raises(oracle.OracleError):
        oracle.count([1], [2], [5], [4])


def test_sort_equals_numpy():
    rng = np.random.default_rng(9)
    for n in (0, 1, 2, 1000, 65537):
        k = rng.integers(0, 2**32, n, dtype=np.uint64).astype(np.uint32)
        assert np.array_equal(oracle.sort_u32(k), np.sort(k))


# ----------------------------------------------------------------------------- placement
GEN = W.genome_offsets(W.GENOME24_LENGTHS)


def py_place(x, d, off):
    """SURVEY.md 8(c) step 3 in Python big integers: V, u = (x*V) >> 64, chromosome walk."""
    off = [int(v) for v in off]
    v = [max(off[c + 1] - off[c] - d, 0) for c in range(len(off) - 1)]
    V = sum(v)
    u = (x * V) >> 64
    for c, vc in enumerate(v):
        if u < vc:
            return off[c] + u
        u -= vc
    raise AssertionError("u >= V")


def test_place_from_bits_matches_bigint():
    rng = np.random.default_rng(21)
    small = np.array([0, 10, 25, 1000, 1003, 5000], dtype=np.uint32)    # lengths 10,15,975,3,3997
    for off in (GEN, small, np.array([0, 1_000_000], dtype=np.uint32)):
        for _ in range(400):
            x = int(rng.integers(0, 2**64, dtype=np.uint64))
            d = int(rng.integers(0, 20)) if off is small else int(rng.integers(0, 100_000))
            assert oracle.place_from_bits(x, d, off) == py_place(x, d, off)


def test_place_boundaries():
    small = np.array([0, 10, 25, 1000, 1003, 5000], dtype=np.uint32)
    # d = 12: chromosome 0 (len 10) and 3 (len 3) cannot hold it; first usable is chromosome 1.
    assert oracle.place_from_bits(0, 12, small) == 10
    # x = 2^64-1 -> last valid start of the last usable chromosome: 5000 - 1 - 12
    assert oracle.place_from_bits(2**64 - 1, 12, small) == 5000 - 1 - 12
    assert oracle.place_from_bits(0, 0, GEN) == 0
    assert oracle.place_from_bits(2**64 - 1, 0, GEN) == int(GEN[-1]) - 1
    with pytest.raises(oracle.OracleError):
        oracle.place_from_bits(5, 4000, small)       # longer than every chromosome


def test_place_round_counter_layout(curand_philox):
    # counter = (i >> 1, round, tag, 0), key = (seed lo, seed hi); interval i takes words
    # 2h, 2h+1 with h = i & 1.  Rebuilt from cuRAND's routine + big ints.
    rng = np.random.default_rng(4)
    spans = rng.integers(0, 50_000, 41).astype(np.uint32)
    seed, rnd, tag = 0x1234_5678_9ABC_DEF1, 77, 1
    s, e = oracle.place_round(spans, GEN, seed, rnd, tag)
    for i in range(spans.size):
        o = curand_philox([i >> 1, rnd, tag, 0], [seed & 0xFFFFFFFF, seed >> 32])
        h = i & 1
        x = int(o[2 * h]) | (int(o[2 * h + 1]) << 32)
        want = py_place(x, int(spans[i]), GEN)
        assert int(s[i]) == want and int(e[i]) == want + int(spans[i])


def test_place_round_structure():
    rng = np.random.default_rng(8)
    spans = np.clip(np.rint(1000 * np.exp(rng.standard_normal(20_000))), 20, 100_000).astype(np.uint32) - 1
    s, e = oracle.place_round(spans, GEN, 1, 3, 0)
    assert np.array_equal(e - s, spans)                                   # lengths kept
    cs = np.searchsorted(GEN, s, side="right") - 1
    ce = np.searchsorted(GEN, e, side="right") - 1
    assert np.array_equal(cs, ce)                                         # chromosome ends respected
    s2, _ = oracle.place_round(spans, GEN, 1, 4, 0)
    s3, _ = oracle.place_round(spans, GEN, 2, 3, 0)
    s4, _ = oracle.place_round(spans, GEN, 1, 3, 1)
    assert (s != s2).mean() > 0.99 and (s != s3).mean() > 0.99 and (s != s4).mean() > 0.99
    # occupancy per chromosome ~ (L_c - d): chi-square against the exact expectation (d ~ 1e3 << L_c)
    L = np.diff(GEN.astype(np.int64))
    exp = spans.size * L / L.sum()
    obs = np.bincount(cs, minlength=24)
    chi2 = ((obs - exp) ** 2 / exp).sum()
    assert chi2 < 60.0                                                    # 23 dof; P(chi2 > 60) ~ 4e-5


def test_place_hit_probability_closed_form():
    # one chromosome of length L, fixed b=[s,e], span d: P(hit) = (min(e, L-1-d) - max(0, s-d) + 1)/(L-d)
    L, d, s, e = 100_000, 400, 30_000, 31_000
    off = np.array([0, L], dtype=np.uint32)
    n, R = 2_000, 60
    spans = np.full(n, d, dtype=np.uint32)
    a_s, a_e = np.zeros(n, dtype=np.uint32), spans.copy()
    _, rc = oracle.mc_rounds(a_s, a_e, [s], [e], off, 0, 99, 0, R)
    p = (min(e, L - 1 - d) - max(0, s - d) + 1) / (L - d)
    mean, sd = n * R * p, np.sqrt(n * R * p * (1 - p))
    assert abs(int(rc.sum()) - mean) < 4.5 * sd


# ----------------------------------------------------------------------------- Monte Carlo
def test_mc_config1_fully_brute_forced():
    w = W.make_config(1)
    obs, rc = oracle.mc_rounds(w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets, 0, w.mc_seed, 0, 100)
    assert obs == int(brute_counts(w.a_start, w.a_end, w.b_start, w.b_end).sum())
    spans = w.a_end - w.a_start
    for r in range(100):
        s, e = oracle.place_round(spans, w.chrom_offsets, w.mc_seed, r, 0)
        assert int(rc[r]) == int(brute_counts(s, e, w.b_start, w.b_end).sum())


def test_mc_permute_b_brute_forced():
    rng = np.random.default_rng(13)
    off = np.array([0, 40_000, 90_000, 100_000], dtype=np.uint32)
    ls = rng.integers(0, 3, 300)
    a_s = off[ls] + rng.integers(0, 5_000, 300)
    a_e = a_s + rng.integers(0, 900, 300)
    lb = rng.integers(0, 3, 500)
    b_s = off[lb] + rng.integers(0, 5_000, 500)
    b_e = b_s + rng.integers(0, 2_000, 500)
    obs, rc = oracle.mc_rounds(a_s, a_e, b_s, b_e, off, 1, 5, 10, 20)
    assert obs == int(brute_counts(a_s, a_e, b_s, b_e).sum())
    for k in range(20):
        s, e = oracle.place_round(b_e - b_s, off, 5, 10 + k, 1)
        assert int(rc[k]) == int(brute_counts(a_s, a_e, s, e).sum())


def test_mc_round_slicing_is_bit_identical():
    w = W.make_config(1)
    args = (w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets)
    for which in (0, 1):
        _, full = oracle.mc_rounds(*args, which, 1, 0, 30)
        _, lo = oracle.mc_rounds(*args, which, 1, 0, 11)
        _, hi = oracle.mc_rounds(*args, which, 1, 11, 19)
        assert np.array_equal(full, np.concatenate([lo, hi]))


def test_mc_empty_sets():
    off = np.array([0, 1000], dtype=np.uint32)
    for which in (0, 1):
        obs, rc = oracle.mc_rounds([], [], [1], [5], off, which, 1, 0, 4)
        assert obs == 0 and not rc.any()
        obs, rc = oracle.mc_rounds([1], [5], [], [], off, which, 1, 0, 4)
        assert obs == 0 and not rc.any()


def test_pvalue():
    assert oracle.pvalue(10, [], 0) == 1.0
    assert oracle.pvalue(10, [1, 2, 3], 0) == 1 / 4
    assert oracle.pvalue(10, [1, 2, 3], 1) == 1.0
    assert oracle.pvalue(2, [1, 2, 3, 2], 0) == 4 / 5
    assert oracle.pvalue(2, [1, 2, 3, 2], 1) == 4 / 5
    assert oracle.pvalue(0, [5] * 99, 1) == 1 / 100


def test_decide_equals_brute_force_existence():
    """PAPER.md:47 decision sub-problem against the closed predicate written out."""
    rng = np.random.default_rng(77)
    for trial in range(60):
        n_a, n_b = int(rng.integers(0, 12)), int(rng.integers(0, 12))
        a_s = rng.integers(0, 400, n_a); a_e = a_s + rng.integers(0, 15, n_a)
        b_s = rng.integers(0, 400, n_b); b_e = b_s + rng.integers(0, 15, n_b)
        want = any(a_s[i] <= b_e[j] and a_e[i] >= b_s[j] for i in range(n_a) for j in range(n_b))
        assert oracle.decide(a_s, a_e, b_s, b_e) == want
    assert oracle.decide([10], [20], [20], [30]) is True          # shared end point: closed intervals meet
    assert oracle.decide([10], [20], [21], [30]) is False
    assert oracle.decide([], [], [1], [2]) is False


def test_enumerate_pairs_agrees_with_counts_and_a_worked_example():
    """PAPER.md:47 enumeration: the pair set has c(a_i) pairs per a_i (the BITS counts) and matches a hand-made case
    with containment (Fig. 1B situation)."""
    a = ([5, 100], [9, 100])
    b = ([0, 6, 9, 10, 50], [200, 7, 9, 12, 60])               # [0,200] contains everything
    assert oracle.enumerate_pairs(*a, *b).tolist() == [[0, 0], [0, 1], [0, 2], [1, 0]]
    rng = np.random.default_rng(5)
    a_s = rng.integers(0, 5000, 300); a_e = a_s + rng.integers(0, 200, 300)
    b_s = rng.integers(0, 5000, 400); b_e = b_s + rng.integers(0, 900, 400)
    pairs = oracle.enumerate_pairs(a_s, a_e, b_s, b_e)
    total, counts = oracle.count_per_interval(a_s, a_e, b_s, b_e)
    assert len(pairs) == total and np.array_equal(np.bincount(pairs[:, 0], minlength=300), counts)


def test_enrichment_score_closed_cases():
    """log2(observed / median): odd and even numbers of rounds, zero cases."""
    import math
    assert oracle.enrichment(8, [1, 2, 3]) == 2.0                       # median 2
    assert oracle.enrichment(5, [4, 1, 3, 2]) == 1.0                    # median (2 + 3) / 2 = 2.5
    assert oracle.enrichment(1, [4, 4, 4, 4, 4]) == -2.0
    assert oracle.enrichment(3, [0, 0, 0]) == math.inf and math.isnan(oracle.enrichment(0, [0, 0]))
    assert oracle.enrichment(0, [2, 2]) == -math.inf and math.isnan(oracle.enrichment(5, []))
    rng = np.random.default_rng(1)
    x = rng.integers(1, 10**9, 1001)
    assert oracle.enrichment(12345, x) == math.log2(12345 / float(np.median(x)))


# ------------------------------------------------------------------------------------- screen
def test_place_round_stream_is_the_fourth_counter_word(curand_philox):
    # counter = (i >> 1, round, tag, stream): rebuilt from cuRAND's routine + big ints, as for stream 0 above
    rng = np.random.default_rng(40)
    spans = rng.integers(0, 50_000, 23).astype(np.uint32)
    seed, rnd, tag, stream = 0xCAFE_F00D_0BAD_BEEF, 9, 0, 25_280
    s, e = oracle.place_round(spans, GEN, seed, rnd, tag, stream)
    for i in range(spans.size):
        o = curand_philox([i >> 1, rnd, tag, stream], [seed & 0xFFFFFFFF, seed >> 32])
        h = i & 1
        want = py_place(int(o[2 * h]) | (int(o[2 * h + 1]) << 32), int(spans[i]), GEN)
        assert int(s[i]) == want and int(e[i]) == want + int(spans[i])
    s0, _ = oracle.place_round(spans, GEN, seed, rnd, tag)
    assert np.array_equal(s0, oracle.place_round(spans, GEN, seed, rnd, tag, 0)[0]) and (s0 != s).mean() > 0.9


def test_screen_brute_forced():
    """oracle.screen on K = 3 small tracks: every observed count and every round count by
    O(N*M) brute force on placements rebuilt with the pair's own stream id i*K + j; the score from numpy's median."""
    rng = np.random.default_rng(41)
    off = np.array([0, 30_000, 50_000, 90_000], dtype=np.uint32)
    tracks = []
    for n, max_len in ((120, 900), (200, 300), (75, 2500)):
        c = rng.integers(0, 3, n)
        ln = rng.integers(1, max_len, n)
        lo, hi = off[:-1][c].astype(np.int64), off[1:][c].astype(np.int64)
        st = lo + (rng.random(n) * (hi - lo - ln)).astype(np.int64)
        tracks.append((st.astype(np.uint32), (st + ln - 1).astype(np.uint32)))
    K, R, r0, seed = 3, 7, 100, 12
    obs, rc, enr = oracle.screen(tracks, off, seed, r0, R)
    for i in range(K):
        for j in range(K):
            assert int(obs[i, j]) == int(brute_counts(*tracks[i], *tracks[j]).sum())
            spans = tracks[i][1] - tracks[i][0]
            for k in range(R):
                s, e = oracle.place_round(spans, off, seed, r0 + k, 0, i * K + j)
                assert int(rc[i, j, k]) == int(brute_counts(s, e, *tracks[j]).sum())
            med = float(np.median(rc[i, j].astype(np.float64)))
            want = np.log2(float(obs[i, j]) / med) if med > 0 else (np.inf if obs[i, j] else np.nan)
            assert enr[i, j] == want or (np.isnan(enr[i, j]) and np.isnan(want))
    # pair (0, 0) draws from stream 0: the plain Monte Carlo job on (T_0, T_0)
    _, plain = oracle.mc_rounds(*tracks[0], *tracks[0], off, 0, seed, r0, R)
    assert np.array_equal(rc[0, 0], plain)
    # the other pairs have their own null: track 0's draws differ between partners
    assert not np.array_equal(oracle.place_round(tracks[0][1] - tracks[0][0], off, seed, r0, 0, 1)[0],
                              oracle.place_round(tracks[0][1] - tracks[0][0], off, seed, r0, 0, 2)[0])


# ------------------------------------------------------------------------------------- golden round counts
def _golden():
    import importlib.util
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "make_golden.py")
    spec = importlib.util.spec_from_file_location("make_golden", path)
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


@pytest.mark.parametrize("config,slices", [(3, ((0, 40), (3333, 25), (9983, 17))), (5, ((0, 1), (437, 1), (999, 1)))])
def test_golden_round_counts_are_the_oracles(config, slices):
    """tests/golden/cfg{3,5}_seed1_rounds.txt (written by tests/golden/make_golden.py from the oracle over disjoint
    round slices): the inputs are the ones workloads.make_config builds today (checksums), a few slices re-derived
    here from the oracle -- at other slice boundaries than the file was written with -- give the same counts, and
    the stored p-values follow from the stored integers."""
    g = _golden()
    header, counts = g.load(config)
    w = W.make_config(config)
    assert header["checksums"] == w.checksums() and header["chrom_offsets_checksum"] == W.array_checksum(w.chrom_offsets)
    assert header["n_rounds"] == w.n_rounds == counts.size and header["which"] == w.which and header["mc_seed"] == w.mc_seed
    for r0, n in slices:
        obs, rc = oracle.mc_rounds(w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets, w.which, w.mc_seed, r0, n)
        assert obs == header["observed"]
        assert np.array_equal(rc, counts[r0:r0 + n])
    assert header["p_enrich"] == oracle.pvalue(header["observed"], counts, 0)
    assert header["p_deplete"] == oracle.pvalue(header["observed"], counts, 1)
    ge = int((counts >= header["observed"]).sum())
    assert header["p_enrich"] == (ge + 1) / (counts.size + 1)
