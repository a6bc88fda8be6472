"""C-ABI checks that need no GPU: the library builds, loads, exports every symbol include/bits.h
declares, sizes workspaces, and rejects bad arguments on the host before any CUDA call."""
import ctypes as C
import math
import os
import re

import numpy as np
import pytest

from paper_1208_3407_b200 import bits

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "bits.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(bits_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported_and_bound():
    names = declared_symbols()
    assert len(names) >= 15
    raw = C.CDLL(bits.lib_path() if os.path.exists(bits.lib_path()) else bits.lib()._name)
    bits.lib()
    for n in names:
        assert hasattr(raw, n), f"{n} declared in bits.h but not exported"
    assert set(names) == set(bits.EXPORTS)


def test_version_and_strerror():
    assert "sm_100a" in bits.version()
    assert bits.strerror(0) == "ok"
    for s in range(1, 9):
        assert bits.strerror(s) not in ("ok", "unknown status")
    assert bits.strerror(99) == "unknown status"


def test_workspace_sizes():
    w = bits.workspace_bytes
    assert w(99, 1, 1) == 0
    assert w(bits.FN_COUNT, 2**32, 1) == 0
    assert w(bits.FN_COUNT, 2**28, 1) == 0 and w(bits.FN_COUNT, 1, 2**28) == 0      # the documented bound: n < 2^28
    assert w(bits.FN_COUNT, 2**28 - 1, 2**28 - 1) > 16 * (2**28 - 1)
    small, big = w(bits.FN_COUNT, 10, 1000), w(bits.FN_COUNT, 10, 10_000_000)
    assert 0 < small < big
    assert big >= 4 * 4 * 10_000_000                      # two arrays, ping + pong
    assert big % 256 == 0
    mc_a = w(bits.FN_MC_ROUNDS, 10_000, 1_000_000, 24, bits.PERMUTE_A)
    mc_b = w(bits.FN_MC_ROUNDS, 10_000, 1_000_000, 24, bits.PERMUTE_B)
    assert mc_b > mc_a > w(bits.FN_SORT, 0, 1_000_000)
    # where the count path can bin the queries by B's buckets (both sets large, B not already sorted) the workspace also
    # holds the queries in bucket order: 12 bytes per query with per-interval counts, 8 without ...
    na, nb = 1 << 20, 3 << 20
    assert w(bits.FN_COUNT_PER_INTERVAL, na, nb) - w(bits.FN_COUNT, na, nb) >= 4 * na - 4096
    assert w(bits.FN_COUNT, na, nb) - w(bits.FN_COUNT, 0, nb) >= 8 * na
    # ... and nowhere else: smaller sets and BITS_B_SORTED calls take the index path, whose workspace does not grow with n_a
    assert w(bits.FN_COUNT, na, nb, 0, 0, bits.B_SORTED) == w(bits.FN_COUNT, 0, nb)
    assert w(bits.FN_COUNT_PER_INTERVAL, 10_000_000, 1_000_000) == w(bits.FN_COUNT, 0, 1_000_000)
    assert w(bits.FN_COUNT, na - 1, nb) == w(bits.FN_COUNT, 0, nb)
    assert w(bits.FN_MC_ROUNDS, 0, 0, 1, 0) > 0
    assert bits.host_staging_bytes(bits.FN_MC_ROUNDS, 1000, 1000, 100) >= 4 * 4 * 1000 + 8 * 100


def test_enrichment_matches_the_oracle_formula():
    """bits_enrichment is host arithmetic on integers: it must equal the oracle's double bit for bit (tolerance 0;
    both are log2 of one double division of the observed count by the median)."""
    import math
    import oracle
    rng = np.random.default_rng(9)
    for n in (1, 2, 3, 10, 999, 1000):
        rc = rng.integers(0, 50_000, n).astype(np.uint64)
        for obs in (0, 1, 777, 10**7):
            a, b = bits.enrichment(obs, rc), oracle.enrichment(obs, rc)
            assert (math.isnan(a) and math.isnan(b)) or a == b
    assert math.isnan(bits.enrichment(5, [])) and bits.enrichment(3, [0, 0, 0]) == math.inf


def test_pvalue():
    assert bits.pvalue(10, [], 0) == 1.0
    assert bits.pvalue(10, [1, 2, 3], 0) == 1 / 4
    assert bits.pvalue(10, [1, 2, 3], 1) == 1.0
    assert bits.pvalue(2, [1, 2, 3, 2], 0) == 4 / 5
    assert bits.pvalue(0, [5] * 99, 1) == 1 / 100
    assert math.isnan(bits.pvalue(1, [1], 2))
    big = 2**63 + 5                                        # uint64 range, not int64
    assert bits.pvalue(big, np.array([big - 1, big, big + 1], dtype=np.uint64), 0) == 3 / 4


def test_set_option_rejects_unknown():
    with pytest.raises(bits.BitsError):
        bits.set_option("no_such_knob", 1)
    bits.set_option("grid_mult", 8)
    with pytest.raises(bits.BitsError):
        bits.set_option("grid_mult", 0)


def test_host_side_argument_checks_return_before_cuda():
    L = bits.lib()
    fake = 0x1000  # never dereferenced: every call below must fail in the host checks
    ws = 256 * 4
    off = np.array([0, 100], dtype=np.uint32)
    st = L.bits_count(fake, fake, 2**32, fake, fake, 1, 0, ws, 1 << 40, fake, None)
    assert st == 2                                         # BITS_ERR_SIZE
    assert L.bits_count(fake, fake, 1, fake, fake, 1, 8, ws, 1 << 40, fake, None) == 6     # flags
    assert L.bits_count(None, fake, 1, fake, fake, 1, 0, ws, 1 << 40, fake, None) == 1     # null
    assert L.bits_count(fake, fake, 1, fake, fake, 1, 0, ws, 1 << 40, None, None) == 1     # null out
    assert L.bits_count(fake, fake, 1, fake, fake, 1, 0, None, 0, fake, None) == 5         # workspace
    assert L.bits_count(fake, fake, 1, fake, fake, 1, 0, ws + 8, 1 << 40, fake, None) == 5  # misaligned
    assert L.bits_count(fake, fake, 1, fake, fake, 1, 0, ws, 16, fake, None) == 5          # too small
    assert L.bits_count_per_interval(fake, fake, 1, fake, fake, 1, 0, ws, 1 << 40, None, fake, None) == 1
    mc = lambda o, nch, which, rb, nr: L.bits_mc_rounds(fake, fake, 1, fake, fake, 1, o, nch, which, 1, rb, nr, 0,
                                                        ws, 1 << 40, fake, fake, None)
    assert mc(off.ctypes.data, 1, 2, 0, 1) == 6                                            # which
    assert mc(None, 1, 0, 0, 1) == 1
    assert mc(off.ctypes.data, 0, 0, 0, 1) == 3                                            # n_chrom == 0
    assert mc(off.ctypes.data, 1, 0, 2**32 - 1, 2) == 2                                    # round overflow
    # independently sorted B has lost the pairing of starts and ends, so its lengths cannot be kept
    assert L.bits_mc_rounds(fake, fake, 1, fake, fake, 1, off.ctypes.data, 1, bits.PERMUTE_B, 1, 0, 1, bits.B_SORTED,
                            ws, 1 << 40, fake, fake, None) == 6
    bad1 = np.array([1, 100], dtype=np.uint32)
    bad2 = np.array([0, 100, 100], dtype=np.uint32)
    assert mc(bad1.ctypes.data, 1, 0, 0, 1) == 3
    assert mc(bad2.ctypes.data, 2, 0, 0, 1) == 3
    assert L.bits_place(fake, 4, bad1.ctypes.data, 1, 1, 0, 0, ws, 1 << 40, fake, fake, None) == 3
    assert L.bits_sort_u32(None, fake, 4, ws, 1 << 40, None) == 1
    assert L.bits_sort_u32(fake, fake, 2**32, ws, 1 << 40, None) == 2


def test_new_entry_points_reject_bad_arguments_on_the_host():
    """bits_decide / bits_enumerate / bits_workspace_sorted_offset: argument errors come back before any CUDA call."""
    L = bits.lib()
    one = (C.c_uint32 * 4)(1, 2, 3, 4)
    p = C.addressof(one)
    tot = C.c_uint64(0)
    # NULL outputs
    assert L.bits_decide(p, p, 1, p, p, 1, 0, 0, 0, 0, 0) == 1
    assert L.bits_enumerate(p, p, 1, p, p, 1, 0, 0, 0, 0, 0, 0, 0, 0) == 1
    assert L.bits_enumerate(p, p, 1, p, p, 1, 0, 0, 0, 0, 0, 5, C.addressof(tot), 0) == 1      # capacity without arrays
    # independently sorted B has lost the pairing of starts and ends: enumeration refuses it
    assert L.bits_enumerate(p, p, 1, p, p, 1, bits.B_SORTED, 0, 0, p, p, 4, C.addressof(tot), 0) == 6
    # unknown flag bits, sizes
    assert L.bits_decide(p, p, 1, p, p, 1, 64, 0, 0, p, 0) == 6
    assert L.bits_decide(p, p, 2**32, p, p, 1, 0, 0, 0, p, 0) == 2
    # workspace missing
    assert L.bits_decide(p, p, 1, p, p, 1, 0, 0, 0, p, 0) == 5
    assert L.bits_enumerate(p, p, 1, p, p, 1, 0, 0, 0, 0, 0, 0, C.addressof(tot), 0) == 5
    assert bits.workspace_bytes(bits.FN_ENUMERATE, 1000, 1000) > bits.workspace_bytes(bits.FN_SORT, 0, 1000) + 1000 * 24
    off = C.c_size_t(0)
    assert L.bits_workspace_sorted_offset(bits.FN_COUNT, 10, 1000, 0, 0, 1, C.addressof(off)) == 0 and off.value > 0
    assert L.bits_workspace_sorted_offset(bits.FN_SORT, 10, 1000, 0, 0, 0, C.addressof(off)) == 6
    assert L.bits_workspace_sorted_offset(bits.FN_COUNT, 10, 1000, 0, 0, 2, C.addressof(off)) == 6


def test_options_are_thread_local():
    """bits_set_option state belongs to the calling host thread (bits.h, "Threads")."""
    import threading
    L = bits.lib()
    assert L.bits_set_option(b"grid_mult", 3) == 0
    seen = {}
    def other():
        seen["rc"] = L.bits_set_option(b"grid_mult", 99)          # out of range: this thread's value stays at its default
        seen["bad"] = L.bits_set_option(b"no_such_knob", 1)
    t = threading.Thread(target=other); t.start(); t.join()
    assert seen == {"rc": 6, "bad": 6}
    assert L.bits_set_option(b"grid_mult", 8) == 0
    assert L.bits_set_option(b"mc_shift_bias", 9) == 6 and L.bits_set_option(b"mc_shift_bias", 0) == 0


def test_screen_rejects_bad_arguments_on_the_host():
    """bits_screen / bits_screen_workspace_bytes / bits_screen_enrichment: argument errors before any CUDA call."""
    L = bits.lib()
    one = (C.c_uint32 * 4)(1, 2, 3, 4)
    p = C.addressof(one)
    off = np.array([0, 100], dtype=np.uint32)
    good = np.array([0, 2, 4], dtype=np.uint64)
    wsb = lambda t, k: L.bits_screen_workspace_bytes(t.ctypes.data if t is not None else None, k, 1)
    assert wsb(good, 2) > 0 and wsb(good, 2) % 256 == 0
    assert wsb(None, 2) == 0 and wsb(good, 0) == 0 and wsb(good[:2], 65536) == 0
    assert wsb(np.array([1, 2, 4], dtype=np.uint64), 2) == 0                      # [0] != 0
    assert wsb(np.array([0, 3, 2], dtype=np.uint64), 2) == 0                      # decreasing
    assert wsb(np.array([0, 2, 2**32], dtype=np.uint64), 2) == 0                  # too many intervals
    assert wsb(np.array([0, 0, 0], dtype=np.uint64), 2) > 0                       # empty tracks are legal
    big = wsb(np.array([0, 100_000, 200_000, 300_000], dtype=np.uint64), 3)
    assert big > 3 * 100_000 * 4 * 2
    scr = lambda t, k, o, nch, rb, nr, fl, obs, rc: L.bits_screen(p, p, t.ctypes.data if t is not None else None, k,
                                                                  o.ctypes.data if o is not None else None, nch, 1, rb, nr, fl,
                                                                  0, 0, obs, rc, None)
    assert scr(None, 2, off, 1, 0, 1, 0, p, p) == 1
    assert scr(good, 0, off, 1, 0, 1, 0, p, p) == 2
    assert scr(good, 2, off, 1, 0, 1, 1, p, p) == 6                               # BITS_B_SORTED means nothing here
    assert scr(good, 2, off, 1, 0, 1, 0, None, p) == 1
    assert scr(good, 2, off, 1, 0, 1, 0, p, None) == 1
    assert scr(good, 2, off, 1, 2**32 - 1, 2, 0, p, p) == 2
    assert scr(good, 2, None, 1, 0, 1, 0, p, p) == 1
    assert scr(good, 2, off, 0, 0, 1, 0, p, p) == 3
    assert scr(good, 2, off, 1, 0, 1, 0, p, p) == 5                               # no workspace
    # enrichment of every pair on the host
    obs = np.array([8, 0, 5], dtype=np.uint64)
    rc = np.array([[2, 2, 4], [0, 0, 0], [0, 0, 1]], dtype=np.uint64)
    out = np.zeros(3)
    assert L.bits_screen_enrichment(obs.ctypes.data, rc.ctypes.data, 3, 3, out.ctypes.data) == 0
    assert out[0] == 2.0 and math.isnan(out[1]) and out[2] == math.inf
    assert L.bits_screen_enrichment(None, rc.ctypes.data, 3, 3, out.ctypes.data) == 1
    assert np.array_equal(bits.screen_enrichment(obs, rc), out, equal_nan=True)
