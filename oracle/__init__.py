"""ctypes loader for the CPU oracle (oracle/bits_oracle.cpp).

TEST INFRASTRUCTURE ONLY: tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this.  The product package never does, and this module
never imports the product's binding or kernels.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bits_oracle.cpp")
# BITS_ORACLE_SANITIZE=1: the same source under AddressSanitizer + UndefinedBehaviorSanitizer (run the pins with
# LD_PRELOAD="$(gcc -print-file-name=libasan.so) $(gcc -print-file-name=libubsan.so)")
_SANITIZE = bool(os.environ.get("BITS_ORACLE_SANITIZE"))
_LIB = os.path.join(_HERE, "libbits_oracle_san.so" if _SANITIZE else "libbits_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with g++ -O3 -march=native (single-threaded C++17)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        opt = (["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"]
               if _SANITIZE else ["-O3", "-march=native"])
        subprocess.check_call(["g++", "-std=c++17", *opt, "-fPIC", "-shared", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


_u32p = C.POINTER(C.c_uint32)
_u64p = C.POINTER(C.c_uint64)


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.oracle_philox4x32_10.argtypes = [_u32p, _u32p, _u32p]
        L.oracle_sort_u32.argtypes = [_u32p, C.c_uint64]
        L.oracle_count_per_interval.argtypes = [_u32p, _u32p, C.c_uint64, _u32p, _u32p, C.c_uint64, _u32p, _u64p]
        L.oracle_place_from_bits.argtypes = [C.c_uint64, C.c_uint32, _u32p, C.c_uint32, _u32p]
        L.oracle_place_round.argtypes = [_u32p, C.c_uint64, _u32p, C.c_uint32, C.c_uint64, C.c_uint32,
                                         C.c_uint32, _u32p, _u32p]
        L.oracle_place_round_stream.argtypes = [_u32p, C.c_uint64, _u32p, C.c_uint32, C.c_uint64, C.c_uint32,
                                                C.c_uint32, C.c_uint32, _u32p, _u32p]
        L.oracle_mc_rounds.argtypes = [_u32p, _u32p, C.c_uint64, _u32p, _u32p, C.c_uint64, _u32p, C.c_uint32,
                                       C.c_int, C.c_uint64, C.c_uint32, C.c_uint32, _u64p, _u64p]
        L.oracle_mc_rounds_stream.argtypes = [_u32p, _u32p, C.c_uint64, _u32p, _u32p, C.c_uint64, _u32p, C.c_uint32,
                                              C.c_int, C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, _u64p, _u64p]
        L.oracle_pvalue.argtypes = [C.c_uint64, _u64p, C.c_uint32, C.c_int]
        L.oracle_pvalue.restype = C.c_double
        L.oracle_enrichment.argtypes = [C.c_uint64, _u64p, C.c_uint32]
        L.oracle_enrichment.restype = C.c_double
        _lib = L
    return _lib


class OracleError(RuntimeError):
    pass


_ERR = {1: "malformed interval (start > end)", 2: "no valid placement (span >= every chromosome)", 3: "bad argument"}


def _chk(rc):
    if rc != 0:
        raise OracleError(_ERR.get(rc, f"oracle error {rc}"))


def _a32(x):
    a = np.ascontiguousarray(x, dtype=np.uint32)
    return a, a.ctypes.data_as(_u32p)


def philox4x32_10(ctr, key) -> np.ndarray:
    c, cp = _a32(ctr)
    k, kp = _a32(key)
    out = np.zeros(4, dtype=np.uint32)
    _chk(lib().oracle_philox4x32_10(cp, kp, out.ctypes.data_as(_u32p)))
    return out


def sort_u32(keys) -> np.ndarray:
    a = np.array(keys, dtype=np.uint32, copy=True)
    _chk(lib().oracle_sort_u32(a.ctypes.data_as(_u32p), a.size))
    return a


def count_per_interval(a_start, a_end, b_start, b_end, want_counts: bool = True):
    """-> (total:int, counts:uint32[n_a] or None)."""
    a_s, asp = _a32(a_start)
    a_e, aep = _a32(a_end)
    b_s, bsp = _a32(b_start)
    b_e, bep = _a32(b_end)
    assert a_s.size == a_e.size and b_s.size == b_e.size
    counts = np.zeros(a_s.size, dtype=np.uint32) if want_counts else None
    total = C.c_uint64(0)
    _chk(lib().oracle_count_per_interval(asp, aep, a_s.size, bsp, bep, b_s.size,
                                         counts.ctypes.data_as(_u32p) if want_counts else None,
                                         C.byref(total)))
    return int(total.value), counts


def count(a_start, a_end, b_start, b_end) -> int:
    return count_per_interval(a_start, a_end, b_start, b_end, want_counts=False)[0]


def decide(a_start, a_end, b_start, b_end) -> bool:
    """Decision problem (sub-problem 1): does at least one interval of A intersect one of B?
    Answered the way PAPER.md:91 states it -- from the sizes |I(B, a_i)|: true iff some per-interval
    count is non-zero.  Pinned by brute force from the closed predicate (tests/test_oracle_pins.py)."""
    _, counts = count_per_interval(a_start, a_end, b_start, b_end, want_counts=True)
    return bool(np.any(counts != 0))


def enumerate_pairs(a_start, a_end, b_start, b_end):
    """Enumeration problem (sub-problem 4): the set I(A, B) itself, straight from the closed
    predicate a.start <= b.end and a.end >= b.start, as an (n, 2) int64 array of
    (index in A, index in B) sorted lexicographically.  O(|A| * |B|): for small inputs only."""
    a_s = np.asarray(a_start, dtype=np.int64); a_e = np.asarray(a_end, dtype=np.int64)
    b_s = np.asarray(b_start, dtype=np.int64); b_e = np.asarray(b_end, dtype=np.int64)
    out = []
    for i in range(a_s.size):
        j = np.nonzero((a_s[i] <= b_e) & (a_e[i] >= b_s))[0]
        out.append(np.stack([np.full(j.size, i, dtype=np.int64), j.astype(np.int64)], axis=1))
    return np.concatenate(out, axis=0) if out else np.zeros((0, 2), dtype=np.int64)


def place_from_bits(x: int, d: int, chrom_offsets) -> int:
    off, offp = _a32(chrom_offsets)
    s = C.c_uint32(0)
    _chk(lib().oracle_place_from_bits(C.c_uint64(x), C.c_uint32(d), offp, off.size - 1, C.byref(s)))
    return int(s.value)


def place_round(spans, chrom_offsets, seed: int, rnd: int, tag: int, stream: int = 0):
    """One round's placement; `stream` is the fourth Philox counter word (0 = a single job, pair id in the screen)."""
    sp, spp = _a32(spans)
    off, offp = _a32(chrom_offsets)
    s = np.zeros(sp.size, dtype=np.uint32)
    e = np.zeros(sp.size, dtype=np.uint32)
    _chk(lib().oracle_place_round_stream(spp, sp.size, offp, off.size - 1, C.c_uint64(seed), C.c_uint32(rnd),
                                         C.c_uint32(tag), C.c_uint32(stream), s.ctypes.data_as(_u32p),
                                         e.ctypes.data_as(_u32p)))
    return s, e


def mc_rounds(a_start, a_end, b_start, b_end, chrom_offsets, which: int, seed: int,
              round_begin: int, n_rounds: int, stream: int = 0):
    """-> (observed:int, round_counts:uint64[n_rounds]).  stream: fourth Philox counter word of every draw."""
    a_s, asp = _a32(a_start)
    a_e, aep = _a32(a_end)
    b_s, bsp = _a32(b_start)
    b_e, bep = _a32(b_end)
    off, offp = _a32(chrom_offsets)
    obs = C.c_uint64(0)
    rc = np.zeros(max(n_rounds, 1), dtype=np.uint64)
    _chk(lib().oracle_mc_rounds_stream(asp, aep, a_s.size, bsp, bep, b_s.size, offp, off.size - 1, which,
                                       C.c_uint64(seed), C.c_uint32(stream), C.c_uint32(round_begin),
                                       C.c_uint32(n_rounds), C.byref(obs), rc.ctypes.data_as(_u64p)))
    return int(obs.value), rc[:n_rounds]


def screen(tracks, chrom_offsets, seed: int, round_begin: int, n_rounds: int):
    """The paper's co-localisation screen (Sec. 3.3: every pairwise comparison of K interval
    sets by the Monte Carlo simulation; Fig. 3 caption :224: score = log2(observed / median of the simulated
    counts)).  For every ORDERED pair (i, j), in row-major order: observed = |I(T_i, T_j)|; per round track i
    is re-placed (lengths kept, chromosome ends respected) and counted against the fixed track j; the draws of
    pair (i, j) come from Philox stream (fourth counter word) i * K + j, so every pair has its own null
    (reading R24).  `tracks` = [(start, end), ...].
    -> (observed uint64[K, K], round_counts uint64[K, K, n_rounds], enrichment float64[K, K])."""
    K = len(tracks)
    obs = np.zeros((K, K), dtype=np.uint64)
    rc = np.zeros((K, K, n_rounds), dtype=np.uint64)
    enr = np.full((K, K), np.nan, dtype=np.float64)
    for i in range(K):
        for j in range(K):
            o, r = mc_rounds(tracks[i][0], tracks[i][1], tracks[j][0], tracks[j][1], chrom_offsets, 0, seed,
                             round_begin, n_rounds, stream=i * K + j)
            obs[i, j], rc[i, j] = o, r
            enr[i, j] = enrichment(o, r)
    return obs, rc, enr


def enrichment(observed: int, round_counts) -> float:
    rc = np.ascontiguousarray(round_counts, dtype=np.uint64)
    return float(lib().oracle_enrichment(C.c_uint64(observed), rc.ctypes.data_as(_u64p), rc.size))


def pvalue(observed: int, round_counts, tail: int = 0) -> float:
    rc = np.ascontiguousarray(round_counts, dtype=np.uint64)
    return float(lib().oracle_pvalue(C.c_uint64(observed), rc.ctypes.data_as(_u64p), rc.size, tail))
