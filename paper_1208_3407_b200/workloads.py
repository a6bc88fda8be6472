"""Seeded synthetic interval sets shaped like the paper's workloads.

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA
path (``paper_1208_3407_b200.bits``): it produces inputs and nothing else.  It
holds none of the method's arithmetic (no intersection counting, no Philox
placement, no sorting of B_S/B_E) and imports neither side.

The paper measured on 1000 Genomes NA12878 alignments, RefSeq exons and
ENCODE/UCSC tracks (PAPER.md:137-139 §3.1, :151 Fig. 2, :167 §3.3) at 1e5..1e7
intervals per set (Table 1).  None of those datasets is
available; the five configurations of BASELINE.json stand in for them with the
same set sizes, read-like fixed lengths vs feature-like lognormal lengths, and
uniform vs clustered ("exome-like") placement.  The exact
recipe is stated in DESIGN.md §"Input recipe".

Coordinates are 0-based CLOSED intervals [start, end] already projected to the
1-D genome (§2.1): chromosome c occupies [off[c], off[c+1]-1].
Arrays are delivered in generation order (unsorted), as uint32.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

__all__ = [
    "GENOME24_LENGTHS", "genome_offsets", "Workload", "make_config", "CONFIG_NAMES",
    "array_checksum",
]

# 24 chromosomes, lengths linearly spaced 249,000,000 .. 48,000,000 bp (BASELINE.json configs[1]).
GENOME24_LENGTHS = tuple(249_000_000 - (c * 201_000_000) // 23 for c in range(24))

CONFIG_NAMES = {
    1: "cfg1_tiny",
    2: "cfg2_genome_count_1M",
    3: "cfg3_mc_permuteA_1e4x1M",
    4: "cfg4_large_count_10M",
    5: "cfg5_mc_permuteB_sort_1Mx10M",
}


def genome_offsets(lengths) -> np.ndarray:
    """Cumulative chromosome offsets off[0..C], off[0]=0, off[C]=G (uint32)."""
    off = np.zeros(len(lengths) + 1, dtype=np.uint64)
    off[1:] = np.cumsum(np.asarray(lengths, dtype=np.uint64))
    assert int(off[-1]) <= 2**32 - 1, "genome does not fit the uint32 coordinate space"
    return off.astype(np.uint32)


def array_checksum(x: np.ndarray) -> int:
    """Order-sensitive 64-bit checksum of a uint32 array (for golden-file input identity)."""
    v = np.ascontiguousarray(x, dtype=np.uint32).astype(np.uint64)
    idx = np.arange(1, v.size + 1, dtype=np.uint64)
    with np.errstate(over="ignore"):
        h = (v + np.uint64(0x9E3779B97F4A7C15)) * (idx * np.uint64(0xBF58476D1CE4E5B9) | np.uint64(1))
        h ^= h >> np.uint64(29)
        return int(np.bitwise_xor.reduce(h) ^ np.uint64(v.size)) if v.size else 0


@dataclass
class Workload:
    name: str
    a_start: np.ndarray
    a_end: np.ndarray
    b_start: np.ndarray
    b_end: np.ndarray
    chrom_offsets: np.ndarray            # uint32[C+1]
    which: int | None = None             # 0 = permute A, 1 = permute B, None = counting only
    n_rounds: int = 0
    mc_seed: int = 1
    spec: dict = field(default_factory=dict)

    @property
    def n_a(self) -> int:
        return int(self.a_start.size)

    @property
    def n_b(self) -> int:
        return int(self.b_start.size)

    def checksums(self) -> dict:
        return {k: array_checksum(getattr(self, k)) for k in ("a_start", "a_end", "b_start", "b_end")}


def _rng(seed: int, stream: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[np.uint64(seed), np.uint64(stream)]))


def _lognormal_lengths(rng, n, median, sigma, lo=20, hi=100_000) -> np.ndarray:
    z = rng.standard_normal(n)
    ell = np.rint(median * np.exp(sigma * z))
    return np.clip(ell, lo, hi).astype(np.int64)


def _chrom_of(pos: np.ndarray, off: np.ndarray) -> np.ndarray:
    return np.searchsorted(off, pos, side="right") - 1


def _place_uniform(rng, lengths: np.ndarray, off_u32: np.ndarray):
    """Global position uniform in [0,G) picks chromosome and start together
    (length-weighted); redraw if the interval crosses the chromosome end."""
    off = off_u32.astype(np.int64)
    G = int(off[-1])
    n = lengths.size
    start = np.empty(n, dtype=np.int64)
    todo = np.arange(n)
    while todo.size:
        pos = rng.integers(0, G, size=todo.size, dtype=np.int64)
        c = _chrom_of(pos, off)
        ok = pos + lengths[todo] - 1 <= off[c + 1] - 1
        start[todo[ok]] = pos[ok]
        todo = todo[~ok]
    return start, start + lengths - 1


def _place_clustered(rng, lengths: np.ndarray, off_u32: np.ndarray, n_clusters: int, sd: float):
    """K centres uniform in [0,G); pick a centre uniformly, midpoint = centre +
    round(sd*z); redraw if the interval leaves the centre's chromosome."""
    off = off_u32.astype(np.int64)
    G = int(off[-1])
    centres = rng.integers(0, G, size=n_clusters, dtype=np.int64)
    cchrom = _chrom_of(centres, off)
    n = lengths.size
    start = np.empty(n, dtype=np.int64)
    todo = np.arange(n)
    while todo.size:
        pick = rng.integers(0, n_clusters, size=todo.size)
        mid = centres[pick] + np.rint(sd * rng.standard_normal(todo.size)).astype(np.int64)
        ell = lengths[todo]
        s = mid - ell // 2
        e = s + ell - 1
        c = cchrom[pick]
        ok = (s >= off[c]) & (e <= off[c + 1] - 1)
        start[todo[ok]] = s[ok]
        todo = todo[~ok]
    return start, start + lengths - 1


def _u32(*arrs):
    out = []
    for a in arrs:
        assert a.min(initial=0) >= 0 and a.max(initial=0) <= 2**32 - 1
        out.append(np.ascontiguousarray(a.astype(np.uint32)))
    return out


def make_config(k: int, scale: float = 1.0, seed: int | None = None) -> Workload:
    """Build configuration k (1..5) of BASELINE.json.

    ``scale`` multiplies the set sizes (and cluster counts) only; shapes, genome,
    length and placement distributions stay as in the full configuration.  Data
    seed defaults to k (streams 0 = A, 1 = B); the Monte Carlo seed is 1.
    """
    if seed is None:
        seed = k
    ra, rb = _rng(seed, 0), _rng(seed, 1)
    sz = lambda n: max(1, int(round(n * scale)))
    if k == 1:
        off = genome_offsets([1_000_000])
        na, nb = sz(1_000), sz(1_000)
        la = ra.integers(50, 501, size=na, dtype=np.int64)
        lb = rb.integers(50, 501, size=nb, dtype=np.int64)
        sa = ra.integers(0, 1_000_000 - la + 1, dtype=np.int64)
        sb = rb.integers(0, 1_000_000 - lb + 1, dtype=np.int64)
        a_s, a_e, b_s, b_e = _u32(sa, sa + la - 1, sb, sb + lb - 1)
        return Workload(CONFIG_NAMES[1], a_s, a_e, b_s, b_e, off, which=0, n_rounds=100,
                        spec=dict(config=1, scale=scale, seed=seed))
    off = genome_offsets(GENOME24_LENGTHS)
    if k == 2:
        na, nb = sz(1_000_000), sz(1_000_000)
        la = _lognormal_lengths(ra, na, 1000, 1.0)
        lb = _lognormal_lengths(rb, nb, 1000, 1.0)
        sa, ea = _place_uniform(ra, la, off)
        sb, eb = _place_uniform(rb, lb, off)
        which, rounds = None, 0
    elif k == 3:
        na, nb = sz(10_000), sz(1_000_000)
        la = _lognormal_lengths(ra, na, 500, 0.8)
        lb = _lognormal_lengths(rb, nb, 2000, 1.2)
        sa, ea = _place_uniform(ra, la, off)
        sb, eb = _place_clustered(rb, lb, off, sz(5_000), 200_000.0)
        which, rounds = 0, 10_000
    elif k == 4:
        na, nb = sz(10_000_000), sz(10_000_000)
        la = np.full(na, 100, dtype=np.int64)
        lb = _lognormal_lengths(rb, nb, 2000, 1.2)
        sa, ea = _place_uniform(ra, la, off)
        nu = nb // 2
        sbu, ebu = _place_uniform(rb, lb[:nu], off)
        sbc, ebc = _place_clustered(rb, lb[nu:], off, sz(20_000), 100_000.0)
        sb, eb = np.concatenate([sbu, sbc]), np.concatenate([ebu, ebc])
        perm = rb.permutation(nb)            # interleave the uniform and clustered halves
        sb, eb = sb[perm], eb[perm]
        which, rounds = None, 0
    elif k == 5:
        na, nb = sz(1_000_000), sz(10_000_000)
        la = _lognormal_lengths(ra, na, 1000, 1.0)
        lb = _lognormal_lengths(rb, nb, 300, 0.7)
        sa, ea = _place_uniform(ra, la, off)
        sb, eb = _place_uniform(rb, lb, off)
        which, rounds = 1, 1_000
    else:
        raise ValueError(f"unknown config {k}")
    a_s, a_e, b_s, b_e = _u32(sa, ea, sb, eb)
    return Workload(CONFIG_NAMES[k], a_s, a_e, b_s, b_e, off, which=which, n_rounds=rounds,
                    spec=dict(config=k, scale=scale, seed=seed))
