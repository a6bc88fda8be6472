"""Front end (host side, off the hot path): BED files -> the library's coordinates.

PAPER.md:111 (Sec. 2.1): the intervals of every chromosome are projected onto one linear coordinate space
("a one-dimensional genome") so that one pair of sorted arrays serves the whole genome; the
Monte Carlo rounds draw starts "from 1 to total genome size".  The library takes 0-based CLOSED intervals
already projected (reading R3): chromosome c occupies [off[c], off[c+1] - 1].

BED is 0-based half-open: a line `chrom  start  end` is the closed interval [start, end - 1] on `chrom`,
i.e. [off[c] + start, off[c] + end - 1] after projection.  Nothing here touches the GPU.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

__all__ = ["Genome", "read_genome", "read_bed", "FrontEndError"]


class FrontEndError(ValueError):
    pass


@dataclass
class Genome:
    names: list            # chromosome names in table order
    lengths: np.ndarray    # uint64[C]
    offsets: np.ndarray    # uint32[C + 1], offsets[0] = 0, offsets[C] = G <= 2^32 - 1

    def index(self) -> dict:
        return {n: i for i, n in enumerate(self.names)}


def read_genome(path: str) -> Genome:
    """A 'genome file': one `name <whitespace> length` line per chromosome, in the order of the projection."""
    names, lengths = [], []
    with open(path) as f:
        for ln, line in enumerate(f, 1):
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            parts = line.split()
            if len(parts) < 2 or not parts[1].isdigit() or int(parts[1]) <= 0:
                raise FrontEndError(f"{path}:{ln}: expected 'name length' with a positive length")
            if parts[0] in names:
                raise FrontEndError(f"{path}:{ln}: chromosome {parts[0]!r} listed twice")
            names.append(parts[0])
            lengths.append(int(parts[1]))
    if not names:
        raise FrontEndError(f"{path}: no chromosomes")
    off = np.zeros(len(names) + 1, dtype=np.uint64)
    off[1:] = np.cumsum(np.asarray(lengths, dtype=np.uint64))
    if int(off[-1]) > 2**32 - 1:
        raise FrontEndError(f"{path}: the genome ({int(off[-1])} bp) does not fit the uint32 coordinate space")
    return Genome(names, np.asarray(lengths, dtype=np.uint64), off.astype(np.uint32))


def read_bed(path: str, genome: Genome, skip_unknown: bool = False):
    """(start, end) uint32 arrays of the projected closed intervals of a BED file, in file order.

    Lines starting with '#', 'track' or 'browser' and empty lines are skipped.  A chromosome that is not in
    the genome file is an error unless skip_unknown.  start < end <= chromosome length is required (an empty
    BED interval has no closed counterpart)."""
    idx = genome.index()
    off = genome.offsets.astype(np.int64)
    starts, ends = [], []
    with open(path) as f:
        for ln, line in enumerate(f, 1):
            if not line.strip() or line.startswith(("#", "track", "browser")):
                continue
            parts = line.split()
            if len(parts) < 3:
                raise FrontEndError(f"{path}:{ln}: a BED line needs chrom, start, end")
            c = idx.get(parts[0])
            if c is None:
                if skip_unknown:
                    continue
                raise FrontEndError(f"{path}:{ln}: chromosome {parts[0]!r} is not in the genome file")
            try:
                s, e = int(parts[1]), int(parts[2])
            except ValueError:
                raise FrontEndError(f"{path}:{ln}: start and end must be integers") from None
            if not (0 <= s < e <= int(genome.lengths[c])):
                raise FrontEndError(f"{path}:{ln}: need 0 <= start < end <= {int(genome.lengths[c])} on {parts[0]}")
            starts.append(off[c] + s)          # half-open [s, e) on the chromosome ...
            ends.append(off[c] + e - 1)        # ... is the closed [off + s, off + e - 1] on the projected genome
    return np.asarray(starts, dtype=np.uint32), np.asarray(ends, dtype=np.uint32)
