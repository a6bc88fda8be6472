"""Round sharding for multi-GPU Monte Carlo jobs (host logic only, no arithmetic of the method).

Rounds are independent and addressed by (seed, round) (include/bits.h, bits_mc_rounds), so a job of
`total_rounds` rounds shards over `world` ranks by contiguous round slices with A and B replicated
and no data-path collective; the only exchange is the gather of the per-round counts at the end.
"""
from __future__ import annotations


def round_slice(rank: int, world: int, total_rounds: int, round_begin: int = 0) -> tuple[int, int]:
    """(first round, number of rounds) of `rank`: contiguous, balanced to within one round."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    base, extra = divmod(total_rounds, world)
    n = base + (1 if rank < extra else 0)
    first = round_begin + rank * base + min(rank, extra)
    return first, n


def weak_slice(rank: int, rounds_per_rank: int, round_begin: int = 0) -> tuple[int, int]:
    """Weak scaling (bench.py --gpus N): every rank runs its own `rounds_per_rank` rounds."""
    return round_begin + rank * rounds_per_rank, rounds_per_rank
