"""Seeded selection of chunk subsets — the only thing shared by the product's bench/tests and the
oracle-side tests.  Holds none of the method's arithmetic (SplitMix64 is a generic generator)."""
from __future__ import annotations

SEED = 150700315
_M64 = (1 << 64) - 1


class SplitMix64:
    def __init__(self, seed: int = SEED):
        self.s = seed & _M64

    def next(self) -> int:
        self.s = (self.s + 0x9E3779B97F4A7C15) & _M64
        z = self.s
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _M64
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _M64
        return z ^ (z >> 31)


def sample_chunks(chunk_bits: int, count: int, seed: int = SEED, salt: int = 0):
    """`count` distinct chunk indices in [0, 2^chunk_bits), seeded, always including the first and
    the last chunk (the all-(+1) and all-(-1) prefixes) when count >= 2."""
    total = 1 << chunk_bits
    count = min(count, total)
    rng = SplitMix64(seed ^ (salt * 0x9E3779B97F4A7C15 & _M64))
    picked = []
    if count >= 2:
        picked = [0, total - 1]
    while len(picked) < count:
        c = rng.next() % total
        if c not in picked:
            picked.append(c)
    return sorted(picked)


def sample_range_starts(chunk_bits: int, runs: int, run_len: int, seed: int = SEED):
    """`runs` seeded, non-overlapping, run_len-aligned runs of contiguous chunks (BASELINE config 5:
    "a fixed seeded 1/64 subset of chunks")."""
    slots = (1 << chunk_bits) // run_len
    runs = min(runs, slots)
    rng = SplitMix64(seed + 1)
    picked = set()
    while len(picked) < runs:
        picked.add(rng.next() % slots)
    return [s * run_len for s in sorted(picked)]
