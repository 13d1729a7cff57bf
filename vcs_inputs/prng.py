"""splitmix64 — the only PRNG behind seeds, ROM bytes and action streams.

This package (`vcs_inputs`) is the seeded synthetic-input generator shared by the oracle tests
and the CUDA path's tests/bench.  It holds none of the emulator's arithmetic: it only produces
ROM images, env seeds and action streams.
"""
from __future__ import annotations

import numpy as np

MASK = (1 << 64) - 1
GAMMA = 0x9E3779B97F4A7C15


def _mix_int(z: int) -> int:
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & MASK
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & MASK
    return z ^ (z >> 31)


class SplitMix64:
    """Sequential stream: next() advances the state by GAMMA and mixes it."""

    def __init__(self, seed: int):
        self.s = seed & MASK

    def next(self) -> int:
        self.s = (self.s + GAMMA) & MASK
        return _mix_int(self.s)

    def rnd(self, k: int) -> int:
        return self.next() % k

    def choice(self, seq):
        return seq[self.rnd(len(seq))]

    def chance(self, num: int, den: int) -> bool:
        return self.rnd(den) < num


def draws(seeds: np.ndarray, index: np.ndarray | int) -> np.ndarray:
    """Vectorised: the `index`-th draw (0-based) of the streams seeded `seeds` (uint64 arrays).

    splitmix64 is counter based: draw i of seed s is mix(s + (i+1)*GAMMA)."""
    seeds = np.asarray(seeds, dtype=np.uint64)
    idx = np.asarray(index, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = seeds + (idx + np.uint64(1)) * np.uint64(GAMMA)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        return z ^ (z >> np.uint64(31))


def env_seeds(config_index: int, batch: int) -> np.ndarray:
    """seed[e] = e-th draw of the stream seeded 0xA7A2600 + config_index (G.0)."""
    base = np.full(batch, 0xA7A2600 + config_index, dtype=np.uint64)
    return draws(base, np.arange(batch, dtype=np.uint64))
