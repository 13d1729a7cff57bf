"""The five BASELINE.json configs as concrete seeded inputs.

Everything here is input generation: ROM images, env->ROM map, env seeds, action streams."""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

from . import prng
from .romgen import FEATURES, make_rom


@dataclass
class Workload:
    index: int
    batch: int
    roms: list[bytes]
    env_rom: np.ndarray            # int32 [batch]
    seeds: np.ndarray              # uint64 [batch]
    frameskip: int
    steps: int
    action_kind: str               # "noop" | "uniform" | "sticky"
    name: str = ""
    _act_seeds: np.ndarray = field(default=None, repr=False)

    def actions(self, t0: int, t1: int) -> np.ndarray:
        """uint8 [t1-t0][batch] actions for steps t0..t1-1 (pure function of the seeds)."""
        n = t1 - t0
        if self.action_kind == "noop":
            return np.zeros((n, self.batch), dtype=np.uint8)
        s = self._act_seeds
        if self.action_kind == "uniform":
            t = np.arange(t0, t1, dtype=np.uint64)[:, None]
            return (prng.draws(s[None, :], t) % np.uint64(18)).astype(np.uint8)
        # sticky: two draws per step; repeat the previous action when draw1 % 4 == 0 and t > 0
        out = np.zeros((t1, self.batch), dtype=np.uint8)
        prev = np.zeros(self.batch, dtype=np.uint8)
        for t in range(t1):
            d1 = prng.draws(s, np.uint64(2 * t))
            d2 = prng.draws(s, np.uint64(2 * t + 1))
            fresh = (d2 % np.uint64(18)).astype(np.uint8)
            rep = ((d1 % np.uint64(4)) == 0) & (t > 0)
            prev = np.where(rep, prev, fresh)
            out[t] = prev
        return out[t0:t1]


def rom_seed(config_index: int, r: int) -> int:
    return int(prng.draws(np.array([0x520D0000 + config_index], dtype=np.uint64), r)[0])


def make_workload(index: int, batch: int | None = None, n_roms: int | None = None) -> Workload:
    """index in 1..4.  `batch`/`n_roms` override the config's size (tests use smaller batches of the
    same recipe; bench uses the full size)."""
    full = {1: 1, 2: 1024, 3: 16384, 4: 65536}[index]
    batch = full if batch is None else batch
    seeds = prng.env_seeds(index, batch)
    act_seeds = seeds ^ np.uint64(0xAC7100000000)
    if index == 1:
        roms = [make_rom(rom_seed(1, 0), FEATURES[1])]
        env_rom = np.zeros(batch, dtype=np.int32)
        return Workload(1, batch, roms, env_rom, seeds, 1, 10, "noop", "config1", act_seeds)
    if index == 2:
        roms = [make_rom(rom_seed(2, 0), FEATURES[2])]
        return Workload(2, batch, roms, np.zeros(batch, dtype=np.int32), seeds, 4, 500, "uniform", "config2", act_seeds)
    if index == 3:
        roms = [make_rom(rom_seed(3, 0), FEATURES[3])]
        return Workload(3, batch, roms, np.zeros(batch, dtype=np.int32), seeds, 4, 2000, "sticky", "config3", act_seeds)
    if index == 4:
        n_roms = 256 if n_roms is None else n_roms
        assert batch % n_roms == 0
        per = batch // n_roms
        roms = [make_rom(rom_seed(4, r), FEATURES["4a"] if r < n_roms // 2 else FEATURES["4b"]) for r in range(n_roms)]
        env_rom = (np.arange(batch, dtype=np.int32) // per).astype(np.int32)
        return Workload(4, batch, roms, env_rom, seeds, 4, 1000, "uniform", "config4", act_seeds)
    raise ValueError(index)
