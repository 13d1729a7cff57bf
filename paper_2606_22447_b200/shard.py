"""Multi-GPU host logic: environments are independent, so a job over N GPUs is N
shards of whole ROM groups with NO collective on the data path.  The only cross-rank traffic is bookkeeping:
the max-over-ranks step time and the sum of emulated cycles that bench.py reports (one small all_reduce each)."""
from __future__ import annotations

import numpy as np


def shard_range(n_groups: int, world: int, rank: int) -> tuple[int, int]:
    """Contiguous [lo, hi) range of ROM groups (blocks of envs that share a cartridge) owned by `rank`; sizes differ by
    at most one group and every group is owned exactly once."""
    if world < 1 or not (0 <= rank < world) or n_groups < 0:
        raise ValueError("bad shard arguments")
    base, extra = divmod(n_groups, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def shard_envs(env_rom: np.ndarray, group: int, world: int, rank: int) -> np.ndarray:
    """Indices of the envs of a global batch that `rank` runs: whole groups of `group` consecutive envs (one ROM each)."""
    n = len(env_rom)
    if n % group:
        raise ValueError("batch is not a whole number of ROM groups")
    lo, hi = shard_range(n // group, world, rank)
    return np.arange(lo * group, hi * group, dtype=np.int64)


def rank_seeds(seeds: np.ndarray, rank: int) -> np.ndarray:
    """Weak scaling: every rank runs the same workload shape with its own env seeds."""
    return seeds ^ np.uint64(0x1000000 * rank)


def reduce_job(dist, total_ms: float, cycles: float, device=None) -> tuple[float, float]:
    """(max over ranks of the timed region in ms, sum over ranks of emulated cycles); identity when not distributed."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return total_ms, cycles
    import torch
    t = torch.tensor([total_ms], dtype=torch.float64, device=device)
    c = torch.tensor([cycles], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return float(t.item()), float(c.item())
