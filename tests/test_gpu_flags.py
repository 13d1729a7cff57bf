"""-m gpu: vcs_config.flags (include/vcs.h VCS_F_*) change launch shape and decode, never results: every switch, alone
and combined, steps the same bytes as the default handle, and the default handle matches the oracle."""
import os

import numpy as np
import pytest

from vcs_inputs import make_workload

pytestmark = pytest.mark.gpu
NCPU = os.cpu_count() or 1


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


def _flags():
    from paper_2606_22447_b200 import binding as B
    return [("no_spin", B.VCS_F_NO_SPIN), ("no_fuse", B.VCS_F_NO_FUSE), ("no_regroup", B.VCS_F_NO_REGROUP),
            ("rom_global", B.VCS_F_ROM_GLOBAL), ("no_balance", B.VCS_F_NO_BALANCE), ("no_promote", B.VCS_F_NO_PROMOTE), ("block64", B.VCS_F_BLOCK_64),
            ("block128", B.VCS_F_BLOCK_128), ("block256", B.VCS_F_BLOCK_256),
            ("all_off+block64", B.VCS_F_NO_SPIN | B.VCS_F_NO_FUSE | B.VCS_F_NO_REGROUP | B.VCS_F_ROM_GLOBAL | B.VCS_F_NO_BALANCE | B.VCS_F_NO_PROMOTE | B.VCS_F_BLOCK_64),
            ("rom_global+block256", B.VCS_F_ROM_GLOBAL | B.VCS_F_BLOCK_256)]


def test_every_flag_steps_the_same_bytes(torch):
    from paper_2606_22447_b200 import VCS
    from oracle.ovcs_py import OracleVCS
    from test_gpu_parity import compare
    w = make_workload(4, batch=1024, n_roms=4)                      # 256 envs per ROM: 4K and F8 carts, regrouping blocks
    acts = w.actions(0, 8)
    dacts = torch.from_numpy(acts).cuda()
    ref = VCS(w.roms, w.seeds, w.env_rom)
    o = OracleVCS(w.roms, w.seeds, w.env_rom)
    others = [(name, VCS(w.roms, w.seeds, w.env_rom, flags=f)) for name, f in _flags()]
    for t in range(8):
        ref.step(dacts[t], 4)
        o.step(acts[t], 4, threads=NCPU)
        for name, g in others:
            g.step(dacts[t], 4)
    compare(ref, o, "default flags vs oracle")
    ram, regs, scr = ref.get_ram(), ref.get_regs(), ref.get_screen()
    for name, g in others:
        assert (g.get_ram() == ram).all() and (g.get_regs() == regs).all() and (g.get_screen() == scr).all(), name


def test_flags_on_timer_loops_and_unknown_flag(torch):
    from paper_2606_22447_b200 import VCS, binding as B
    w = make_workload(3, batch=200)
    dacts = torch.from_numpy(w.actions(0, 6)).cuda()
    ref = VCS(w.roms, w.seeds, w.env_rom)
    g = VCS(w.roms, w.seeds, w.env_rom, flags=B.VCS_F_NO_SPIN | B.VCS_F_NO_FUSE | B.VCS_F_BLOCK_64)
    for t in range(6):
        ref.step(dacts[t], 4); g.step(dacts[t], 4)
    assert (g.get_ram() == ref.get_ram()).all() and (g.get_regs() == ref.get_regs()).all() and (g.get_screen() == ref.get_screen()).all()
    with pytest.raises(B.VcsError):
        VCS(w.roms, w.seeds, w.env_rom, flags=1 << 20)
