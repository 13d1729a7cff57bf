"""-m gpu: vcs_step_instructions — the paper's step unit, "one step = one CPU instruction" (Table 8:
3,000-instruction rollouts) — against the oracle's single-instruction stepping: RAM and every
vcs_regs field (cycle counter, beam, frame count, timer) after each call, for instruction counts from 1 to 3,000, on
the config-3 / config-4 generators, the TIA/RIOT chaos ROM, a halting ROM and small frame caps."""
import os

import numpy as np
import pytest

from vcs_inputs import make_workload, hand_rom, env_seeds, TIA_W

pytestmark = pytest.mark.gpu
NCPU = os.cpu_count() or 1


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


def same_cpu_state(g, o, tag):
    gr, orr = g.regs_host(), o.regs()
    for f in gr.dtype.names:
        bad = np.nonzero((gr[f] != orr[f]).reshape(len(orr), -1).any(axis=1))[0]
        assert bad.size == 0, f"{tag}: regs.{f} differs for envs {bad[:8]}: gpu {gr[f][bad[:4]]} oracle {orr[f][bad[:4]]}"
    bad = np.nonzero((g.ram_host() != o.ram()).any(axis=1))[0]
    assert bad.size == 0, f"{tag}: RAM differs for envs {bad[:8]}"


@pytest.mark.parametrize("cfg,kw", [(3, dict(batch=200)), (4, dict(batch=512, n_roms=4)), (2, dict(batch=33))])
def test_instruction_steps_match_the_oracle(torch, cfg, kw):
    from paper_2606_22447_b200 import VCS
    from oracle.ovcs_py import OracleVCS
    from test_gpu_parity import compare
    w = make_workload(cfg, **kw)
    g, o = VCS(w.roms, w.seeds, w.env_rom), OracleVCS(w.roms, w.seeds, w.env_rom)
    acts = w.actions(0, 12)
    scr0 = g.screen_host().copy()
    for t, n in enumerate([1, 1, 2, 7, 100, 3000, 333, 3000, 1]):
        g.step_instructions(torch.from_numpy(acts[t]).cuda(), n); o.step_instructions(acts[t], n, threads=NCPU)
        same_cpu_state(g, o, f"config{cfg} call {t} ({n} instructions)")
    assert (g.screen_host() == scr0).all()                       # the front screen belongs to vcs_step
    # back to frames: two frames on, the screen vcs_step shows lies wholly inside that call
    g.step(torch.from_numpy(acts[10]).cuda(), 2); o.step(acts[10], 2, threads=NCPU)
    compare(g, o, f"config{cfg} vcs_step after instruction steps")
    g.step_instructions(torch.from_numpy(acts[11]).cuda(), 500); o.step_instructions(acts[11], 500, threads=NCPU)
    same_cpu_state(g, o, f"config{cfg} instructions after vcs_step")


def test_instruction_steps_on_chaos_halt_and_cap(torch):
    from paper_2606_22447_b200 import VCS
    from oracle.ovcs_py import OracleVCS
    from test_gpu_parity import _chaos_rom

    def halting(a):
        a.org(0xF000); a.op("LDX", "imm", 5); a.label("l"); a.op("STA", "zp", TIA_W["WSYNC"]); a.op("DEX"); a.op("BNE", "rel", "l"); a.byte(0x02)
    for rom, kw in ((_chaos_rom(1004), dict(max_lines=40)), (_chaos_rom(1001), dict(max_lines=300, y0=20)), (hand_rom(halting), dict(max_lines=7))):
        seeds = env_seeds(5, 40)
        g, o = VCS([rom], seeds, **kw), OracleVCS([rom], seeds, **kw)
        for t, n in enumerate([3, 50, 1, 1, 1200, 2, 700]):
            a = np.array([(e + t) % 18 for e in range(40)], np.uint8)
            g.step_instructions(torch.from_numpy(a).cuda(), n); o.step_instructions(a, n, threads=NCPU)
            same_cpu_state(g, o, f"call {t} ({n} instructions) {kw}")


def test_instruction_step_argument_checks(torch):
    from paper_2606_22447_b200 import VCS, VcsError
    w = make_workload(2, batch=8)
    g = VCS(w.roms, w.seeds, w.env_rom)
    a = torch.zeros(8, dtype=torch.uint8, device="cuda")
    for n in (0, -1, 1000001):
        with pytest.raises(VcsError):
            g.step_instructions(a, n)
