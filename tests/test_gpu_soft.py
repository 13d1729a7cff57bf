"""-m gpu: SOFT-STE forward mode (vcs_step_soft; BASELINE config 5) against the oracle's soft
mode and against hard mode.  PAPER.md Theorem 1/3 (L140, L320): the soft forward state equals the hard one bit for
bit, tolerance 0, at any finite alpha and T; the soft values themselves (relaxed reads, branch gates) are compared
as per-env sums with the oracle's (float32 on the GPU, float64 in the oracle: relative 2e-4)."""
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


def same_state(a, b, tag):
    ra, rb = a.regs_host(), (b.regs_host() if hasattr(b, "regs_host") else b.regs())
    for f in ra.dtype.names:
        assert (ra[f] == rb[f]).all(), f"{tag}: regs.{f} differs"
    assert (a.ram_host() == (b.ram_host() if hasattr(b, "ram_host") else b.ram())).all(), f"{tag}: RAM differs"
    assert (a.screen_host() == (b.screen_host() if hasattr(b, "screen_host") else b.screen())).all(), f"{tag}: screen differs"


@pytest.mark.parametrize("cfg,kw", [(3, dict(batch=24)), (4, dict(batch=256, n_roms=2))])   # config 4 with 128 envs per ROM: staged ROM, F8 regroup
@pytest.mark.parametrize("T,alpha", [(0.1, 2.0), (1.0, 6.0), (10.0, 20.0)])
def test_soft_three_way(torch, cfg, kw, T, alpha):
    from paper_2606_22447_b200 import VCS
    from oracle.ovcs_py import OracleVCS
    w = make_workload(cfg, **kw)
    idx = np.arange(0, w.batch, max(1, w.batch // 12))                       # oracle soft mode is slow: a strided sample
    g, gs = VCS(w.roms, w.seeds, w.env_rom), VCS(w.roms, w.seeds, w.env_rom)
    o = OracleVCS(w.roms, w.seeds[idx], w.env_rom[idx])
    acts = w.actions(0, 3)
    for t in range(3):
        a = torch.from_numpy(acts[t]).cuda()
        g.step(a, 4)
        so = gs.step_soft(a, 4, T, alpha).cpu().numpy().astype(np.float64)
        oo = o.step_soft(acts[t][idx], 4, T, alpha, threads=NCPU)
        same_state(gs, g, f"cfg{cfg} T={T} step {t} soft vs hard")
        assert (gs.ram_host()[idx] == o.ram()).all() and (gs.screen_host()[idx] == o.screen()).all()
        assert (so[:, 6] == 0).all() and (oo[:, 6] == 0).all()               # no rounded STE value ever differed from hard
        assert (so[idx, 3:6] == oo[:, 3:6]).all()                            # the same reads and branches went through the soft path
        assert np.allclose(so[idx, 0:3], oo[:, 0:3], rtol=2e-4, atol=0)      # and produced the same soft values
        assert np.allclose(so[idx, 7], oo[:, 7], rtol=1e-4, atol=2e-4)       # |soft - hard| of float32 values up to 255: a few ulp(255) = 3e-5 each


def test_config5_soft_forward_equals_hard(torch):
    """BASELINE config 5: batch 4096 on config 2's ROM, 200 steps of frameskip 4 at T in {0.1, 1, 10}; forward
    RAM / regs / screen of soft mode == hard mode, every env, tolerance 0 (checked every 20 steps and at the end), and
    == the oracle's hard mode on a 64-env sample at the same checkpoints."""
    from paper_2606_22447_b200 import VCS
    from oracle.ovcs_py import OracleVCS
    w = make_workload(2, batch=4096)
    steps = 200
    acts_host = w.actions(0, steps)
    acts = torch.from_numpy(acts_host).cuda()
    g = VCS(w.roms, w.seeds, w.env_rom)
    softs = {T: VCS(w.roms, w.seeds, w.env_rom) for T in (0.1, 1.0, 10.0)}
    idx = np.arange(64) * 64 + (np.arange(64) * 7) % 64
    o = OracleVCS(w.roms, w.seeds[idx], w.env_rom[idx])
    out = torch.empty((4096, 8), dtype=torch.float32, device="cuda")
    bad = torch.zeros((), dtype=torch.float32, device="cuda")
    for t in range(steps):
        g.step(acts[t], 4)
        o.step(acts_host[t][idx], 4, threads=NCPU)
        for T, gs in softs.items():
            gs.step_soft(acts[t], 4, T, 6.0, out=out)
            bad += out[:, 6].sum()
        if t % 20 == 19 or t == steps - 1:
            oregs = o.regs()
            for T, gs in softs.items():
                same_state(gs, g, f"config5 T={T} step {t}")
                assert (gs.ram_host()[idx] == o.ram()).all() and (gs.screen_host()[idx] == o.screen()).all(), f"T={T} step {t} vs oracle"
                assert all((gs.regs_host()[idx][f] == oregs[f]).all() for f in oregs.dtype.names), f"T={T} step {t} regs vs oracle"
    assert float(bad.item()) == 0.0


def test_soft_at_other_launch_shapes(torch):
    """The soft kernel always runs 128 envs per block in env order, whatever shape and block placement the handle's
    hard steps use: a 32,768-env handle (256-env blocks) and a handle with 64-env blocks whose placement has been
    re-computed by a few plain steps must both step soft == hard, every env."""
    from paper_2606_22447_b200 import VCS
    from paper_2606_22447_b200.binding import VCS_F_BLOCK_64
    from oracle.ovcs_py import OracleVCS
    w = make_workload(2, batch=32768)
    acts_host = w.actions(0, 4); acts = torch.from_numpy(acts_host).cuda()
    g, gs = VCS(w.roms, w.seeds, w.env_rom), VCS(w.roms, w.seeds, w.env_rom)
    idx = np.arange(32) * 1024 + (np.arange(32) * 37) % 1024
    o = OracleVCS(w.roms, w.seeds[idx], w.env_rom[idx])
    for t in range(4):
        g.step(acts[t], 4); o.step(acts_host[t][idx], 4, threads=NCPU)
        if t < 2: gs.step(acts[t], 4)
        else: gs.step_soft(acts[t], 4, 1.0, 6.0)
    same_state(gs, g, "soft at batch 32768")
    assert (gs.ram_host()[idx] == o.ram()).all() and (gs.screen_host()[idx] == o.screen()).all()
    g.close(); gs.close()
    w = make_workload(4, batch=512, n_roms=8)                                # 64 envs per ROM
    acts = torch.from_numpy(w.actions(0, 8)).cuda()
    g, gs = VCS(w.roms, w.seeds, w.env_rom, flags=VCS_F_BLOCK_64), VCS(w.roms, w.seeds, w.env_rom, flags=VCS_F_BLOCK_64)
    for t in range(8):
        g.step(acts[t], 4)
        if t < 6: gs.step(acts[t], 4)                                         # plain steps 2.. re-place the blocks
        else: gs.step_soft(acts[t], 4, 10.0, 2.0)
    _, perm = gs.block_times()
    assert sorted(perm.tolist()) == list(range(8))
    same_state(gs, g, "soft after a re-placement with 64-env blocks")


def test_soft_argument_checks(torch):
    from paper_2606_22447_b200 import VCS, VcsError
    w = make_workload(2, batch=8)
    g = VCS(w.roms, w.seeds, w.env_rom)
    a = torch.zeros(8, dtype=torch.uint8, device="cuda")
    for T, alpha in ((0.0, 6.0), (-1.0, 6.0), (61.0, 6.0), (1.0, float("nan"))):
        with pytest.raises(VcsError):
            g.step_soft(a, 4, T, alpha)
    with pytest.raises(VcsError):
        g.step_soft(a, 0, 1.0, 6.0)
