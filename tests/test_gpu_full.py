"""-m gpu: vcs_step_instructions_soft — the soft modes in the paper's step unit — against the oracle.
  * FULL mode (appendix D, Table 3; reading R18): the casts decide what the machine reads and where it branches,
    so the CUDA path must take every cast as the oracle does — inside the exact corner (alpha >= 6, T <= 0.14), on the
    two boundaries where the trajectory leaves the hard one, and far outside, where the consoles run whatever the
    pulled bytes decode to (illegal opcodes, code in RAM, wild branches): RAM and every register after each call.
  * SOFT-STE per instruction: state == vcs_step_instructions == oracle, soft sums against the oracle's.
T and alpha go to both sides as the float32 values the C ABI takes."""
import os

import numpy as np
import pytest

from test_gpu_instructions import same_cpu_state, torch  # noqa: F401
from vcs_inputs import make_workload

pytestmark = pytest.mark.gpu
NCPU = os.cpu_count() or 1
CALLS = [1, 1, 2, 5, 40, 300, 1000, 1651]                     # 3,000 instructions from reset, as Table 3 runs them


def f32(x):
    return float(np.float32(x))


def pair(cfg, **kw):
    from paper_2606_22447_b200 import VCS
    from oracle.ovcs_py import OracleVCS
    w = make_workload(cfg, **kw)
    return w, VCS(w.roms, w.seeds, w.env_rom), OracleVCS(w.roms, w.seeds, w.env_rom)


@pytest.mark.parametrize("alpha,T", [(6.0, 0.14), (6.0, 0.08), (5.0, 0.14), (3.0, 0.14), (2.0, 0.05), (6.0, 0.15), (6.0, 0.2), (4.0, 1.0), (1.0, 10.0)])
@pytest.mark.parametrize("cfg,kw", [(3, dict(batch=160)), (4, dict(batch=256, n_roms=4))])
def test_full_mode_takes_the_oracles_casts(torch, cfg, kw, alpha, T):
    w, g, o = pair(cfg, **kw)
    alpha, T = f32(alpha), f32(T)
    acts = w.actions(0, len(CALLS))
    casts_off = 0
    for t, n in enumerate(CALLS):
        so = g.step_instructions_soft(torch.from_numpy(acts[t]).cuda(), n, T, alpha, True).cpu().numpy()
        oo = o.step_instructions_soft(acts[t], n, T, alpha, True, threads=NCPU)
        same_cpu_state(g, o, f"FULL alpha={alpha} T={T} config{cfg} call {t} ({n} instructions)")
        assert (so[:, 3:7] == oo[:, 3:7]).all(), f"call {t}: read / branch / failed-cast counts differ"
        assert np.allclose(so[:, 0:3], oo[:, 0:3], rtol=2e-4, atol=1e-3) and np.allclose(so[:, 7], oo[:, 7], rtol=1e-4, atol=1e-4)
        casts_off += int(oo[:, 6].sum())
    if alpha >= 6.0 and T <= f32(0.14):
        assert casts_off == 0                                 # the corner: exact on every program (L459)
        from oracle.ovcs_py import OracleVCS
        h = OracleVCS(w.roms, w.seeds, w.env_rom)
        for t, n in enumerate(CALLS): h.step_instructions(acts[t], n, threads=NCPU)
        same_cpu_state(g, h, "FULL in the corner == HARD")
    if alpha <= 3.0 or T >= f32(0.2):
        assert casts_off > 0                                  # outside it the casts do fail (and both sides fail alike)
    g.close(); o.close()


def test_full_mode_on_an_f8_handle_and_after_frames(torch):
    """a FULL rollout that starts from a state reached by ordinary frame steps, on bank-switching carts"""
    w, g, o = pair(4, batch=300, n_roms=2)
    acts = w.actions(0, 6)
    for t in range(2):
        g.step(torch.from_numpy(acts[t]).cuda(), 3); o.step(acts[t], 3, threads=NCPU)
    for t, (n, alpha, T) in enumerate([(700, 6.0, 0.14), (900, 3.0, 0.12), (500, 6.0, 0.17)]):
        alpha, T = f32(alpha), f32(T)
        g.step_instructions_soft(torch.from_numpy(acts[2 + t]).cuda(), n, T, alpha, True)
        o.step_instructions_soft(acts[2 + t], n, T, alpha, True, threads=NCPU)
        same_cpu_state(g, o, f"FULL after frames, call {t}")
    g.step(torch.from_numpy(acts[5]).cuda(), 2); o.step(acts[5], 2, threads=NCPU)              # and back to hard frames
    same_cpu_state(g, o, "hard frames after FULL")
    assert (g.screen_host() == o.screen()).all()
    g.close(); o.close()


@pytest.mark.parametrize("T", [0.1, 1.0, 10.0])
def test_soft_ste_per_instruction(torch, T):
    from oracle.ovcs_py import OracleVCS
    w, g, o = pair(3, batch=130)
    h = OracleVCS(w.roms, w.seeds, w.env_rom)
    T, alpha = f32(T), f32(4.0)
    acts = w.actions(0, 5)
    for t, n in enumerate([1, 3, 250, 3000, 77]):
        so = g.step_instructions_soft(torch.from_numpy(acts[t]).cuda(), n, T, alpha, False).cpu().numpy()
        oo = o.step_instructions_soft(acts[t], n, T, alpha, False, threads=NCPU); h.step_instructions(acts[t], n, threads=NCPU)
        same_cpu_state(g, h, f"SOFT-STE T={T} call {t}: state == hard")
        assert (so[:, 3:7] == oo[:, 3:7]).all() and (so[:, 6] == 0).all()
        assert np.allclose(so[:, 0:3], oo[:, 0:3], rtol=2e-4, atol=1e-3)
    g.close(); o.close(); h.close()


def test_arguments(torch):
    from paper_2606_22447_b200 import VCS
    from vcs_inputs import superchip_rom, env_seeds
    w = make_workload(2, batch=8)
    g = VCS(w.roms, w.seeds, w.env_rom)
    a = torch.zeros(8, dtype=torch.uint8, device="cuda")
    for bad in (dict(n=0, T=0.1, alpha=6.0), dict(n=5, T=0.0, alpha=6.0), dict(n=5, T=0.1, alpha=float("nan")), dict(n=2000000, T=0.1, alpha=1.0)):
        with pytest.raises(RuntimeError):
            g.step_instructions_soft(a, bad["n"], bad["T"], bad["alpha"], True)
    g.close()
    g = VCS([superchip_rom("F8SC", 3)], env_seeds(1, 8), mappers=["F8SC"])
    with pytest.raises(RuntimeError):
        g.step_instructions_soft(a, 10, 0.1, 6.0, True)
    g.close()
