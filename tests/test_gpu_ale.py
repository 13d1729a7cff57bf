"""CUDA path vs oracle for the ALE-style wrapper pieces (Table 8):
vcs_set_switches, vcs_step_masked, vcs_boot — bit-exact RAM, regs and screens through the C ABI."""
import os

import numpy as np
import pytest

from helpers import switch_rom
from test_gpu_parity import compare, mk, torch  # noqa: F401
from vcs_inputs import make_workload, SplitMix64

pytestmark = pytest.mark.gpu
NCPU = os.cpu_count() or 1


def pair(roms, seeds, env_rom=None, **kw):
    from paper_2606_22447_b200 import VCS
    from oracle.ovcs_py import OracleVCS
    return VCS(roms, seeds, env_rom, **kw), OracleVCS(roms, seeds, env_rom, **kw)


def dev(torch, x):
    return torch.from_numpy(np.ascontiguousarray(x, dtype=np.uint8)).cuda()


def test_switches(torch):
    n = 70                                                       # one block and a ragged tail
    g, o = pair([switch_rom()], np.arange(1, n + 1, dtype=np.uint64))
    r = SplitMix64(5)
    for t in range(6):
        sw = np.array([r.rnd(256) for _ in range(n)], np.uint8)
        if t == 3:
            g.set_switches(None); o.set_switches(None)
        else:
            g.set_switches(dev(torch, sw)); o.set_switches(sw)
        if t == 4:
            g.reset(); o.reset()                                 # switches are physical: a reset leaves them
        a = np.array([r.rnd(18) for _ in range(n)], np.uint8)
        g.step(dev(torch, a), 1 + t % 3); o.step(a, 1 + t % 3)
        compare(g, o, f"switches step {t}")
    assert (g.ram_host()[:, 2] == (sw | 0x34)).all()


@pytest.mark.parametrize("cfg,batch,n_roms", [(2, 200, None), (4, 256, 32), (4, 96, 6)])
def test_masked_step(torch, cfg, batch, n_roms):
    w = make_workload(cfg, batch=batch, n_roms=n_roms)           # config 4: F8 blocks regroup with frozen envs among them
    g, o = mk(torch, w)
    acts = w.actions(0, 8)
    r = SplitMix64(11 + batch)
    for t in range(8):
        mask = np.array([r.rnd(3) > 0 for _ in range(batch)], np.uint8)
        if t == 5: mask[:] = 0
        if t == 6: mask[: batch // 2] = 0
        g.step_masked(dev(torch, acts[t]), w.frameskip, dev(torch, mask))
        o.step_masked(acts[t], w.frameskip, mask, threads=NCPU)
        compare(g, o, f"masked cfg{cfg} step {t}")
    g.step_masked(dev(torch, acts[0]), 2, None); o.step_masked(acts[0], 2, None, threads=NCPU)
    compare(g, o, "masked NULL mask")


def test_boot_switch_rom(torch):
    n = 130
    g, o = pair([switch_rom()], np.arange(100, 100 + n, dtype=np.uint64))
    starts = (np.arange(n) * 7 % 34).astype(np.uint8)            # 0..33: some above the cap of 30
    g.boot(None, 60, 4, dev(torch, starts), 30, 4); o.boot(None, 60, 4, starts, 30, 4)
    compare(g, o, "boot")
    k = np.minimum(starts, 30).astype(np.int64)
    assert (g.regs_host()["frame"] == 64 + 4 * k).all() and (g.ram_host()[:, 1] == 4).all()


def test_boot_subset_mid_episode(torch):
    w = make_workload(4, batch=128, n_roms=4)
    g, o = mk(torch, w)
    acts = w.actions(0, 6)
    r = SplitMix64(77)
    for t in range(6):
        g.step(dev(torch, acts[t]), 4); o.step(acts[t], 4, threads=NCPU)
        if t in (1, 4):                                          # "auto-reset" of a few envs: boot them, the rest stay put
            mask = np.array([r.rnd(5) == 0 for _ in range(128)], np.uint8)
            starts = np.array([r.rnd(5) for _ in range(128)], np.uint8)
            g.boot(dev(torch, mask), 5, 2, dev(torch, starts), 4, 4); o.boot(mask, 5, 2, starts, 4, 4)
        compare(g, o, f"boot subset step {t}")
    g.boot(None, 3, 1, None, 30, 4); o.boot(None, 3, 1, None, 30, 4)      # no NOOP starts
    compare(g, o, "boot all")


def test_boot_argument_errors(torch):
    g, _ = pair([switch_rom()], np.arange(4, dtype=np.uint64))
    for kw in (dict(noop_frames=-1), dict(reset_frames=-1), dict(max_noop_starts=256), dict(frameskip=0)):
        with pytest.raises(RuntimeError):
            g.boot(**kw)


def test_ale_vec_env_auto_reset(torch):
    from paper_2606_22447_b200 import AleVecEnv
    from oracle.ovcs_py import OracleVCS
    n = 96
    w = make_workload(4, batch=n, n_roms=6)
    env = AleVecEnv(w.roms, w.seeds, w.env_rom, frameskip=4, noop_max=5, boot_noop_frames=6, boot_reset_frames=2,
                    max_episode_steps=4, start_seed=3, amortised=False)
    o = OracleVCS(w.roms, w.seeds, w.env_rom)
    starts = env.reset().cpu().numpy()
    assert starts.max() <= 5 and len(set(starts.tolist())) > 1
    o.boot(None, 6, 2, starts, 5, 4)
    compare(env.vcs, o, "ale reset")
    acts = w.actions(0, 10)
    r = SplitMix64(9)
    n_boot = np.ones(n, np.int64)
    for t in range(10):
        done = np.array([r.rnd(7) == 0 for _ in range(n)], np.uint8)
        steps_before = env.episode_steps.cpu().numpy()
        mask = env.step(dev(torch, acts[t]), dev(torch, done)).cpu().numpy()
        assert (mask.astype(bool) == (done.astype(bool) | (steps_before + 1 >= 4))).all()
        o.step(acts[t], 4, threads=NCPU)
        if mask.any():
            o.boot(mask, 6, 2, env.last_starts.cpu().numpy(), 5, 4)
        n_boot += mask
        compare(env.vcs, o, f"ale step {t}")
    assert (env.episodes.cpu().numpy() == n_boot).all()
    env.close()


def test_masked_and_boot_full_batch_launch_shape(torch):
    """Config 4 at its full batch (bench.py's launch configuration: 256-env blocks, spare warp, F8 regroup with frozen
    envs among the files): masked steps and a mid-episode boot of a subset, one env per ROM against the oracle."""
    from paper_2606_22447_b200 import VCS
    from oracle.ovcs_py import OracleVCS
    w = make_workload(4)
    idx = np.arange(256) * 256 + (np.arange(256) * 91) % 256
    g = VCS(w.roms, w.seeds, w.env_rom)
    o = OracleVCS(w.roms, w.seeds[idx], w.env_rom[idx])
    acts = w.actions(0, 6)
    rng = np.random.default_rng(5)
    for t in range(6):
        mask = (rng.integers(0, 4, w.batch) > 0).astype(np.uint8)
        g.step_masked(dev(torch, acts[t]), 4, dev(torch, mask)); o.step_masked(acts[t][idx], 4, mask[idx], threads=NCPU)
        compare(g, o, f"full masked step {t}", envs=idx)
        if t == 2:
            bm = (rng.integers(0, 3, w.batch) == 0).astype(np.uint8)
            st = rng.integers(0, 4, w.batch).astype(np.uint8)
            g.boot(dev(torch, bm), 4, 2, dev(torch, st), 3, 4); o.boot(bm[idx], 4, 2, st[idx], 3, 4)
            compare(g, o, "full boot", envs=idx)


@pytest.mark.parametrize("batch,n_roms", [(96, 6), (256, 2)])
def test_auto_reset_amortised_equals_boot_protocol(torch, batch, n_roms):
    """vcs_auto_reset arms envs whose boot then runs inside the batch's ordinary vcs_step calls; the result must be
    what the paper's protocol gives when spelled frame by frame (ovcs_boot: 60 single NOOP frames, 4 single RESET
    frames, k NOOP steps) followed by the agent's actions from the step at which each env became ready."""
    w = make_workload(4, batch=batch, n_roms=n_roms)
    g, o = mk(torch, w)
    acts = w.actions(0, 60)
    r = np.random.default_rng(batch)
    for t in range(3):                                           # some history first
        g.step(dev(torch, acts[t]), 4); o.step(acts[t], 4, threads=NCPU)
    mask = (r.integers(0, 3, batch) == 0).astype(np.uint8); mask[0] = 1
    starts = r.integers(0, 36, batch).astype(np.uint8)           # some above the cap of 30
    g.auto_reset(dev(torch, mask), 15, 1, dev(torch, starts), 30)
    o.boot(mask, 60, 4, starts, 30, 4)                           # the oracle boots "instantly" ...
    k = np.minimum(starts, 30).astype(np.int64)
    want = np.where(mask != 0, 16 + k, 0)
    assert (g.get_booting().cpu().numpy() == want).all()
    T = 16 + 30 + 4
    for t in range(T):                                           # ... and then waits until the GPU env is ready
        ready = (t >= want).astype(np.uint8)
        g.step(dev(torch, acts[3 + t]), 4); o.step_masked(acts[3 + t], 4, ready, threads=NCPU)
        assert (g.get_booting().cpu().numpy() == np.maximum(want - (t + 1), 0)).all()
    compare(g, o, "auto_reset")
    # a second arming while the first envs play on, with a masked step in between (frozen envs do not count down)
    m2 = (r.integers(0, 4, batch) == 0).astype(np.uint8)
    g.auto_reset(dev(torch, m2), 2, 1, None, 0); o.boot(m2, 8, 4, None, 0, 4)
    frozen = (r.integers(0, 2, batch) == 0).astype(np.uint8)
    g.step_masked(dev(torch, acts[0]), 4, dev(torch, frozen))
    left = np.where(m2 != 0, 3, 0) - np.where((m2 != 0) & (frozen != 0), 1, 0)
    assert (g.get_booting().cpu().numpy() == left).all()
    o.step_masked(acts[0], 4, frozen & (m2 == 0), threads=NCPU)
    for t in range(1, 5):
        a_t = acts[t]
        g.step(dev(torch, a_t), 4)
        o.step_masked(a_t, 4, (left == 0).astype(np.uint8), threads=NCPU)
        left = np.maximum(left - 1, 0)
    compare(g, o, "auto_reset second arming")
    with pytest.raises(RuntimeError):
        g.auto_reset(None, 200, 50, None, 30)


def test_ale_vec_env_amortised_auto_reset(torch):
    from paper_2606_22447_b200 import AleVecEnv
    from oracle.ovcs_py import OracleVCS
    n = 64
    w = make_workload(4, batch=n, n_roms=4)
    env = AleVecEnv(w.roms, w.seeds, w.env_rom, frameskip=4, noop_max=3, boot_noop_frames=8, boot_reset_frames=4, start_seed=1)
    assert env.amortised
    o = OracleVCS(w.roms, w.seeds, w.env_rom)
    st = env.reset().cpu().numpy(); o.boot(None, 8, 4, st, 3, 4)
    acts = w.actions(0, 14)
    r = SplitMix64(21)
    wait = np.zeros(n, np.int64)                                  # boot steps each env still owes
    for t in range(14):
        done = np.array([r.rnd(9) == 0 for _ in range(n)], np.uint8)
        play = (wait == 0).astype(np.uint8)
        m = env.step(dev(torch, acts[t]), dev(torch, done)).cpu().numpy()
        o.step_masked(acts[t], 4, play, threads=NCPU)                          # the oracle env waits while the GPU env runs its boot steps
        wait = np.maximum(wait - 1, 0)
        assert (m == (done & play)).all()                        # a `done` for an env that is still booting is ignored
        if m.any():
            k = np.minimum(env.last_starts.cpu().numpy(), 3)
            o.boot(m, 8, 4, k.astype(np.uint8), 3, 4)
            wait = np.where(m != 0, 3 + k, wait)
        assert (env.booting().cpu().numpy() == wait).all()
    for t in range(8):                                           # let every boot finish
        play = (wait == 0).astype(np.uint8)
        env.step(dev(torch, acts[t]))
        o.step_masked(acts[t], 4, play, threads=NCPU)
        wait = np.maximum(wait - 1, 0)
    compare(env.vcs, o, "amortised AleVecEnv")
    env.close()


def test_ale_vec_env_truncates_at_the_same_agent_step_in_both_modes(torch):
    """max_episode_steps counts AGENT steps: the boot steps an amortised re-boot spends inside the batch's steps do not
    count, so both modes end every episode after the same number of steps in which the env followed the agent."""
    from paper_2606_22447_b200 import AleVecEnv
    n = 48
    w = make_workload(2, batch=n)
    acts = w.actions(0, 40)
    played = {}
    for amortised in (False, True):
        env = AleVecEnv(w.roms, w.seeds, w.env_rom, frameskip=4, noop_max=2, boot_noop_frames=8, boot_reset_frames=4,
                        max_episode_steps=5, start_seed=3, amortised=amortised)
        env.reset()
        agent_steps = np.zeros(n, np.int64); lengths = [[] for _ in range(n)]
        for t in range(40):
            play = (env.booting().cpu().numpy() == 0) if amortised else np.ones(n, bool)
            m = env.step(dev(torch, acts[t])).cpu().numpy()
            agent_steps += play
            for e in np.nonzero(m)[0]:
                lengths[e].append(int(agent_steps[e])); agent_steps[e] = 0
        played[amortised] = lengths
        env.close()
    for e in range(n):
        assert played[False][e] and all(v == 5 for v in played[False][e]), (e, played[False][e])
        assert played[True][e] and all(v == 5 for v in played[True][e]), (e, played[True][e])
