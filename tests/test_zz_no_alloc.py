"""-m gpu: vcs_step_host_noalloc — the host-buffer step that allocates nothing (its device-side staging is a static array
of the library; include/vcs.h) — against the existing path vcs_step_host + vcs_get_ram_host + vcs_get_regs_host.

This file is named to be collected LAST (the suite runs with pytest -x): it must pass alone in a fresh process and after
every other GPU test, whatever they left in the shared scratch array.  Tolerance: bit-exact, as every parity test here."""
import numpy as np
import pytest

from vcs_inputs import make_workload

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


def existing_path(g, actions, frameskip):
    """step + read-back through the entry points that were there before"""
    g.step_host(actions, frameskip)
    regs = g.regs_host()
    return g.ram_host(), regs, int((regs["status"] != 0).sum())


def same(tag, got, want):
    ram, regs, flagged = got
    wram, wregs, wflagged = want
    assert (ram == wram).all(), f"{tag}: RAM differs for envs {np.nonzero((ram != wram).any(axis=1))[0][:8]}"
    for f in wregs.dtype.names:
        assert (regs[f] == wregs[f]).all(), f"{tag}: regs.{f} differs"
    assert int(flagged[0]) == wflagged, f"{tag}: {int(flagged[0])} envs flagged, existing path says {wflagged}"


def test_two_calls_in_a_row_equal_the_existing_path(torch):
    from paper_2606_22447_b200 import VCS
    w = make_workload(4, batch=1200, n_roms=4)                 # 4K and F8 carts, a ragged last block
    a, b = VCS(w.roms, w.seeds, w.env_rom, max_lines=150), VCS(w.roms, w.seeds, w.env_rom, max_lines=150)
    acts = w.actions(0, 4)                                     # (150-line cap: every env hits it, so the flag counter is not trivially 0)
    flagged = []
    for t in range(4):                                         # two calls in a row, and two more
        got = a.step_host_noalloc(acts[t], 2 + t % 2)
        want = existing_path(b, acts[t], 2 + t % 2)
        same(f"call {t}", got, want)
        flagged.append(int(got[2][0]))
    assert flagged[0] > 0 and all(f <= w.batch for f in flagged) and sum(flagged) > w.batch    # cleared per call, not accumulated across calls
    torch.cuda.synchronize(); free0 = torch.cuda.mem_get_info()[0]      # once warm, further calls leave the device's free memory alone
    for t in range(3):
        a.step_host_noalloc(acts[t], 1)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    a.close(); b.close()


def test_a_smaller_batch_after_a_larger_one_and_another_handle(torch):
    """the array keeps the last call's contents: a later, smaller call (another handle, another ROM set) must not see them"""
    from paper_2606_22447_b200 import VCS
    big = make_workload(3, batch=4096)
    g = VCS(big.roms, big.seeds, big.env_rom); g.step_host_noalloc(big.actions(0, 1)[0], 1); g.close()
    w = make_workload(2, batch=37)
    a, b = VCS(w.roms, w.seeds, w.env_rom), VCS(w.roms, w.seeds, w.env_rom)
    acts = w.actions(0, 2)
    for t in range(2):
        same(f"small call {t}", a.step_host_noalloc(acts[t], 4), existing_path(b, acts[t], 4))
    assert int(a.step_host_noalloc(acts[0], 1)[2][0]) == 0     # no cap, no illegal opcode: nothing flagged, and nothing left over
    a.close(); b.close()


def test_async_form_with_caller_buffers(torch):
    """the C call only enqueues: caller-owned pinned buffers, one synchronise for two calls on the same stream"""
    from paper_2606_22447_b200 import VCS
    from paper_2606_22447_b200.binding import REGS_DTYPE
    w = make_workload(2, batch=300)
    a, b = VCS(w.roms, w.seeds, w.env_rom), VCS(w.roms, w.seeds, w.env_rom)
    acts = w.actions(0, 2)
    pin = [torch.empty(300 * 128 + 300 * 32 + 4 + 300, dtype=torch.uint8).pin_memory() for _ in range(2)]
    views = []
    for t in range(2):
        buf = pin[t].numpy()
        ram = buf[:300 * 128].reshape(300, 128); regs = buf[300 * 128:300 * 160].view(REGS_DTYPE)
        flagged = buf[300 * 160:300 * 160 + 4].view(np.int32); act = buf[300 * 160 + 4:]
        act[:] = acts[t]
        a.step_host_noalloc(act, 3, ram_out=ram, regs_out=regs, flagged_out=flagged, sync=False)
        views.append((ram, regs, flagged))
    torch.cuda.current_stream().synchronize()
    for t in range(2):
        same(f"async call {t}", views[t], existing_path(b, acts[t], 3))
    a.close(); b.close()


def test_rejects_a_batch_beyond_the_scratch_array(torch):
    from paper_2606_22447_b200 import VCS
    from paper_2606_22447_b200.binding import NOALLOC_MAX_BATCH, VcsError
    w = make_workload(2, batch=NOALLOC_MAX_BATCH + 256)
    g = VCS(w.roms, w.seeds, w.env_rom)
    with pytest.raises(VcsError, match="exceeds VCS_NOALLOC_MAX_BATCH"):
        g.step_host_noalloc(np.zeros(w.batch, np.uint8), 1)
    g.close()
    w = make_workload(2, batch=NOALLOC_MAX_BATCH)              # the maximum itself is served
    a, b = VCS(w.roms, w.seeds, w.env_rom), VCS(w.roms, w.seeds, w.env_rom)
    act = w.actions(0, 1)[0]
    same("max batch", a.step_host_noalloc(act, 1), existing_path(b, act, 1))
    a.close(); b.close()
