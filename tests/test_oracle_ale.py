"""Oracle pins for the ALE-style wrapper pieces (Table 8): console
switches on SWCHB, the masked step, the boot protocol.  Expected values follow from the test program's text
(tests/helpers.switch_rom) and the protocol's frame counts, not from the oracle."""
import numpy as np

from helpers import switch_rom
from oracle.ovcs_py import OracleVCS

SEEDS = np.arange(1, 7, dtype=np.uint64)


def mk(n=6):
    return OracleVCS([switch_rom()], SEEDS[:n])


def test_switch_pins_read_through_swchb():
    o = mk()
    sw = np.array([0x3F, 0x3E, 0x37, 0xBF, 0x7D, 0x00], np.uint8)          # released / RESET / b&w / P1 A / P0 A + SELECT / all low
    o.set_switches(sw)
    for _ in range(3):
        o.step(np.zeros(6, np.uint8), 1)
    ram = o.ram()
    want = sw | 0x34                                                        # pins 2, 4, 5 are not connected: read 1
    assert (ram[:, 2] == want).all()
    assert (ram[:, 0] == 2).all()                                           # $80 == frames - 1
    assert (ram[:, 1] == 2 * ((want & 1) == 0)).all()                       # RESET seen low in both sampled frames
    p = ram[:, 6]
    assert (((p >> 7) & 1) == (want >> 7)).all() and (((p >> 6) & 1) == ((want >> 6) & 1)).all()   # BIT: N = bit 7, V = bit 6
    scr = o.screen()
    for e in range(6):
        assert (scr[e][:150] == (0x4A if want[e] & 8 else 0x0E)).all()         # the program draws ~204 lines: rows below stay 0
    o.set_switches(None)
    o.step(np.zeros(6, np.uint8), 1)
    assert (o.ram()[:, 2] == 0x3F).all()


def test_switches_survive_reset_and_ddr_outputs_win():
    o = mk(2)
    o.set_switches(np.array([0x37, 0x3F], np.uint8))
    o.reset()
    o.step(np.zeros(2, np.uint8), 2)
    assert o.ram()[:, 2].tolist() == [0x37, 0x3F]


def test_masked_step_freezes_the_rest():
    a, b = mk(), mk()
    acts = np.array([0, 1, 2, 3, 4, 5], np.uint8)
    mask = np.array([1, 0, 1, 1, 0, 1], np.uint8)
    a.step(acts, 2); b.step(acts, 2)
    r0, ram0, s0 = b.regs().copy(), b.ram().copy(), b.screen().copy()
    a.step(acts, 3); b.step_masked(acts, 3, mask)
    on = mask.astype(bool)
    assert (a.ram()[on] == b.ram()[on]).all() and (a.regs()[on] == b.regs()[on]).all() and (a.screen()[on] == b.screen()[on]).all()
    assert (b.ram()[~on] == ram0[~on]).all() and (b.regs()[~on] == r0[~on]).all() and (b.screen()[~on] == s0[~on]).all()


def test_boot_protocol_counts():
    o = mk()
    o.step(np.full(6, 3, np.uint8), 5)                                      # some history the boot must wipe
    starts = np.array([0, 1, 7, 30, 31, 200], np.uint8)
    o.boot(None, 60, 4, starts, 30, 4)
    k = np.minimum(starts, 30).astype(np.int64)
    r, ram = o.regs(), o.ram()
    assert (r["frame"] == 64 + 4 * k).all()
    assert (ram[:, 0] == (63 + 4 * k) & 0xFF).all()                         # $80 == frames - 1
    assert (ram[:, 1] == 4).all()                                           # RESET read low in exactly the 4 RESET frames
    assert (ram[:, 2] == np.where(k > 0, 0x3F, 0x3E)).all()                 # the last sample: released again once a NOOP step ran
    assert (ram[:, 5] == 0xFF).all()                                        # NOOP: no joystick direction pressed


def test_boot_mask_leaves_others_alone_and_equals_manual_sequence():
    o, m = mk(), mk()
    acts = np.array([2, 3, 4, 5, 6, 7], np.uint8)
    o.step(acts, 3); m.step(acts, 3)
    mask = np.array([0, 1, 0, 0, 1, 0], np.uint8)
    starts = np.array([9, 2, 9, 9, 0, 9], np.uint8)
    keep = (o.ram().copy(), o.regs().copy(), o.screen().copy())
    o.boot(mask, 6, 2, starts, 30, 2)
    off = ~mask.astype(bool)
    assert (o.ram()[off] == keep[0][off]).all() and (o.regs()[off] == keep[1][off]).all() and (o.screen()[off] == keep[2][off]).all()
    # the same thing spelled with the primitives
    z = np.zeros(6, np.uint8)
    m.reset(mask)
    for _ in range(6): m.step_masked(z, 1, mask)
    m.set_switches(np.full(6, 0x3E, np.uint8))
    for _ in range(2): m.step_masked(z, 1, mask)
    m.set_switches(None)
    for k in range(2): m.step_masked(z, 2, mask & (starts > k))
    assert (o.ram() == m.ram()).all() and (o.regs() == m.regs()).all() and (o.screen() == m.screen()).all()


def test_boot_frames_equal_boot_steps_when_inputs_change_every_fourth_frame():
    """60 single NOOP frames + 4 single RESET frames + k NOOP steps (the protocol as ovcs_boot spells it) == 15 + 1 + k
    env-steps of frameskip 4 with the same inputs: inputs are latched per step and only change at those frame counts.
    This is the identity the amortised vcs_auto_reset rests on."""
    import vcs_inputs
    w = vcs_inputs.make_workload(4, batch=8, n_roms=4)
    a = OracleVCS(w.roms, w.seeds, w.env_rom); b = OracleVCS(w.roms, w.seeds, w.env_rom)
    starts = np.array([0, 1, 2, 3, 5, 8, 13, 30], np.uint8)
    a.boot(None, 60, 4, starts, 30, 4)
    z = np.zeros(8, np.uint8)
    b.reset()
    for t in range(16 + 30):
        b.set_switches(np.full(8, 0x3E if t == 15 else 0x3F, np.uint8))
        b.step_masked(z, 4, (t < 16 + starts.astype(np.int64)).astype(np.uint8))
    assert (a.ram() == b.ram()).all() and (a.regs() == b.regs()).all() and (a.screen() == b.screen()).all()
