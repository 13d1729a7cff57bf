"""Seeded input generators: PRNG check values and the generated cartridges' frame
structure (G.1: every frame exactly 262 lines = 19,912 cycles, never a halt or a frame cap)."""
import ctypes as C

import numpy as np
import pytest

from oracle.ovcs_py import OracleVCS
from vcs_inputs import SplitMix64, draws, env_seeds, make_rom, make_workload, FEATURES
from vcs_inputs.configs import rom_seed


def test_splitmix64_check_values(oracle_lib):
    s = SplitMix64(0)
    assert [s.next() for _ in range(3)] == [0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4, 0x06C45D188009454F]
    s = SplitMix64(1)
    assert [s.next() for _ in range(2)] == [0x910A2DEC89025CC1, 0xBEEB8DA1658EEC67]
    # vectorised form and the oracle's own C implementation agree with the sequential one
    assert [int(v) for v in draws(np.zeros(3, np.uint64), np.arange(3))] == [0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4, 0x06C45D188009454F]
    st = C.c_uint64(1)
    assert oracle_lib.ovcs_splitmix64(C.byref(st)) == 0x910A2DEC89025CC1
    s = SplitMix64(0xA7A2600 + 2)
    assert [int(v) for v in env_seeds(2, 4)] == [s.next() for _ in range(4)]


def test_power_on_ram_is_the_env_seed_stream():
    w = make_workload(1)
    o = OracleVCS(w.roms, w.seeds)
    s = SplitMix64(int(w.seeds[0])); want = b"".join(s.next().to_bytes(8, "little") for _ in range(16))
    assert bytes(o.ram()[0]) == want
    r = o.regs()[0]
    assert (r["a"], r["x"], r["y"], r["sp"], r["p"], r["pc"], r["cycles"]) == (0, 0, 0, 0xFD, 0x24, 0xF000, 0)
    assert r["intim"] == 0xFF and r["timint"] == 0


@pytest.mark.parametrize("key", [1, 2, 3, "4a", "4b"])
def test_generated_roms_make_exact_262_line_frames(key):
    feat = FEATURES[key]
    for r in range(6):
        rom = make_rom(rom_seed(90 + (key if isinstance(key, int) else 4), r), feat)
        assert len(rom) == feat.size
        seeds = env_seeds(7, 3)
        o = OracleVCS([rom], seeds)
        rng = SplitMix64(r)
        o.step(np.zeros(3, np.uint8), 1)                       # short first frame (entry code)
        prev = o.regs()["cycles"].copy()
        banks = set()
        for t in range(6):
            o.step(np.array([rng.rnd(18) for _ in range(3)], np.uint8), 1)
            g = o.regs()
            assert (g["cycles"] - prev == 262 * 76).all(), (key, r, t)
            assert (g["status"] == 0).all() and (g["line"] == 0).all() and (g["cyc_in_line"] == 5).all()
            prev = g["cycles"].copy(); banks |= set(g["bank"].tolist())
        scr = o.screen()
        # VBLANK opens at the start of line 36 (row 2, store-free) and closes in line 229 (G.1 line accounting)
        assert (scr[:, :2] == 0).all() and (scr[:, 195:] == 0).all() and scr[:, 3:195].any()


def test_f8_roms_really_switch_banks():
    seen = set()
    for r in range(4):
        rom = make_rom(rom_seed(4, 200 + r), FEATURES["4b"])
        o = OracleVCS([rom], env_seeds(4, 8))
        for t in range(8):
            o.step(np.full(8, t % 18, np.uint8), 1); seen |= set(o.regs()["bank"].tolist())
    assert seen == {0, 1}


def test_workloads_and_action_streams():
    w2 = make_workload(2, batch=16)
    a = w2.actions(0, 50)
    assert a.shape == (50, 16) and a.max() <= 17 and len(np.unique(a)) == 18
    assert (w2.actions(10, 20) == a[10:20]).all()              # pure function of (seed, t)
    s = SplitMix64(int(w2.seeds[5]) ^ 0xAC7100000000); assert [s.next() % 18 for _ in range(50)] == a[:, 5].tolist()
    w3 = make_workload(3, batch=64)
    a3 = w3.actions(0, 400)
    rep = (a3[1:] == a3[:-1]).mean()
    assert 0.25 < rep < 0.35                                   # sticky: 0.25 + 0.75/18
    w4 = make_workload(4, batch=32, n_roms=4)
    assert [len(r) for r in w4.roms] == [4096, 4096, 8192, 8192] and w4.env_rom.tolist() == [i // 8 for i in range(32)]
    assert len(set(w4.roms)) == 4
