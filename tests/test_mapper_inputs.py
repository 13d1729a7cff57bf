"""The Superchip / E0 / FE test cartridges (vcs_inputs/mapper_roms.py) on the oracle: they run, stay alive, and really
use what is particular to their format; and the two independent format guesses (oracle/ and the library's
vcs_detect_mapper, a host call) agree on every generated cartridge."""
import numpy as np
import pytest

from oracle.ovcs_py import OracleVCS, detect_mapper as oracle_detect
from vcs_inputs import superchip_rom, e0_rom, fe_rom, make_workload, env_seeds, SplitMix64
from vcs_inputs.romgen import FEATURES, make_rom

CARTS = [("F8SC", lambda: superchip_rom("F8SC", 11)), ("F6SC", lambda: superchip_rom("F6SC", 12)), ("F4SC", lambda: superchip_rom("F4SC", 13)),
         ("E0", lambda: e0_rom(14)), ("FE", lambda: fe_rom(15))]


def _run(kind, rom, n=24, steps=6):
    o = OracleVCS([rom], env_seeds(3, n), mappers=[kind], max_lines=200)
    r = SplitMix64(9)
    seen = set()
    for t in range(steps):
        o.step(np.array([r.rnd(18) for _ in range(n)], np.uint8), 1 + t % 2, threads=4)
        regs = o.regs()
        seen |= set(zip(regs["bank"].tolist(), regs["pad"][:, 0].tolist()))
    return o, seen


@pytest.mark.parametrize("kind,make", CARTS, ids=[k for k, _ in CARTS])
def test_cart_runs_and_uses_its_format(kind, make):
    o, seen = _run(kind, make())
    regs, ram = o.regs(), o.ram()
    assert (regs["status"] == 0).all() and (regs["frame"] >= 8).all()               # nobody halted, no frame cap
    if kind.endswith("SC"):
        assert len({b for b, _ in seen}) > 1                                        # banks were switched
        assert len({bytes(x) for x in o.cart_ram()}) > 1 and (ram[:, 0x05] > 0).all()   # cart RAM differs per env; the stub in cart RAM ran (INC $85)
        assert (ram[:, 0x40:0x50] != 0).any()                                       # the seeded cart RAM was copied out at start
    if kind == "E0":
        assert len(seen) > 4 and (ram[:, 0x07] > 0).all()                           # many window combinations
        assert ((ram[:, 0x04] & 0x0F) == 5).all() and ((ram[:, 0x05] & 0x0F) == 5).all()     # the subroutines behind the windows ran
    if kind == "FE":
        assert {b for b, _ in seen} == {0, 1} or len(set(ram[:, 0x06].tolist())) > 1          # both pages reached at run time
        assert set(ram[:, 0x04].tolist()) <= {0x41 + 0x09, 0x40 + 0x08, 0x41 + 0x08, 0x40 + 0x09} and (ram[:, 0x07] > 0).all()


def test_both_format_guesses_agree():
    from paper_2606_22447_b200.binding import detect_mapper as lib_detect
    carts = [(k, m()) for k, m in CARTS]
    carts += [("2K", make_rom(1, FEATURES[1])), ("4K", make_rom(2, FEATURES[3])), ("F8", make_rom(3, FEATURES["4b"])),
              ("F6", make_rom(4, FEATURES["f6"])), ("F4", make_rom(5, FEATURES["f4"]))]
    carts += [("", r) for r in make_workload(4, batch=2048, n_roms=8).roms]
    for want, rom in carts:
        a, b = oracle_detect(rom), lib_detect(rom)
        assert a == b and (want == "" or a == want), (want, a, b)
    r = SplitMix64(5)
    for size in (8192, 8192, 8192, 16384, 32768):                                  # random bytes: whatever the answer, the same one
        img = bytes(r.rnd(256) for _ in range(size))
        assert oracle_detect(img) == lib_detect(img)
    assert lib_detect(bytes(3000)) == "" and oracle_detect(bytes(3000)) == ""
