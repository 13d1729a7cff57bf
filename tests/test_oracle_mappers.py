"""Oracle pins for the F6 / F4 mappers: every bank holds the same code and
its own marker bytes, so what the program stores says which bank answered each access."""
import numpy as np
import pytest

from helpers import regs, run_instr
from oracle.ovcs_py import OracleVCS
from vcs_inputs import hand_rom


def banked_image(build, nb):
    code = hand_rom(build)
    banks = []
    for b in range(nb):
        img = bytearray([b]) * 4096
        img[:0x100] = code[:0x100]; img[0xFFC:] = code[0xFFC:]
        img[0x800] = 0xA0 + b                                       # marker read through $F800
        for k in range(0xFF0, 0xFFC): img[k] = 0x50 + b             # what a read of a hotspot address returns
        banks.append(img)
    return bytes(b"".join(banks))


@pytest.mark.parametrize("nb,lo", [(4, 0xFFF6), (8, 0xFFF4)])
def test_every_hotspot_selects_its_bank(nb, lo):
    def build(a):
        a.org(0xF000)
        for k in range(nb):
            a.op("LDA", "abs", lo + k); a.op("STA", "zp", 0x80 + k)           # the read itself already sees bank k
            a.op("LDA", "abs", 0xF800); a.op("STA", "zp", 0x90 + k)
        a.label("end"); a.op("JMP", "abs", "end")
    o = OracleVCS([banked_image(build, nb)], np.array([3], dtype=np.uint64))
    assert regs(o)["bank"] == 0                                     # F6 / F4 power up in bank 0 (reading R15)
    for k in range(nb):
        run_instr(o, 4)
        assert regs(o)["bank"] == k
    ram = o.ram()[0]
    assert ram[0:nb].tolist() == [0x50 + k for k in range(nb)]
    assert ram[0x10:0x10 + nb].tolist() == [0xA0 + k for k in range(nb)]


@pytest.mark.parametrize("nb,lo", [(4, 0xFFF6), (8, 0xFFF4)])
def test_writes_dummy_reads_and_neighbours(nb, lo):
    def build(a):
        a.org(0xF000)
        a.op("STA", "abs", lo + nb - 1); a.op("LDA", "abs", 0xF800); a.op("STA", "zp", 0x80)     # a write selects too
        a.op("LDA", "abs", lo - 1); a.op("LDA", "abs", 0xF800); a.op("STA", "zp", 0x81)          # one below the range: no switch
        a.op("LDA", "abs", lo + nb); a.op("LDA", "abs", 0xF800); a.op("STA", "zp", 0x82)         # one above: no switch
        a.op("LDX", "imm", 0xFF); a.op("LDA", "abx", lo + 1 - 0xFF)                             # no page cross: only $lo+1 is read
        a.op("LDA", "abs", 0xF800); a.op("STA", "zp", 0x83)
        a.op("LDX", "imm", 0xFF); a.op("LDA", "abx", lo + 2 - 0x100 - 0xFF + 0x100)             # same page again -> bank 2
        a.op("LDA", "abs", 0xF800); a.op("STA", "zp", 0x84)
        a.op("LDY", "imm", 0x10); a.op("LDA", "aby", lo - 0x10)                                 # $FFEx + $10 = lo: bank 0
        a.op("LDA", "abs", 0xF800); a.op("STA", "zp", 0x85)
        a.label("end"); a.op("JMP", "abs", "end")
    o = OracleVCS([banked_image(build, nb)], np.array([3], dtype=np.uint64))
    run_instr(o, 22)
    ram = o.ram()[0]
    assert ram[0] == 0xA0 + nb - 1 and ram[1] == 0xA0 + nb - 1 and ram[2] == 0xA0 + nb - 1
    assert ram[3] == 0xA1 and ram[4] == 0xA2 and ram[5] == 0xA0


def test_sizes_accepted_and_rejected():
    for size in (16384, 32768):
        OracleVCS([bytes(size)], np.array([1], dtype=np.uint64)).close()
    with pytest.raises(RuntimeError):
        OracleVCS([bytes(12288)], np.array([1], dtype=np.uint64))
