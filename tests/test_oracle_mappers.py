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


# ---------------------------------------------------------------------------------------------- Superchip, E0, FE, detection
# (PAPER.md L69 / L469: F8SC, F6SC, F4SC, E0, FE are among the ports' formats; L197: Superchip RAM must
# be seeded.)  Expectations are hand-derived from the board descriptions restated in oracle/ovcs.h.
from oracle.ovcs_py import detect_mapper
from vcs_inputs import SplitMix64


def _sc_image(nb):
    def build(a):
        a.org(0xF100)                                               # (the first 256 bytes of a bank are the RAM ports)
        a.op("LDA", "abs", 0xF085); a.op("STA", "zp", 0x80)           # read port: power-on content of cell 5
        a.op("LDA", "imm", 0x5A); a.op("STA", "abs", 0xF005)          # write port
        a.op("LDA", "abs", 0xF085); a.op("STA", "zp", 0x81)           # -> $5A
        a.op("LDA", "abs", 0xF005); a.op("STA", "zp", 0x82)           # a read of the write port: the cell, unchanged [R]
        a.op("LDA", "abs", 0xF085); a.op("STA", "zp", 0x83)
        a.op("LDX", "imm", 0x7F); a.op("LDA", "imm", 0xC3); a.op("STA", "abx", 0xF000); a.op("LDA", "abx", 0xF080); a.op("STA", "zp", 0x84)   # last cell, indexed
        a.op("LDA", "abs", 0xF100); a.op("STA", "zp", 0x85)           # just above the ports: ROM again
        a.op("LDA", "abs", 0xFFFA - nb + 1); a.op("LDA", "abs", 0xF085); a.op("STA", "zp", 0x86)     # another bank (hotspot of bank 1): the same RAM
        a.op("LDA", "abs", 0xF800); a.op("STA", "zp", 0x87)
        a.label("end"); a.op("JMP", "abs", "end")
    code = hand_rom(build, entry=0xF100)
    banks = []
    for b in range(nb):
        img = bytearray([0xEE]) * 4096                               # Superchip images carry a filler where the ports sit
        img[0x100:0x200] = code[0x100:0x200]; img[0xFFC:] = code[0xFFC:]; img[0x800] = 0xA0 + b
        banks.append(img)
    return bytes(b"".join(banks))


@pytest.mark.parametrize("kind,nb", [("F8SC", 2), ("F6SC", 4), ("F4SC", 8)])
def test_superchip_ports_seed_and_banks(kind, nb):
    img = _sc_image(nb)
    hot0 = {2: 0xFFF8, 4: 0xFFF6, 8: 0xFFF4}[nb]
    img = img.replace(bytes([0xAD, (0xFFFA - nb + 1) & 0xFF, 0xFF]), bytes([0xAD, (hot0 + 1) & 0xFF, 0xFF]))    # LDA hotspot of bank 1
    o = OracleVCS([img], np.array([77], dtype=np.uint64), mappers=[kind], f8_start_bank=0)
    r = SplitMix64(77); draws = [r.next() for _ in range(32)]
    want_ram = b"".join(int(z).to_bytes(8, "little") for z in draws[:16]); want_sc = b"".join(int(z).to_bytes(8, "little") for z in draws[16:])
    assert bytes(o.ram()[0]) == want_ram and bytes(o.cart_ram()[0]) == want_sc     # RIOT RAM: draws 1-16 (C.2); Superchip RAM: draws 17-32
    run_instr(o, 26)
    ram = o.ram()[0]
    assert ram[0] == want_sc[5] and ram[1] == 0x5A and ram[2] == 0x5A and ram[3] == 0x5A and ram[4] == 0xC3
    assert ram[5] == img[0x100] and ram[6] == 0x5A and ram[7] == 0xA1 and regs(o)["bank"] == 1
    sc = o.cart_ram()[0]; assert sc[5] == 0x5A and sc[0x7F] == 0xC3 and bytes(sc[6:0x7F]) == want_sc[6:0x7F]
    # the plain format of the same size has no RAM there: the same program reads the filler
    o2 = OracleVCS([img], np.array([77], dtype=np.uint64), f8_start_bank=0); run_instr(o2, 6)
    assert o2.ram()[0][0] == 0xEE and o2.ram()[0][1] == 0xEE and (o2.cart_ram() == 0).all()


def _e0_image(build):
    code = hand_rom(build, entry=0xFC00)
    slices = []
    for k in range(8):
        img = bytearray([0x10 * k + 1]) * 1024; img[0] = 0xE0 + k      # a marker at the start of every slice
        slices.append(img)
    slices[7][:] = code[0xC00:0x1000]                                  # slice 7 is the fixed window at $1C00: code + vectors
    return bytes(b"".join(slices))


def test_e0_windows_and_hotspots():
    def build(a):
        a.org(0xFC00)
        for i, w in enumerate((0xF000, 0xF400, 0xF800)): a.op("LDA", "abs", w); a.op("STA", "zp", 0x80 + i)       # power-up slices 4, 5, 6 [R]
        a.op("LDA", "abs", 0xFFE2); a.op("STA", "abs", 0xFFEB); a.op("BIT", "abs", 0xFFF0)                          # read, write, read hotspots: 2, 3, 0
        for i, w in enumerate((0xF000, 0xF400, 0xF800)): a.op("LDA", "abs", w); a.op("STA", "zp", 0x84 + i)
        a.op("LDX", "imm", 7); a.op("LDA", "abx", 0xFFE0); a.op("LDA", "abx", 0xFFE8); a.op("LDA", "abx", 0xFFF0)   # every window on slice 7
        for i, w in enumerate((0xF000, 0xF400, 0xF800)): a.op("LDA", "abs", w); a.op("STA", "zp", 0x88 + i)
        a.op("LDA", "abs", 0xFFF8); a.op("LDA", "abs", 0xFFDF); a.op("LDA", "abs", 0xF800); a.op("STA", "zp", 0x8C)  # $1FF8 / $1FDF are no hotspots here
        a.label("end"); a.op("JMP", "abs", "end")
    o = OracleVCS([_e0_image(build)], np.array([1], dtype=np.uint64), mappers=["E0"])
    r = regs(o); assert r["pc"] == 0xFC00 and r["bank"] == (4 | 5 << 3) and r["pad"][0] == 6
    run_instr(o, 6); assert o.ram()[0][:3].tolist() == [0xE4, 0xE5, 0xE6]
    run_instr(o, 3); r = regs(o); assert r["bank"] == (2 | 3 << 3) and r["pad"][0] == 0
    run_instr(o, 6); assert o.ram()[0][4:7].tolist() == [0xE2, 0xE3, 0xE0]
    run_instr(o, 10); assert o.ram()[0][8:11].tolist() == [0xAD, 0xAD, 0xAD]                  # slice 7 holds the program: its first byte is LDA abs
    run_instr(o, 4); assert o.ram()[0][12] == 0xAD and regs(o)["bank"] == (7 | 7 << 3) and regs(o)["pad"][0] == 7


def test_fe_bank_follows_the_byte_after_the_stack_cell_01fe():
    def build(a):
        a.org(0xF000); a.op("LDX", "imm", 0xFF); a.op("TXS")
        a.op("JSR", "abs", 0xD100)                                     # pushes $01FF, $01FE; then the target's high byte $D1 (bit 5 = 0): bank 1
        a.op("STA", "zp", 0x81); a.op("STX", "zp", 0x82)
        a.op("LDA", "imm", 0x11); a.op("STA", "abs", 0x01FE); a.byte(0x8A)        # TXA = $8A: bit 5 clear -> bank 1 (whose byte there is INX)
        a.op("STX", "zp", 0x83); a.op("STA", "abs", 0x01FE); a.op("NOP")          # NOP = $EA: bit 5 set -> bank 0
        a.op("STA", "zp", 0x84)
        a.label("end"); a.op("JMP", "abs", "end")
        a.org(0xF100); a.op("LDA", "imm", 0xB0); a.op("STA", "zp", 0x80); a.op("LDX", "imm", 0xC0); a.op("RTS")
    b0 = bytearray(hand_rom(build)); b1 = bytearray(b0)
    b1[0x101] = 0xB1; b1[0x105] = 0xC1                                  # bank 1's subroutine loads other constants
    tx = bytes(b0).index(bytes([0x8D, 0xFE, 0x01, 0x8A])) + 3
    b1[tx] = 0xE8                                                       # ... and has INX where bank 0 has TXA
    o = OracleVCS([bytes(b0 + b1)], np.array([2], dtype=np.uint64), mappers=["FE"])
    assert regs(o)["bank"] == 0
    run_instr(o, 3); r = regs(o); assert r["pc"] == 0xD100 and r["bank"] == 1 and r["sp"] == 0xFD and r["pad"][0] == 0
    run_instr(o, 3); assert o.ram()[0][0] == 0xB1 and regs(o)["x"] == 0xC1           # bank 1's code ran
    run_instr(o); r = regs(o); assert r["pc"] == 0xF006 and r["bank"] == 0           # RTS: $01FE then $01FF = $F0 (bit 5 set)
    run_instr(o, 4); assert regs(o)["pad"][0] == 1                                   # STA $01FE: waiting for the next access
    # the next access is the opcode fetch at $F00F: it still reads bank 0's byte, $8A = TXA, whose bit 5 is clear -> bank 1
    run_instr(o); r = regs(o); assert r["bank"] == 1 and r["a"] == 0xC1 and r["x"] == 0xC1 and r["pad"][0] == 0
    run_instr(o, 2); run_instr(o); assert regs(o)["bank"] == 0                       # ... and after the second STA $01FE, NOP = $EA: bit 5 set
    run_instr(o); assert o.ram()[0][4] == 0xC1 and o.ram()[0][3] == 0xC1


def test_detect_mapper_rules():
    import vcs_inputs
    assert detect_mapper(bytes(2048)) == "2K" and detect_mapper(bytes(4096)) == "4K" and detect_mapper(bytes(1000)) == ""
    for n, plain, sc in ((2, "F8", "F8SC"), (4, "F6", "F6SC"), (8, "F4", "F4SC")):
        img = bytearray(_sc_image(n)); assert detect_mapper(bytes(img)) == sc
        img[0x1010] ^= 0xFF; assert detect_mapper(bytes(img)) == plain                # one bank without the filler: no Superchip
    img = bytearray([0xEA]) * 8192; img[5] = 0x00                                                    # (no filler in the port area)
    assert detect_mapper(bytes(img)) == "F8"
    img[0x100:0x103] = bytes([0xAD, 0xE3, 0xFF]); img[0x200:0x203] = bytes([0x8D, 0xF1, 0x1F])       # LDA $FFE3, STA $1FF1
    assert detect_mapper(bytes(img)) == "E0"
    img[0x300:0x303] = bytes([0x2C, 0xF8, 0xFF]); img[0x310:0x313] = bytes([0x2C, 0xF9, 0xFF])       # as many F8 hotspot accesses: F8 wins a tie
    assert detect_mapper(bytes(img)) == "F8"
    img = bytearray([0xEA]) * 8192; img[5] = 0x00
    img[0x100:0x103] = bytes([0x20, 0x00, 0xD1]); img[0x200:0x203] = bytes([0x4C, 0x40, 0xD2])       # JSR $D100, JMP $D240
    assert detect_mapper(bytes(img)) == "FE"
    img[0x300:0x303] = bytes([0xAD, 0xF9, 0x1F]); assert detect_mapper(bytes(img)) == "F8"
    for cfg in (1, 2, 3):                                                                            # the generated carts are what their size says
        rom = vcs_inputs.make_workload(cfg, batch=1).roms[0]
        assert detect_mapper(rom) == {2048: "2K", 4096: "4K"}[len(rom)]
    w = vcs_inputs.make_workload(4, batch=512, n_roms=4)
    assert [detect_mapper(r) for r in w.roms] == ["4K", "4K", "F8", "F8"]
