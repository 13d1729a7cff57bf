"""Seeded test cartridges for the Superchip (F8SC / F6SC / F4SC), E0 and FE formats (PAPER.md L69,
L469).  Input generation only: they emit bytes, no emulator arithmetic lives here.  Each is a small frame loop (VSYNC
pulse, work that depends on the env's seeded RAM and on the joystick, a few WSYNC lines that put results on the
screen) written to exercise what is particular to its format:
  * Superchip: cartridge RAM read before it is written (its seeded power-on contents), indexed stores into the write
    port and loads from the read port, a read-modify-write on the write port, code copied into cartridge RAM and
    called there, bank hotspots reached by indexed reads;
  * E0: all three windows re-pointed every frame (by an indexed read, an indexed store and a plain read), subroutines
    and tables reached through the windows, the fixed window holding the main program;
  * FE: JSR / RTS between the $F000 and $D000 pages with the stack at $01FF / $01FE, nested calls that do NOT touch
    $01FE, and a return address whose page is computed at run time."""
from __future__ import annotations

from .asm6502 import Asm, TIA_W, RIOT
from .prng import SplitMix64


def _vsync(a: Asm):
    a.op("LDA", "imm", 2); a.op("STA", "zp", TIA_W["VSYNC"]); a.op("STA", "zp", TIA_W["WSYNC"])
    a.op("LDA", "imm", 0); a.op("STA", "zp", TIA_W["VSYNC"]); a.op("STA", "zp", TIA_W["VBLANK"])


def _lines(a: Asm, n: int, table: int):
    """n WSYNC lines whose colours / playfield come from `table`,Y and RAM"""
    a.op("LDY", "imm", n); lp = a.newlabel("L"); a.label(lp)
    a.op("STA", "zp", TIA_W["WSYNC"]); a.op("LDA", "aby", table); a.op("STA", "zp", TIA_W["COLUBK"])
    a.op("LDA", "zpx", 0x80); a.op("STA", "zp", TIA_W["PF1"]); a.op("TYA"); a.op("STA", "zp", TIA_W["COLUPF"])
    a.op("DEY"); a.op("BNE", "rel", lp)


def superchip_rom(kind: str, seed: int) -> bytes:
    nb = {"F8SC": 2, "F6SC": 4, "F4SC": 8}[kind]
    hot = {2: 0xFFF8, 4: 0xFFF6, 8: 0xFFF4}[nb]
    r = SplitMix64(seed)
    a = Asm(4096, 0xF000, fill=0xFF)
    a.org(0xF100); a.label("entry")
    a.op("SEI"); a.op("CLD"); a.op("LDX", "imm", 0xFF); a.op("TXS")
    a.op("LDX", "imm", 15); a.label("c"); a.op("LDA", "abx", 0xF080); a.op("STA", "zpx", 0xC0); a.op("DEX"); a.op("BPL", "rel", "c")   # seeded cart RAM -> RIOT RAM
    stub = [0xA5, 0x80, 0x49, r.rnd(256), 0x85, 0x81, 0xE6, 0x85, 0x60]          # LDA $80 ; EOR #k ; STA $81 ; INC $85 ; RTS
    for i, b in enumerate(stub): a.op("LDA", "imm", b); a.op("STA", "abs", 0xF040 + i)                                                   # ... into cart RAM cells $40..
    a.label("frame"); _vsync(a)
    a.op("LDA", "abs", RIOT["SWCHA"]); a.op("EOR", "zp", 0x80); a.op("STA", "zp", 0x80)
    a.op("AND", "imm", 0x3F); a.op("TAX"); a.op("LDA", "zp", 0x80); a.op("STA", "abx", 0xF000)        # write port, indexed (cells $00-$3F)
    a.op("LDA", "abx", 0xF080); a.op("CLC"); a.op("ADC", "zp", 0x82); a.op("STA", "zp", 0x82)         # read port
    a.op("INC", "abs", 0xF010 + r.rnd(16)); a.op("LDA", "abx", 0xF000); a.op("STA", "zp", 0x86)       # RMW on / read of the write port
    a.op("LDY", "zp", 0x82); a.op("LDA", "aby", 0xF080); a.op("STA", "zp", 0x87)                      # runs past the ports into ROM for large Y
    a.op("JSR", "abs", 0xF0C0)                                                                        # code in cartridge RAM (read port + $40)
    a.op("LDA", "zp", 0x81); a.op("AND", "imm", nb - 1); a.op("TAX"); a.op("LDA", "abx", hot)         # bank hotspot by an indexed read
    a.op("LDA", "abs", 0xF800); a.op("STA", "zp", 0x83)                                               # this bank's marker
    a.op("LDX", "imm", 3); _lines(a, 24, 0xF080)
    a.op("JMP", "abs", "frame")
    img = bytearray(a.finish())
    for off in (0xFFC, 0xFFE): img[off] = a.labels["entry"] & 0xFF; img[off + 1] = a.labels["entry"] >> 8
    banks = []
    for b in range(nb):
        bk = bytearray(img); bk[0x800] = 0xA0 + b
        for i in range(0x810, 0x900): bk[i] = r.rnd(256) if b == 0 else banks[0][i]      # a shared data table
        banks.append(bk)
    return bytes(b"".join(banks))


def e0_rom(seed: int) -> bytes:
    r = SplitMix64(seed)
    a = Asm(1024, 0xFC00, fill=0xEA)                       # slice 7: the fixed window
    a.org(0xFC00); a.label("entry")
    a.op("SEI"); a.op("CLD"); a.op("LDX", "imm", 0xFF); a.op("TXS")
    a.label("frame"); _vsync(a)
    a.op("LDA", "abs", RIOT["SWCHA"]); a.op("EOR", "zp", 0x80); a.op("STA", "zp", 0x80)
    a.op("AND", "imm", 3); a.op("TAX"); a.op("LDA", "abx", 0xFFE0)                                     # window $1000 <- slice 0..3, by an indexed read
    a.op("LDA", "zp", 0x80); a.op("LSR", "acc"); a.op("LSR", "acc"); a.op("AND", "imm", 3); a.op("CLC"); a.op("ADC", "imm", 2)
    a.op("TAX"); a.op("STA", "abx", 0xFFE8)                                                            # window $1400 <- slice 2..5, by an indexed store
    a.op("LDA", "zp", 0x81); a.op("AND", "imm", 1); a.op("BEQ", "rel", "w2b"); a.op("BIT", "abs", 0xFFF6); a.op("JMP", "abs", "w2d")
    a.label("w2b"); a.op("BIT", "abs", 0xFFF3); a.label("w2d")                                         # window $1800 <- slice 6 or 3
    a.op("JSR", "abs", 0xF000); a.op("STA", "zp", 0x84); a.op("JSR", "abs", 0xF400); a.op("STA", "zp", 0x85)
    a.op("JSR", "abs", 0xF800); a.op("STA", "zp", 0x86)
    a.op("LDY", "zp", 0x80); a.op("LDA", "aby", 0xF010); a.op("EOR", "aby", 0xF410); a.op("CLC"); a.op("ADC", "aby", 0xF810)
    a.op("STA", "zp", 0x81); a.op("INC", "zp", 0x87)
    a.op("LDX", "imm", 1); _lines(a, 24, 0xF410)
    a.op("JMP", "abs", "frame")
    s7 = bytearray(a.finish())
    for off in (0x3FC, 0x3FE): s7[off] = a.labels["entry"] & 0xFF; s7[off + 1] = a.labels["entry"] >> 8
    slices = []
    for k in range(7):
        sl = bytearray(r.rnd(256) for _ in range(1024))
        sl[0:5] = bytes([0xA9, 0x10 * k + 5, 0xE6, 0x88 + k, 0x60])         # LDA #id ; INC $88+k ; RTS  (the same entry point in every window)
        slices.append(sl)
    return bytes(b"".join(slices) + s7)


def fe_rom(seed: int) -> bytes:
    r = SplitMix64(seed)

    def bank(which: int) -> bytearray:
        a = Asm(4096, 0xF000, fill=0xEA)
        a.org(0xF000); a.label("entry")
        a.op("SEI"); a.op("CLD"); a.op("LDX", "imm", 0xFF); a.op("TXS")
        a.label("frame"); _vsync(a)
        a.op("LDX", "imm", 0xFF); a.op("TXS")
        a.op("LDA", "abs", RIOT["SWCHA"]); a.op("EOR", "zp", 0x80); a.op("STA", "zp", 0x80)
        a.op("JSR", "abs", 0xD200); a.op("STA", "zp", 0x84)                  # pushes at $01FF / $01FE: lands in bank 1
        a.op("JSR", "abs", 0xF280); a.op("STA", "zp", 0x85)                  # a call inside the $F000 page
        a.op("LDA", "zp", 0x80); a.op("AND", "imm", 0x20); a.op("ORA", "imm", 0xD3); a.op("PHA")          # return address $D3xx or $F3xx ...
        a.op("LDA", "imm", 0x0F); a.op("PHA"); a.op("RTS")                                                  # ... - 1 low: "returns" to $x310 of the page chosen at run time
        a.org(0xF1C0); a.label("back"); a.op("STA", "zp", 0x86); a.op("INC", "zp", 0x87)
        a.op("LDX", "imm", 2); _lines(a, 24, 0xFA00)
        a.op("JMP", "abs", "frame")
        a.org(0xF200)                                                         # sub A (entered as $D200 in bank 1)
        a.op("LDA", "imm", 0x40 + which); a.op("JSR", "abs", 0xF2C0)          # nested: SP = $FD, $01FE is not touched, the bank stays
        a.op("RTS")
        a.org(0xF280); a.op("LDA", "imm", 0x50 + which); a.op("PHA"); a.op("PLA"); a.op("RTS")              # PHA / PLA at $01FD
        a.org(0xF2C0); a.op("CLC"); a.op("ADC", "imm", 0x08 + which); a.op("RTS")
        a.org(0xF310); a.op("LDX", "imm", 0xFF); a.op("TXS"); a.op("LDA", "imm", 0x60 + which)
        a.op("JMP", "abs", 0xF1C0 if which == 0 else 0xD1C0)                  # (a JMP does not switch: bank 1 carries the same tail)
        for i in range(0xA00, 0xB00): a.img[i] = 0                            # table filled below
        img = bytearray(a.finish())
        for off in (0xFFC, 0xFFE): img[off] = 0x00; img[off + 1] = 0xF0
        return img
    b0, b1 = bank(0), bank(1)
    tab = bytes(r.rnd(256) for _ in range(256))
    b0[0xA00:0xB00] = tab; b1[0xA00:0xB00] = tab
    return bytes(b0 + b1)
