"""Seeded synthetic cartridge generator (DESIGN.md §4 "input recipe").

Stands in for the copyrighted ROMs the paper measures on: 2/4/8 KB images
with 2K/4K/F8 mapping and a 262-line NTSC frame kernel (3 VSYNC + VBLANK timed by the RIOT timer
+ 192 WSYNC-paced visible lines with a few TIA stores each + 30 overscan lines), joystick polling
once per frame, random documented-opcode blocks with forward branches.  No real ROM byte or game
logic is reproduced.  Emits bytes only — no emulator arithmetic lives here.
"""
from __future__ import annotations

from dataclasses import dataclass

from .asm6502 import Asm, TIA_W, TIA_R, RIOT
from .prng import SplitMix64

ORIGIN = 0xF000
SUBS_ORG, TABLES_ORG, TABLES_END, TRAMP2_ORG = 0xF800, 0xFA00, 0xFE00, 0xFE00


@dataclass(frozen=True)
class Features:
    size: int = 2048          # 2048 | 4096 | 8192 (F8) | 16384 (F6) | 32768 (F4)
    joystick: bool = False    # config 2+: SWCHA / INPT4 reads, object update, RESP0 timing, CX reads
    extended: bool = False    # config 3+: indexed/indirect, JSR/RTS, stack, BCD, all timer divisors


FEATURES = {
    1: Features(2048, False, False),
    2: Features(4096, True, False),
    3: Features(4096, True, True),
    "4a": Features(4096, True, True),
    "4b": Features(8192, True, True),
    "f6": Features(16384, True, True),      # F6: four 4 KB banks, hotspots $1FF6-$1FF9
    "f4": Features(32768, True, True),      # F4: eight 4 KB banks, hotspots $1FF4-$1FFB
}


def _banks(size: int) -> int:
    return max(1, size // 4096)


def _hotspot_lo(size: int) -> int:
    return {8192: 0x1FF8, 16384: 0x1FF6, 32768: 0x1FF4}[size]

BAND_REGS_1 = ["COLUBK", "COLUPF", "PF0", "PF1", "PF2", "GRP0", "GRP1", "COLUP0", "RESP0", "HMP0", "HMOVE"]
BAND_REGS_2 = BAND_REGS_1 + ["COLUP1", "NUSIZ0", "NUSIZ1", "CTRLPF", "REFP0", "REFP1", "RESP1", "RESM0",
                             "RESM1", "RESBL", "ENAM0", "ENAM1", "ENABL", "HMP1", "HMM0", "HMM1", "HMBL",
                             "VDELP0", "VDELP1", "VDELBL", "HMCLR", "RESMP0", "RESMP1"]

# pointer table set up at entry for config 3+:  zp address -> (target, kind, Y range for writes)
POINTERS = [
    (0x90, 0xFAF0, "rom"),    # reads cross a page when Y >= 0x10
    (0x92, 0xFB80, "rom"),
    (0x94, 0x00A0, "ramlo"),  # writes with Y in [0x00,0x4F] stay in scratch $A0-$EF
    (0x96, 0x00F8, "ramhi"),  # writes with Y in [0xA8,0xF7] cross into the $0180 mirror = $A0-$EF
    (0x98, 0xFCFF, "rom"),    # crosses for every Y >= 1
    (0x9A, 0xFB10, "rom"),
    (0x9C, 0x0080, "ramrd"),  # read-only use
    (0x9E, 0xFC40, "rom"),
]


class _Gen:
    def __init__(self, a: Asm, rng: SplitMix64, feat: Features):
        self.a, self.rng, self.f = a, rng, feat
        self.subs: list[tuple[str, int]] = []      # (label, worst-case cycles incl. JSR+RTS)
        self.scratch = (0xA0, 0xEF) if feat.extended else (0x80, 0xFF)

    # ---- operand pickers ----------------------------------------------------------
    def zp_any(self) -> int:
        return 0x80 + self.rng.rnd(0x80)

    def zp_scratch(self) -> int:
        lo, hi = self.scratch
        return lo + self.rng.rnd(hi - lo + 1)

    def rom_table_addr(self) -> int:
        return TABLES_ORG + self.rng.rnd(0x300)     # +255 of index stays below TABLES_END

    # ---- items --------------------------------------------------------------------
    def item_base(self):
        a, r = self.a, self.rng
        k = r.rnd(10)
        if k < 2:
            a.op(r.choice(["LDA", "LDX", "LDY"]), *(("imm", r.rnd(256)) if r.chance(1, 2) else ("zp", self.zp_any())))
        elif k < 4:
            a.op(r.choice(["STA", "STA", "STX", "STY"]), "zp", self.zp_scratch())
        elif k < 7:
            mn = r.choice(["ADC", "SBC", "AND", "ORA", "EOR", "CMP"])
            if mn in ("ADC", "SBC") and r.chance(1, 3):
                a.op(r.choice(["CLC", "SEC"]))
            a.op(mn, *(("imm", r.rnd(256)) if r.chance(1, 2) else ("zp", self.zp_any())))
        else:
            mn = r.choice(["INC", "DEC", "ASL", "LSR", "ROL", "ROR"])
            if mn not in ("INC", "DEC") and r.chance(1, 3):
                a.op(mn, "acc")
            else:
                a.op(mn, "zp", self.zp_scratch())

    def item_extended(self):
        a, r = self.a, self.rng
        k = r.rnd(16)
        if k == 0:      # zp,X / zp,Y read with whatever index is live (page-0 wrap; TIA reads are harmless)
            mn = r.choice(["LDA", "ADC", "EOR", "CMP", "LDY", "ORA"])
            a.op(mn, "zpx", self.zp_any())
        elif k == 1:    # zp,X store with a pinned index, target in scratch
            t = self.zp_scratch(); i = r.rnd(min(16, t - self.scratch[0] + 1))
            a.op("LDX", "imm", i); a.op(r.choice(["STA", "STY"]), "zpx", t - i)
        elif k == 2:    # abs,X / abs,Y read from a ROM table (page crossings by chance)
            mn = r.choice(["LDA", "ADC", "SBC", "AND", "CMP", "EOR", "ORA"])
            a.op(mn, r.choice(["abx", "aby"]), self.rom_table_addr())
        elif k == 3:    # LDX abs,Y / LDY abs,X
            if r.chance(1, 2): a.op("LDX", "aby", self.rom_table_addr())
            else: a.op("LDY", "abx", self.rom_table_addr())
        elif k == 4:    # abs store / abs,X store / abs,Y store into scratch (pinned index)
            t = self.zp_scratch(); i = r.rnd(min(16, t - self.scratch[0] + 1))
            m = r.rnd(3)
            if m == 0: a.op(r.choice(["STA", "STX", "STY"]), "abs", t)
            elif m == 1: a.op("LDX", "imm", i); a.op("STA", "abx", t - i)
            else: a.op("LDY", "imm", i); a.op("STA", "aby", t - i)
        elif k == 5:    # abs RMW in scratch, abs,X RMW with pinned index
            t = self.zp_scratch(); mn = r.choice(["INC", "DEC", "ASL", "LSR", "ROL", "ROR"])
            if r.chance(1, 2): a.op(mn, "abs", t)
            else:
                i = r.rnd(min(16, t - self.scratch[0] + 1)); a.op("LDX", "imm", i)
                a.op(mn, r.choice(["abx", "zpx"]), t - i)
        elif k == 6:    # (zp),Y read through any pointer
            p = r.choice(POINTERS)
            a.op("LDY", "imm", r.rnd(256))
            a.op(r.choice(["LDA", "ADC", "SBC", "AND", "CMP", "EOR", "ORA"]), "izy", p[0])
        elif k == 7:    # (zp),Y store through a write-safe pointer
            if r.chance(1, 2): a.op("LDY", "imm", r.rnd(0x50)); a.op("STA", "izy", 0x94)
            else: a.op("LDY", "imm", 0xA8 + r.rnd(0x50)); a.op("STA", "izy", 0x96)
        elif k == 8:    # (zp,X) read / store
            j = r.rnd(len(POINTERS))
            if r.chance(1, 3):
                a.op("LDX", "imm", 4); a.op("STA", "izx", 0x90)      # through ($94) -> $00A0 (scratch)
            else:
                a.op("LDX", "imm", 2 * j); a.op(r.choice(["LDA", "ADC", "EOR", "CMP", "ORA", "AND", "SBC"]), "izx", 0x90)
        elif k == 9 and self.subs:
            lab, cost = r.choice(self.subs); a.op("JSR", "abs", lab); a.cycles += cost - 6
        elif k == 10:   # stack pair around a simple item
            if r.chance(1, 2): a.op("PHA"); self.item_base(); a.op("PLA")
            else: a.op("PHP"); self.item_base(); a.op("PLP")
        elif k == 11:   # BCD section on uniform random bytes (invalid BCD included)
            a.op("SED"); a.op(r.choice(["CLC", "SEC"]))
            a.op("LDA", *(("imm", r.rnd(256)) if r.chance(1, 2) else ("zp", self.zp_any())))
            for _ in range(1 + r.rnd(3)):
                a.op(r.choice(["ADC", "SBC"]), *(("imm", r.rnd(256)) if r.chance(1, 2) else ("zp", self.zp_any())))
            a.op("STA", "zp", self.zp_scratch()); a.op("CLD")
        elif k == 12:   # timer / port reads (never after an underflow: blocks are shorter than the timer)
            a.op("LDA", "abs", r.choice([RIOT["INTIM"], RIOT["TIMINT"], RIOT["SWCHB"], RIOT["SWCHA"]]))
        elif k == 13:   # transfers and index arithmetic
            a.op(r.choice(["TAX", "TAY", "TXA", "TYA", "INX", "INY", "DEX", "DEY", "TSX", "CLV", "NOP"]))
        elif k == 14:   # BIT / CPX / CPY
            mn = r.choice(["BIT", "CPX", "CPY"])
            if mn == "BIT": a.op("BIT", *(("zp", self.zp_any()) if r.chance(1, 2) else ("abs", self.rom_table_addr())))
            else: a.op(mn, *(("imm", r.rnd(256)) if r.chance(1, 2) else ("zp", self.zp_any())))
        else:
            self.item_base()

    def item(self):
        if self.f.extended and self.rng.chance(1, 2):
            self.item_extended()
        else:
            self.item_base()

    def block(self, cyc_budget: int, byte_limit_addr: int, item_reserve: int = 110):
        """Random block: items + forward branches skipping 1-4 whole items (G.1)."""
        a, r = self.a, self.rng
        start_cycles = a.cycles
        pending: list[list] = []           # [items still to skip, label]
        while (a.cycles - start_cycles) + item_reserve <= cyc_budget and a.pc + 48 <= byte_limit_addr:
            if r.chance(1, 5):
                lab = a.newlabel("B")
                a.op(r.choice(["BCC", "BCS", "BEQ", "BNE", "BMI", "BPL", "BVC", "BVS"]), "rel", lab)
                pending.append([1 + r.rnd(4) + 1, lab])     # +1: this branch item itself is counted below
            else:
                self.item()
            for p in pending:
                p[0] -= 1
            for p in [p for p in pending if p[0] <= 0]:
                a.label(p[1]); pending.remove(p)
        for p in pending:
            a.label(p[1])
        return a.cycles - start_cycles


def _prologue(a: Asm, feat: Features):
    """entry + frame head; byte-identical in both banks of an F8 image (no randomness)."""
    a.org(ORIGIN)
    a.label("entry")
    a.op("SEI"); a.op("CLD"); a.op("LDX", "imm", 0xFF); a.op("TXS")
    if feat.extended:
        for zp, target, _ in POINTERS:
            a.op("LDA", "imm", target & 0xFF); a.op("STA", "zp", zp)
            a.op("LDA", "imm", target >> 8); a.op("STA", "zp", zp + 1)
    a.label("frame")
    a.op("LDA", "imm", 2); a.op("STA", "zp", TIA_W["VBLANK"]); a.op("STA", "zp", TIA_W["VSYNC"])
    for _ in range(3):
        a.op("STA", "zp", TIA_W["WSYNC"])
    a.op("LDA", "imm", 0); a.op("STA", "zp", TIA_W["VSYNC"])          # frame-end event, cycle 4 of line 0
    a.op("LDA", "imm", 43); a.op("STA", "abs", RIOT["TIM64T"])        # written in cycle 10
    if feat.size == 8192:                                              # trampoline 1 (bank by a RAM bit)
        a.op("LDA", "zp", 0xA7); a.op("EOR", "zp", 0x80); a.op("LSR", "acc")
        a.op("BCS", "rel", "t1_b1"); a.op("BIT", "abs", 0x1FF8); a.op("BCC", "rel", "t1_c")
        a.label("t1_b1"); a.op("BIT", "abs", 0x1FF9)
        a.label("t1_c")
    elif feat.size > 8192:                                             # F6 / F4: bank = RAM bits, selected by an indexed read
        a.op("LDA", "zp", 0xA7); a.op("EOR", "zp", 0x80); a.op("AND", "imm", _banks(feat.size) - 1); a.op("TAX")
        a.op("LDA", "abx", _hotspot_lo(feat.size))


def _input_block(a: Asm, g: _Gen):
    """config 2+: joystick -> object state -> RESP0 timing / colour / graphics (G.1 INPUT block)."""
    r = g.rng
    a.op("LDA", "abs", RIOT["SWCHA"])
    for mn, zp in (("INC", 0x80), ("DEC", 0x80), ("INC", 0x81), ("DEC", 0x81)):   # bits 7 R, 6 L, 5 D, 4 U
        lab = a.newlabel("J")
        a.op("ASL", "acc"); a.op("BCS", "rel", lab); a.op(mn, "zp", zp); a.label(lab)
    lab = a.newlabel("F")
    a.op("BIT", "zp", TIA_R["INPT4"]); a.op("BMI", "rel", lab); a.op("INC", "zp", 0x82); a.label(lab)
    a.op("INC", "zp", 0x83)                                                       # frame counter
    # collision latches feed RAM, then clear
    a.op("LDA", "zp", TIA_R[r.choice(["CXP0FB", "CXP1FB", "CXM0P", "CXM1P", "CXPPMM", "CXBLPF", "CXM0FB", "CXM1FB"])])
    a.op("STA", "zp", 0x84)
    a.op("LDA", "zp", TIA_R[r.choice(["CXP0FB", "CXP1FB", "CXM0P", "CXM1P", "CXPPMM", "CXBLPF"])])
    a.op("ORA", "zp", 0x85); a.op("STA", "zp", 0x85)
    a.op("STA", "zp", TIA_W["CXCLR"])
    # bounded delay loop then RESP0: horizontal position follows the joystick
    d = a.newlabel("D")
    a.op("STA", "zp", TIA_W["WSYNC"])
    a.op("LDA", "zp", 0x80); a.op("AND", "imm", 15); a.op("TAX")
    a.label(d); a.op("DEX"); a.op("BPL", "rel", d)
    a.op("STA", "zp", TIA_W["RESP0"])
    a.op("LDA", "zp", 0x81); a.op("STA", "zp", TIA_W[r.choice(["COLUP0", "COLUP1", "COLUPF"])])
    a.op("LDA", "zp", 0x82); a.op("STA", "zp", TIA_W[r.choice(["GRP0", "GRP1", "PF1"])])
    a.op("LDA", "zp", 0x80); a.op("STA", "zp", TIA_W[r.choice(["HMP0", "HMP1", "HMBL"])])
    # the worst case of the delay loop (16 iterations of DEX/BPL) beyond the single pass counted by Asm
    a.cycles += 15 * 5 + 76


def _bands(a: Asm, g: _Gen):
    r = g.rng
    regs = BAND_REGS_2 if g.f.joystick else BAND_REGS_1
    for _ in range(8):
        lab = a.newlabel("V")
        a.op("LDY", "imm", 24)
        a.label(lab)
        a.op("STA", "zp", TIA_W["WSYNC"])
        for _ in range(2 + r.rnd(5)):
            use_x = r.chance(1, 2)
            if g.f.joystick and r.chance(1, 4):
                a.op("LDX" if use_x else "LDA", "zp", 0x80 + r.rnd(16))
            else:
                a.op("LDX" if use_x else "LDA", "imm", r.rnd(256))
            a.op("STX" if use_x else "STA", "zp", TIA_W[r.choice(regs)])
        a.op("DEY"); a.op("BNE", "rel", lab)


def _overscan(a: Asm, g: _Gen):
    """30 lines (229..258).  config 1-2: WSYNC-counted; config 3+: paced by a random timer divisor."""
    r = g.rng
    a.op("STA", "zp", TIA_W["WSYNC"]); a.op("LDA", "imm", 2); a.op("STA", "zp", TIA_W["VBLANK"])   # line 229, cycle 5
    limit = SUBS_ORG - 80 if g.f.size != 2048 else ORIGIN + 2048 - 40
    if not g.f.extended:
        g.block(60, limit, item_reserve=12)
        lab = a.newlabel("O")
        a.op("LDY", "imm", 30); a.label(lab); a.op("STA", "zp", TIA_W["WSYNC"]); a.op("DEY"); a.op("BNE", "rel", lab)
        return
    div = r.choice(["TIM1T", "TIM8T", "TIM64T", "T1024T"])
    if div == "TIM1T":
        g.block(55, limit, item_reserve=12)
        t, w = a.newlabel("T"), a.newlabel("W")
        a.op("LDY", "imm", 29); a.label(t); a.op("STA", "zp", TIA_W["WSYNC"])
        a.op("LDA", "imm", 40); a.op("STA", "abs", RIOT["TIM1T"])
        a.label(w); a.op("BIT", "abs", RIOT["TIMINT"]); a.op("BPL", "rel", w)
        a.op("DEY"); a.op("BNE", "rel", t)
        a.op("STA", "zp", TIA_W["WSYNC"])
        return
    n, shift = {"TIM8T": (250, 3), "TIM64T": (35, 6), "T1024T": (2, 10)}[div]
    a.op("LDA", "imm", n); a.op("STA", "abs", RIOT[div])           # write lands in cycle 10 of line 229
    cu = 10 + 1 + (n << shift)                                      # underflow cycle (C.7 closed form)
    line_idx, cyc_in_line = divmod(cu, 76)
    assert 5 <= cyc_in_line <= 55 and line_idx <= 29, (div, cu)
    g.block(min(600, cu - 200), limit)
    w = a.newlabel("W")
    a.label(w); a.op("BIT", "abs", RIOT["TIMINT"]); a.op("BPL", "rel", w)
    for _ in range(1 + (29 - line_idx)):
        a.op("STA", "zp", TIA_W["WSYNC"])


def _gen_bank(seed: int, feat: Features, bank: int) -> bytes:
    rng = SplitMix64(seed ^ (0xB4 * (bank + 1)))
    size = 2048 if feat.size == 2048 else 4096
    a = Asm(size, ORIGIN)
    g = _Gen(a, rng, feat)
    if feat.size != 2048:                     # data tables + subroutines first (their costs are needed)
        a.org(TABLES_ORG)
        for _ in range(TABLES_END - TABLES_ORG):
            a.byte(rng.rnd(256))
    if feat.extended:
        a.org(SUBS_ORG)
        for k in range(4 + rng.rnd(5)):
            lab = f"sub{k}"
            a.label(lab); c0 = a.cycles
            saved, g.subs = g.subs, []          # no nested JSR
            g.block(70, TABLES_ORG - 8, item_reserve=30)
            g.subs = saved
            a.op("RTS")
            g.subs.append((lab, a.cycles - c0 + 6))
        assert a.pc <= TABLES_ORG
    _prologue(a, feat)
    # BLOCK_A (+ input block) must fit well inside the 43*64-cycle VBLANK timer
    a.cycles = 0
    limit = (SUBS_ORG if size == 4096 else ORIGIN + 2048) - 800
    # JSR items cost up to 6 + 70 + 6; reserve accordingly
    g.block(1900, limit, item_reserve=130 if feat.extended else 40)
    if feat.joystick:
        _input_block(a, g)
    assert a.cycles <= 2400, a.cycles
    a.label("wait"); a.op("LDA", "abs", RIOT["INTIM"]); a.op("BNE", "rel", "wait")
    a.op("STA", "zp", TIA_W["WSYNC"]); a.op("STA", "zp", TIA_W["VBLANK"])          # A = 0
    _bands(a, g)
    if feat.size >= 8192:                      # trampoline 2 at a fixed address, landing differs per bank
        a.op("JMP", "abs", TRAMP2_ORG)
        a.label("after_t2")
    _overscan(a, g)
    a.op("JMP", "abs", "frame")
    assert a.pc <= (SUBS_ORG if size == 4096 else ORIGIN + 2048 - 4), hex(a.pc)
    if feat.size == 8192:
        a.org(TRAMP2_ORG)
        a.op("LDA", "zp", 0xB3); a.op("EOR", "zp", 0x83); a.op("LSR", "acc"); a.op("LSR", "acc")
        a.op("BCS", "rel", "t2_b1"); a.op("BIT", "abs", 0x1FF8); a.op("BCC", "rel", "t2_c")
        a.label("t2_b1"); a.op("BIT", "abs", 0x1FF9)
        a.label("t2_c"); a.op("JMP", "abs", "after_t2")
    elif feat.size > 8192:
        a.org(TRAMP2_ORG)
        a.op("LDA", "zp", 0xB3); a.op("EOR", "zp", 0x83); a.op("LSR", "acc"); a.op("AND", "imm", _banks(feat.size) - 1); a.op("TAY")
        a.op("STA", "aby", _hotspot_lo(feat.size))                     # a write selects the bank as well (any bus access does)
        a.op("JMP", "abs", "after_t2")
    img = bytearray(a.finish())
    entry = a.labels["entry"]
    for off in (size - 4, size - 2):
        img[off] = entry & 0xFF; img[off + 1] = entry >> 8
    return bytes(img)


def make_rom(seed: int, feat: Features) -> bytes:
    """One cartridge image of feat.size bytes from `seed`."""
    return b"".join(_gen_bank(seed, feat, b) for b in range(_banks(feat.size)))
