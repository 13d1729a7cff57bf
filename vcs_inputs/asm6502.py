"""A tiny two-pass 6502 assembler used by the ROM generator and by hand-written test programs.

Input-generation tooling only (it emits bytes; it does not emulate anything).  The opcode
table is the documented NMOS 6502 set (151 opcodes, SURVEY.md §8(c) C.5 [D]).
Cycle figures are (base, +1-on-page-cross) and are used only to budget generated code so that
frames keep their line count (SURVEY §8(d) G.1 "worst-case cycles").
"""
from __future__ import annotations

# mnemonic -> mode -> (opcode, base cycles, page-cross penalty)
OPCODES = {
    "ADC": {"imm": (0x69, 2, 0), "zp": (0x65, 3, 0), "zpx": (0x75, 4, 0), "abs": (0x6D, 4, 0), "abx": (0x7D, 4, 1), "aby": (0x79, 4, 1), "izx": (0x61, 6, 0), "izy": (0x71, 5, 1)},
    "AND": {"imm": (0x29, 2, 0), "zp": (0x25, 3, 0), "zpx": (0x35, 4, 0), "abs": (0x2D, 4, 0), "abx": (0x3D, 4, 1), "aby": (0x39, 4, 1), "izx": (0x21, 6, 0), "izy": (0x31, 5, 1)},
    "ASL": {"acc": (0x0A, 2, 0), "zp": (0x06, 5, 0), "zpx": (0x16, 6, 0), "abs": (0x0E, 6, 0), "abx": (0x1E, 7, 0)},
    "BCC": {"rel": (0x90, 2, 0)}, "BCS": {"rel": (0xB0, 2, 0)}, "BEQ": {"rel": (0xF0, 2, 0)}, "BMI": {"rel": (0x30, 2, 0)},
    "BNE": {"rel": (0xD0, 2, 0)}, "BPL": {"rel": (0x10, 2, 0)}, "BVC": {"rel": (0x50, 2, 0)}, "BVS": {"rel": (0x70, 2, 0)},
    "BIT": {"zp": (0x24, 3, 0), "abs": (0x2C, 4, 0)},
    "BRK": {"imp": (0x00, 7, 0)},
    "CLC": {"imp": (0x18, 2, 0)}, "CLD": {"imp": (0xD8, 2, 0)}, "CLI": {"imp": (0x58, 2, 0)}, "CLV": {"imp": (0xB8, 2, 0)},
    "CMP": {"imm": (0xC9, 2, 0), "zp": (0xC5, 3, 0), "zpx": (0xD5, 4, 0), "abs": (0xCD, 4, 0), "abx": (0xDD, 4, 1), "aby": (0xD9, 4, 1), "izx": (0xC1, 6, 0), "izy": (0xD1, 5, 1)},
    "CPX": {"imm": (0xE0, 2, 0), "zp": (0xE4, 3, 0), "abs": (0xEC, 4, 0)},
    "CPY": {"imm": (0xC0, 2, 0), "zp": (0xC4, 3, 0), "abs": (0xCC, 4, 0)},
    "DEC": {"zp": (0xC6, 5, 0), "zpx": (0xD6, 6, 0), "abs": (0xCE, 6, 0), "abx": (0xDE, 7, 0)},
    "DEX": {"imp": (0xCA, 2, 0)}, "DEY": {"imp": (0x88, 2, 0)},
    "EOR": {"imm": (0x49, 2, 0), "zp": (0x45, 3, 0), "zpx": (0x55, 4, 0), "abs": (0x4D, 4, 0), "abx": (0x5D, 4, 1), "aby": (0x59, 4, 1), "izx": (0x41, 6, 0), "izy": (0x51, 5, 1)},
    "INC": {"zp": (0xE6, 5, 0), "zpx": (0xF6, 6, 0), "abs": (0xEE, 6, 0), "abx": (0xFE, 7, 0)},
    "INX": {"imp": (0xE8, 2, 0)}, "INY": {"imp": (0xC8, 2, 0)},
    "JMP": {"abs": (0x4C, 3, 0), "ind": (0x6C, 5, 0)},
    "JSR": {"abs": (0x20, 6, 0)},
    "LDA": {"imm": (0xA9, 2, 0), "zp": (0xA5, 3, 0), "zpx": (0xB5, 4, 0), "abs": (0xAD, 4, 0), "abx": (0xBD, 4, 1), "aby": (0xB9, 4, 1), "izx": (0xA1, 6, 0), "izy": (0xB1, 5, 1)},
    "LDX": {"imm": (0xA2, 2, 0), "zp": (0xA6, 3, 0), "zpy": (0xB6, 4, 0), "abs": (0xAE, 4, 0), "aby": (0xBE, 4, 1)},
    "LDY": {"imm": (0xA0, 2, 0), "zp": (0xA4, 3, 0), "zpx": (0xB4, 4, 0), "abs": (0xAC, 4, 0), "abx": (0xBC, 4, 1)},
    "LSR": {"acc": (0x4A, 2, 0), "zp": (0x46, 5, 0), "zpx": (0x56, 6, 0), "abs": (0x4E, 6, 0), "abx": (0x5E, 7, 0)},
    "NOP": {"imp": (0xEA, 2, 0)},
    "ORA": {"imm": (0x09, 2, 0), "zp": (0x05, 3, 0), "zpx": (0x15, 4, 0), "abs": (0x0D, 4, 0), "abx": (0x1D, 4, 1), "aby": (0x19, 4, 1), "izx": (0x01, 6, 0), "izy": (0x11, 5, 1)},
    "PHA": {"imp": (0x48, 3, 0)}, "PHP": {"imp": (0x08, 3, 0)}, "PLA": {"imp": (0x68, 4, 0)}, "PLP": {"imp": (0x28, 4, 0)},
    "ROL": {"acc": (0x2A, 2, 0), "zp": (0x26, 5, 0), "zpx": (0x36, 6, 0), "abs": (0x2E, 6, 0), "abx": (0x3E, 7, 0)},
    "ROR": {"acc": (0x6A, 2, 0), "zp": (0x66, 5, 0), "zpx": (0x76, 6, 0), "abs": (0x6E, 6, 0), "abx": (0x7E, 7, 0)},
    "RTI": {"imp": (0x40, 6, 0)}, "RTS": {"imp": (0x60, 6, 0)},
    "SBC": {"imm": (0xE9, 2, 0), "zp": (0xE5, 3, 0), "zpx": (0xF5, 4, 0), "abs": (0xED, 4, 0), "abx": (0xFD, 4, 1), "aby": (0xF9, 4, 1), "izx": (0xE1, 6, 0), "izy": (0xF1, 5, 1)},
    "SEC": {"imp": (0x38, 2, 0)}, "SED": {"imp": (0xF8, 2, 0)}, "SEI": {"imp": (0x78, 2, 0)},
    "STA": {"zp": (0x85, 3, 0), "zpx": (0x95, 4, 0), "abs": (0x8D, 4, 0), "abx": (0x9D, 5, 0), "aby": (0x99, 5, 0), "izx": (0x81, 6, 0), "izy": (0x91, 6, 0)},
    "STX": {"zp": (0x86, 3, 0), "zpy": (0x96, 4, 0), "abs": (0x8E, 4, 0)},
    "STY": {"zp": (0x84, 3, 0), "zpx": (0x94, 4, 0), "abs": (0x8C, 4, 0)},
    "TAX": {"imp": (0xAA, 2, 0)}, "TAY": {"imp": (0xA8, 2, 0)}, "TSX": {"imp": (0xBA, 2, 0)},
    "TXA": {"imp": (0x8A, 2, 0)}, "TXS": {"imp": (0x9A, 2, 0)}, "TYA": {"imp": (0x98, 2, 0)},
}

MODE_LEN = {"imp": 1, "acc": 1, "imm": 2, "zp": 2, "zpx": 2, "zpy": 2, "rel": 2, "izx": 2, "izy": 2,
            "abs": 3, "abx": 3, "aby": 3, "ind": 3}

# TIA write / read and RIOT register addresses (SURVEY §8(c) C.7/C.8 register maps [D])
TIA_W = dict(VSYNC=0x00, VBLANK=0x01, WSYNC=0x02, RSYNC=0x03, NUSIZ0=0x04, NUSIZ1=0x05, COLUP0=0x06,
             COLUP1=0x07, COLUPF=0x08, COLUBK=0x09, CTRLPF=0x0A, REFP0=0x0B, REFP1=0x0C, PF0=0x0D,
             PF1=0x0E, PF2=0x0F, RESP0=0x10, RESP1=0x11, RESM0=0x12, RESM1=0x13, RESBL=0x14,
             AUDC0=0x15, AUDC1=0x16, AUDF0=0x17, AUDF1=0x18, AUDV0=0x19, AUDV1=0x1A, GRP0=0x1B,
             GRP1=0x1C, ENAM0=0x1D, ENAM1=0x1E, ENABL=0x1F, HMP0=0x20, HMP1=0x21, HMM0=0x22,
             HMM1=0x23, HMBL=0x24, VDELP0=0x25, VDELP1=0x26, VDELBL=0x27, RESMP0=0x28, RESMP1=0x29,
             HMOVE=0x2A, HMCLR=0x2B, CXCLR=0x2C)
TIA_R = dict(CXM0P=0x00, CXM1P=0x01, CXP0FB=0x02, CXP1FB=0x03, CXM0FB=0x04, CXM1FB=0x05, CXBLPF=0x06,
             CXPPMM=0x07, INPT0=0x08, INPT1=0x09, INPT2=0x0A, INPT3=0x0B, INPT4=0x0C, INPT5=0x0D)
RIOT = dict(SWCHA=0x0280, SWACNT=0x0281, SWCHB=0x0282, SWBCNT=0x0283, INTIM=0x0284, TIMINT=0x0285,
            TIM1T=0x0294, TIM8T=0x0295, TIM64T=0x0296, T1024T=0x0297)


def worst_cycles(mn: str, mode: str) -> int:
    """Worst-case cycle count of one instruction (page-cross and branch penalties included)."""
    _, base, px = OPCODES[mn][mode]
    return base + px + (2 if mode == "rel" else 0)


class Asm:
    """Assembles into a flat image of `size` bytes whose byte 0 sits at CPU address `origin`."""

    def __init__(self, size: int, origin: int, fill: int = 0xEA):
        self.size, self.origin = size, origin
        self.img = bytearray([fill]) * size
        self.pc = origin
        self.labels: dict[str, int] = {}
        self.fixups: list[tuple[int, str, str]] = []   # (image offset, kind, label)
        self.cycles = 0                                   # running worst-case total (callers may reset)
        self._uid = 0

    # -- placement ------------------------------------------------------------------
    def org(self, addr: int):
        assert self.origin <= addr < self.origin + self.size, hex(addr)
        self.pc = addr

    def label(self, name: str):
        assert name not in self.labels, name
        self.labels[name] = self.pc

    def newlabel(self, stem: str = "L") -> str:
        self._uid += 1
        return f"{stem}_{self._uid}"

    def _put(self, b: int):
        off = self.pc - self.origin
        assert 0 <= off < self.size, f"image overflow at {self.pc:#x}"
        self.img[off] = b & 0xFF
        self.pc += 1

    def byte(self, *vals: int):
        for v in vals:
            self._put(v)

    def word_at(self, addr: int, value: int):
        off = addr - self.origin
        self.img[off] = value & 0xFF
        self.img[off + 1] = (value >> 8) & 0xFF

    # -- instructions ---------------------------------------------------------------
    def op(self, mn: str, mode: str = "imp", arg=None):
        """Emit one instruction.  `arg` is an int, or a label name for rel/abs/ind modes."""
        code, _, _ = OPCODES[mn][mode]
        self.cycles += worst_cycles(mn, mode)
        self._put(code)
        n = MODE_LEN[mode]
        if n == 1:
            return
        if isinstance(arg, str):
            if mode == "rel":
                self.fixups.append((self.pc - self.origin, "rel", arg))
                self._put(0)
            else:
                assert n == 3, (mn, mode)
                self.fixups.append((self.pc - self.origin, "abs", arg))
                self._put(0); self._put(0)
            return
        assert arg is not None, (mn, mode)
        if n == 2:
            if mode == "rel":
                assert -128 <= arg <= 127
            self._put(arg & 0xFF)
        else:
            self._put(arg & 0xFF); self._put((arg >> 8) & 0xFF)

    def finish(self) -> bytes:
        for off, kind, name in self.fixups:
            target = self.labels[name]
            if kind == "rel":
                d = target - (self.origin + off + 1)
                assert -128 <= d <= 127, f"branch to {name} out of range ({d})"
                self.img[off] = d & 0xFF
            else:
                self.img[off] = target & 0xFF
                self.img[off + 1] = (target >> 8) & 0xFF
        self.fixups.clear()
        return bytes(self.img)


def hand_rom(build, size: int = 4096, origin: int = 0xF000, entry: str | int = 0xF000) -> bytes:
    """Helper for tests: run `build(asm)` and set reset + BRK vectors to `entry`."""
    a = Asm(size, origin)
    build(a)
    img = bytearray(a.finish())
    e = a.labels[entry] if isinstance(entry, str) else entry
    for off in (size - 4, size - 2):     # $FFFC reset, $FFFE BRK (mirrored for 2 KB images)
        img[off] = e & 0xFF
        img[off + 1] = (e >> 8) & 0xFF
    return bytes(img)
