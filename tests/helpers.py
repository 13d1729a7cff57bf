"""Shared test helpers: hand-assembled programs on the oracle, golden-file parsing."""
from __future__ import annotations

import os

import numpy as np

from oracle.ovcs_py import OracleVCS
from vcs_inputs import Asm, hand_rom, TIA_W, TIA_R, RIOT  # noqa: F401

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def oracle_for(build, size=4096, seed=0, entry=0xF000, **kw) -> OracleVCS:
    """One oracle console running the program assembled by build(asm) at $F000."""
    rom = hand_rom(build, size=size, entry=entry)
    return OracleVCS([rom], np.array([seed], dtype=np.uint64), **kw)


def run_instr(o: OracleVCS, n=1):
    ev = 0
    for _ in range(n):
        ev += o.step_instruction(0)
    return ev


def regs(o: OracleVCS):
    return o.regs()[0]


def load_opcode_matrix():
    """-> {opcode: (mnemonic, mode, cycles, pagecross)} from tests/golden/opcode_matrix.txt"""
    cols = None
    out = {}
    for line in open(os.path.join(GOLDEN, "opcode_matrix.txt")):
        if line.startswith("#") or not line.strip():
            continue
        toks = line.split()
        if toks[0] == "x0":
            cols = [int(t[1], 16) for t in toks]
            continue
        hi = int(toks[0][0], 16)
        cells = toks[1:]
        assert len(cells) == len(cols), line
        for lo, cell in zip(cols, cells):
            if cell == "-":
                continue
            name, cyc = cell.split("/")
            px = cyc.endswith("+")
            cyc = int(cyc.rstrip("+"))
            if "." in name:
                mn, mode = name.split(".")
                mode = {"A": "acc"}.get(mode, mode)
            else:
                mn = name
                mode = "rel" if mn in ("BPL", "BMI", "BVC", "BVS", "BCC", "BCS", "BNE", "BEQ") else \
                       "abs" if mn == "JSR" else "imp"
            out[hi * 16 + lo] = (mn, mode, cyc, px)
    return out


def load_undocumented():
    """-> {opcode: (mnemonic, mode, cycles, pagecross)} from tests/golden/undocumented_opcodes.txt"""
    out = {}
    for line in open(os.path.join(GOLDEN, "undocumented_opcodes.txt")):
        if line.startswith("#") or not line.strip():
            continue
        code, mn, mode, cyc = line.split()
        out[int(code, 16)] = (mn, mode, int(cyc.rstrip("+")), cyc.endswith("+"))
    return out


def switch_rom() -> bytes:
    """A frame loop that samples the console switches once per frame (NEXT-4 tests).  After the VSYNC that ends frame
    n (n >= 1) it runs: $80 += 1 (frames seen), $82 = SWCHB, $81 += 1 if RESET (bit 0) reads low, COLUBK = $4A when the
    colour switch (bit 3) reads high else $0E, $85 = SWCHA, $86 = P after BIT SWCHB (N = bit 7, V = bit 6), then 200
    WSYNC lines.  $80 / $81 are cleared at power-on, so after f frames $80 == f - 1."""
    def build(a):
        a.org(0xF000); a.op("LDX", "imm", 0xFF); a.op("TXS"); a.op("LDA", "imm", 0); a.op("STA", "zp", 0x80); a.op("STA", "zp", 0x81)
        a.label("frame")
        a.op("LDA", "imm", 2); a.op("STA", "zp", TIA_W["VSYNC"])
        for _ in range(3): a.op("STA", "zp", TIA_W["WSYNC"])
        a.op("LDA", "imm", 0); a.op("STA", "zp", TIA_W["VSYNC"])
        a.op("INC", "zp", 0x80)
        a.op("LDA", "abs", RIOT["SWCHB"]); a.op("STA", "zp", 0x82)
        a.op("LSR", "acc"); a.op("BCS", "rel", "held_not"); a.op("INC", "zp", 0x81); a.label("held_not")
        a.op("LDA", "zp", 0x82); a.op("AND", "imm", 0x08); a.op("BEQ", "rel", "bw")
        a.op("LDA", "imm", 0x4A); a.op("JMP", "abs", "setc"); a.label("bw"); a.op("LDA", "imm", 0x0E)
        a.label("setc"); a.op("STA", "zp", TIA_W["COLUBK"])
        a.op("LDA", "abs", RIOT["SWCHA"]); a.op("STA", "zp", 0x85)
        a.op("BIT", "abs", RIOT["SWCHB"]); a.op("PHP"); a.op("PLA"); a.op("STA", "zp", 0x86)
        a.op("LDY", "imm", 200); a.label("line"); a.op("STA", "zp", TIA_W["WSYNC"]); a.op("DEY"); a.op("BNE", "rel", "line")
        a.op("JMP", "abs", "frame")
    return hand_rom(build)
