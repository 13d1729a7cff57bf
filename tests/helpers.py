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
