"""CPU-only checks of the boundary: libvcsb200.so loads, exports every symbol include/vcs.h declares, its
decode table matches the documented opcode matrix, and host-side validation answers before any launch."""
import ctypes as C
import re
import os

import numpy as np

from helpers import load_opcode_matrix, load_undocumented

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _lib():
    import __graft_entry__ as g
    g.build()
    from paper_2606_22447_b200 import load_library
    return load_library()


def test_library_exports_every_declared_symbol():
    L = _lib()
    hdr = open(os.path.join(ROOT, "include", "vcs.h")).read()
    declared = set(re.findall(r"\b(vcs_[a-z_0-9]+)\s*\(", hdr))
    from paper_2606_22447_b200 import EXPORTS
    assert declared == set(EXPORTS), declared ^ set(EXPORTS)
    for name in declared:
        assert hasattr(L, name), name


def test_decode_table_matches_documented_matrix():
    from paper_2606_22447_b200 import optable
    tab = optable()
    matrix = load_opcode_matrix()
    modes = ["imp", "acc", "imm", "zp", "zpx", "zpy", "abs", "abx", "aby", "izx", "izy", "rel", "spc"]
    ops = ["ILL", "LDA", "LDX", "LDY", "AND", "ORA", "EOR", "ADC", "SBC", "CMP", "CPX", "CPY", "BIT", "LAX", "NOPR",
           "STA", "STX", "STY", "SAX", "ASL", "LSR", "ROL", "ROR", "INC", "DEC", "CLC", "SEC", "CLD", "SED", "CLI", "SEI", "CLV", "NOP", "DEX", "DEY",
           "INX", "INY", "TAX", "TAY", "TSX", "TXA", "TYA", "TXS", "BPL", "BMI", "BVC", "BVS", "BCC", "BCS", "BNE", "BEQ",
           "JMP", "JMPI", "JSR", "RTS", "RTI", "PHA", "PHP", "PLA", "PLP", "BRK"]
    special = {"JMP", "JMPI", "JSR", "RTS", "RTI", "PHA", "PHP", "PLA", "PLP", "BRK"}
    stores, rmws = {"STA", "STX", "STY", "SAX"}, {"ASL", "LSR", "ROL", "ROR", "INC", "DEC"}
    undoc = load_undocumented()
    n_doc = 0
    for code in range(256):
        ent = int(tab[code]); mode, op, kind = modes[ent & 15], ops[(ent >> 4) & 63], ent >> 10
        if code in undoc:
            mn, mmode, _, _ = undoc[code]
            if mn == "NOP" and mmode != "imp": mn = "NOPR"
        elif code not in matrix:
            assert op == "ILL", hex(code); continue
        else:
            n_doc += 1
            mn, mmode, _, _ = matrix[code]
        if mn == "JMP" and mmode == "ind": mn = "JMPI"
        assert op == mn, (hex(code), op, mn)
        if op in special: assert mode == "spc"
        else: assert mode == mmode, (hex(code), mode, mmode)
        want_kind = 2 if op in stores else 3 if (op in rmws and mode != "acc") else 0 if (mode in ("imp", "acc", "rel", "spc")) else 1
        assert kind == want_kind, (hex(code), op, mode, kind)
    assert n_doc == 151


def test_host_side_validation_without_gpu():
    L = _lib()
    from paper_2606_22447_b200.binding import VcsRom, VcsConfig
    h = C.c_void_p()
    seeds = np.zeros(1, np.uint64)
    buf = (C.c_uint8 * 1000)()
    rom = (VcsRom * 1)(); rom[0].data = C.cast(buf, C.POINTER(C.c_uint8)); rom[0].size = 1000
    assert L.vcs_create(C.byref(h), 1, rom, 1, None, seeds.ctypes.data, None) == -4          # VCS_EROM
    assert L.vcs_create(C.byref(h), 0, rom, 1, None, seeds.ctypes.data, None) == -1          # VCS_EINVAL
    assert L.vcs_create(None, 1, rom, 1, None, seeds.ctypes.data, None) == -1
    rom[0].size = 2048
    big = (C.c_uint8 * 2048)(); rom[0].data = C.cast(big, C.POINTER(C.c_uint8))
    bad = VcsConfig(1, 320, 1, 0)
    assert L.vcs_create(C.byref(h), 1, rom, 1, None, seeds.ctypes.data, C.byref(bad)) == -1   # y0 < 2
    er = np.array([3], np.int32)
    assert L.vcs_create(C.byref(h), 1, rom, 1, er.ctypes.data, seeds.ctypes.data, None) == -1
    assert L.vcs_step(None, None, 4, None) == -1 and L.vcs_destroy(None) == -1
    assert L.vcs_last_error(None) == b""
    import torch
    if not torch.cuda.is_available():                                                           # no CPU fallback
        assert L.vcs_create(C.byref(h), 1, rom, 1, None, seeds.ctypes.data, None) == -2        # VCS_ECUDA
        from paper_2606_22447_b200 import VCS, VcsError
        try:
            VCS([bytes(2048)], seeds); raise AssertionError("must fail loudly without a GPU")
        except VcsError:
            pass
