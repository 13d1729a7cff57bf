"""Pins for the oracle's TIA, cartridge and inputs: hand-assembled
programs with hand-derived rows.  y0 = 0 is used so that row == scanline and `back` can be read mid-frame."""
import numpy as np
import pytest

from helpers import oracle_for, run_instr, regs, TIA_W, TIA_R, RIOT
from oracle.ovcs_py import OracleVCS
from vcs_inputs import hand_rom

W = TIA_W


def sta(a, reg, v=None):
    if v is not None:
        a.op("LDA", "imm", v)
    a.op("STA", "zp", W[reg])


def run_to_line(o, line):
    while regs(o)["line"] < line:
        run_instr(o)


def prog(lines_fn, **kw):
    """program = setup on line 0, then WSYNC-separated lines; ends in a tight loop"""
    def build(a):
        a.org(0xF000); lines_fn(a); a.label("end"); a.op("JMP", "abs", "end")
    return oracle_for(build, y0=0, **kw)


def test_background_and_write_timing():
    # write COLUBK in cycle n=30 of line 1 -> first affected pixel x = 3*(n+1)-68 = 25 (C.4)
    def lines(a):
        sta(a, "WSYNC")                                   # line 1 starts
        for _ in range(13): a.op("NOP")                   # cycles 0..25
        sta(a, "COLUBK", 0x87)                            # LDA 26,27 ; STA 28,29,30 -> write in cycle 30
        sta(a, "WSYNC")
    o = prog(lines); run_to_line(o, 2)
    row = o.back(0)[1]
    assert (row[:25] == 0).all() and (row[25:] == 0x86).all()           # value & 0xFE


def test_playfield_bit_order_and_reflection():
    def lines(a):
        sta(a, "COLUPF", 0x0E); sta(a, "PF0", 0x10); sta(a, "PF1", 0x80); sta(a, "PF2", 0x01)
        sta(a, "WSYNC"); sta(a, "WSYNC")                 # line 1 drawn with REF=0
        sta(a, "CTRLPF", 0x01); sta(a, "WSYNC"); sta(a, "WSYNC")   # line 3 fully drawn with REF=1
    o = prog(lines); run_to_line(o, 4)
    b = o.back(0)
    lit = lambda row: set(np.nonzero(row)[0].tolist())
    left = set(range(0, 4)) | set(range(16, 20)) | set(range(48, 52))
    assert lit(b[1]) == left | {x + 80 for x in left}                    # copy
    assert lit(b[3]) == left | {159 - x for x in left}                   # mirror: PF0=0x10 -> x 156..159


def test_position_strobes_and_fresh():
    def lines(a):
        sta(a, "COLUP0", 0x1E); sta(a, "GRP0", 0xFF)
        sta(a, "WSYNC"); sta(a, "RESP0")                 # line 1: write in cycle 2 (HBLANK) -> pos 3
        sta(a, "RESBL"); sta(a, "RESM0")                 # still HBLANK -> 2, 2
        sta(a, "WSYNC"); sta(a, "WSYNC")                 # line 2 complete
        for _ in range(12): a.op("NOP")                  # line 3: cycles 0..23
        sta(a, "RESP0")                                  # write in cycle 26, x_now = 13 -> pos 18
        sta(a, "WSYNC"); sta(a, "WSYNC")                 # lines 3 (strobe line) and 4
    o = prog(lines); run_to_line(o, 2)
    d = o.debug(0); assert (d.posP0, d.posBL, d.posM0) == (3, 2, 2) and d.fresh == 0   # fresh cleared at line start
    run_to_line(o, 5)
    assert o.debug(0).posP0 == 18
    b = o.back(0)
    assert set(np.nonzero(b[2])[0]) == set(range(3, 11))
    assert set(np.nonzero(b[3])[0]) == set(range(3, 11))    # strobe line: old position until the strobe, no main copy after
    assert set(np.nonzero(b[4])[0]) == set(range(18, 26))


def test_nusiz_copies_sizes_reflect_vdel():
    def lines(a):
        sta(a, "COLUP0", 0x2E); sta(a, "COLUP1", 0x4E)
        sta(a, "WSYNC"); sta(a, "RESP0"); sta(a, "RESP1")           # P0 pos 3, P1 pos 3
        sta(a, "GRP0", 0b11010000); sta(a, "NUSIZ0", 0x03)           # three copies close: +0,+16,+32
        sta(a, "WSYNC"); sta(a, "WSYNC")                             # line 2
        sta(a, "NUSIZ0", 0x05); sta(a, "REFP0", 0x08)                # double size, reflected
        sta(a, "WSYNC"); sta(a, "WSYNC")                             # line 4
        sta(a, "NUSIZ0", 0x07); sta(a, "REFP0", 0x00)                # quad size
        sta(a, "WSYNC"); sta(a, "WSYNC")                             # line 6
        sta(a, "NUSIZ0", 0x00); sta(a, "VDELP0", 0x01)               # VDEL: old copy (0 until GRP1 written)
        sta(a, "WSYNC"); sta(a, "WSYNC")                             # line 8: nothing
        sta(a, "GRP1", 0x00)                                         # GRP0_old := GRP0_new
        sta(a, "WSYNC"); sta(a, "WSYNC")                             # line 10: 0b11010000 at pos 3
    o = prog(lines); run_to_line(o, 11); b = o.back(0)
    lit = lambda r: set(np.nonzero(b[r])[0].tolist())
    base = {3, 4, 6}                                                  # bits 7,6,4 -> d = 0,1,3
    assert lit(2) == base | {x + 16 for x in base} | {x + 32 for x in base}
    # reflected, double: bit b lit at d/2 == b -> bits 4,6,7 -> d in {8,9,12,13,14,15}
    assert lit(4) == {3 + d for d in (8, 9, 12, 13, 14, 15)}
    assert lit(6) == {3 + d for d in (0, 1, 2, 3, 4, 5, 6, 7, 12, 13, 14, 15)}      # quad: bits 7,6,4
    assert lit(8) == set() and lit(10) == base


def test_missile_ball_widths_and_resmp():
    def lines(a):
        sta(a, "COLUP0", 0x2E); sta(a, "COLUPF", 0x6E)
        sta(a, "WSYNC"); sta(a, "RESM0"); sta(a, "RESBL")            # both at 2
        sta(a, "NUSIZ0", 0x20); sta(a, "ENAM0", 0x02)                 # missile width 4
        sta(a, "CTRLPF", 0x30); sta(a, "ENABL", 0x02)                 # ball width 8 (same pixels, P0/M0 on top)
        sta(a, "WSYNC"); sta(a, "WSYNC")                              # line 2
        sta(a, "RESMP0", 0x02)                                        # missile hidden while locked
        sta(a, "WSYNC"); sta(a, "WSYNC")                              # line 4
        for _ in range(20): a.op("NOP")
        sta(a, "RESP0")                                               # line 5: cycle 40+2 -> x_now=3*43-68=61 -> pos 66
        sta(a, "RESMP0", 0x00)                                        # 1->0: posM0 = 66 + 4
        sta(a, "WSYNC"); sta(a, "WSYNC")                              # line 6
    o = prog(lines); run_to_line(o, 7); b = o.back(0)
    assert (b[2][2:6] == 0x2E).all() and (b[2][6:10] == 0x6E).all() and (b[2][10:] == 0).all()
    assert (b[4][2:10] == 0x6E).all()                                 # missile not drawn while RESMP=1
    assert o.debug(0).posP0 == 66 and o.debug(0).posM0 == 70
    assert (b[6][70:74] == 0x2E).all() and b[6][74] == 0 and b[6][69] == 0


@pytest.mark.parametrize("hm,shift", [(0x10, -1), (0xF0, +1), (0x80, +8), (0x70, -7), (0x00, 0)])
def test_hmove_direction_and_blank(hm, shift):
    def lines(a):
        sta(a, "COLUBK", 0x04); sta(a, "COLUP0", 0x2E); sta(a, "GRP0", 0x80)
        sta(a, "WSYNC")
        for _ in range(15): a.op("NOP")
        sta(a, "RESP0")                                   # cycle 30+2=32 -> x_now = 31 -> pos 36
        sta(a, "HMP0", hm)
        sta(a, "WSYNC"); sta(a, "HMOVE")                  # line 2, cycle 2: in HBLANK -> blank x 0..7
        sta(a, "WSYNC"); sta(a, "WSYNC")                  # line 3 complete, no blank
    o = prog(lines); run_to_line(o, 4); b = o.back(0)
    assert o.debug(0).posP0 == 36 + shift
    assert (b[2][:8] == 0).all() and (b[2][8:36 + shift] == 0x04).all() and b[2][36 + shift] == 0x2E
    assert (b[3][:8] == 0x04).all() and b[3][36 + shift] == 0x2E


def test_priority_score_pfp():
    # P0 at 3 (8 px), PF covers x 0..15 (PF0=0xF0), ball at 2..9; check one pixel per branch of the colour rule
    def lines(a):
        sta(a, "COLUBK", 0x02); sta(a, "COLUP0", 0x20); sta(a, "COLUP1", 0x40); sta(a, "COLUPF", 0x60)
        sta(a, "PF0", 0xF0); sta(a, "GRP0", 0xF0); sta(a, "GRP1", 0xFF)
        sta(a, "WSYNC"); sta(a, "RESP0"); sta(a, "RESP1")               # P0 pos 3 (x 3..6 lit), P1 pos 3 (x 3..10)
        sta(a, "WSYNC"); sta(a, "WSYNC")                                 # line 2: normal priority
        sta(a, "CTRLPF", 0x04); sta(a, "WSYNC"); sta(a, "WSYNC")         # line 4: PFP
        sta(a, "CTRLPF", 0x02); sta(a, "WSYNC"); sta(a, "WSYNC")         # line 6: SCORE
    o = prog(lines); run_to_line(o, 7); b = o.back(0)
    # normal: P0 > P1 > PF > BK
    assert b[2][4] == 0x20 and b[2][8] == 0x40 and b[2][12] == 0x60 and b[2][20] == 0x02 and b[2][84] == 0x60
    # PFP: PF on top of players where PF is lit; players elsewhere
    assert b[4][4] == 0x60 and b[4][12] == 0x60 and b[4][20] == 0x02
    # SCORE: left-half PF in COLUP0, right-half PF in COLUP1; players keep their colours
    assert b[6][12] == 0x20 and b[6][84] == 0x40 and b[6][8] == 0x20 and b[6][20] == 0x02


def test_collisions_latch_clear_and_vblank():
    def lines(a):
        sta(a, "PF0", 0xF0); sta(a, "GRP0", 0xFF); sta(a, "COLUP0", 0x20)
        sta(a, "VBLANK", 0x02)
        sta(a, "WSYNC"); sta(a, "RESP0"); sta(a, "WSYNC"); sta(a, "WSYNC")   # overlap under VBLANK: no latch
        a.op("LDA", "zp", TIA_R["CXP0FB"]); a.op("STA", "zp", 0x80)
        sta(a, "VBLANK", 0x00); sta(a, "WSYNC"); sta(a, "WSYNC")
        a.op("LDA", "zp", TIA_R["CXP0FB"]); a.op("STA", "zp", 0x81)
        a.op("LDA", "zp", TIA_R["CXPPMM"]); a.op("STA", "zp", 0x82)
        sta(a, "CXCLR"); a.op("LDA", "zp", TIA_R["CXP0FB"]); a.op("STA", "zp", 0x83)
    o = prog(lines)
    run_instr(o, 60)                                                  # runs into the final JMP loop
    ram = o.ram()[0]
    assert ram[0] == 0x00 and ram[1] == 0x80 and ram[2] == 0x00 and ram[3] == 0x00
    assert o.debug(0).cx == 1 << 4                                    # re-latched (P0.PF only) on the following lines


def test_collision_read_sees_pixels_up_to_its_own_cycle():
    # P0 at x 3..10 overlaps PF (x 0..15).  A CXP0FB read whose cycle ends before clock 68+3 sees 0.
    def lines(a):
        sta(a, "PF0", 0xF0); sta(a, "GRP0", 0xFF)
        sta(a, "WSYNC"); sta(a, "RESP0"); sta(a, "WSYNC")                # line 2 begins, fresh cleared
        sta(a, "CXCLR")                                                   # cycles 0,1,2
        for _ in range(9): a.op("NOP")                                    # cycles 3..20
        a.op("LDA", "zp", TIA_R["CXP0FB"])                                # cycles 21,22,23: read renders through clock 71 -> x 0..3
        a.op("STA", "zp", 0x80)
        a.op("LDX", "zp", TIA_R["CXP0FB"]); a.op("STX", "zp", 0x81)
    o = prog(lines); run_to_line(o, 2)
    run_instr(o, 14)
    ram = o.ram()[0]
    assert ram[0] == 0x80 and ram[1] == 0x80                             # x=3 is the first overlap pixel (clock 71)
    # same program with one NOP fewer: read in cycle 21 renders through clock 65 only -> no overlap yet
    def lines2(a):
        sta(a, "PF0", 0xF0); sta(a, "GRP0", 0xFF)
        sta(a, "WSYNC"); sta(a, "RESP0"); sta(a, "WSYNC")
        sta(a, "CXCLR")
        for _ in range(8): a.op("NOP")
        a.op("LDA", "zp", TIA_R["CXP0FB"]); a.op("STA", "zp", 0x80)
    o = prog(lines2); run_to_line(o, 2); run_instr(o, 11)
    assert o.ram()[0][0] == 0x00


def test_f8_hotspots_by_read_write_and_dummy_read():
    b0 = bytearray([0x00]) * 4096; b1 = bytearray([0x11]) * 4096
    def build(a):
        a.org(0xF000)
        a.op("LDA", "abs", 0xFFF8); a.op("STA", "zp", 0x80)       # read hotspot: returns the new bank's byte
        a.op("STA", "abs", 0xFFF9); a.op("LDA", "abs", 0xF800); a.op("STA", "zp", 0x81)
        a.op("LDX", "imm", 0x01); a.op("LDA", "abx", 0xFFF7)       # operand read @ $FFF8 -> bank 0
        a.op("LDA", "abs", 0xF800); a.op("STA", "zp", 0x82)
        a.op("LDX", "imm", 0xFA); a.op("LDA", "abx", 0xFEFF)       # dummy read @ $FEF9, real read @ $FFF9 -> bank 1
        a.op("LDA", "abs", 0xF800); a.op("STA", "zp", 0x83)
        a.label("end"); a.op("JMP", "abs", "end")
    code = hand_rom(build)
    n = 0x60
    for b, fillv in ((b0, 0xA0), (b1, 0xB1)):
        b[:n] = code[:n]; b[0xFFC:] = code[0xFFC:]; b[0x800] = fillv; b[0xFF8] = fillv + 1; b[0xFF9] = fillv + 2
    o = OracleVCS([bytes(b0 + b1)], np.array([5], dtype=np.uint64))
    assert regs(o)["bank"] == 1                                    # cfg.f8_start_bank default [R]
    for _ in range(14): run_instr(o)
    ram = o.ram()[0]
    assert ram[0] == 0xA1            # LDA $FFF8 switched to bank 0 before returning data
    assert ram[1] == 0xB1 and ram[2] == 0xA0 and ram[3] == 0xB1
    assert regs(o)["bank"] == 1


def test_actions_to_pins_and_fire_latch():
    def build(a):
        a.org(0xF000)
        a.op("LDA", "abs", RIOT["SWCHA"]); a.op("STA", "zp", 0x80)
        a.op("LDA", "zp", TIA_R["INPT4"]); a.op("STA", "zp", 0x81)
        a.op("LDA", "abs", RIOT["SWCHB"]); a.op("STA", "zp", 0x82)
        a.op("JMP", "abs", 0xF000)
    want = {0: (0xFF, 0x80), 1: (0xFF, 0x00), 2: (0xEF, 0x80), 3: (0x7F, 0x80), 4: (0xBF, 0x80), 5: (0xDF, 0x80),
            6: (0x6F, 0x80), 7: (0xAF, 0x80), 8: (0x5F, 0x80), 9: (0x9F, 0x80), 10: (0xEF, 0x00), 11: (0x7F, 0x00),
            12: (0xBF, 0x00), 13: (0xDF, 0x00), 14: (0x6F, 0x00), 15: (0xAF, 0x00), 16: (0x5F, 0x00), 17: (0x9F, 0x00),
            18: (0xFF, 0x80), 255: (0xFF, 0x80)}
    o = oracle_for(build)
    for act, (swcha, inpt4) in want.items():
        o.set_action(0, act); run_instr(o, 7)
        ram = o.ram()[0]; assert (ram[0], ram[1], ram[2]) == (swcha, inpt4, 0x3F), act
    # latched mode: a press drops the latch until VBLANK bit 6 is cleared
    def build2(a):
        a.org(0xF000); sta(a, "VBLANK", 0x40)
        a.op("LDA", "zp", TIA_R["INPT4"]); a.op("STA", "zp", 0x80)
        a.op("LDA", "zp", TIA_R["INPT4"]); a.op("STA", "zp", 0x81)
        sta(a, "VBLANK", 0x00); a.op("LDA", "zp", TIA_R["INPT4"]); a.op("STA", "zp", 0x82)
    o = oracle_for(build2); run_instr(o, 2)
    o.set_action(0, 1); run_instr(o, 2); o.set_action(0, 0); run_instr(o, 2); run_instr(o, 4)
    ram = o.ram()[0]; assert (ram[0], ram[1], ram[2]) == (0x00, 0x00, 0x80)


def test_riot_port_direction_registers():
    def build(a):
        a.org(0xF000)
        a.op("LDA", "imm", 0xF0); a.op("STA", "abs", RIOT["SWACNT"]); a.op("LDA", "imm", 0x5A); a.op("STA", "abs", RIOT["SWCHA"])
        a.op("LDA", "abs", RIOT["SWCHA"]); a.op("STA", "zp", 0x80); a.op("LDA", "abs", RIOT["SWACNT"]); a.op("STA", "zp", 0x81)
    o = oracle_for(build); o.set_action(0, 3); run_instr(o, 8)            # RIGHT: ina = 0x7F
    ram = o.ram()[0]; assert ram[0] == (0x5A & 0xF0) | (0x7F & 0x0F) and ram[1] == 0xF0
