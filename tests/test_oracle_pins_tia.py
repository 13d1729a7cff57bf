"""More pins for the oracle's TIA: every collision latch and its place in the read map, missile
copies and `fresh`, VDELBL / ENABL_old, HMOVE on all five objects + HMCLR, RESMP with double / quad players, the
player-1 / missile-1 strobes, INPT5, sprites wrapping at the right edge.  Every expectation below is derived by hand
from the C.8 text (register map, position constants 3 / +5 and 2 / +4, copy offsets O(m), HM sign convention), none is
produced by running anything.  y0 = 0, so row == scanline and `back` can be read mid-frame."""
import numpy as np
import pytest

from helpers import oracle_for, run_instr, regs, TIA_W, TIA_R

W = TIA_W


def sta(a, reg, v=None):
    if v is not None:
        a.op("LDA", "imm", v)
    a.op("STA", "zp", W[reg])


def prog(lines_fn, **kw):
    def build(a):
        a.org(0xF000); lines_fn(a); a.label("end"); a.op("JMP", "abs", "end")
    return oracle_for(build, y0=0, **kw)


def run_to_line(o, line):
    while regs(o)["line"] < line:
        run_instr(o)


def run_to_end(o, limit=4000):
    """until the program sits in its final `JMP end` loop"""
    last = -1
    for _ in range(limit):
        run_instr(o)
        pc = int(regs(o)["pc"])
        if pc == last:
            return
        last = pc
    raise AssertionError("program did not reach its end loop")


def lit(row):
    return set(np.nonzero(row)[0].tolist())


# ---------------------------------------------------------------------------------------------- collisions
# C.8 read map, typed out by hand: register index -> (pair behind bit 7, pair behind bit 6)
READ_MAP = {
    0: (("M0", "P1"), ("M0", "P0")),      # CXM0P
    1: (("M1", "P0"), ("M1", "P1")),      # CXM1P
    2: (("P0", "PF"), ("P0", "BL")),      # CXP0FB
    3: (("P1", "PF"), ("P1", "BL")),      # CXP1FB
    4: (("M0", "PF"), ("M0", "BL")),      # CXM0FB
    5: (("M1", "PF"), ("M1", "BL")),      # CXM1FB
    6: (("BL", "PF"), None),              # CXBLPF
    7: (("P0", "P1"), ("M0", "M1")),      # CXPPMM
}
OBJECTS = ["P0", "P1", "M0", "M1", "BL", "PF"]
PAIRS = [(OBJECTS[i], OBJECTS[j]) for i in range(6) for j in range(i + 1, 6)]
ENABLE = {"P0": ("GRP0", 0xFF), "P1": ("GRP1", 0xFF), "M0": ("ENAM0", 0x02), "M1": ("ENAM1", 0x02),
          "BL": ("ENABL", 0x02), "PF": ("PF0", 0xF0)}


def test_the_read_map_names_each_of_the_15_pairs_once():
    named = [frozenset(p) for pairs in READ_MAP.values() for p in pairs if p]
    assert len(named) == 15 and len(set(named)) == 15 and set(named) == {frozenset(p) for p in PAIRS}


@pytest.mark.parametrize("pair", PAIRS, ids=["".join(p) for p in PAIRS])
def test_each_collision_latch_alone_and_where_it_reads(pair):
    """Players at x 3..10, missiles and ball (8 wide) at x 2..9, playfield x 0..15: any two of them overlap at x 3..9.
    Exactly the two objects of `pair` are switched on; all eight CXxx registers are read; one bit may be set."""
    def lines(a):
        sta(a, "NUSIZ0", 0x30); sta(a, "NUSIZ1", 0x30); sta(a, "CTRLPF", 0x30)           # missiles / ball 8 clocks wide
        sta(a, "WSYNC")
        for r in ("RESP0", "RESP1", "RESM0", "RESM1", "RESBL"): sta(a, r)                 # writes in cycles 2..14: HBLANK -> 3,3,2,2,2
        sta(a, "WSYNC")
        sta(a, "CXCLR")
        for ob in pair: sta(a, *ENABLE[ob])
        sta(a, "WSYNC"); sta(a, "WSYNC")                                                  # one complete line with both on
        for r in range(8):
            a.op("LDA", "zp", r); a.op("STA", "zp", 0x80 + r)
    o = prog(lines); run_to_end(o)
    d = o.debug(0)
    assert (d.posP0, d.posP1, d.posM0, d.posM1, d.posBL) == (3, 3, 2, 2, 2)
    got = o.ram()[0][:8].tolist()
    want = [0] * 8
    for r, (p7, p6) in READ_MAP.items():
        if p7 and frozenset(p7) == frozenset(pair): want[r] = 0x80
        if p6 and frozenset(p6) == frozenset(pair): want[r] = 0x40
    assert sum(1 for v in want if v) == 1
    assert got == want, (pair, [hex(v) for v in got])
    assert bin(d.cx).count("1") == 1                                                      # one latch, whatever its internal number


def test_all_objects_on_sets_all_15_and_low_bits_read_zero():
    def lines(a):
        sta(a, "NUSIZ0", 0x30); sta(a, "NUSIZ1", 0x30); sta(a, "CTRLPF", 0x30)
        sta(a, "WSYNC")
        for r in ("RESP0", "RESP1", "RESM0", "RESM1", "RESBL"): sta(a, r)
        sta(a, "WSYNC")
        for ob in OBJECTS: sta(a, *ENABLE[ob])
        sta(a, "WSYNC"); sta(a, "WSYNC")
        for r in range(16):
            a.op("LDA", "zp", r); a.op("STA", "zp", 0x80 + r)
    o = prog(lines); run_to_end(o)
    got = o.ram()[0][:16].tolist()
    assert got[:8] == [0xC0, 0xC0, 0xC0, 0xC0, 0xC0, 0xC0, 0x80, 0xC0]                    # CXBLPF has no bit 6
    assert got[8:12] == [0, 0, 0, 0]                                                       # INPT0-3: no paddles [R]
    assert got[12] == 0x80 and got[13] == 0x80 and got[14:] == [0, 0]                      # INPT4 / INPT5 released; E, F read 0


# ---------------------------------------------------------------------------------------------- missiles
COPIES = {0: [0], 1: [0, 16], 2: [0, 32], 3: [0, 16, 32], 4: [0, 64], 5: [0], 6: [0, 32, 64], 7: [0]}      # O(m), C.8 [D]


@pytest.mark.parametrize("p", [0, 1])
@pytest.mark.parametrize("mode,wcode", [(0, 0), (1, 1), (2, 2), (3, 0), (4, 3), (5, 1), (6, 2), (7, 3)])
def test_missile_copies_widths_fresh_for_both_missiles(p, mode, wcode):
    colour = (0x2E, 0x4E)[p]
    def lines(a):
        sta(a, "COLUP0", 0x2E); sta(a, "COLUP1", 0x4E); sta(a, "WSYNC")
        sta(a, f"RESM{p}")                                                                 # line 1, cycle 2 -> pos 2
        sta(a, f"NUSIZ{p}", (wcode << 4) | mode); sta(a, f"ENAM{p}", 0x02); sta(a, "WSYNC")
        sta(a, "WSYNC")                                                                    # line 2: every copy
        sta(a, f"RESM{p}"); sta(a, "WSYNC")                                                # line 3: strobe line, main copy held back
        sta(a, "WSYNC")                                                                    # line 4: every copy again
    o = prog(lines); run_to_line(o, 5); b = o.back(0)
    w = 1 << wcode
    full = {2 + off + k for off in COPIES[mode] for k in range(w)}
    extra = {2 + off + k for off in COPIES[mode] if off for k in range(w)}
    assert lit(b[2]) == full and lit(b[4]) == full
    assert lit(b[3]) == extra                                                              # fresh: no main copy on the strobe line
    assert all(b[2][x] == colour for x in full)
    assert (o.debug(0).posM0, o.debug(0).posM1)[p] == 2


def test_missile_needs_enam_and_m1_uses_nusiz1():
    def lines(a):
        sta(a, "COLUP1", 0x4E); sta(a, "WSYNC")
        sta(a, "RESM1"); sta(a, "NUSIZ0", 0x33); sta(a, "NUSIZ1", 0x10); sta(a, "ENAM1", 0x02); sta(a, "WSYNC")
        sta(a, "WSYNC")                                                                    # line 2: M1 two clocks wide, one copy (NUSIZ0 is not its register)
        sta(a, "ENAM1", 0x00); sta(a, "ENAM0", 0x02); sta(a, "COLUP0", 0x2E); sta(a, "WSYNC")
        sta(a, "WSYNC")                                                                    # line 4: M1 off; M0 (pos 0 since reset) 8 wide x 3 copies close
    o = prog(lines); run_to_line(o, 5); b = o.back(0)
    assert lit(b[2]) == {2, 3} and b[2][2] == 0x4E
    assert lit(b[4]) == {k + off for off in (0, 16, 32) for k in range(8)} and b[4][0] == 0x2E


# ---------------------------------------------------------------------------------------------- ball
def test_vdelbl_and_the_grp1_copy_of_enabl():
    def lines(a):
        sta(a, "COLUPF", 0x6E); sta(a, "CTRLPF", 0x10); sta(a, "WSYNC")                    # ball 2 clocks wide
        sta(a, "RESBL"); sta(a, "ENABL", 0x02); sta(a, "WSYNC")                            # line 1: pos 2, ENABL_new = 1
        sta(a, "WSYNC")                                                                    # line 2: lit
        sta(a, "VDELBL", 0x01); sta(a, "WSYNC"); sta(a, "WSYNC")                           # line 4: delayed copy (still 0) -> dark
        sta(a, "GRP0", 0x00); sta(a, "WSYNC"); sta(a, "WSYNC")                             # line 6: a GRP0 write copies nothing of the ball
        sta(a, "GRP1", 0x00); sta(a, "WSYNC"); sta(a, "WSYNC")                             # line 8: GRP1 write: ENABL_old := ENABL_new = 1 -> lit
        sta(a, "ENABL", 0x00); sta(a, "WSYNC"); sta(a, "WSYNC")                            # line 10: new = 0, old = 1 -> still lit
        sta(a, "GRP1", 0x00); sta(a, "WSYNC"); sta(a, "WSYNC")                             # line 12: old := 0 -> dark
        sta(a, "VDELBL", 0x00); sta(a, "ENABL", 0x02); sta(a, "WSYNC"); sta(a, "WSYNC")    # line 14: undelayed again -> lit
    o = prog(lines); run_to_line(o, 15); b = o.back(0)
    on = {2, 3}
    assert [lit(b[r]) for r in (2, 4, 6, 8, 10, 12, 14)] == [on, set(), set(), on, on, set(), on]
    assert b[2][2] == 0x6E


def test_resbl_restarts_the_ball_on_the_strobe_line():
    def lines(a):
        sta(a, "COLUPF", 0x6E); sta(a, "CTRLPF", 0x30); sta(a, "ENABL", 0x02); sta(a, "WSYNC")
        for _ in range(12): a.op("NOP")                                                    # cycles 0..23
        sta(a, "RESBL")                                                                    # write in cycle 26: x_now = 13 -> pos 17
        sta(a, "WSYNC"); sta(a, "WSYNC")
    o = prog(lines); run_to_line(o, 3); b = o.back(0)
    assert o.debug(0).posBL == 17
    # strobe line (1): the old position 0 shows x 0..7 (all before x_now = 13), and the ball restarts at 17 at once (no `fresh` for the ball)
    assert lit(b[1]) == set(range(0, 8)) | set(range(17, 25))
    assert lit(b[2]) == set(range(17, 25))


# ---------------------------------------------------------------------------------------------- HMOVE
def test_hmove_moves_all_five_objects_by_their_own_hm_and_hmclr_zeroes_them():
    def lines(a):
        sta(a, "WSYNC")
        for _ in range(15): a.op("NOP")                                                    # line 1, cycles 0..29
        for r in ("RESP0", "RESP1", "RESM0", "RESM1", "RESBL"): sta(a, r)                  # writes in cycles 32, 35, 38, 41, 44
        sta(a, "HMP0", 0x10); sta(a, "HMP1", 0xF0); sta(a, "HMM0", 0x70); sta(a, "HMM1", 0x80); sta(a, "HMBL", 0x20)
        sta(a, "WSYNC"); a.op("NOP"); sta(a, "HMOVE")                                      # line 2 (the NOP's fetch is the line's first cycle)
        sta(a, "WSYNC"); a.op("NOP"); sta(a, "HMOVE")                                      # line 3: the same shifts once more
        sta(a, "WSYNC"); a.op("NOP"); sta(a, "HMCLR"); sta(a, "HMOVE")                     # line 4: all HM = 0 -> nothing moves
        sta(a, "WSYNC"); a.op("NOP")
    o = prog(lines)
    pos = lambda: (o.debug(0).posP0, o.debug(0).posP1, o.debug(0).posM0, o.debug(0).posM1, o.debug(0).posBL)
    run_to_line(o, 2)
    # x_now = 3 (n + 1) - 68 = 31, 40, 49, 58, 67 ; players + 5, missiles / ball + 4
    assert pos() == (36, 45, 53, 62, 71)
    run_instr(o)                                                                           # HMOVE #1: 1 left, 1 right, 7 left, 8 right, 2 left
    assert pos() == (35, 46, 46, 70, 69) and o.debug(0).hmove_blank == 1
    run_to_line(o, 3); run_instr(o)
    assert pos() == (34, 47, 39, 78, 67)
    run_to_line(o, 4); run_instr(o, 2)
    assert pos() == (34, 47, 39, 78, 67)
    run_to_line(o, 5)
    assert o.debug(0).hmove_blank == 0                                                     # the comb lasts for its own line only


def test_hmove_wraps_positions_mod_160():
    def lines(a):
        sta(a, "WSYNC")
        sta(a, "RESM0"); sta(a, "RESBL")                                                   # line 1: HBLANK -> 2, 2
        for _ in range(32): a.op("NOP")                                                    # cycles 6..69
        sta(a, "RESP0")                                                                    # write in cycle 72: x_now = 151 -> pos 156
        sta(a, "WSYNC")
        sta(a, "HMM0", 0x70); sta(a, "HMBL", 0x30); sta(a, "HMP0", 0x80)                   # 7 left, 3 left, 8 right
        sta(a, "WSYNC"); sta(a, "HMOVE"); sta(a, "WSYNC")
    o = prog(lines); run_to_line(o, 2)
    assert (o.debug(0).posP0, o.debug(0).posM0, o.debug(0).posBL) == (156, 2, 2)
    run_to_line(o, 4)
    assert (o.debug(0).posP0, o.debug(0).posM0, o.debug(0).posBL) == ((156 + 8) % 160, (2 - 7) % 160, (2 - 3) % 160) == (4, 155, 159)


def test_hmove_in_the_visible_part_moves_without_blank():
    def lines(a):
        sta(a, "COLUBK", 0x04); sta(a, "HMP0", 0x20); sta(a, "WSYNC")
        for _ in range(12): a.op("NOP")
        sta(a, "HMOVE")                                                                    # write in cycle 26: x_now = 13 >= 0
        sta(a, "WSYNC")
    o = prog(lines); run_to_line(o, 2)
    assert o.debug(0).posP0 == (0 - 2) % 160 and (o.back(0)[1] == 0x04).all()              # shifted at once [R], no comb


# ---------------------------------------------------------------------------------------------- RESMP, player 1 / missile 1 strobes
@pytest.mark.parametrize("p", [0, 1])
@pytest.mark.parametrize("mode,mid", [(0, 4), (5, 8), (7, 16), (3, 4)])
def test_resmp_snaps_the_missile_to_its_players_middle(p, mode, mid):
    def lines(a):
        sta(a, "WSYNC")
        for _ in range(20): a.op("NOP")                                                    # cycles 0..39
        sta(a, f"RESP{p}")                                                                 # write in cycle 42: x_now = 61 -> pos 66
        sta(a, "WSYNC")
        sta(a, f"NUSIZ{p}", mode); sta(a, f"RESMP{p}", 0x02); sta(a, f"RESMP{p}", 0x00)
    o = prog(lines); run_to_end(o)
    d = o.debug(0)
    assert (d.posP0, d.posP1)[p] == 66 and (d.posM0, d.posM1)[p] == 66 + mid
    assert (d.posM0, d.posM1)[1 - p] == 0                                                  # the other missile is not touched


def test_resmp_0_to_0_and_1_to_1_do_not_move_the_missile():
    def lines(a):
        sta(a, "WSYNC"); sta(a, "RESP0")                                                   # P0 -> 3
        for _ in range(12): a.op("NOP")
        sta(a, "RESM0")                                                                    # NOPs in cycles 3..26, write in 29: x_now = 22 -> 26
        sta(a, "RESMP0", 0x00); sta(a, "RESMP0", 0x02); sta(a, "RESMP0", 0x02)
    o = prog(lines); run_to_end(o)
    assert o.debug(0).posM0 == 26                                                          # only the 1 -> 0 edge snaps [R]


def test_player1_missile1_strobe_constants():
    def lines(a):
        sta(a, "WSYNC"); sta(a, "RESP1"); sta(a, "RESM1")                                  # cycles 2, 5: HBLANK -> 3, 2
        sta(a, "WSYNC")
        for _ in range(12): a.op("NOP")
        sta(a, "RESP1"); sta(a, "RESM1")                                                   # cycles 26, 29: x_now = 13, 22 -> 18, 26
        sta(a, "WSYNC")
    o = prog(lines); run_to_line(o, 2)
    assert (o.debug(0).posP1, o.debug(0).posM1) == (3, 2) and (o.debug(0).posP0, o.debug(0).posM0) == (0, 0)
    run_to_line(o, 3)
    assert (o.debug(0).posP1, o.debug(0).posM1) == (18, 26)


def test_last_strobe_cycles_of_hblank_and_first_visible_one():
    # x_now = 3 (n + 1) - 68 is still negative for a write in cycle n = 21 (-2) and is 1 for n = 22
    def lines(a):
        sta(a, "WSYNC"); a.op("LDA", "zp", 0x80)                                           # 3 cycles: 0..2
        for _ in range(8): a.op("NOP")                                                     # 3..18
        sta(a, "RESP0"); sta(a, "RESBL"); sta(a, "WSYNC")                                  # writes in cycles 21, 24: x_now = -2 -> 3 ; 7 -> 11
    o = prog(lines); run_to_line(o, 2); assert (o.debug(0).posP0, o.debug(0).posBL) == (3, 11)
    def lines(a):
        sta(a, "WSYNC")
        for _ in range(10): a.op("NOP")                                                    # 0..19
        sta(a, "RESP0"); sta(a, "WSYNC")                                                   # write in cycle 22: x_now = 1 -> 6
    o = prog(lines); run_to_line(o, 2); assert o.debug(0).posP0 == 6


@pytest.mark.parametrize("reg,field,want74,want75", [("RESP0", "posP0", 2, 5), ("RESP1", "posP1", 2, 5), ("RESM0", "posM0", 1, 4),
                                                     ("RESM1", "posM1", 1, 4), ("RESBL", "posBL", 1, 4)])
def test_strobes_in_the_last_two_cycles_of_a_line_wrap_mod_160(reg, field, want74, want75):
    # cycle 74: x_now = 157 -> players 162 % 160 = 2, missiles / ball 161 % 160 = 1 ; cycle 75: x_now = 160 -> 5 / 4
    def lines(a):
        sta(a, "WSYNC")
        for _ in range(36): a.op("NOP")                                                    # cycles 0..71
        sta(a, reg)                                                                        # write in cycle 74
        a.op("NOP")
    o = prog(lines); run_to_end(o); assert getattr(o.debug(0), field) == want74
    def lines(a):
        sta(a, "WSYNC"); a.op("LDA", "zp", 0x80)                                           # cycles 0..2
        for _ in range(35): a.op("NOP")                                                    # 3..72
        sta(a, reg)                                                                        # write in cycle 75
        a.op("NOP")
    o = prog(lines); run_to_end(o); assert getattr(o.debug(0), field) == want75


# ---------------------------------------------------------------------------------------------- right-edge wrap
def test_sprites_wrap_at_the_right_edge():
    def lines(a):
        sta(a, "COLUP0", 0x2E); sta(a, "GRP0", 0xFF); sta(a, "NUSIZ0", 0x30); sta(a, "WSYNC")
        for _ in range(34): a.op("NOP")                                                    # cycles 0..67
        a.op("LDA", "imm", 0x02)                                                           # 68, 69
        sta(a, "RESP0")                                                                    # write in cycle 72: x_now = 151 -> 156
        sta(a, "WSYNC"); sta(a, "WSYNC")                                                   # line 2: P0 only
        sta(a, "GRP0", 0x00); sta(a, "ENAM0", 0x02)
        for _ in range(28): a.op("NOP")                                                    # line 3: cycles 10..65
        a.op("LDA", "zp", 0x80)                                                            # 66..68
        sta(a, "RESM0")                                                                    # write in cycle 71: x_now = 148 -> 152
        sta(a, "WSYNC"); sta(a, "WSYNC")                                                   # line 4: M0 only, 8 wide
    o = prog(lines); run_to_line(o, 5); b = o.back(0)
    assert o.debug(0).posP0 == 156 and o.debug(0).posM0 == 152
    assert lit(b[2]) == {156, 157, 158, 159, 0, 1, 2, 3}
    assert lit(b[4]) == set(range(152, 160))
    # a three-copy player whose last copy wraps: pos 156, copies at +16, +32 -> 172 % 160 = 12, 188 % 160 = 28
    def lines2(a):
        sta(a, "COLUP0", 0x2E); sta(a, "GRP0", 0x81); sta(a, "NUSIZ0", 0x03); sta(a, "WSYNC")
        for _ in range(34): a.op("NOP")
        a.op("LDA", "imm", 0x02)
        sta(a, "RESP0"); sta(a, "WSYNC"); sta(a, "WSYNC")
    o = prog(lines2); run_to_line(o, 3); b = o.back(0)
    assert lit(b[2]) == {156, 163 % 160, 12, 19, 28, 35}


# ---------------------------------------------------------------------------------------------- INPT5
def test_inpt5_is_never_pressed_latched_or_not():
    def build(a):
        a.org(0xF000)
        a.op("LDA", "zp", TIA_R["INPT5"]); a.op("STA", "zp", 0x80)
        sta(a, "VBLANK", 0x40)                                                             # latched mode
        a.op("LDA", "zp", TIA_R["INPT5"]); a.op("STA", "zp", 0x81)
        a.op("LDA", "zp", TIA_R["INPT4"]); a.op("STA", "zp", 0x82)
        a.op("LDA", "zp", TIA_R["INPT5"]); a.op("STA", "zp", 0x83)
        a.label("end"); a.op("JMP", "abs", "end")
    o = oracle_for(build); run_instr(o, 6)
    o.set_action(0, 1)                                                                     # FIRE: drops INPT4's latch only
    run_instr(o, 6)
    assert o.ram()[0][:4].tolist() == [0x80, 0x80, 0x00, 0x80]
