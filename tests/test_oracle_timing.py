"""Pins for the oracle's clocking: 3 colour clocks per CPU cycle,
76-cycle / 228-clock lines, WSYNC, the RIOT timer against its closed form, frame ends and the cap."""
import numpy as np
import pytest

from helpers import oracle_for, run_instr, regs, TIA_W, RIOT
from oracle.ovcs_py import OracleVCS
from vcs_inputs import make_workload


def test_three_clocks_per_cycle_and_76_cycle_lines():
    w = make_workload(2, batch=1)
    o = OracleVCS(w.roms, w.seeds)
    last_line, last_cyc = 0, 0
    for i in range(4000):
        run_instr(o)
        r, d = regs(o), o.debug(0)
        assert d.clocks_rendered == 3 * int(r["cycles"])             # PAPER.md L21 "cycle by cycle"; 3:1
        assert int(r["cyc_in_line"]) == int(r["cycles"]) % 76         # the beam is never re-phased
    # line counter: +1 per 76 cycles between frame ends
    o = OracleVCS(w.roms, w.seeds)
    for _ in range(300):
        o.tick(0)
    r = regs(o)
    assert r["cycles"] == 300 and r["line"] == (300 - 1) // 76       # line k covers cycles 76k..76k+75


@pytest.mark.parametrize("k", list(range(0, 74)))
def test_wsync_resumes_at_line_start(k):
    def build(a):
        a.org(0xF000); a.op("STA", "zp", TIA_W["WSYNC"]); a.op("NOP"); a.op("NOP")
    o = oracle_for(build)
    for _ in range(k):
        o.tick(0)                                                    # STA WSYNC then writes in cycle n = k + 2
    run_instr(o)                                                     # the store itself is never stalled
    assert regs(o)["cycles"] == k + 3 and o.debug(0).wsync == (1 if k + 2 < 75 else 1)
    run_instr(o)                                                     # NOP: fetch must be cycle 0 of the next line
    r = regs(o)
    assert r["cycles"] == 76 + 2 and r["cyc_in_line"] == 2 and r["line"] == 1
    assert o.debug(0).wsync == 0
    if k + 2 == 75:
        assert True                                                  # write in cycle 75: zero stall cycles (76 = k+3)


def test_wsync_does_not_stall_write_cycles():
    # RMW on WSYNC: R old (sets nothing), W old -> wsync, W new must run unstalled; next read stalls
    def build(a):
        a.org(0xF000); a.op("INC", "zp", TIA_W["WSYNC"]); a.op("NOP")
    o = oracle_for(build)
    run_instr(o); assert regs(o)["cycles"] == 5
    run_instr(o); assert regs(o)["cycles"] == 78


SHIFT = {"TIM1T": 0, "TIM8T": 3, "TIM64T": 6, "T1024T": 10}


def _closed_form(N, shift, dt):
    """value, flag at dt = c - c0 >= 1 cycles after the write (C.7 closed form)."""
    D = 1 << shift
    cu = 1 + N * D
    if dt < cu:
        return N - 1 - ((dt - 1) >> shift), 0
    return (0xFF - (dt - cu)) & 0xFF, 1


@pytest.mark.parametrize("reg", list(SHIFT))
@pytest.mark.parametrize("N", [0, 1, 2, 3, 5, 43, 200, 255])
def test_riot_timer_tick_rule_equals_closed_form(reg, N):
    if reg == "T1024T" and N > 5:
        N = N % 4
    if reg == "TIM64T" and N > 43:
        N = 43

    def build(a):
        a.org(0xF000); a.op("LDA", "imm", N); a.op("STA", "abs", RIOT[reg])
    o = oracle_for(build); run_instr(o, 2)
    d = o.debug(0); assert d.timer == N and d.tflag == 0
    for dt in range(1, (N << SHIFT[reg]) + 601):
        o.tick(0); d = o.debug(0)
        assert (d.timer, d.tflag) == _closed_form(N, SHIFT[reg], dt), (reg, N, dt)


@pytest.mark.parametrize("reg,want_off", [("TIM64T", 1), ("TIM1T", 4), ("TIM8T", 1), ("T1024T", 1)])
def test_lda_intim_after_store(reg, want_off):
    for N in (7, 43, 255):
        def build(a):
            a.org(0xF000); a.op("LDA", "imm", N); a.op("STA", "abs", RIOT[reg]); a.op("LDA", "abs", RIOT["INTIM"])
        o = oracle_for(build); run_instr(o, 3)
        assert regs(o)["a"] == N - want_off                           # C.7: N-1 with TIM64T, N-4 with TIM1T


def test_timint_and_represcale_after_intim_read():
    def build(a):
        a.org(0xF000); a.op("LDA", "imm", 2); a.op("STA", "abs", RIOT["TIM8T"])          # c0 = 5 (cycle index)
        for _ in range(10): a.op("NOP")                                                    # 20 cycles -> past underflow (17)
        a.op("BIT", "abs", RIOT["TIMINT"]); a.op("LDA", "abs", RIOT["INTIM"]); a.op("BIT", "abs", RIOT["TIMINT"])
    o = oracle_for(build); run_instr(o, 12)
    c0 = 5
    assert regs(o)["timint"] == 0x80
    run_instr(o); assert regs(o)["p"] & 0x80                          # TIMINT bit 7 -> N; does not clear
    assert o.debug(0).tflag == 1
    run_instr(o)                                                      # LDA INTIM at cycle index 33: 0xFF-(33-(c0+17))
    read_cycle = int(regs(o)["cycles"]) - 1
    assert regs(o)["a"] == (0xFF - (read_cycle - (c0 + 1 + 16))) & 0xFF and o.debug(0).tflag == 0
    run_instr(o); assert not (regs(o)["p"] & 0x80)
    # prescaled decrements resume where (c - c0 - 1) % 8 == 0
    v = o.debug(0).timer
    for _ in range(40):
        before = int(regs(o)["cycles"]); o.tick(0); d = o.debug(0)
        if (before - c0 - 1) % 8 == 0:
            v = (v - 1) & 0xFF
        assert d.timer == v


def _frame_prog(a, visible_colour=None):
    a.org(0xF000); a.op("SEI"); a.op("CLD"); a.op("LDX", "imm", 0xFF); a.op("TXS")
    a.label("frame")
    a.op("LDA", "imm", 2); a.op("STA", "zp", TIA_W["VBLANK"]); a.op("STA", "zp", TIA_W["VSYNC"])
    for _ in range(3): a.op("STA", "zp", TIA_W["WSYNC"])
    a.op("LDA", "imm", 0); a.op("STA", "zp", TIA_W["VSYNC"])
    a.op("LDY", "imm", 37); a.label("vb"); a.op("STA", "zp", TIA_W["WSYNC"]); a.op("DEY"); a.op("BNE", "rel", "vb")
    if visible_colour is not None:
        a.op("LDA", "imm", visible_colour); a.op("STA", "zp", TIA_W["COLUBK"])
    a.op("LDA", "imm", 0); a.op("STA", "zp", TIA_W["VBLANK"])
    a.op("LDY", "imm", 192); a.label("vis"); a.op("STA", "zp", TIA_W["WSYNC"]); a.op("DEY"); a.op("BNE", "rel", "vis")
    a.op("LDA", "imm", 2); a.op("STA", "zp", TIA_W["VBLANK"])
    a.op("LDY", "imm", 30); a.label("os"); a.op("STA", "zp", TIA_W["WSYNC"]); a.op("DEY"); a.op("BNE", "rel", "os")
    a.op("JMP", "abs", "frame")


def test_solid_colour_frame_geometry():
    """C.13: COLUBK=v, VBLANK off for lines 37..228 -> rows 3..194 all v&0xFE, other rows 0 (y0 = 34)."""
    o = oracle_for(lambda a: _frame_prog(a, 0x4B))
    o.step(np.zeros(1, np.uint8), 3)
    r = regs(o); assert r["frame"] == 3 and r["line"] == 0 and r["cyc_in_line"] == 5
    c1 = int(r["cycles"]); o.step(np.zeros(1, np.uint8), 1)
    assert int(regs(o)["cycles"]) - c1 == 262 * 76                    # [D] 262-line frame
    scr = o.screen()[0]
    # VBLANK goes off in line 37 at cycle 9+: the rest of line 37 (row 3) from x = 3*(n+1)-68 on is coloured
    assert (scr[:3] == 0).all() and (scr[195:] == 0).all()
    assert (scr[4:195] == 0x4A).all()
    row3 = scr[3]; first = int(np.argmax(row3 != 0))
    assert (row3[first:] == 0x4A).all() and (row3[:first] == 0).all() and first == 0   # still in HBLANK
    assert regs(o)["status"] == 0


def test_frame_cap_ends_frames_without_vsync():
    def build(a):
        a.org(0xF000); a.label("l"); a.op("JMP", "abs", "l")
    o = oracle_for(build, max_lines=100)
    o.step(np.zeros(1, np.uint8), 2)
    r = regs(o)
    assert r["frame"] == 2 and r["status"] & 2
    assert 2 * 7600 <= r["cycles"] <= 2 * 7600 + 6                    # first instruction boundary past the cap


def test_halted_env_idles_to_the_cap():
    def build(a):
        a.org(0xF000); a.byte(0x02)
    o = oracle_for(build, max_lines=50)
    o.step(np.zeros(1, np.uint8), 3)
    r = regs(o); assert r["status"] == 3 and r["frame"] == 3 and r["pc"] == 0xF000 and r["cycles"] == 3 * 3800


def test_step_instructions_is_n_single_instruction_steps():
    """SURVEY §8(f) NEXT-2 / PAPER.md L582: n instructions of a NOP sled are 2n cycles and n bytes of PC; a WSYNC stall
    belongs to the instruction that follows it; the call latches the action first."""
    def build(a):
        a.org(0xF000)
        for _ in range(20): a.op("NOP")
        a.op("STA", "zp", TIA_W["WSYNC"]); a.op("LDA", "abs", RIOT["SWCHA"]); a.op("STA", "zp", 0x80)
    o = oracle_for(build)
    o.step_instructions(np.array([3], np.uint8), 7)                  # RIGHT
    r = regs(o); assert r["cycles"] == 14 and r["pc"] == 0xF007
    o.step_instructions(np.array([3], np.uint8), 14)                 # 13 NOPs + STA WSYNC (3 cycles, written in cycle 42)
    r = regs(o); assert r["cycles"] == 14 + 26 + 3 and r["pc"] == 0xF016
    o.step_instructions(np.array([3], np.uint8), 2)                  # LDA SWCHA waits for the line end first: 76 + 4, then STA 3
    r = regs(o); assert r["cycles"] == 76 + 4 + 3 and o.ram()[0][0] == 0x7F
