"""Pins for the oracle's FULL mode — the fully relaxed forward of PAPER.md appendix D (L425-459, Table 2,
Table 3, forward part; reading R18) — against what the paper fixes for ANY program:
  * a crisp-flag branch keeps its rounded soft PC on the hard target iff |delta| < tau_b(alpha) = (1 + e^alpha) / 2 (L429);
  * a temperature-T read is exact iff the neighbour pull stays below 1/2, which T <= 1 / ln(4 * 255) ~ 0.144 guarantees
    for every byte pattern, while just above it a byte between extreme neighbours is pulled off (L459);
  * so (alpha >= 6, T <= 0.14) is bit-exact on every program and "the first-divergence step" is the first cast that
    does not round to the hard value (L435: "measurement and model agree").
Expected values are worked by hand from these closed forms or derived from the HARD trajectory by the paper's cast-margin
rule, never from the FULL-mode code.  The paper's own N_div numbers (Table 3) need the Space Invaders ROM: not here."""
import math

import numpy as np
import pytest

from helpers import oracle_for
from oracle.ovcs_py import OracleVCS
from vcs_inputs import make_workload

BRANCH = {0x10, 0x30, 0x50, 0x70, 0x90, 0xB0, 0xD0, 0xF0}
NOOP = np.zeros(1, np.uint8)


def full(o, n, T, alpha):
    return o.step_instructions_soft(np.zeros(o.batch, np.uint8), n, T, alpha, True)


# ---- branch casts, by hand: sigma(2) = 0.880797, sigma(-2) = 0.119203
@pytest.mark.parametrize("a_imm,delta,pc_full", [
    (0x00, 4, 0xF008),       # BEQ taken, 4 * 0.8808 = 3.52 -> 4: on the hard target $F004 + 4
    (0x00, 5, 0xF008),       # 5 * 0.8808 = 4.40 -> 4: one short of $F009 (|delta| = 5 > tau_b(2) = 4.19)
    (0x00, 100, 0xF05C),     # 88.08 -> 88: $F004 + 88
    (0x00, -6, 0xEFFF),      # -5.28 -> -5: $F004 - 5 (hard: $EFFE)
    (0x01, 4, 0xF004),       # BEQ not taken, 4 * 0.1192 = 0.48 -> 0: stays on the fall-through address
    (0x01, 5, 0xF005),       # 0.596 -> 1: one past it
    (0x01, -128, 0xEFF5),    # -15.26 -> -15
])
def test_branch_cast_alpha2(a_imm, delta, pc_full):
    def prog(a):
        a.org(0xF000); a.op("LDA", "imm", a_imm); a.byte(0xF0); a.byte(delta & 0xFF)       # LDA #imm ; BEQ delta
    o = oracle_for(prog); h = oracle_for(prog)
    out = full(o, 2, 0.05, 2.0); h.step_instructions(NOOP, 2)                                # (T = 0.05: every read exact)
    taken = a_imm == 0
    pc_hard = 0xF004 + (delta if taken else 0)
    assert int(h.regs()[0]["pc"]) == pc_hard & 0xFFFF
    assert int(o.regs()[0]["pc"]) == pc_full
    assert int(out[0, 6]) == (0 if pc_full == pc_hard & 0xFFFF else 1)                       # the failed cast is counted
    assert o.regs()[0]["cycles"] == h.regs()[0]["cycles"]                                    # R18: timing follows the hard decision


@pytest.mark.parametrize("alpha", [5.54, 6.0, 8.0])
def test_every_branch_offset_is_exact_from_alpha_min(alpha):
    """alpha >= ln(2 * 127 - 1) = 5.533: tau_b > 127 (L459); -128 needs tau_b > 128, i.e. alpha >= ln(255) = 5.541"""
    for delta in (127, -127, 1, -1, 64) + ((-128,) if alpha >= 5.55 else ()):
        for a_imm in (0, 1):
            def prog(a):
                a.org(0xF000); a.op("LDA", "imm", a_imm); a.byte(0xF0); a.byte(delta & 0xFF)
            o = oracle_for(prog); h = oracle_for(prog)
            out = full(o, 2, 0.05, alpha); h.step_instructions(NOOP, 2)
            assert o.regs()[0] == h.regs()[0] and out[0, 6] == 0, (alpha, delta, a_imm)


# ---- read casts, by hand.  A RAM cell holding 0 between cells holding 255 (the worst case of L459):
#   T = 0.14: w_1 = e^{-1/0.14} = 7.90e-4, pull = 255 (1 - w_0) = 255 * 2(w_1 + w_2 + w_3) / (1 + ...) = 0.402 -> reads 0
#   T = 0.15: w_1 = e^{-1/0.15} = 1.273e-3, pull = 255 * 0.0025494 / 1.0025494 = 0.648 -> reads 1
#   one neighbour 255, the rest 0, T = 0.20: 255 e^{-5} / (1 + 2 (e^{-5} + e^{-10} + ...)) = 1.695 -> reads 2 (L437: "~1.7")
@pytest.mark.parametrize("T,cells,expect", [
    (0.14, {k: 255 for k in range(0x0C, 0x15) if k != 0x10}, 0),
    (0.15, {k: 255 for k in range(0x0C, 0x15) if k != 0x10}, 1),
    (0.12, {k: 255 for k in range(0x0C, 0x15) if k != 0x10}, 0),
    (0.15, {0x11: 255}, 0),                                      # one neighbour at T = 0.15: 255 * 1.27e-3 = 0.32
])
def test_read_cast_between_extreme_neighbours(T, cells, expect):
    def prog(a):
        a.org(0xF000); a.op("LDA", "zp", 0x90); a.op("STA", "zp", 0xA0)       # code bytes A5 90 85 A0: no extreme neighbours
    o = oracle_for(prog)
    for k in range(0x08, 0x18): o.poke_ram(0, k, cells.get(k, 0))
    out = full(o, 2, T, 6.0)
    assert int(o.regs()[0]["a"]) == expect and int(o.ram()[0, 0x20]) == expect
    assert int(out[0, 6]) == (1 if expect else 0)


def test_single_neighbour_at_T020_reads_two():
    def prog(a):
        a.org(0xF000); a.op("LDX", "zp", 0x90); a.byte(0x7A)
    o = oracle_for(prog)
    for k in range(0x08, 0x18): o.poke_ram(0, k, 255 if k == 0x11 else 0)
    # the instruction's own bytes are reads at T = 0.20 too.  A6 sits at the edge of the bank tensor with 90 to its right:
    # pull (0x90 - 0xA6) e^{-5} = -0.15; 90 sits between A6 and 7A: (0xA6 + 0x7A - 2 * 0x90) e^{-5} = 0 -> both exact
    out = full(o, 1, 0.20, 6.0)
    assert int(o.regs()[0]["pc"]) == 0xF002 and int(o.regs()[0]["x"]) == 2 and out[0, 6] == 1


def test_an_operand_byte_is_a_read_too():
    """the same load with the assembler's $FF fill behind it: the OPERAND fetch is pulled by (0xA6 + 0xFF - 2 * 0x90) e^{-5}
    = 0.89 to $91, so the load reads the neighbour cell (255, itself pulled by -2 * 255 e^{-5} = -3.4 -> 252)"""
    def prog(a):
        a.org(0xF000); a.op("LDX", "zp", 0x90)
    o = oracle_for(prog)
    for k in range(0x08, 0x18): o.poke_ram(0, k, 255 if k == 0x11 else 0)
    out = full(o, 1, 0.20, 6.0)
    assert int(o.regs()[0]["x"]) == 252 and out[0, 6] == 2


# ---- the corner is exact on every program: Table 3 rows "exact" (alpha = 6, T = 0.08 .. 0.14), L459
@pytest.mark.parametrize("cfg", [2, 3, 4])
@pytest.mark.parametrize("T", [0.08, 0.14])
def test_corner_is_bit_exact_over_3000_instructions(cfg, T):
    w = make_workload(cfg, batch=4, n_roms=4) if cfg == 4 else make_workload(cfg, batch=3)
    o = OracleVCS(w.roms, w.seeds, w.env_rom); h = OracleVCS(w.roms, w.seeds, w.env_rom)
    a = w.actions(0, 1)[0]
    out = o.step_instructions_soft(a, 3000, T, 6.0, True); h.step_instructions(a, 3000)
    assert (o.ram() == h.ram()).all() and (o.screen() == h.screen()).all()
    assert all((o.regs()[f] == h.regs()[f]).all() for f in h.regs().dtype.names)
    assert (out[:, 6] == 0).all() and (out[:, 3] > 3000).all()


def first_divergence(w, e, T, alpha, n=3000):
    """(measured N_div, predicted N_div): step the FULL and the HARD console one instruction at a time; the prediction is
    the first conditional branch of the HARD trajectory whose cast leaves the hard target by the tau_b rule"""
    o = OracleVCS(w.roms, w.seeds[e:e + 1], w.env_rom[e:e + 1]); h = OracleVCS(w.roms, w.seeds[e:e + 1], w.env_rom[e:e + 1])
    rom = w.roms[int(w.env_rom[e])]
    a = w.actions(0, 1)[0][e:e + 1]
    miss_unit = 1.0 / (1.0 + math.exp(alpha))                              # sigma(-alpha): the share of delta the cast loses
    measured = predicted = None
    for i in range(1, n + 1):
        r = h.regs()[0]; pc, bank = int(r["pc"]), int(r["bank"])
        if predicted is None and pc & 0x1000:
            opc = rom[(bank * 4096 + (pc & 0xFFF)) % len(rom)]
            if opc in BRANCH:
                d = rom[(bank * 4096 + ((pc + 1) & 0xFFF)) % len(rom)]; d = d - 256 if d >= 128 else d
                miss = abs(d) * miss_unit
                assert abs(miss - 0.5) > 1e-3
                if miss > 0.5: predicted = i
        o.step_instructions_soft(a, 1, T, alpha, True); h.step_instructions(a, 1)
        if measured is None and (o.regs()[0] != h.regs()[0] or (o.ram() != h.ram()).any()): measured = i
        if measured is not None and predicted is not None: break
    return measured, predicted


@pytest.mark.parametrize("alpha", [2.0, 3.0, 4.0])
def test_first_divergence_is_the_first_failed_branch_cast(alpha):
    """the forward is bit-exact precisely while every cast margin holds.  T = 0.05 keeps every read exact,
    so the first divergence must be the first executed branch with |delta| sigma(-alpha) > 1/2 (|delta| >= tau_b)."""
    w = make_workload(3, batch=4)
    for e in range(2):
        measured, predicted = first_divergence(w, e, 0.05, alpha)
        assert measured == predicted, (alpha, e, measured, predicted)        # (both None: no such branch in 3000 instructions -> exact)
        assert predicted is not None or alpha >= 4.0


def test_above_T_max_the_forward_leaves_the_trajectory_early():
    """Table 3: T = 0.18 / 0.20 diverge after a couple of instructions on a real game; on the synthetic cartridges too"""
    w = make_workload(3, batch=4)
    m, _ = first_divergence(w, 0, 0.20, 6.0, n=400)
    assert m is not None and m < 400
