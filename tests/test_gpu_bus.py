"""-m gpu: bus patterns outside "code in ROM, stack and pointers in RAM" — every access is decoded by address (SURVEY
§8(c) C.3 / C.5; one shared 13-bit bus to cartridge, RIOT and TIA), so the stack may sit on TIA registers
(SP < $80), zero-page pointers and JMP() vectors may be read from TIA / RIOT addresses, and code may run from RAM, from
the TIA's read addresses or from the RIOT's ports.  The CUDA interpreter against the per-cycle oracle, bit-exact on RAM,
registers (cycle counter included) and screens after every step."""
import os

import numpy as np
import pytest

from vcs_inputs import hand_rom, SplitMix64, TIA_W, TIA_R, RIOT, env_seeds

pytestmark = pytest.mark.gpu
NCPU = os.cpu_count() or 1


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


def _compare(g, o, tag):
    from test_gpu_parity import compare
    compare(g, o, tag)


def _run(torch, rom, n_envs, steps, seed, actions=None, fs=None, **kw):
    from paper_2606_22447_b200 import VCS
    from oracle.ovcs_py import OracleVCS
    seeds = env_seeds(seed, n_envs)
    g, o = VCS([rom], seeds, **kw), OracleVCS([rom], seeds, **kw)
    rng = SplitMix64(seed ^ 0x5EED)
    for t in range(steps):
        a = np.array([rng.rnd(18) for _ in range(n_envs)], np.uint8) if actions is None else np.full(n_envs, actions, np.uint8)
        f = (1 + t % 3) if fs is None else fs
        g.step(torch.from_numpy(a).cuda(), f); o.step(a, f, threads=NCPU)
        _compare(g, o, f"step {t}")
    return g, o


def _frame(a, body, lines=40):
    """a short frame: VSYNC pulse, `body`, a few WSYNC lines with a picture"""
    a.label("frame")
    a.op("LDA", "imm", 2); a.op("STA", "zp", TIA_W["VSYNC"]); a.op("STA", "zp", TIA_W["WSYNC"]); a.op("LDA", "imm", 0); a.op("STA", "zp", TIA_W["VSYNC"])
    a.op("STA", "zp", TIA_W["VBLANK"])
    body(a)
    a.op("LDX", "imm", 0xFF); a.op("TXS")
    a.op("LDY", "imm", lines); lp = a.newlabel("L"); a.label(lp)
    a.op("STA", "zp", TIA_W["WSYNC"]); a.op("LDA", "zp", 0x90); a.op("STA", "zp", TIA_W["COLUBK"])
    a.op("TYA"); a.op("STA", "zp", TIA_W["PF1"]); a.op("DEY"); a.op("BNE", "rel", lp)
    a.op("JMP", "abs", "frame")


def test_classic_clear_loop_sweeps_the_stack_through_the_tia(torch):
    """LDX #0 / TXA / DEX / TXS / PHA / BNE: SP runs $FF -> $00, so PHA writes A to RAM and then to every TIA register
    (WSYNC stalls, VSYNC / VBLANK, the strobes, HMOVE, CXCLR ...).  A second sweep pushes a per-env random byte."""
    def build(a):
        a.org(0xF000); a.op("SEI"); a.op("CLD")
        a.op("LDX", "imm", 0); a.op("TXA")
        a.label("clr"); a.op("DEX"); a.op("TXS"); a.op("PHA"); a.op("BNE", "rel", "clr")
        def body(a):
            a.op("LDA", "zp", 0x90); a.op("ADC", "zp", 0x91); a.op("STA", "zp", 0x90); a.op("INC", "zp", 0x91)    # a changing byte
            a.op("LDX", "imm", 0x80)
            s = a.newlabel("S"); a.label(s); a.op("DEX"); a.op("TXS"); a.op("PHA"); a.op("PHP"); a.op("BNE", "rel", s)   # SP $7F..$00: all pushes hit the TIA
            a.op("LDX", "imm", 0x45); a.op("TXS"); a.op("PLA"); a.op("STA", "zp", 0x92); a.op("PLP"); a.op("PLA"); a.op("STA", "zp", 0x93)   # pulls read CXxx / INPTx
            a.op("PHP"); a.op("PLA"); a.op("STA", "zp", 0x94)
        _frame(a, body)
    rom = hand_rom(build)
    from paper_2606_22447_b200 import VCS
    from oracle.ovcs_py import OracleVCS
    seeds = env_seeds(11, 40)
    g, o = VCS([rom], seeds, max_lines=150), OracleVCS([rom], seeds, max_lines=150)
    # before the first step both hold the seeded power-on RAM; the clear loop must leave RAM zero on both sides
    a0 = np.zeros(40, np.uint8)
    g.step(torch.from_numpy(a0).cuda(), 1); o.step(a0, 1, threads=NCPU)
    _compare(g, o, "clear loop")
    assert not (g.regs_host()["status"] & 1).any()
    for t in range(6):
        a = np.array([(3 * e + t) % 18 for e in range(40)], np.uint8)
        g.step(torch.from_numpy(a).cuda(), 1 + t % 3); o.step(a, 1 + t % 3, threads=NCPU)
        _compare(g, o, f"tia stack step {t}")


def test_jsr_rts_brk_rti_with_the_stack_in_tia_space(torch):
    """JSR / BRK push onto TIA registers (two of the pushed addresses are WSYNC and VSYNC: the read that follows the
    pushes stalls, a frame can end in mid-instruction); RTS / RTI then pull collision latches as a return address and
    land in TIA / RAM-mirror space, where the bytes executed are TIA reads, until a BRK (opcode $00) vectors back."""
    def build(a):
        a.org(0xF000); a.op("SEI"); a.op("CLD"); a.op("LDX", "imm", 0xFF); a.op("TXS")
        def body(a):
            a.op("LDA", "imm", 0)                                                                                       # return addresses pulled from the TIA are
            for cell in (0x81, 0x82, 0xC1, 0xC2): a.op("STA", "zp", cell)                                               # $xx01 / 41 / 81 / C1: BRK waits in RAM there
            a.op("INC", "zp", 0xA0); a.op("LDA", "zp", 0xA0); a.op("AND", "imm", 0x3F); a.op("TAX"); a.op("TXS")        # SP = 0..$3F, one more each frame
            a.op("LDA", "imm", 0xFF); a.op("STA", "zp", TIA_W["GRP0"]); a.op("STA", "zp", TIA_W["PF0"])                 # so that some latches are set
            a.op("JSR", "abs", "sub")
            a.op("LDA", "zp", 0xA0); a.op("EOR", "imm", 0x55); a.op("AND", "imm", 0x7F); a.op("TAX"); a.op("TXS")
            a.op("PHA"); a.op("PHP"); a.op("JSR", "abs", "sub2"); a.op("NOP")
        _frame(a, body)
        a.label("sub"); a.op("INC", "zp", 0xA1); a.op("RTS")
        a.label("sub2"); a.op("INC", "zp", 0xA2); a.op("PLA"); a.op("PLA"); a.op("JMP", "abs", "back")
        a.label("back"); a.op("LDX", "imm", 0x02); a.op("TXS"); a.op("BRK"); a.byte(0xEA)          # pushes to VBLANK... / WSYNC / VSYNC then reads the vector
        a.org(0xF400); a.label("irq"); a.op("INC", "zp", 0xA3); a.op("LDX", "imm", 0xFF); a.op("TXS"); a.op("JMP", "abs", "frame")
    rom = bytearray(hand_rom(build))
    rom[0xFFE] = 0x00; rom[0xFFF] = 0xF4                                  # BRK vector -> irq
    _run(torch, bytes(rom), 36, 8, seed=21, max_lines=120)


def test_pointers_and_vectors_read_from_tia_and_riot(torch):
    """(zp),Y / (zp,X) with the pointer cells below $80 (the pointer bytes are collision-latch reads), pointers whose
    target is the RIOT (an indexed page crossing does a dummy read of INTIM, which clears the underflow flag), and
    JMP ($0284): the vector bytes are INTIM and TIMINT."""
    def build(a):
        a.org(0xF000); a.op("SEI"); a.op("CLD"); a.op("LDX", "imm", 0xFF); a.op("TXS")
        # pointers in RAM aimed at the RIOT and at RAM / ROM
        for zp, target in ((0xB0, 0x02F0), (0xB2, 0x0284), (0xB4, 0xF7F0), (0xB6, 0x00F8)):
            a.op("LDA", "imm", target & 0xFF); a.op("STA", "zp", zp); a.op("LDA", "imm", target >> 8); a.op("STA", "zp", zp + 1)
        def body(a):
            a.op("LDA", "imm", 0xFF); a.op("STA", "zp", TIA_W["GRP0"]); a.op("STA", "zp", TIA_W["GRP1"]); a.op("STA", "zp", TIA_W["PF0"])
            a.op("STA", "zp", TIA_W["ENABL"]); a.op("STA", "zp", TIA_W["ENAM0"])
            a.op("LDA", "imm", 3); a.op("STA", "abs", RIOT["TIM8T"])
            a.op("STA", "zp", TIA_W["WSYNC"]); a.op("STA", "zp", TIA_W["WSYNC"])
            for i, (mn, mode, zp) in enumerate([("LDA", "izy", 0x02), ("LDA", "izy", 0x06), ("LDA", "izx", 0x00), ("ADC", "izy", 0x0C),
                                                ("LDA", "izy", 0xB0), ("LDA", "izy", 0xB2), ("ORA", "izx", 0xB2), ("LDA", "izy", 0xB4),
                                                ("STA", "izy", 0x03), ("STA", "izx", 0x07), ("STA", "izy", 0xB0), ("STA", "izy", 0xB6), ("STA", "izx", 0xB6)]):
                a.op("LDY", "zp", 0xA0); a.op("LDX", "imm", (2 * i) & 6)
                a.op(mn, mode, zp); a.op("STA", "zp", 0xC0 + i); a.op("PHP"); a.op("PLA"); a.op("STA", "zp", 0xD0 + i)
            a.op("INC", "zp", 0xA0); a.op("INC", "zp", 0xA0); a.op("INC", "zp", 0xA0)
            a.op("LDA", "zp", 0xA0); a.op("AND", "imm", 1); a.op("BNE", "rel", "novec")
            a.op("LDA", "imm", 0); a.op("LDX", "imm", 15); f = a.newlabel("F"); a.label(f); a.op("STA", "zpx", 0xE0); a.op("DEX"); a.op("BPL", "rel", f)   # BRKs at $E0-$EF
            a.op("LDA", "imm", 0xF0); a.op("STA", "abs", RIOT["TIM1T"])                     # INTIM = $E8 by the time of the jump: the vector is $00E8 (RAM)
            a.op("JMP", "ind", 0x0284)
            a.label("novec")
        _frame(a, body)
    rom = bytearray(hand_rom(build))
    _run(torch, bytes(rom), 40, 8, seed=31, max_lines=140)


def test_code_running_from_ram_tia_and_riot_space(torch):
    """A routine copied to RAM and called there (it modifies its own operand and its stack overlaps it), a jump into
    the TIA's read addresses (opcodes = collision latches: $00 BRK, $40 RTI, $80 NOP #, $C0 CPY #) and a jump to $0280
    with port A and B as outputs (SWCHA / SWACNT / SWCHB read back as JMP $F0FF)."""
    def build(a):
        a.org(0xF000); a.op("SEI"); a.op("CLD"); a.op("LDX", "imm", 0xFF); a.op("TXS")
        a.op("LDX", "imm", 15); a.label("cp"); a.op("LDA", "abx", "ramcode"); a.op("STA", "zpx", 0xE0); a.op("DEX"); a.op("BPL", "rel", "cp")
        def body(a):
            a.op("LDA", "imm", 0xFF); a.op("STA", "zp", TIA_W["GRP0"]); a.op("STA", "zp", TIA_W["PF0"]); a.op("STA", "zp", TIA_W["ENAM1"]); a.op("STA", "zp", TIA_W["GRP1"])
            a.op("STA", "zp", TIA_W["WSYNC"])
            a.op("LDX", "imm", 0xFF); a.op("TXS"); a.op("JSR", "abs", 0x00E0)               # RAM routine, ordinary stack
            a.op("LDX", "imm", 0xEE); a.op("TXS"); a.op("JSR", "abs", 0x00E0)               # the pushes land inside the routine's own bytes
            a.op("LDA", "zp", 0xA5); a.op("CLC"); a.op("ADC", "imm", 1); a.op("STA", "zp", 0xA5); a.op("AND", "imm", 3)
            a.op("BEQ", "rel", "tia"); a.op("CMP", "imm", 1); a.op("BEQ", "rel", "riot"); a.op("JMP", "abs", "done")
            a.label("tia"); a.op("LDX", "imm", 0x9F); a.op("TXS"); a.op("JMP", "abs", 0x0030)   # $30..: reads of CXM0P.. mirrors
            a.label("riot")
            a.op("LDA", "imm", 0xFF); a.op("STA", "abs", RIOT["SWACNT"]); a.op("STA", "abs", RIOT["SWBCNT"])
            a.op("LDA", "imm", 0x4C); a.op("STA", "abs", RIOT["SWCHA"]); a.op("LDA", "imm", 0xF0); a.op("STA", "abs", RIOT["SWCHB"])
            a.op("JMP", "abs", 0x0280)                                                       # executes 4C FF F0 = JMP $F0FF from the ports
            a.label("done")
            a.op("LDA", "imm", 0x00); a.op("STA", "abs", RIOT["SWACNT"]); a.op("STA", "abs", RIOT["SWBCNT"])
        _frame(a, body)
        a.label("ramcode")                                                                    # 16 bytes, runs at $E0
        a.op("INC", "zp", 0xE3)                                                               # E0: bumps the operand of the next instruction
        a.op("LDA", "imm", 0x10)                                                              # E2
        a.op("STA", "zp", 0xA8); a.op("INC", "zp", 0xA9); a.op("LDA", "zp", 0xEE); a.op("STA", "zp", 0xAA)   # E4..EB
        a.op("RTS")                                                                           # EC
        a.byte(0xEA, 0xEA, 0xEA)
        a.org(0xF0FF); a.op("INC", "zp", 0xAB); a.op("JMP", "abs", "done")
        a.org(0xF500); a.label("irq"); a.op("INC", "zp", 0xAC); a.op("LDX", "imm", 0xFF); a.op("TXS"); a.op("JMP", "abs", "done")
    rom = bytearray(hand_rom(build))
    rom[0xFFE] = 0x00; rom[0xFFF] = 0xF5
    _run(torch, bytes(rom), 36, 10, seed=41, max_lines=130)


def test_code_in_the_last_16_bytes_of_a_bank_and_opcode_fetches_on_f8_hotspots(torch):
    """The CPU runs through $FFF0-$FFFB: the opcode fetch at $FFF8 selects bank 0 (and returns ITS byte), the dummy read
    of that one-byte instruction at $FFF9 selects bank 1 again, the fetch at $FFF9 executes bank 1's byte; the JMP at
    $FFFA takes its high byte from the reset vector ($00) and lands in a RAM stub."""
    def build(a):
        a.org(0xF000); a.op("SEI"); a.op("CLD"); a.op("LDX", "imm", 0xFF); a.op("TXS")
        for i, b in enumerate((0x4C, 0x00, 0xF1)): a.op("LDA", "imm", b); a.op("STA", "zp", 0x80 + i)    # RAM stub: JMP $F100
        def body(a):
            a.op("INC", "zp", 0x90); a.op("LDY", "zp", 0x90); a.op("JMP", "abs", 0xFFF0)
            a.label("after")
        _frame(a, body)
        a.org(0xF100); a.op("STX", "zp", 0x91); a.op("STY", "zp", 0x92); a.op("JMP", "abs", "after")
        a.org(0xFFF0)
        for _ in range(6): a.op("NOP")
        a.op("LDX", "imm", 0x11)                                                                         # $FFF6
        a.byte(0xCA, 0xC8)                                                                               # $FFF8 DEX, $FFF9 INY (bank 1's bytes)
        a.byte(0x4C, 0x80)                                                                               # $FFFA JMP $0080 (high byte = $FFFC = $00)
    b1 = bytearray(hand_rom(build)); b0 = bytearray(b1)
    b0[0xFF8] = 0xE8; b0[0xFF9] = 0x88                                                                   # bank 0: INX, DEY
    from paper_2606_22447_b200 import VCS
    from oracle.ovcs_py import OracleVCS
    roms = [bytes(b0 + b1), bytes(b1)]                                                                   # the F8 cart and the same code as a plain 4K cart
    seeds = env_seeds(77, 64); env_rom = (np.arange(64) % 2).astype(np.int32)
    g, o = VCS(roms, seeds, env_rom, max_lines=120), OracleVCS(roms, seeds, env_rom, max_lines=120)
    for t in range(5):
        a = np.zeros(64, np.uint8)
        g.step(torch.from_numpy(a).cuda(), 2); o.step(a, 2, threads=NCPU)
        _compare(g, o, f"bank end step {t}")
    ram = g.ram_host()
    assert (ram[0::2, 0x11] == 0x12).all() and (ram[1::2, 0x11] == 0x10).all()                          # F8: INX from bank 0; 4K: DEX
    assert not (g.regs_host()["status"] & 1).any()


def _soup_rom(seed: int) -> bytes:
    """Random instruction soup with the stack pointer, the pointer cells and the jump vectors anywhere: TXS with random X,
    pushes / pulls / JSR / RTS / BRK at any SP, every indirect mode with any zero-page cell, JMP () through any page,
    stores and RMWs anywhere in $0000-$03FF.  Whatever happens (garbage return addresses, code in RAM / TIA / RIOT space,
    halts on undocumented opcodes) must happen identically on both sides; BRK and the frame cap bring control back."""
    r = SplitMix64(seed)
    READ = ["LDA", "ADC", "SBC", "AND", "ORA", "EOR", "CMP"]

    def build(a):
        a.org(0xF000); a.op("SEI"); a.op("CLD"); a.op("LDX", "imm", 0xFF); a.op("TXS")
        a.label("top")
        a.op("LDA", "imm", 2); a.op("STA", "zp", TIA_W["VSYNC"]); a.op("LDA", "imm", 0); a.op("STA", "zp", TIA_W["VSYNC"])
        for i in range(230):
            k = r.rnd(24)
            if k < 4: a.op("LDX", "imm", r.rnd(256)); a.op("TXS")
            elif k < 7: a.op(r.choice(["PHA", "PHP", "PLA", "PLP"]))
            elif k < 9: a.op("JSR", "abs", r.choice(["s0", "s1", "s2"]))
            elif k < 10: a.op("LDA", "imm", r.rnd(256)); a.op("PHA"); a.op("LDA", "imm", r.rnd(256)); a.op("PHA"); a.op("RTS" if r.chance(2, 3) else "RTI")
            elif k < 13: a.op("LDY", "imm", r.rnd(256)); a.op(r.choice(READ), "izy", r.rnd(256)); a.op("STA", "zp", 0x80 + r.rnd(128))
            elif k < 15: a.op("LDX", "imm", r.rnd(256)); a.op(r.choice(READ), "izx", r.rnd(256)); a.op("STA", "zp", 0x80 + r.rnd(128))
            elif k < 17: a.op("LDY", "imm", r.rnd(256)); a.op("LDA", "imm", r.rnd(256)); a.op("STA", r.choice(["izy", "izx"]), r.rnd(256))
            elif k < 18:
                v = r.choice([0x0000 + r.rnd(0x100), 0x0280 + r.rnd(8), 0x01F0 + r.rnd(16), 0xF7FF, 0x00FF])
                a.op("JMP", "ind", v)
            elif k < 20: a.op(r.choice(["INC", "DEC", "ASL", "ROR"]), "abx", r.rnd(0x400)); a.op("LDX", "imm", r.rnd(256))
            elif k < 21: a.op("LDA", "imm", r.rnd(256)); a.op("STA", "abs", RIOT[r.choice(["TIM1T", "TIM8T", "TIM64T", "SWACNT", "SWCHA"])])
            elif k < 22: a.op("BRK"); a.byte(r.rnd(256))
            elif k < 23: a.op("STA", "zp", TIA_W[r.choice(["WSYNC", "GRP0", "GRP1", "PF1", "ENABL", "ENAM0", "RESP0", "RESBL", "HMOVE", "COLUBK"])])
            else: a.op(r.choice(["LDA", "LDX", "LDY"]), "imm", r.rnd(256))
        a.op("JMP", "abs", "top")
        a.label("s0"); a.op("RTS")
        a.label("s1"); a.op("PLA"); a.op("TAY"); a.op("PLA"); a.op("PHA"); a.op("TYA"); a.op("PHA"); a.op("RTS")
        a.label("s2"); a.op("PHP"); a.op("PLA"); a.op("STA", "zp", 0xBF); a.op("RTS")
        a.org(0xFE00); a.label("irq"); a.op("INC", "zp", 0xBE); a.op("LDX", "imm", 0xFF); a.op("TXS"); a.op("CLD"); a.op("JMP", "abs", "top")
    rom = bytearray(hand_rom(build))
    rom[0xFFE] = 0x00; rom[0xFFF] = 0xFE
    return bytes(rom)


@pytest.mark.parametrize("seed", range(8))
def test_bus_soup(torch, seed):
    _run(torch, _soup_rom(7000 + seed), 48, 8, seed=60 + seed, max_lines=100 + 20 * seed, y0=2 + 4 * seed)
