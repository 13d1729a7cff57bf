"""Pins for the oracle's 6507: opcode matrix, cycle counts from the
bus sequences, ALU brute force against wide-integer / base-100 definitions, hand programs."""
import ctypes as C

import numpy as np
import pytest

from helpers import oracle_for, run_instr, regs, load_opcode_matrix, load_undocumented
from vcs_inputs import OPCODES

fC, fZ, fI, fD, fV, fN = 1, 2, 4, 8, 0x40, 0x80
MATRIX = load_opcode_matrix()
UNDOC = load_undocumented()          # the paper's 38 undocumented bytes: executed, not halted
BR_FLAG = {"BPL": (fN, 0), "BMI": (fN, 1), "BVC": (fV, 0), "BVS": (fV, 1), "BCC": (fC, 0), "BCS": (fC, 1), "BNE": (fZ, 0), "BEQ": (fZ, 1)}


def test_matrix_is_151_and_matches_assembler_table():
    assert len(MATRIX) == 151
    flat = {}
    for mn, modes in OPCODES.items():
        for mode, (code, cyc, px) in modes.items():
            assert code not in flat
            flat[code] = (mn, mode, cyc, bool(px))
    assert flat == MATRIX                                       # two independently typed encodings agree


def _one(opcode, mode, cross, p=0x24):
    """Run one instruction of `opcode` in `mode`; return (cycles, regs, oracle)."""
    operand = {"imp": [], "acc": [], "imm": [0x12], "zp": [0x80], "zpx": [0x80], "zpy": [0x80], "rel": [0x10],
               "abs": [0x80, 0x00], "abx": [0xFF if cross else 0x00, 0xFA], "aby": [0xFF if cross else 0x00, 0xFA],
               "izx": [0x90], "izy": [0x90], "ind": [0x00, 0xFA]}[mode]
    if MATRIX.get(opcode, ("",))[0] in ("JMP", "JSR") and mode == "abs":
        operand = [0x10, 0xF0]

    def build(a):
        a.org(0xF000); a.byte(opcode, *operand)
        a.org(0xFA00); a.byte(0x10, 0xF0)                        # JMP (ind) vector
    o = oracle_for(build)
    o.set_cpu(0, a=0x55, x=1, y=1, sp=0xFD, p=p, pc=0xF000)
    o.poke_ram(0, 0x10, 0xFF if cross else 0x00); o.poke_ram(0, 0x11, 0xFA)     # ($90) -> $FAxx
    if mode == "izx":
        o.set_cpu(0, x=0)
    c0 = regs(o)["cycles"]
    run_instr(o)
    return int(regs(o)["cycles"] - c0), regs(o), o


@pytest.mark.parametrize("opcode", range(256))
def test_cycles_from_bus_sequences_match_matrix(opcode):
    if opcode in UNDOC:
        mn, mode, cyc, px = UNDOC[opcode]
        n, r, _ = _one(opcode, mode, False)
        assert n == cyc and not (r["status"] & 1), (hex(opcode), mn, mode)
        n2, _, _ = _one(opcode, mode, True)
        assert n2 == cyc + (1 if px else 0), (hex(opcode), "page cross")
        assert r["pc"] == 0xF000 + {"imp": 1, "abs": 3, "abx": 3, "aby": 3}.get(mode, 2)
        return
    if opcode not in MATRIX:                                    # C.12: halt, PC stays, status bit 0
        n, r, o = _one(opcode, "imp", False)
        assert n == 1 and r["status"] & 1 and r["pc"] == 0xF000
        c = r["cycles"]; run_instr(o, 5)                        # then idle ticks only
        assert regs(o)["cycles"] == c + 5 and regs(o)["pc"] == 0xF000
        return
    mn, mode, cyc, px = MATRIX[opcode]
    if mode == "rel":
        flag, want = BR_FLAG[mn]
        n, r, _ = _one(opcode, mode, False, p=0x24 | (0 if want else flag))   # not taken
        assert n == 2 and r["pc"] == 0xF002
        n, r, _ = _one(opcode, mode, False, p=0x24 | (flag if want else 0))   # taken, same page
        assert n == 3 and r["pc"] == 0xF012
        return
    n, r, _ = _one(opcode, mode, False)
    assert n == cyc, (mn, mode)
    assert not (r["status"] & 1)
    n2, _, _ = _one(opcode, mode, True)
    assert n2 == cyc + (1 if px else 0), (mn, mode, "page cross")
    if mn not in ("JMP", "JSR", "RTS", "RTI", "BRK"):
        assert r["pc"] == 0xF000 + {"imp": 1, "acc": 1, "abs": 3, "abx": 3, "aby": 3, "ind": 3}.get(mode, 2)


def test_branch_page_cross_is_4_cycles():
    def build(a):
        a.org(0xF0FC); a.op("SEC"); a.op("BCS", "rel", 0x10)    # next instr at $F0FF, target $F10F
        a.org(0xF100); a.op("CLC"); a.op("BCC", "rel", -0x10)   # backwards across a page: $F103-0x10=$F0F3
    o = oracle_for(build); o.set_cpu(0, pc=0xF0FC); run_instr(o)
    c = regs(o)["cycles"]; run_instr(o)
    assert regs(o)["cycles"] - c == 4 and regs(o)["pc"] == 0xF10F
    o.set_cpu(0, pc=0xF100); run_instr(o); c = regs(o)["cycles"]; run_instr(o)
    assert regs(o)["cycles"] - c == 4 and regs(o)["pc"] == 0xF0F3


def _adc_ref_binary(a, m, c):
    s = a + m + c
    sv = (a - 256 if a > 127 else a) + (m - 256 if m > 127 else m) + c
    return s & 0xFF, int(s > 255), int(sv < -128 or sv > 127)


def test_adc_sbc_binary_bruteforce(oracle_lib):
    ao, po = C.c_int(), C.c_int()
    for c in (0, 1):
        for a in range(256):
            for m in range(256):
                oracle_lib.ovcs_alu_adc(a, m, 0x24 | c, C.byref(ao), C.byref(po))
                r, cy, v = _adc_ref_binary(a, m, c)
                assert (ao.value, po.value & fC, (po.value & fV) >> 6) == (r, cy, v)
                assert bool(po.value & fZ) == (r == 0) and bool(po.value & fN) == (r > 127)
                assert po.value & 0x3C == 0x24                  # I, D, bit5 untouched
                # SBC: A - M - (1-C) over wide integers
                oracle_lib.ovcs_alu_sbc(a, m, 0x24 | c, C.byref(ao), C.byref(po))
                d = a - m - (1 - c)
                dv = (a - 256 if a > 127 else a) - (m - 256 if m > 127 else m) - (1 - c)
                assert ao.value == d & 0xFF and (po.value & fC) == int(d >= 0)
                assert bool(po.value & fV) == (dv < -128 or dv > 127)
                assert bool(po.value & fZ) == ((d & 0xFF) == 0) and bool(po.value & fN) == ((d & 0xFF) > 127)


def test_adc_sbc_decimal_valid_bcd_is_base100(oracle_lib):
    ao, po = C.c_int(), C.c_int()
    bcd = [t * 16 + u for t in range(10) for u in range(10)]
    for c in (0, 1):
        for ia, a in enumerate(bcd):
            for im, m in enumerate(bcd):
                oracle_lib.ovcs_alu_adc(a, m, 0x2C | c, C.byref(ao), C.byref(po))
                s = ia + im + c
                assert ao.value == bcd[s % 100] and (po.value & fC) == int(s >= 100)
                assert bool(po.value & fZ) == (((a + m + c) & 0xFF) == 0)      # Z from the binary sum (NMOS)
                assert po.value & fD
                oracle_lib.ovcs_alu_sbc(a, m, 0x2C | c, C.byref(ao), C.byref(po))
                d = ia - im - (1 - c)
                assert ao.value == bcd[d % 100] and (po.value & fC) == int(d >= 0)
                bd = a - m - (1 - c)                                             # flags exactly as binary
                assert bool(po.value & fZ) == ((bd & 0xFF) == 0) and bool(po.value & fN) == ((bd & 0xFF) > 127)


def test_decimal_hand_cases(oracle_lib):
    ao, po = C.c_int(), C.c_int()
    oracle_lib.ovcs_alu_adc(0x99, 0x01, 0x2C, C.byref(ao), C.byref(po))
    assert ao.value == 0x00 and po.value & fC and not (po.value & fZ)
    oracle_lib.ovcs_alu_adc(0x79, 0x00, 0x2D, C.byref(ao), C.byref(po))
    assert ao.value == 0x80 and po.value & fN and po.value & fV
    # invalid BCD (pinned by the cited algorithm only): 0x0F + 0x00 -> low-nibble fix-up gives 0x15
    oracle_lib.ovcs_alu_adc(0x0F, 0x00, 0x2C, C.byref(ao), C.byref(po))
    assert ao.value == 0x15 and not (po.value & fC)


@pytest.mark.parametrize("mn", ["ASL", "LSR", "ROL", "ROR"])
def test_shift_rotate_arithmetic_definitions(mn):
    def build(a):
        a.org(0xF000); a.op(mn, "acc")
    o = oracle_for(build)
    for c in (0, 1):
        for v in range(256):
            o.set_cpu(0, a=v, p=0x24 | c, pc=0xF000); run_instr(o)
            r = regs(o); res, cy = int(r["a"]), int(r["p"]) & 1
            if mn == "ASL": want, wc = (2 * v) % 256, v // 128
            elif mn == "LSR": want, wc = v // 2, v % 2
            elif mn == "ROL": want, wc = (2 * v + c) % 256, v // 128
            else: want, wc = v // 2 + 128 * c, v % 2
            assert (res, cy) == (want, wc)
            assert bool(r["p"] & fZ) == (want == 0) and bool(r["p"] & fN) == (want >= 128)
            assert r["p"] & 0x7C == 0x24                         # V, bit5, D, I untouched


def test_compare_and_bit_flags():
    def build(a):
        a.org(0xF000); a.op("CMP", "zp", 0x80); a.op("CPX", "zp", 0x80); a.op("CPY", "zp", 0x80); a.op("BIT", "zp", 0x80)
    o = oracle_for(build)
    for rv in range(0, 256, 3):
        for m in range(0, 256, 5):
            o.poke_ram(0, 0, m)
            for pc, reg in ((0xF000, "a"), (0xF002, "x"), (0xF004, "y")):
                o.set_cpu(0, p=0x64, pc=pc, **{reg: rv}); run_instr(o); p = int(regs(o)["p"])
                assert bool(p & fC) == (rv >= m) and bool(p & fZ) == (rv == m) and bool(p & fN) == (((rv - m) % 256) >= 128)
                assert p & fV                                    # V untouched (was set)
            o.set_cpu(0, a=rv, p=0x24, pc=0xF006); run_instr(o); p = int(regs(o)["p"])
            assert bool(p & fZ) == ((rv & m) == 0) and bool(p & fN) == (m >= 128) and bool(p & fV) == bool(m & 0x40)
            assert regs(o)["a"] == rv


def test_php_plp_pha_pla_and_stack_lands_in_ram():
    def build(a):
        a.org(0xF000); a.op("PHP"); a.op("PLA"); a.op("PHA"); a.op("PLP"); a.op("LDA", "imm", 0x7E); a.op("PHA")
    o = oracle_for(build); o.set_cpu(0, sp=0xFF, p=0xE5, pc=0xF000)
    run_instr(o)
    assert o.ram()[0][0x7F] == 0xE5 | 0x30 and regs(o)["sp"] == 0xFE          # pushed with B and bit5; ram[SP&0x7F]
    run_instr(o); assert regs(o)["a"] == 0xF5 and regs(o)["sp"] == 0xFF
    run_instr(o); run_instr(o)
    assert regs(o)["p"] == 0xE5                                               # bit4 dropped, bit5 forced
    run_instr(o, 2); assert o.ram()[0][0x7F] == 0x7E


def test_stack_wrap_and_tia_stack():
    def build(a):
        a.org(0xF000); a.op("PHA"); a.op("PHA"); a.op("PLA"); a.op("PLA")
    o = oracle_for(build); o.set_cpu(0, a=0x42, sp=0x80, pc=0xF000)
    run_instr(o); assert o.ram()[0][0] == 0x42 and regs(o)["sp"] == 0x7F
    run_instr(o); assert regs(o)["sp"] == 0x7E                 # $017F decodes to the TIA: no RAM change
    run_instr(o); run_instr(o); assert regs(o)["a"] == 0x42 and regs(o)["sp"] == 0x80


def test_jmp_indirect_page_wrap_and_jsr_rts():
    def build(a):
        a.org(0xF000); a.op("JMP", "ind", 0xFAFF)
        a.org(0xFAFF); a.byte(0x34)              # low byte at $FAFF, high byte taken from $FA00 (no carry)
        a.org(0xFA00); a.byte(0xF1)
        a.org(0xFB00); a.byte(0xF9)              # would be used if the carry propagated
        a.org(0xF134); a.op("JSR", "abs", 0xF200)
        a.op("NOP")
        a.org(0xF200); a.op("RTS")
    o = oracle_for(build); o.set_cpu(0, sp=0xFF, pc=0xF000)
    run_instr(o); assert regs(o)["pc"] == 0xF134
    c = regs(o)["cycles"]; run_instr(o)
    assert regs(o)["pc"] == 0xF200 and regs(o)["cycles"] - c == 6
    ram = o.ram()[0]; assert (ram[0x7F], ram[0x7E]) == (0xF1, 0x36)           # address of the JSR's 3rd byte
    run_instr(o); assert regs(o)["pc"] == 0xF137 and regs(o)["sp"] == 0xFF


def test_brk_rti():
    def build(a):
        a.org(0xF000); a.op("BRK"); a.byte(0xEA); a.op("NOP")
        a.org(0xF300); a.op("RTI")
    import vcs_inputs
    rom = bytearray(vcs_inputs.hand_rom(build)); rom[0xFFE] = 0x00; rom[0xFFF] = 0xF3
    from oracle.ovcs_py import OracleVCS
    o = OracleVCS([bytes(rom)], np.array([1], dtype=np.uint64)); o.set_cpu(0, sp=0xFF, p=0x61, pc=0xF000)
    c = regs(o)["cycles"]; run_instr(o)
    r = regs(o); assert r["pc"] == 0xF300 and r["cycles"] - c == 7 and r["p"] & fI and r["sp"] == 0xFC
    ram = o.ram()[0]; assert (ram[0x7F], ram[0x7E], ram[0x7D]) == (0xF0, 0x02, 0x61 | 0x30)
    run_instr(o); r = regs(o); assert r["pc"] == 0xF002 and r["p"] == 0x61 and r["sp"] == 0xFF


def test_ram_mirrors_and_zero_page_wrap():
    def build(a):
        a.org(0xF000); a.op("LDA", "imm", 0x5A); a.op("STA", "zp", 0x80); a.op("LDA", "abs", 0x0180)
        a.op("LDX", "imm", 0x90); a.op("LDY", "zpx", 0xF0)      # ($F0+$90)&$FF = $80, stays in page 0
        a.op("LDA", "imm", 0x33); a.op("STA", "abs", 0x0480); a.op("LDA", "zp", 0x80)
    o = oracle_for(build); run_instr(o, 3); assert regs(o)["a"] == 0x5A
    run_instr(o, 2); assert regs(o)["y"] == 0x5A
    run_instr(o, 3); assert regs(o)["a"] == 0x33


def test_izy_izx_pointer_wrap_in_zero_page():
    def build(a):
        a.org(0xF000); a.op("LDY", "imm", 0); a.op("LDA", "izy", 0xFF)        # pointer bytes at $FF and $00 (TIA read -> 0)
        a.op("LDX", "imm", 0x10); a.op("LDA", "izx", 0xEF)                    # pointer at ($EF+$10)&$FF = $FF,$00
    o = oracle_for(build); o.poke_ram(0, 0x7F, 0x80); o.poke_ram(0, 0, 0x77)  # -> $0080 = ram[0]
    run_instr(o, 2); assert regs(o)["a"] == 0x77
    o.set_cpu(0, a=0); run_instr(o, 2); assert regs(o)["a"] == 0x77


def test_undocumented_family_is_38_and_disjoint():
    assert len(UNDOC) == 38 and not (set(UNDOC) & set(MATRIX))             # 151 + USBC + 37 = 189
    assert sum(1 for v in UNDOC.values() if v[0] == "NOP") == 27 and sum(1 for v in UNDOC.values() if v[0] == "LAX") == 6
    assert sum(1 for v in UNDOC.values() if v[0] == "SAX") == 4 and UNDOC[0xEB][0] == "SBC"


def test_undocumented_behaviour():
    """NOPs change nothing but PC and time; LAX loads A and X with N,Z; SAX stores A & X without flags; USBC == SBC."""
    for code, (mn, mode, _, _) in UNDOC.items():
        n, r, o = _one(code, mode, False, p=0x24 | fC)
        ram = o.ram()[0]
        # operand value seen by the instruction in _one(): imm $12; zp/zpx/zpy -> RAM cell; abs $0080 -> RAM[0]; abx/aby $FA00+1 -> ROM $10/$F0; (zp,X)/(zp),Y -> $FA00(+1)
        if mn == "NOP":
            assert (r["a"], r["x"], r["y"], r["sp"], r["p"]) == (0x55, 0 if mode == "izx" else 1, 1, 0xFD, 0x24 | fC), hex(code)
        elif mn == "LAX":
            assert r["a"] == r["x"], hex(code)
            assert bool(r["p"] & fZ) == (r["a"] == 0) and bool(r["p"] & fN) == bool(r["a"] & 0x80)
        elif mn == "SAX":
            assert r["p"] == 0x24 | fC and r["a"] == 0x55                    # no flags, registers kept
    # LAX zp with a known byte; SAX zp stores A & X
    def build(a):
        a.org(0xF000); a.byte(0xA7, 0x90); a.byte(0x87, 0x91); a.byte(0xA7, 0x92)
    o = oracle_for(build)
    o.set_cpu(0, a=0, x=0, y=0, sp=0xFD, p=0x24, pc=0xF000); o.poke_ram(0, 0x10, 0xC3); o.poke_ram(0, 0x12, 0x00)
    run_instr(o); r = regs(o); assert r["a"] == 0xC3 and r["x"] == 0xC3 and r["p"] & fN and not r["p"] & fZ
    o.set_cpu(0, a=0xF0, x=0x3C); run_instr(o); assert o.ram()[0][0x11] == 0x30 and regs(o)["p"] & fN     # flags untouched by SAX
    run_instr(o); r = regs(o); assert r["a"] == 0 and r["x"] == 0 and r["p"] & fZ
    # USBC ($EB) == SBC #imm ($E9) on a sample of operands, binary and decimal
    rng = np.random.default_rng(7)
    for _ in range(200):
        a_, m_, p_ = int(rng.integers(256)), int(rng.integers(256)), 0x24 | int(rng.integers(2)) | (8 if rng.integers(2) else 0)
        res = []
        for opc in (0xE9, 0xEB):
            def build(a, opc=opc): a.org(0xF000); a.byte(opc, m_)
            o = oracle_for(build); o.set_cpu(0, a=a_, x=0, y=0, sp=0xFD, p=p_, pc=0xF000); run_instr(o)
            r = regs(o); res.append((int(r["a"]), int(r["p"]), int(r["cycles"])))
        assert res[0] == res[1]
