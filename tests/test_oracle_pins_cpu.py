"""More pins for the oracle's 6507 ALU and RIOT timer:
  * decimal ADC / SBC — N, V, Z, C and the value — on hand-worked cases (invalid BCD included) and, over all
    2 x 256 x 256 inputs, against a digit-serial model of the NMOS adder (two 4-bit stages with a decimal-adjust on
    each carry), which is a different construction from the oracle's whole-byte formulation of C.6;
  * N, Z of every load / logic / increment / decrement / transfer / pull, over all 256 results;
  * the per-cycle timer rule against the C.7 closed form for ALL N in 0..255 x 4 divisors, every cycle up to N*D + 600.
Expected values are worked by hand or come from the independent constructions in this file, never from the oracle."""
import ctypes as C

import numpy as np
import pytest

from helpers import oracle_for, run_instr, regs, RIOT, TIA_W

fC, fZ, fI, fD, fV, fN = 1, 2, 4, 8, 0x40, 0x80

# (A, M, C_in) -> (A', N, V, Z, C_out), decimal mode, NMOS.  Worked by hand from C.6: the low digits are added and
# decimal-adjusted first; N and V are those of the sum BEFORE the high digit is adjusted; Z is that of the binary sum.
ADC_DEC = [
    ((0x00, 0x00, 0), (0x00, 0, 0, 1, 0)),
    ((0x00, 0x00, 1), (0x01, 0, 0, 0, 0)),
    ((0x99, 0x01, 0), (0x00, 1, 0, 0, 1)),       # Z = 0 although A' = 0 (binary sum 0x9A)
    ((0x79, 0x00, 1), (0x80, 1, 1, 0, 0)),
    ((0x58, 0x46, 1), (0x05, 1, 1, 0, 1)),       # 58 + 46 + 1 = 105
    ((0x12, 0x34, 0), (0x46, 0, 0, 0, 0)),
    ((0x15, 0x26, 0), (0x41, 0, 0, 0, 0)),
    ((0x81, 0x92, 0), (0x73, 0, 1, 0, 1)),       # 81 + 92 = 173
    ((0x50, 0x50, 0), (0x00, 1, 1, 0, 1)),       # 100: A' = 0 but Z = 0
    ((0x99, 0x99, 1), (0x99, 0, 1, 0, 1)),       # 199
    ((0x49, 0x50, 1), (0x00, 1, 1, 0, 1)),
    ((0x09, 0x01, 0), (0x10, 0, 0, 0, 0)),
    ((0x7F, 0x01, 0), (0x86, 1, 1, 0, 0)),       # invalid low digit F
    ((0x80, 0x80, 0), (0x60, 0, 1, 1, 1)),       # binary sum 0x100 -> Z = 1 while A' = 0x60
    ((0xF0, 0x10, 0), (0x60, 0, 0, 1, 1)),
    ((0x0F, 0x00, 0), (0x15, 0, 0, 0, 0)),       # invalid BCD from here on
    ((0x0A, 0x0A, 0), (0x1A, 0, 0, 0, 0)),
    ((0xFF, 0xFF, 1), (0x55, 1, 0, 0, 1)),
    ((0xA0, 0x00, 0), (0x00, 1, 0, 0, 1)),
    ((0x9A, 0x00, 0), (0x00, 1, 0, 0, 1)),
    ((0x1B, 0x2C, 0), (0x4D, 0, 0, 0, 0)),
    ((0xD5, 0x38, 1), (0x74, 0, 0, 0, 1)),
    ((0x6E, 0x3F, 0), (0x03, 1, 1, 0, 1)),
    ((0x40, 0x3F, 0), (0x85, 1, 1, 0, 0)),
]
# (A, M, C_in) -> (A', N, V, Z, C_out), decimal SBC: the flags are those of the binary subtraction
SBC_DEC = [
    ((0x00, 0x01, 1), (0x99, 1, 0, 0, 0)),
    ((0x46, 0x12, 1), (0x34, 0, 0, 0, 1)),
    ((0x40, 0x13, 1), (0x27, 0, 0, 0, 1)),
    ((0x32, 0x02, 0), (0x29, 0, 0, 0, 1)),
    ((0x12, 0x21, 1), (0x91, 1, 0, 0, 0)),
    ((0x21, 0x34, 1), (0x87, 1, 0, 0, 0)),
    ((0x80, 0x01, 1), (0x79, 0, 1, 0, 1)),       # -128 - 1 overflows
    ((0x00, 0x00, 0), (0x99, 1, 0, 0, 0)),
    ((0x50, 0x50, 1), (0x00, 0, 0, 1, 1)),
    ((0x0A, 0x00, 1), (0x0A, 0, 0, 0, 1)),       # invalid BCD from here on
    ((0x00, 0x0F, 1), (0x9B, 1, 0, 0, 0)),
    ((0x1F, 0x0A, 0), (0x14, 0, 0, 0, 1)),
    ((0xF0, 0x0F, 1), (0xEB, 1, 0, 0, 1)),
]


def _flags(p):
    return (int(bool(p & fN)), int(bool(p & fV)), int(bool(p & fZ)), int(bool(p & fC)))


@pytest.mark.parametrize("inp,want", ADC_DEC, ids=[f"{a:02X}+{m:02X}+{c}" for (a, m, c), _ in ADC_DEC])
def test_decimal_adc_hand_cases(oracle_lib, inp, want):
    ao, po = C.c_int(), C.c_int()
    a, m, c = inp
    oracle_lib.ovcs_alu_adc(a, m, 0x2C | c, C.byref(ao), C.byref(po))
    assert (ao.value,) + _flags(po.value) == want
    assert po.value & 0x3C == 0x2C                                   # D, I, bit 5 untouched


@pytest.mark.parametrize("inp,want", SBC_DEC, ids=[f"{a:02X}-{m:02X}-{1 - c}" for (a, m, c), _ in SBC_DEC])
def test_decimal_sbc_hand_cases(oracle_lib, inp, want):
    ao, po = C.c_int(), C.c_int()
    a, m, c = inp
    oracle_lib.ovcs_alu_sbc(a, m, 0x2C | c, C.byref(ao), C.byref(po))
    assert (ao.value,) + _flags(po.value) == want
    assert po.value & 0x3C == 0x2C


def _digit_serial_adc(a, m, c):
    """The NMOS decimal adder as two 4-bit stages: a stage whose sum exceeds 9 adds 6 and carries 1 into the next.
    N / V are those of the second stage BEFORE its own adjustment, Z that of the plain binary sum."""
    lo = (a & 15) + (m & 15) + c
    half = lo > 9
    if half:
        lo = (lo + 6) & 15
    hi = (a >> 4) + (m >> 4) + (1 if half else 0)
    n = (hi >> 3) & 1
    v = 1 if (((a ^ m) & 0x80) == 0 and ((a >> 7) & 1) != n) else 0       # both operands of one sign, the raw high digit of the other
    z = 1 if ((a + m + c) & 0xFF) == 0 else 0
    carry = hi > 9
    if carry:
        hi = (hi + 6) & 15
    return ((hi & 15) << 4) | lo, n, v, z, int(carry)


def _digit_serial_sbc(a, m, c):
    lo = (a & 15) - (m & 15) - (1 - c)
    borrow = lo < 0
    if borrow:
        lo = (lo - 6) & 15
    hi = (a >> 4) - (m >> 4) - (1 if borrow else 0)
    if hi < 0:
        hi = (hi - 6) & 15
    d = a - m - (1 - c)                                                    # flags: the binary subtraction over wide integers
    dv = (a - 256 if a > 127 else a) - (m - 256 if m > 127 else m) - (1 - c)
    return ((hi & 15) << 4) | lo, ((d & 0xFF) >> 7) & 1, int(dv < -128 or dv > 127), int((d & 0xFF) == 0), int(d >= 0)


def test_digit_serial_models_agree_with_the_hand_cases():
    for (a, m, c), want in ADC_DEC:
        assert _digit_serial_adc(a, m, c) == want, (hex(a), hex(m), c)
    for (a, m, c), want in SBC_DEC:
        assert _digit_serial_sbc(a, m, c) == want, (hex(a), hex(m), c)


def test_decimal_adc_sbc_all_inputs_against_the_digit_serial_adder(oracle_lib):
    ao, po = C.c_int(), C.c_int()
    for c in (0, 1):
        for a in range(256):
            for m in range(256):
                oracle_lib.ovcs_alu_adc(a, m, 0x2C | c, C.byref(ao), C.byref(po))
                assert (ao.value,) + _flags(po.value) == _digit_serial_adc(a, m, c), ("adc", hex(a), hex(m), c)
                oracle_lib.ovcs_alu_sbc(a, m, 0x2C | c, C.byref(ao), C.byref(po))
                assert (ao.value,) + _flags(po.value) == _digit_serial_sbc(a, m, c), ("sbc", hex(a), hex(m), c)


# ---------------------------------------------------------------------------------------------- N, Z of everything else
def _nz(v):
    return (fN if v & 0x80 else 0) | (fZ if v == 0 else 0)


MVALS = [0x00, 0xFF, 0x0F, 0xF0, 0x55, 0xAA, 0x01, 0x02, 0x04, 0x08, 0x10, 0x20, 0x40, 0x80, 0x7F, 0xFE, 0x33, 0xC3]


@pytest.mark.parametrize("mn,fn", [("AND", lambda a, m: a & m), ("ORA", lambda a, m: a | m), ("EOR", lambda a, m: a ^ m)])
def test_logic_ops_value_and_nz(mn, fn):
    def build(a):
        a.org(0xF000); a.op(mn, "zp", 0x80)
    o = oracle_for(build)
    for m in MVALS:
        o.poke_ram(0, 0, m)
        for av in range(256):
            for p0 in (0x24, 0xE7):                                  # every other flag clear / set beforehand
                o.set_cpu(0, a=av, p=p0, pc=0xF000); run_instr(o); r = regs(o)
                want = fn(av, m)
                assert r["a"] == want and r["p"] == (p0 & ~(fN | fZ)) | _nz(want), (mn, hex(av), hex(m))


@pytest.mark.parametrize("mn,reg", [("LDA", "a"), ("LDX", "x"), ("LDY", "y")])
def test_loads_nz(mn, reg):
    def build(a):
        a.org(0xF000); a.op(mn, "zp", 0x80)
    o = oracle_for(build)
    for v in range(256):
        for p0 in (0x24, 0xE7):
            o.poke_ram(0, 0, v); o.set_cpu(0, a=0x11, x=0x22, y=0x33, p=p0, pc=0xF000); run_instr(o); r = regs(o)
            assert r[reg] == v and r["p"] == (p0 & ~(fN | fZ)) | _nz(v)
            assert [int(r[k]) for k in "axy" if k != reg] == [x for k, x in zip("axy", (0x11, 0x22, 0x33)) if k != reg]


@pytest.mark.parametrize("mn,delta", [("INC", 1), ("DEC", -1)])
def test_inc_dec_memory_nz_and_carry_untouched(mn, delta):
    def build(a):
        a.org(0xF000); a.op(mn, "zp", 0x80)
    o = oracle_for(build)
    for v in range(256):
        for p0 in (0x24, 0xE7):
            o.poke_ram(0, 0, v); o.set_cpu(0, a=0x5A, p=p0, pc=0xF000); run_instr(o); r = regs(o)
            want = (v + delta) & 0xFF
            assert o.ram()[0][0] == want and r["p"] == (p0 & ~(fN | fZ)) | _nz(want) and r["a"] == 0x5A


@pytest.mark.parametrize("mn,reg,delta", [("INX", "x", 1), ("INY", "y", 1), ("DEX", "x", -1), ("DEY", "y", -1)])
def test_inx_iny_dex_dey(mn, reg, delta):
    def build(a):
        a.org(0xF000); a.op(mn)
    o = oracle_for(build)
    for v in range(256):
        for p0 in (0x24, 0xE7):
            o.set_cpu(0, a=7, x=v, y=v, p=p0, pc=0xF000); run_instr(o); r = regs(o)
            want = (v + delta) & 0xFF
            other = "y" if reg == "x" else "x"
            assert r[reg] == want and r[other] == v and r["a"] == 7 and r["p"] == (p0 & ~(fN | fZ)) | _nz(want)


@pytest.mark.parametrize("mn,src,dst", [("TAX", "a", "x"), ("TAY", "a", "y"), ("TXA", "x", "a"), ("TYA", "y", "a"), ("TSX", "sp", "x")])
def test_transfers_nz(mn, src, dst):
    def build(a):
        a.org(0xF000); a.op(mn)
    o = oracle_for(build)
    for v in range(256):
        for p0 in (0x24, 0xE7):
            init = dict(a=0x11, x=0x22, y=0x33, sp=0x44); init[src] = v
            o.set_cpu(0, p=p0, pc=0xF000, **init); run_instr(o); r = regs(o)
            init[dst] = v
            assert {k: int(r[k]) for k in init} == init and r["p"] == (p0 & ~(fN | fZ)) | _nz(v)


def test_txs_sets_no_flags_and_pla_sets_nz():
    def build(a):
        a.org(0xF000); a.op("TXS"); a.op("PLA")
    o = oracle_for(build)
    for v in range(256):
        for p0 in (0x24, 0xE7):
            o.set_cpu(0, a=1, x=v, sp=0x10, p=p0, pc=0xF000); run_instr(o); r = regs(o)
            assert r["sp"] == v and r["p"] == p0                      # TXS: no flags (C.6)
            o.poke_ram(0, 0x55, v); o.set_cpu(0, sp=0xD4, p=p0, pc=0xF001); run_instr(o); r = regs(o)     # pulls from $01D5 -> ram[$55]
            assert r["a"] == v and r["sp"] == 0xD5 and r["p"] == (p0 & ~(fN | fZ)) | _nz(v)


def test_flag_instructions_touch_one_bit_each():
    ops = [("CLC", fC, 0), ("SEC", fC, 1), ("CLD", fD, 0), ("SED", fD, 1), ("CLI", fI, 0), ("SEI", fI, 1), ("CLV", fV, 0)]
    def build(a):
        a.org(0xF000)
        for mn, _, _ in ops: a.op(mn)
    o = oracle_for(build)
    for i, (mn, bit, val) in enumerate(ops):
        for p0 in (0x20, 0xEF):
            o.set_cpu(0, p=p0, pc=0xF000 + i); run_instr(o)
            assert regs(o)["p"] == ((p0 | bit) if val else (p0 & ~bit)) | 0x20, mn


# ---------------------------------------------------------------------------------------------- RIOT timer, all N
SHIFT = {"TIM1T": 0, "TIM8T": 3, "TIM64T": 6, "T1024T": 10}


def _closed_form_vec(N, shift, n):
    """C.7 closed form for dt = 1..n cycles after the write: (value, flag) arrays."""
    dt = np.arange(1, n + 1, dtype=np.int64)
    cu = 1 + (N << shift)                                             # the underflow cycle
    before = N - 1 - ((dt - 1) >> shift)
    after = (0xFF - (dt - cu)) & 0xFF
    flag = (dt >= cu).astype(np.uint8)
    return np.where(dt < cu, before, after).astype(np.uint8), flag


@pytest.mark.parametrize("reg", list(SHIFT))
def test_riot_timer_every_n_every_cycle_against_the_closed_form(reg):
    shift = SHIFT[reg]
    for N in range(256):
        def build(a, N=N):
            a.org(0xF000); a.op("LDA", "imm", 2); a.op("STA", "zp", TIA_W["VBLANK"])        # (blanked: the idle cycles render nothing)
            a.op("LDA", "imm", N); a.op("STA", "abs", RIOT[reg])
        o = oracle_for(build); run_instr(o, 4)
        d = o.debug(0); assert d.timer == N and d.tflag == 0 and d.shift == shift
        n = (N << shift) + 600
        t, f = o.tick_trace(n)
        wt, wf = _closed_form_vec(N, shift, n)
        bad = np.nonzero((t != wt) | (f != wf))[0]
        assert bad.size == 0, (reg, N, "first mismatch at dt", int(bad[0]) + 1, int(t[bad[0]]), int(wt[bad[0]]))
