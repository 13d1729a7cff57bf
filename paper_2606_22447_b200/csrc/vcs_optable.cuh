// vcs_optable.cuh — 6507 decode table for the CUDA interpreter, in opcode order.
// The 151 documented NMOS 6502 opcodes (SURVEY.md §8(c) C.5 matrix [D]) plus the 38 undocumented bytes
// of the paper's ports (USBC + the NOP / LAX / SAX family: tests/golden/undocumented_opcodes.txt); every other byte
// decodes to OP_ILL (C.12).  Entry = mode | op<<4 | kind<<10.
#pragma once
#include <stdint.h>

namespace vcs {

enum Mode : uint32_t { MD_IMP = 0, MD_ACC, MD_IMM, MD_ZP, MD_ZPX, MD_ZPY, MD_ABS, MD_ABX, MD_ABY, MD_IZX, MD_IZY,
                       MD_REL, MD_SPC };
enum Kind : uint32_t { K_NONE = 0, K_READ = 1, K_WRITE = 2, K_RMW = 3 };
enum Op : uint32_t {
  OP_ILL = 0,
  // K_READ (operand value v)
  OP_LDA, OP_LDX, OP_LDY, OP_AND, OP_ORA, OP_EOR, OP_ADC, OP_SBC, OP_CMP, OP_CPX, OP_CPY, OP_BIT,
  OP_LAX, OP_NOPR,          // undocumented: A = X = v ; read and discard (NOP with an operand)
  // K_WRITE
  OP_STA, OP_STX, OP_STY, OP_SAX,     // SAX (undocumented): stores A & X
  // K_RMW (or accumulator)
  OP_ASL, OP_LSR, OP_ROL, OP_ROR, OP_INC, OP_DEC,
  // implied
  OP_CLC, OP_SEC, OP_CLD, OP_SED, OP_CLI, OP_SEI, OP_CLV, OP_NOP, OP_DEX, OP_DEY, OP_INX, OP_INY,
  OP_TAX, OP_TAY, OP_TSX, OP_TXA, OP_TYA, OP_TXS,
  // branches: OP_BR + (condition index): flag = idx>>1 (0 N, 1 V, 2 C, 3 Z), taken when flag == idx&1
  OP_BPL, OP_BMI, OP_BVC, OP_BVS, OP_BCC, OP_BCS, OP_BNE, OP_BEQ,
  // special sequences
  OP_JMP, OP_JMPI, OP_JSR, OP_RTS, OP_RTI, OP_PHA, OP_PHP, OP_PLA, OP_PLP, OP_BRK,
  OP_COUNT
};
static_assert(OP_COUNT <= 64, "op field is 6 bits");

#define E(op, md, k) (uint16_t)((md) | ((op) << 4) | ((k) << 10))
#define ILL E(OP_ILL, MD_IMP, K_NONE)
#define RD(op, md) E(OP_##op, MD_##md, K_READ)
#define WRT(op, md) E(OP_##op, MD_##md, K_WRITE)
#define RMW(op, md) E(OP_##op, MD_##md, K_RMW)
#define ACC(op) E(OP_##op, MD_ACC, K_NONE)
#define IMP(op) E(OP_##op, MD_IMP, K_NONE)
#define BR(op) E(OP_##op, MD_REL, K_NONE)
#define SPC(op) E(OP_##op, MD_SPC, K_NONE)

static const uint16_t kOpTable[256] = {
  /*00*/ SPC(BRK), RD(ORA, IZX), ILL, ILL, RD(NOPR, ZP), RD(ORA, ZP), RMW(ASL, ZP), ILL, SPC(PHP), RD(ORA, IMM), ACC(ASL), ILL, RD(NOPR, ABS), RD(ORA, ABS), RMW(ASL, ABS), ILL,
  /*10*/ BR(BPL), RD(ORA, IZY), ILL, ILL, RD(NOPR, ZPX), RD(ORA, ZPX), RMW(ASL, ZPX), ILL, IMP(CLC), RD(ORA, ABY), IMP(NOP), ILL, RD(NOPR, ABX), RD(ORA, ABX), RMW(ASL, ABX), ILL,
  /*20*/ SPC(JSR), RD(AND, IZX), ILL, ILL, RD(BIT, ZP), RD(AND, ZP), RMW(ROL, ZP), ILL, SPC(PLP), RD(AND, IMM), ACC(ROL), ILL, RD(BIT, ABS), RD(AND, ABS), RMW(ROL, ABS), ILL,
  /*30*/ BR(BMI), RD(AND, IZY), ILL, ILL, RD(NOPR, ZPX), RD(AND, ZPX), RMW(ROL, ZPX), ILL, IMP(SEC), RD(AND, ABY), IMP(NOP), ILL, RD(NOPR, ABX), RD(AND, ABX), RMW(ROL, ABX), ILL,
  /*40*/ SPC(RTI), RD(EOR, IZX), ILL, ILL, RD(NOPR, ZP), RD(EOR, ZP), RMW(LSR, ZP), ILL, SPC(PHA), RD(EOR, IMM), ACC(LSR), ILL, SPC(JMP), RD(EOR, ABS), RMW(LSR, ABS), ILL,
  /*50*/ BR(BVC), RD(EOR, IZY), ILL, ILL, RD(NOPR, ZPX), RD(EOR, ZPX), RMW(LSR, ZPX), ILL, IMP(CLI), RD(EOR, ABY), IMP(NOP), ILL, RD(NOPR, ABX), RD(EOR, ABX), RMW(LSR, ABX), ILL,
  /*60*/ SPC(RTS), RD(ADC, IZX), ILL, ILL, RD(NOPR, ZP), RD(ADC, ZP), RMW(ROR, ZP), ILL, SPC(PLA), RD(ADC, IMM), ACC(ROR), ILL, SPC(JMPI), RD(ADC, ABS), RMW(ROR, ABS), ILL,
  /*70*/ BR(BVS), RD(ADC, IZY), ILL, ILL, RD(NOPR, ZPX), RD(ADC, ZPX), RMW(ROR, ZPX), ILL, IMP(SEI), RD(ADC, ABY), IMP(NOP), ILL, RD(NOPR, ABX), RD(ADC, ABX), RMW(ROR, ABX), ILL,
  /*80*/ RD(NOPR, IMM), WRT(STA, IZX), RD(NOPR, IMM), WRT(SAX, IZX), WRT(STY, ZP), WRT(STA, ZP), WRT(STX, ZP), WRT(SAX, ZP), IMP(DEY), RD(NOPR, IMM), IMP(TXA), ILL, WRT(STY, ABS), WRT(STA, ABS), WRT(STX, ABS), WRT(SAX, ABS),
  /*90*/ BR(BCC), WRT(STA, IZY), ILL, ILL, WRT(STY, ZPX), WRT(STA, ZPX), WRT(STX, ZPY), WRT(SAX, ZPY), IMP(TYA), WRT(STA, ABY), IMP(TXS), ILL, ILL, WRT(STA, ABX), ILL, ILL,
  /*A0*/ RD(LDY, IMM), RD(LDA, IZX), RD(LDX, IMM), RD(LAX, IZX), RD(LDY, ZP), RD(LDA, ZP), RD(LDX, ZP), RD(LAX, ZP), IMP(TAY), RD(LDA, IMM), IMP(TAX), ILL, RD(LDY, ABS), RD(LDA, ABS), RD(LDX, ABS), RD(LAX, ABS),
  /*B0*/ BR(BCS), RD(LDA, IZY), ILL, RD(LAX, IZY), RD(LDY, ZPX), RD(LDA, ZPX), RD(LDX, ZPY), RD(LAX, ZPY), IMP(CLV), RD(LDA, ABY), IMP(TSX), ILL, RD(LDY, ABX), RD(LDA, ABX), RD(LDX, ABY), RD(LAX, ABY),
  /*C0*/ RD(CPY, IMM), RD(CMP, IZX), RD(NOPR, IMM), ILL, RD(CPY, ZP), RD(CMP, ZP), RMW(DEC, ZP), ILL, IMP(INY), RD(CMP, IMM), IMP(DEX), ILL, RD(CPY, ABS), RD(CMP, ABS), RMW(DEC, ABS), ILL,
  /*D0*/ BR(BNE), RD(CMP, IZY), ILL, ILL, RD(NOPR, ZPX), RD(CMP, ZPX), RMW(DEC, ZPX), ILL, IMP(CLD), RD(CMP, ABY), IMP(NOP), ILL, RD(NOPR, ABX), RD(CMP, ABX), RMW(DEC, ABX), ILL,
  /*E0*/ RD(CPX, IMM), RD(SBC, IZX), RD(NOPR, IMM), ILL, RD(CPX, ZP), RD(SBC, ZP), RMW(INC, ZP), ILL, IMP(INX), RD(SBC, IMM), IMP(NOP), RD(SBC, IMM), RD(CPX, ABS), RD(SBC, ABS), RMW(INC, ABS), ILL,
  /*F0*/ BR(BEQ), RD(SBC, IZY), ILL, ILL, RD(NOPR, ZPX), RD(SBC, ZPX), RMW(INC, ZPX), ILL, IMP(SED), RD(SBC, ABY), IMP(NOP), ILL, RD(NOPR, ABX), RD(SBC, ABX), RMW(INC, ABX), ILL,
};
#undef E
#undef ILL
#undef RD
#undef WRT
#undef RMW
#undef ACC
#undef IMP
#undef BR
#undef SPC

}  // namespace vcs
