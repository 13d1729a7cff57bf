// vcs_decode.cuh — the pre-decoded instruction stream of the CUDA interpreter (shares nothing with oracle/).
//
// Cartridge ROM is immutable, so vcs_create decodes every byte offset of every bank ONCE into a 32-bit
// word; the interpreter kernel then dispatches on a fused handler id instead of walking opcode -> mode ->
// operation tables per executed instruction (the paper's cost centre is exactly that dispatch: PAPER.md
// L584/L592, a 256-way switch per step).  The decode is purely static: it never changes what an instruction
// does (SURVEY.md C.5 bus sequences), it only picks a specialised handler where the operand address class is
// known from the instruction bytes alone (immediate, zero-page RAM $80-$FF, zero-page TIA register stores).
//
//   bits  7:0   hid      handler id (enum Hid)
//   bits 23:8   payload  immediate | smem byte offset of a RAM cell | TIA register | b1|b2<<8 | branch displacement+2
//   bit  24     leader   a static branch / JMP / JSR target, a JSR return point or the instruction after a static
//                        bank-hotspot access: the warp re-forms its min-key group before executing it
//   bits 29:25  op2      second-level operation of a generic handler (read op 0..11, store 0..2, RMW 0..5),
//                        or the cycles of a taken branch (3 | 4)
//   bits 31:30  len      instruction length in bytes (1..3; 0 for H_SLOW)
//
// Offsets >= 0xFF0 of a bank (wrap-around, F8 hotspots inside the instruction bytes) and every PC outside
// cartridge space decode to H_SLOW: the kernel then fetches byte-wise with side effects and builds the
// word at run time from c_gen[] (generic handlers only).
#pragma once
#include <stdint.h>
#include "vcs_optable.cuh"

namespace vcs {

enum Hid : uint32_t {
  H_SLOW = 0,
  H_IMM0 = 1,        // +0..10: LDA LDX LDY AND ORA EOR ADC SBC CMP CPX CPY #imm
  H_ZR0 = 12,        // +0..11: LDA .. CPY, BIT  zp ($80-$FF: RAM)
  H_STZR0 = 24,      // +0..2 : STA STX STY zp RAM
  H_STZT0 = 27,      // +0..2 : STA STX STY zp TIA register (payload = register, one with an effect)
  H_NOP3 = 30,       // a zp store to a TIA address without effect (audio, RSYNC, $2D-$3F)
  H_MZR0 = 31,       // +0..5 : ASL LSR ROL ROR INC DEC zp RAM
  H_ACC0 = 37,       // +0..3 : ASL LSR ROL ROR A
  H_IMP0 = 41,       // +0..17: CLC SEC CLD SED CLI SEI CLV NOP DEX DEY INX INY TAX TAY TSX TXA TYA TXS
  H_BR0 = 59,        // +0..7 : BPL BMI BVC BVS BCC BCS BNE BEQ
  H_JMP = 67, H_JSR, H_RTS, H_PHA, H_PHP, H_PLA, H_PLP,
  H_R0 = 74,         // generic reads : +0..8  IMM ZP ZPX ZPY ABS ABX ABY IZX IZY   (op2 = read op)
  H_W0 = 83,         // generic stores: +0..7  ZP ZPX ZPY ABS ABX ABY IZX IZY       (op2 = STA STX STY)
  H_M0 = 91,         // generic RMW   : +0..3  ZP ZPX ABS ABX                       (op2 = ASL .. DEC)
  H_JMPI = 95, H_RTI, H_BRK, H_ILL,
  H_COUNT
};

constexpr uint32_t DW_LEADER = 1u << 24;
constexpr int DW_OP2_SHIFT = 25, DW_LEN_SHIFT = 30;
constexpr uint32_t DW_SLOW_LIMIT = 0xFF0;      // bank offsets >= this decode to H_SLOW

// generic (address-class agnostic) decode of one opcode: hid | op2<<8 | len<<13.  Used on the host as the base
// of every decode word and on the device (c_gen) by the byte-wise slow fetch.
inline uint16_t generic_entry(uint32_t opc) {
  const uint32_t ent = kOpTable[opc], mode = ent & 15u, op = (ent >> 4) & 63u, kind = ent >> 10;
  uint32_t hid = H_ILL, op2 = 0, len = 1;
  static const uint8_t mode_len[13] = {1, 1, 2, 2, 2, 2, 3, 3, 3, 2, 2, 2, 1};
  len = mode_len[mode];
  if (op == OP_ILL) { hid = H_ILL; len = 1; }
  else if (mode == MD_SPC) {
    switch (op) {
      case OP_JMP: hid = H_JMP; len = 3; break;   case OP_JMPI: hid = H_JMPI; len = 3; break;
      case OP_JSR: hid = H_JSR; len = 3; break;   case OP_RTS: hid = H_RTS; break;
      case OP_RTI: hid = H_RTI; break;            case OP_PHA: hid = H_PHA; break;
      case OP_PHP: hid = H_PHP; break;            case OP_PLA: hid = H_PLA; break;
      case OP_PLP: hid = H_PLP; break;            default: hid = H_BRK; len = 2; break;
    }
  }
  else if (mode == MD_REL) hid = H_BR0 + (op - OP_BPL);
  else if (mode == MD_IMP) hid = H_IMP0 + (op - OP_CLC);
  else if (mode == MD_ACC) hid = H_ACC0 + (op - OP_ASL);
  else if (kind == K_READ) { hid = H_R0 + (mode - MD_IMM); op2 = op - OP_LDA; }
  else if (kind == K_WRITE) { hid = H_W0 + (mode - MD_ZP); op2 = op - OP_STA; }
  else {                                          // K_RMW: zp, zpx, abs, abx
    const uint32_t mi = (mode == MD_ZP) ? 0u : (mode == MD_ZPX) ? 1u : (mode == MD_ABS) ? 2u : 3u;
    hid = H_M0 + mi; op2 = op - OP_ASL;
  }
  return (uint16_t)(hid | (op2 << 8) | (len << 13));
}

inline bool tia_write_has_effect(uint32_t r) {    // r = address & 0x3F (SURVEY C.8 write map)
  return !(r > 0x2Cu || (r >= 0x15u && r <= 0x1Au) || r == 0x03u);
}

// One bank image (4096 bytes; 2 KB carts are passed mirrored) -> 4096 decode words.  `leader` is the bank-
// independent leader bitmap (4096 flags) filled by mark_leaders() for every bank of the cartridge first.
inline void decode_bank(const uint8_t *img, const uint8_t *leader, int block, uint32_t *out) {
  for (uint32_t off = 0; off < 4096; ++off) {
    if (off >= DW_SLOW_LIMIT) { out[off] = H_SLOW | (leader[off] ? DW_LEADER : 0u); continue; }
    const uint32_t opc = img[off], b1 = img[off + 1], b2 = img[off + 2];
    const uint32_t ent = kOpTable[opc], mode = ent & 15u, op = (ent >> 4) & 63u, kind = ent >> 10;
    const uint16_t g = generic_entry(opc);
    uint32_t hid = g & 0xFFu, op2 = (g >> 8) & 31u;
    const uint32_t len = g >> 13;
    uint32_t payload = (len == 3) ? (b1 | (b2 << 8)) : (len == 2) ? b1 : 0u;
    if (op != OP_ILL) {
      if (mode == MD_IMM) { hid = H_IMM0 + (op - OP_LDA); op2 = 0; }
      else if (mode == MD_ZP && b1 >= 0x80u) {
        payload = ((b1 & 0x7Cu) * (uint32_t)block) | (b1 & 3u);          // byte offset of the cell in the RAM words
        if (kind == K_READ) hid = H_ZR0 + (op - OP_LDA);
        else if (kind == K_WRITE) hid = H_STZR0 + (op - OP_STA);
        else hid = H_MZR0 + (op - OP_ASL);
        op2 = 0;
      }
      else if (mode == MD_ZP && kind == K_WRITE) {                         // b1 < 0x80: a TIA register
        const uint32_t r = b1 & 0x3Fu;
        if (tia_write_has_effect(r)) { hid = H_STZT0 + (op - OP_STA); payload = r; }
        else { hid = H_NOP3; payload = 0; }
        op2 = 0;
      }
      else if (mode == MD_REL) {
        const uint32_t next = 0x1000u + off + 2u, target = (next + (uint32_t)(int32_t)(int8_t)b1) & 0xFFFFu;
        payload = (2u + (uint32_t)(int32_t)(int8_t)b1) & 0xFFFFu;
        op2 = ((target ^ next) & 0xFF00u) ? 4u : 3u;
      }
    }
    out[off] = hid | (payload << 8) | (leader[off] ? DW_LEADER : 0u) | (op2 << DW_OP2_SHIFT) | (len << DW_LEN_SHIFT);
  }
}

// static control-flow targets of one bank image, OR-ed into `leader` (shared by all banks of the cartridge:
// a jump may land in whichever bank is selected at that moment)
inline void mark_leaders(const uint8_t *img, uint8_t *leader) {
  for (uint32_t off = 0; off + 2 < 4096; ++off) {
    const uint32_t opc = img[off], b1 = img[off + 1], b2 = img[off + 2];
    const uint32_t ent = kOpTable[opc], mode = ent & 15u, op = (ent >> 4) & 63u;
    if (op == OP_ILL) continue;
    if (mode == MD_REL) leader[(off + 2u + (uint32_t)(int32_t)(int8_t)b1) & 0xFFFu] = 1;
    else if (op == OP_JMP || op == OP_JSR) {
      const uint32_t a = b1 | (b2 << 8);
      if (a & 0x1000u) leader[a & 0xFFFu] = 1;
      if (op == OP_JSR) leader[(off + 3u) & 0xFFFu] = 1;
    }
    else if (mode == MD_ABS || mode == MD_ABX || mode == MD_ABY) {         // static hotspot access: regroup after it
      const uint32_t a = (b1 | (b2 << 8)) & 0x1FFFu;
      if ((a | 1u) == 0x1FF9u) leader[(off + 3u) & 0xFFFu] = 1;
    }
  }
}

}  // namespace vcs
