// vcs_decode.cuh — the pre-decoded instruction stream of the CUDA interpreter (shares nothing with oracle/).
//
// Cartridge ROM is immutable, so vcs_create decodes every byte offset of every bank ONCE into a 64-bit
// entry; the interpreter kernel then dispatches on a fused handler id instead of walking opcode -> mode ->
// operation tables per executed instruction (the paper's cost centre is exactly that dispatch: PAPER.md
// L584/L592, a 256-way switch per step).  The decode is purely static: it never changes what an instruction
// does (SURVEY.md C.5 bus sequences), it only picks a specialised handler where the operand's address class
// is known from the instruction bytes alone (immediate, RAM, TIA register stores, RIOT timer reads, fixed
// ROM bytes), and it carries the instruction's base cycle count and length so that the kernel adds them
// without looking anything up.
//
//   .x  bits  6:0   hid      handler id (enum Hid)
//       bit   7     leader   a static branch / JMP / JSR target, a JSR return point or the instruction after a
//                            static bank-hotspot access: the warp re-forms its min-key group before executing it
//       bits 15:8   cy       base cycles (0 for the generic handlers, which count their own bus accesses)
//       bits 23:16  len      instruction length in bytes (0 for H_SLOW / H_ILL)
//       bits 31:24  op2      second-level operation of a generic handler (read op 0..11, store 0..2, RMW 0..5),
//                            or the extra cycles of a taken branch (1 | 2)
//   .y  payload     immediate | smem byte offset of a RAM cell | TIA register | b1|b2<<8 | signed branch displacement
//
// Offsets >= 0xFF0 of a bank (wrap-around, F8 hotspots inside the instruction bytes), branches that leave
// the 4 KB window or whose dummy reads can touch a hotspot, and every PC outside cartridge space decode to
// H_SLOW: the kernel then fetches byte-wise with side effects and builds the entry at run time from c_gen[]
// (generic handlers only).
#pragma once
#include <stdint.h>
#include "vcs_optable.cuh"

namespace vcs {

enum Hid : uint32_t {
  H_SLOW = 0,
  H_IMM0 = 1,        // +0..10: LDA LDX LDY AND ORA EOR ADC SBC CMP CPX CPY #imm (also: absolute reads of a fixed ROM byte)
  H_ZR0 = 12,        // +0..11: LDA .. CPY, BIT  RAM cell (zp $80-$FF, or an absolute address that decodes to RAM)
  H_STZR0 = 24,      // +0..2 : STA STX STY RAM cell
  H_STZT0 = 27,      // +0..2 : STA STX STY TIA register (payload = register, one with an effect), written in the last cycle
  H_NOP = 30,        // no effect beyond its cycles (NOP; a store to a TIA address without effect: audio, RSYNC, $2D-$3F)
  H_MZR0 = 31,       // +0..5 : ASL LSR ROL ROR INC DEC RAM cell
  H_ACC0 = 37,       // +0..3 : ASL LSR ROL ROR A
  H_IMP0 = 41,       // +0..17: CLC SEC CLD SED CLI SEI CLV (NOP) DEX DEY INX INY TAX TAY TSX TXA TYA TXS
  H_BR0 = 59,        // +0..7 : BPL BMI BVC BVS BCC BCS BNE BEQ
  H_JMP = 67, H_JSR, H_RTS, H_PHA, H_PHP, H_PLA, H_PLP,
  H_R0 = 74,         // generic reads : +0..8  IMM ZP ZPX ZPY ABS ABX ABY IZX IZY   (op2 = read op)
  H_W0 = 83,         // generic stores: +0..7  ZP ZPX ZPY ABS ABX ABY IZX IZY       (op2 = STA STX STY)
  H_M0 = 91,         // generic RMW   : +0..3  ZP ZPX ABS ABX                       (op2 = ASL .. DEC)
  H_JMPI = 95, H_RTI, H_BRK, H_ILL,
  H_RTIM = 99,       // absolute read of INTIM / TIMINT (payload = address, op2 = read op)
  H_COUNT
};
static_assert(H_COUNT <= 128, "hid is 7 bits");

constexpr uint32_t DW_LEADER = 1u << 7;
// one-bit class flags of the four classes that make up most executed entries (bits 12..15; cy itself is < 16): the
// interpreter tests them before it looks at the class number at all
constexpr uint32_t DW_F_LDST = 1u << 12, DW_F_STTIA = 1u << 13, DW_F_LDIMM = 1u << 14, DW_F_BR = 1u << 15;
constexpr int DW_CY_SHIFT = 8, DW_LEN_SHIFT = 16, DW_OP2_SHIFT = 24;
constexpr uint32_t DW_SLOW_LIMIT = 0xFF0;      // bank offsets >= this decode to H_SLOW

struct DWord { uint32_t x, y; };

constexpr uint32_t dw_x(uint32_t hid, uint32_t cy, uint32_t len, uint32_t op2) {
  return hid | (cy << DW_CY_SHIFT) | (len << DW_LEN_SHIFT) | (op2 << DW_OP2_SHIFT);
}

// generic (address-class agnostic) decode of one opcode in the .x format.  Used on the host as the base of
// every decode entry and on the device (c_gen) by the byte-wise slow fetch.
inline uint32_t generic_entry(uint32_t opc) {
  const uint32_t ent = kOpTable[opc], mode = ent & 15u, op = (ent >> 4) & 63u, kind = ent >> 10;
  static const uint8_t mode_len[13] = {1, 1, 2, 2, 2, 2, 3, 3, 3, 2, 2, 2, 1};
  uint32_t len = mode_len[mode];
  if (op == OP_ILL) return dw_x(H_ILL, 1, 0, 0);
  if (mode == MD_SPC) {
    switch (op) {
      case OP_JMP: return dw_x(H_JMP, 3, 3, 0);    case OP_JMPI: return dw_x(H_JMPI, 5, 3, 0);
      case OP_JSR: return dw_x(H_JSR, 6, 3, 0);    case OP_RTS: return dw_x(H_RTS, 6, 1, 0);
      case OP_RTI: return dw_x(H_RTI, 6, 1, 0);    case OP_PHA: return dw_x(H_PHA, 3, 1, 0);
      case OP_PHP: return dw_x(H_PHP, 3, 1, 0);    case OP_PLA: return dw_x(H_PLA, 4, 1, 0);
      case OP_PLP: return dw_x(H_PLP, 4, 1, 0);    default: return dw_x(H_BRK, 7, 2, 0);
    }
  }
  if (mode == MD_REL) return dw_x(H_BR0 + (op - OP_BPL), 2, 2, 1);
  if (mode == MD_IMP) return (op == OP_NOP) ? dw_x(H_NOP, 2, 1, 0) : dw_x(H_IMP0 + (op - OP_CLC), 2, 1, 0);
  if (mode == MD_ACC) return dw_x(H_ACC0 + (op - OP_ASL), 2, 1, 0);
  if (kind == K_READ) return dw_x(H_R0 + (mode - MD_IMM), 0, len, op - OP_LDA);
  if (kind == K_WRITE) return dw_x(H_W0 + (mode - MD_ZP), 0, len, op - OP_STA);
  const uint32_t mi = (mode == MD_ZP) ? 0u : (mode == MD_ZPX) ? 1u : (mode == MD_ABS) ? 2u : 3u;   // K_RMW
  return dw_x(H_M0 + mi, 0, len, op - OP_ASL);
}

inline bool tia_write_has_effect(uint32_t r) {    // r = address & 0x3F (SURVEY C.8 write map)
  return !(r > 0x2Cu || (r >= 0x15u && r <= 0x1Au) || r == 0x03u);
}
// bank hotspots of an image with nb banks: F8 $1FF8-9, F6 $1FF6-9, F4 $1FF4-B
inline bool is_hotspot(uint32_t a13, int nb) { const uint32_t lo = (nb == 8) ? 0x1FF4u : 0x1FFAu - (uint32_t)nb; return nb >= 2 && a13 - lo < (uint32_t)nb; }

// Second step of the decode: the handler ids above are what the out-of-line ("cold") executor understands.  The
// instructions that make up almost every executed one are re-coded into a handful of data-driven HOT classes run
// inline by the interpreter loop: the CPU registers A,X,Y,SP live packed in one 32-bit word, so "which register"
// is a byte-permute selector carried in the entry instead of a separate handler (LDA/LDX/LDY, STA/STX/STY,
// INX/INY/DEX/DEY, the transfers), and the eight branches share one flag test described by the entry.
// Everything else keeps its id, offset by HC_COLD.
enum HotClass : uint32_t {
  HC_ST_TIA = 1,     // y = TIA register | extract selector << 16
  HC_LD_IMM = 2,     // y = immediate | insert selector << 16
  HC_BR = 3,         // y = signed displacement ; aux = flag bit position in P | wanted value << 3 | extra cycles << 4
  HC_RTIM = 4,       // y = address ; aux = read op
  HC_INCDEC = 5,     // y = extract selector | insert selector << 16 ; aux = delta (1 | 0xFF)
  HC_LD_RAM = 6,     // y = smem byte offset | insert selector << 16
  HC_ST_RAM = 7,     // y = smem byte offset | extract selector << 16
  HC_XFER = 8,       // y = extract selector | insert selector << 16 ; aux = 1: sets N,Z  0: TXS
  HC_ALU_IMM = 9,    // y = immediate ; aux = read op (3..10)
  HC_ALU_RAM = 10,   // y = smem byte offset ; aux = read op (3..11)
  HC_RMW_RAM = 11,   // y = smem byte offset ; aux = RMW op
  HC_ACC = 12,       // aux = RMW op on A
  HC_FLAG = 13,      // y = P bits to clear | P bits to set << 16
  HC_NOP = 14,
  HC_JMP = 15,       // y = target
  HC_SPIN = 16,      // LDA INTIM ; BNE *-3  /  BIT TIMINT ; BPL *-3 : the timer wait loop, fast-forwarded (aux = 0 / 1 ; y = the poll's own entry .x)
  HC_LDST = 17,      // LDx #imm ; STx <TIA register> as one entry: y = imm | (register | source index << 6) << 8 | insert selector << 16 ;
                     // aux = 1 when the store is absolute ; cy / len cover both instructions
  // Indexed / indirect accesses and stack instructions whose bus accesses all turn out, at run time, to be RAM cells or
  // plain cartridge bytes (no TIA / RIOT register, no bank hotspot).  The inline loop checks that first and otherwise
  // hands the instruction, untouched, to the out-of-line executor under its generic handler id.
  HC_IDX_RD = 18,    // zp,X zp,Y abs,X abs,Y reads: y = base | index extract selector << 16 ; aux = read op | zp-indexed << 7
  HC_IZY_RD = 19,    // (zp),Y reads, pointer cells in RAM: y = smem byte offset of cell zp | of cell zp+1 << 15 ; aux = read op
  HC_IZX_RD = 20,    // (zp,X) reads: y = zp ; aux = read op
  HC_IDX_ST = 21,    // zp,X zp,Y abs,X abs,Y stores into RAM: y = base | index extract selector << 16 ; aux = source (0 A, 1 X, 2 Y) | zp-indexed << 7
  HC_IZY_ST = 22,    // (zp),Y stores: y as HC_IZY_RD ; aux = source
  HC_IZX_ST = 23,    // (zp,X) stores: y = zp ; aux = source
  HC_JSR = 24,       // y = target
  HC_RTS = 25,
  HC_STACK = 26,     // aux = 0 PHA, 1 PHP, 2 PLA, 3 PLP
  HC_ST_RIOT = 27,   // absolute store to a RIOT register (ports, timer): y = address | extract selector << 16
  HC_COLD = 28       // + Hid: executed by the out-of-line executor
};
static_assert(HC_COLD + H_COUNT <= 128, "hid is 7 bits");

// smem byte offset of RAM cell `a` (any address that decodes to RAM) in a file of `block` interleaved words
inline uint32_t ram_cell_offset(uint32_t a, int block) { return ((a & 0x7Cu) * (uint32_t)block) | (a & 3u); }

inline void hot_class(uint32_t &x, uint32_t &y, int block, bool promote) {
  const uint32_t hid = x & 0x7Fu, rest = x & 0x00FFFF00u;                  // cy and len stay
  static const uint32_t ins[4] = {0x3214u, 0x3240u, 0x3410u, 0x4210u};     // prmt(axys, v, sel): v -> A, X, Y, SP
  auto ext = [](uint32_t i) { return 0x4440u | i; };                       // prmt(axys, 0, sel): zero-extended byte i
  auto mk = [&](uint32_t hc, uint32_t aux) { x = hc | rest | (aux << DW_OP2_SHIFT); };
  if (hid >= H_STZT0 && hid < H_STZT0 + 3) { y = (y & 0xFFu) | (ext(hid - H_STZT0) << 16); mk(HC_ST_TIA, 0); }
  else if (hid >= H_IMM0 && hid < H_IMM0 + 3) { y = (y & 0xFFu) | (ins[hid - H_IMM0] << 16); mk(HC_LD_IMM, 0); }
  else if (hid >= H_IMM0 + 3 && hid < H_IMM0 + 11) { y &= 0xFFu; mk(HC_ALU_IMM, hid - H_IMM0); }
  else if (hid >= H_ZR0 && hid < H_ZR0 + 3) { y = (y & 0xFFFFu) | (ins[hid - H_ZR0] << 16); mk(HC_LD_RAM, 0); }
  else if (hid >= H_ZR0 + 3 && hid < H_ZR0 + 12) { y &= 0xFFFFu; mk(HC_ALU_RAM, hid - H_ZR0); }
  else if (hid >= H_STZR0 && hid < H_STZR0 + 3) { y = (y & 0xFFFFu) | (ext(hid - H_STZR0) << 16); mk(HC_ST_RAM, 0); }
  else if (hid == H_NOP) { y = 0; mk(HC_NOP, 0); }
  else if (hid >= H_MZR0 && hid < H_MZR0 + 6) { y &= 0xFFFFu; mk(HC_RMW_RAM, hid - H_MZR0); }
  else if (hid >= H_ACC0 && hid < H_ACC0 + 4) { y = 0; mk(HC_ACC, hid - H_ACC0); }
  else if (hid >= H_IMP0 && hid < H_IMP0 + 7) {                            // CLC SEC CLD SED CLI SEI CLV
    static const uint32_t clr[7] = {1, 1, 8, 8, 4, 4, 0x40}, set[7] = {0, 1, 0, 8, 0, 4, 0};
    y = clr[hid - H_IMP0] | (set[hid - H_IMP0] << 16); mk(HC_FLAG, 0);
  }
  else if (hid >= H_IMP0 + 8 && hid < H_IMP0 + 12) {                       // DEX DEY INX INY
    const uint32_t k = hid - H_IMP0 - 8, r = 1u + (k & 1u);
    y = ext(r) | (ins[r] << 16); mk(HC_INCDEC, (k < 2) ? 0xFFu : 1u);
  }
  else if (hid >= H_IMP0 + 12 && hid < H_IMP0 + 18) {                      // TAX TAY TSX TXA TYA TXS
    static const uint32_t src[6] = {0, 0, 3, 1, 2, 1}, dst[6] = {1, 2, 1, 0, 0, 3};
    const uint32_t k = hid - H_IMP0 - 12;
    y = ext(src[k]) | (ins[dst[k]] << 16); mk(HC_XFER, (k == 5) ? 0u : 1u);
  }
  else if (hid >= H_BR0 && hid < H_BR0 + 8) {                              // BPL BMI BVC BVS BCC BCS BNE BEQ
    static const uint32_t pos[4] = {7, 6, 0, 1};                           // N V C Z in the P layout
    const uint32_t k = hid - H_BR0, extra = x >> DW_OP2_SHIFT;
    mk(HC_BR, pos[k >> 1] | ((k & 1u) << 3) | (extra << 4));
  }
  else if (hid == H_JMP) mk(HC_JMP, 0);
  else if (hid == H_RTIM) mk(HC_RTIM, x >> DW_OP2_SHIFT);
  else if (promote && (hid == H_R0 + 2 || hid == H_R0 + 3 || hid == H_R0 + 5 || hid == H_R0 + 6) && (x >> DW_OP2_SHIFT) <= 11u) {
    const bool zpm = hid < H_R0 + 4, useX = (hid == H_R0 + 2 || hid == H_R0 + 5);              // ZPX ZPY ABX ABY reads
    y = (y & 0xFFFFu) | (ext(useX ? 1u : 2u) << 16);
    x = HC_IDX_RD | (4u << DW_CY_SHIFT) | (x & 0x00FF0000u) | (((x >> DW_OP2_SHIFT) | (zpm ? 0x80u : 0u)) << DW_OP2_SHIFT);
  }
  else if (promote && (hid == H_W0 + 1 || hid == H_W0 + 2 || hid == H_W0 + 4 || hid == H_W0 + 5) && (x >> DW_OP2_SHIFT) <= 2u) {
    const bool zpm = hid < H_W0 + 3, useX = (hid == H_W0 + 1 || hid == H_W0 + 4);              // ZPX ZPY ABX ABY stores
    y = (y & 0xFFFFu) | (ext(useX ? 1u : 2u) << 16);
    x = HC_IDX_ST | ((zpm ? 4u : 5u) << DW_CY_SHIFT) | (x & 0x00FF0000u) | (((x >> DW_OP2_SHIFT) | (zpm ? 0x80u : 0u)) << DW_OP2_SHIFT);
  }
  else if (promote && (hid == H_R0 + 8 || hid == H_W0 + 7) && (y & 0xFFu) >= 0x80u && (y & 0xFFu) <= 0xFEu &&
           (x >> DW_OP2_SHIFT) <= (hid == H_R0 + 8 ? 11u : 2u)) {                                // (zp),Y with both pointer cells in RAM
    const uint32_t z = y & 0xFFu;
    y = ram_cell_offset(z, block) | (ram_cell_offset(z + 1u, block) << 15);
    x = (hid == H_R0 + 8 ? (uint32_t)HC_IZY_RD | (5u << DW_CY_SHIFT) : (uint32_t)HC_IZY_ST | (6u << DW_CY_SHIFT)) | (x & 0xFFFF0000u);
  }
  else if (promote && (hid == H_R0 + 7 || hid == H_W0 + 6) && (x >> DW_OP2_SHIFT) <= (hid == H_R0 + 7 ? 11u : 2u)) {    // (zp,X)
    y &= 0xFFu;
    x = (hid == H_R0 + 7 ? (uint32_t)HC_IZX_RD : (uint32_t)HC_IZX_ST) | (6u << DW_CY_SHIFT) | (x & 0xFFFF0000u);
  }
  else if (promote && hid == H_JSR) mk(HC_JSR, 0);
  else if (promote && hid == H_RTS) mk(HC_RTS, 0);
  else if (promote && hid >= H_PHA && hid <= H_PLP) mk(HC_STACK, hid - H_PHA);
  else if (promote && hid == H_W0 + 3 && (x >> DW_OP2_SHIFT) <= 2u && (y & 0x1280u) == 0x0280u) {                      // STx abs -> RIOT
    y = (y & 0x1FFFu) | (ext(x >> DW_OP2_SHIFT) << 16);
    x = HC_ST_RIOT | (4u << DW_CY_SHIFT) | (x & 0x00FF0000u);
  }
  else x += HC_COLD;                                                       // (hid + HC_COLD stays below 128)
  const uint32_t hc = x & 0x7Fu;
  x |= (hc == HC_ST_TIA) ? DW_F_STTIA : (hc == HC_LD_IMM) ? DW_F_LDIMM : (hc == HC_BR) ? DW_F_BR : 0u;
}

// One bank image (4096 bytes; 2 KB carts are passed mirrored) -> 4096 decode entries.  `leader` is the bank-
// independent leader bitmap (4096 flags) filled by mark_leaders() for every bank of the cartridge first.
// sc: a Superchip cart — the first 256 bytes of the bank are RAM ports, not ROM: no instruction there is pre-decoded and
// no operand there is folded into an immediate
inline void decode_bank(const uint8_t *img, const uint8_t *leader, int block, int nb, DWord *out, bool promote = true, bool sc = false) {
  for (uint32_t off = 0; off < 4096; ++off) {
    const uint32_t lead = leader[off] ? DW_LEADER : 0u;
    if (off >= DW_SLOW_LIMIT || (sc && off < 0x100u)) { out[off].x = (HC_COLD + H_SLOW) | lead; out[off].y = 0; continue; }
    const uint32_t opc = img[off], b1 = img[off + 1], b2 = img[off + 2];
    const uint32_t ent = kOpTable[opc], mode = ent & 15u, op = (ent >> 4) & 63u, kind = ent >> 10;
    uint32_t x = generic_entry(opc);
    const uint32_t len = (x >> DW_LEN_SHIFT) & 0xFFu;
    uint32_t payload = (len == 3) ? (b1 | (b2 << 8)) : (len == 2) ? b1 : 0u;
    const uint32_t abs13 = (b1 | (b2 << 8)) & 0x1FFFu;
    const bool zp = (mode == MD_ZP), ab = (mode == MD_ABS);
    const uint32_t cyz = zp ? 0u : 1u;                                     // absolute = zero page + 1 cycle
    if (op != OP_ILL) {
      const uint32_t a13 = zp ? b1 : abs13;
      const bool is_ram = zp ? (b1 >= 0x80u) : (ab && (a13 & 0x1280u) == 0x0080u);
      const bool rd_std = kind == K_READ && op <= OP_BIT, wr_std = kind == K_WRITE && op <= OP_STY;   // (LAX / NOPR / SAX stay generic)
      if (mode == MD_IMM && op <= OP_CPY) x = dw_x(H_IMM0 + (op - OP_LDA), 2, 2, 0);
      else if (mode == MD_IMM) { /* NOP #imm: generic read */ }
      else if ((zp || ab) && is_ram && (rd_std || wr_std || kind == K_RMW)) {
        payload = ((a13 & 0x7Cu) * (uint32_t)block) | (a13 & 3u);          // byte offset of the cell in the RAM words
        if (kind == K_READ) x = dw_x(H_ZR0 + (op - OP_LDA), 3 + cyz, len, 0);
        else if (kind == K_WRITE) x = dw_x(H_STZR0 + (op - OP_STA), 3 + cyz, len, 0);
        else x = dw_x(H_MZR0 + (op - OP_ASL), 5 + cyz, len, 0);
      }
      else if ((zp || ab) && wr_std && (a13 & 0x1080u) == 0) {    // a TIA register
        const uint32_t r = a13 & 0x3Fu;
        if (tia_write_has_effect(r)) { x = dw_x(H_STZT0 + (op - OP_STA), 3 + cyz, len, 0); payload = r; }
        else { x = dw_x(H_NOP, 3 + cyz, len, 0); payload = 0; }
      }
      else if (ab && rd_std && (a13 & 0x1284u) == 0x0284u) {       // INTIM / TIMINT
        x = dw_x(H_RTIM, 4, 3, op - OP_LDA); payload = a13;
      }
      else if (ab && rd_std && op != OP_BIT && (a13 & 0x1000u) && !is_hotspot(a13, nb) && !(sc && (a13 & 0x0F00u) == 0)) {   // a fixed ROM byte
        x = dw_x(H_IMM0 + (op - OP_LDA), 4, 3, 0); payload = img[a13 & 0xFFFu];                        // of this bank
      }
      else if (mode == MD_REL) {
        const int32_t disp = (int32_t)(int8_t)b1;
        const int32_t toff = (int32_t)off + 2 + disp;                      // target offset inside the 4 KB window
        const uint32_t next = 0x1000u + off + 2u, target = (uint32_t)((int32_t)next + disp);
        const uint32_t dummy2 = (next & 0xFF00u) | (target & 0xFFu);
        if (toff < 0 || toff >= 4096 || (is_hotspot(next & 0x1FFFu, nb) || is_hotspot(dummy2 & 0x1FFFu, nb)))
          x = H_SLOW;                                                      // run-time decode keeps every side effect
        else {
          payload = (uint32_t)disp;
          x = (x & 0x00FFFFFFu) | ((((target ^ next) & 0xFF00u) ? 2u : 1u) << DW_OP2_SHIFT);
        }
      }
    }
    if ((x & 0x7Fu) == H_SLOW) { out[off].x = (HC_COLD + H_SLOW) | lead; out[off].y = 0; }
    else { hot_class(x, payload, block, promote); out[off].x = x | lead; out[off].y = payload; }
  }
}

// Timer wait loops — "LDA INTIM ; BNE back" and "BIT TIMINT ; BPL back", the way every kernel waits for the end of
// VBLANK / overscan — are marked so that the interpreter can jump to the loop's exit in closed form (same registers,
// cycles and line ends as running it; see HC_SPIN in vcs_step.cu).  The poll's own entry is kept in .y for the cases
// the closed form does not cover.
inline void mark_spins(const uint8_t *img, DWord *out) {
  for (uint32_t off = 0; off + 5 < DW_SLOW_LIMIT; ++off) {
    const uint32_t a13 = (img[off + 1] | (img[off + 2] << 8)) & 0x1FFFu;
    const bool intim = img[off] == 0xAD && (a13 & 0x1285u) == 0x0284u && img[off + 3] == 0xD0;
    const bool timint = img[off] == 0x2C && (a13 & 0x1285u) == 0x0285u && img[off + 3] == 0x10;
    if (!(intim || timint) || img[off + 4] != 0xFB) continue;                  // branch back to the poll
    if (((0x1000u + off + 5u) ^ (0x1000u + off)) & 0xFF00u) continue;          // taken branch must not cross a page (3 cycles)
    if ((out[off].x & 0x7Fu) != HC_RTIM || (out[off + 3].x & 0x7Fu) != HC_BR) continue;
    out[off].y = out[off].x & ~DW_LEADER;
    out[off].x = HC_SPIN | (out[off].x & DW_LEADER) | ((timint ? 1u : 0u) << DW_OP2_SHIFT);
  }
}

// "LDx #imm ; STx reg" pairs — the body of every display kernel — become ONE entry at the load's offset (the store's
// own entry stays for anyone who jumps to it).  The interpreter still honours the instruction boundary between the
// two: with a line end / cap / WSYNC release pending there, it runs the load alone and the store as its own entry.
inline void fuse_ld_st(DWord *out) {
  for (uint32_t off = 0; off + 5 < DW_SLOW_LIMIT; ++off) {
    const DWord ld = out[off], st = out[off + 2];
    if ((ld.x & 0x7Fu) != HC_LD_IMM || ((ld.x >> DW_LEN_SHIFT) & 0xFFu) != 2u) continue;    // (a fixed-ROM-byte load is 3 bytes: not fused)
    if ((st.x & 0x7Fu) != HC_ST_TIA || (st.x & DW_LEADER)) continue;
    const uint32_t cy2 = (st.x >> DW_CY_SHIFT) & 0xFu, len2 = (st.x >> DW_LEN_SHIFT) & 0xFFu;
    if (off + 2 + len2 >= DW_SLOW_LIMIT) continue;
    const uint32_t reg = st.y & 0x3Fu, src = (st.y >> 16) & 3u;                             // extract selector 0x4440 | src
    out[off].x = HC_LDST | DW_F_LDST | (ld.x & DW_LEADER) | ((2u + cy2) << DW_CY_SHIFT) | ((2u + len2) << DW_LEN_SHIFT) | ((len2 - 2u) << DW_OP2_SHIFT);
    out[off].y = (ld.y & 0xFFu) | ((reg | (src << 6)) << 8) | (ld.y & 0xFFFF0000u);
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
