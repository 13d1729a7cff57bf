// vcs_step.cu — the persistent interpreter kernel behind vcs_step (SURVEY.md §8(a) a1–a16).
//
// One thread = one environment for the whole env-step (all `frameskip` frames).  CPU registers and the beam
// position live in registers; RAM, the TIA/RIOT latches, the cached TIA object masks and the colour-index
// planes live in the thread's shared-memory file; the block's cartridge ROM is staged in shared memory with
// one bulk asynchronous copy (TMA 1-D, cp.async.bulk + mbarrier) when all of the block's envs share a ROM.
//
// Divergence (the measured choice north_star asks for): lanes of a warp are NOT run in lock-step.  Every
// iteration each lane forms the key (frames done, SP, bank, PC); a warp-wide REDUX.MIN picks the smallest
// and only the lanes holding it execute one 6507 instruction — all at the same PC of the same ROM, hence
// the same opcode, the same addressing mode and (for stores) the same TIA register: the decode switch, the
// TIA write switch and the lazy-TIA catch-up are warp-uniform.  Lower SP first returns lanes from
// subroutines, lower PC first re-joins forward branches, the frame count bounds how long a lane can wait.
// On BASELINE config 4 this keeps ~95 % (4 KB ROMs) of the lanes active per iteration versus 18 % active
// threads per instruction for the lock-step kernel it replaced (profiles/r01_*).
//
// Each instruction runs in four phases shared by all opcodes — addressing (switch on 13 modes) -> ONE
// generic operand-read site -> ALU (switch on op) -> ONE generic write site.  Cycle accounting is per bus
// access (C.4/C.5): an access `k` cycles into the instruction happens in cycle `cyc + k`, scanline slot `n + k`.
#include "vcs_tia.cuh"
#include "vcs_optable.cuh"
#include "vcs_step.cuh"

namespace vcs {

__constant__ uint16_t c_optab[256];

void upload_optable() { cudaMemcpyToSymbol(c_optab, kOpTable, sizeof(kOpTable)); }
const uint16_t *host_optable() { return kOpTable; }

constexpr uint32_t IB_SLOW = 0x80000000u;

template <int BLOCK, bool ROMS>
struct Cpu {
  using T = Tia<BLOCK>;
  // ---- CPU
  uint32_t A, X, Y, SP, PC;
  uint32_t fC, fV, fD, fI, zv, nv;     // Z <=> (zv & 0xFF) == 0 ; N <=> nv & 0x80
  uint32_t status;
  // ---- beam / time (cycle counts are relative to the start of this vcs_step call)
  int32_t cyc;        // CPU cycles executed in this step
  int32_t n;          // cycle-in-line of `cyc` (0..76)
  int32_t fstart;     // value of `cyc` at which the current frame began (frame_cyc = cyc - fstart)
  uint32_t fdone;     // frames completed in this step (mirror of S_FDONE)
  bool wsync;         // mirror of TF_WSYNC
  // ---- cart
  uint32_t bank, rom_mask, is_f8;
  uint32_t rom_off;   // ROMS: byte offset of the ROM image inside smem
  const uint8_t *rom_g;   // !ROMS: the image in global memory
  uint32_t ib;        // prefetched opcode | b1<<8 | b2<<16 at PC (IB_SLOW: fetch byte-wise with side effects)

  static DEV uint32_t &S(int i) { return T::S(i); }

  // ------------------------------------------------------------------ RAM (smem, conflict-free)
  DEV uint32_t ram_rd(uint32_t a) const { return reinterpret_cast<const uint8_t *>(smem)[(((a & 0x7Cu) * BLOCK) | (a & 3u)) + 4 * threadIdx.x]; }
  DEV void ram_wr(uint32_t a, uint32_t v) { reinterpret_cast<uint8_t *>(smem)[(((a & 0x7Cu) * BLOCK) | (a & 3u)) + 4 * threadIdx.x] = (uint8_t)v; }

  // ------------------------------------------------------------------ ROM
  DEV uint32_t rom_byte(uint32_t off) const {
    if constexpr (ROMS) return reinterpret_cast<const uint8_t *>(smem)[rom_off + off];
    else return __ldg(rom_g + off);
  }
  DEV uint32_t rom_rd(uint32_t a) {            // a = addr & 0x1FFF with A12 set
    if (is_f8 && (a | 1u) == 0x1FF9u) bank = a & 1u;
    return rom_byte((bank << 12) + (a & rom_mask));
  }
  DEV void hotspot(uint32_t a) { if (is_f8 && (a | 1u) == 0x1FF9u) bank = a & 1u; }
  // the three bytes at PC in one go when no fetch can have a side effect (cartridge space, below the hotspots)
  DEV void prefetch() {
    const uint32_t a = PC & 0x1FFFu;
    if ((a & 0x1000u) && (a & rom_mask) < rom_mask - 10u) {
      const uint32_t off = (bank << 12) + (a & rom_mask);
      uint32_t w0, w1;
      if constexpr (ROMS) { const uint32_t *r = reinterpret_cast<const uint32_t *>(reinterpret_cast<const uint8_t *>(smem) + rom_off) + (off >> 2); w0 = r[0]; w1 = r[1]; }
      else { const uint32_t *r = reinterpret_cast<const uint32_t *>(rom_g) + (off >> 2); w0 = __ldg(r); w1 = __ldg(r + 1); }
      ib = __funnelshift_r(w0, w1, (off & 3u) * 8u) & 0x00FFFFFFu;
    } else ib = IB_SLOW;
  }

  // ------------------------------------------------------------------ RIOT timer, closed form (C.7)
  // advance the (timer, sub, tflag) state in smem to "after `ticks` cycles of this step" and return it unpacked
  DEV void timer_sync(int32_t ticks, uint32_t &timer, uint32_t &sub, uint32_t &shift, uint32_t &tflag) {
    const uint32_t w = S(S_TMR);
    timer = w & 0xFFu; shift = (w >> 8) & 0xFu; tflag = (w >> 12) & 1u; sub = w >> 16;
    const uint32_t d = (uint32_t)(ticks - (int32_t)S(S_TTICKS));
    if ((int32_t)d <= 0) return;
    S(S_TTICKS) = (uint32_t)ticks;
    const uint32_t mask = (1u << shift) - 1u;
    if (tflag) { timer = (timer - d) & 0xFFu; sub = (sub + d) & mask; return; }
    const uint32_t k = (sub + d) >> shift;            // prescaler wraps (decrement events) in d ticks
    if (k <= timer) { timer -= k; }
    else {                                            // event number timer+1 is the underflow
      const uint32_t iu = ((timer + 1u) << shift) - sub;    // tick index (1-based) of the underflow
      timer = (0xFFu - (d - iu)) & 0xFFu; tflag = 1;
    }
    sub = (sub + d) & mask;
  }
  DEV void timer_put(uint32_t timer, uint32_t sub, uint32_t shift, uint32_t tflag) { S(S_TMR) = timer | (shift << 8) | (tflag << 12) | (sub << 16); }
  DEV uint32_t riot_read(uint32_t a, int32_t c) {     // access in cycle index c (tick c happened first)
    if ((a & 4u) == 0) {
      const uint32_t ports = S(S_PORTS);
      const uint32_t ora = byte_of(ports, 0), ddra = byte_of(ports, 1), orb = byte_of(ports, 2), ddrb = byte_of(ports, 3);
      switch (a & 3u) {
        case 0: return (ora & ddra) | (S(S_INP) & ~ddra & 0xFFu);
        case 1: return ddra;
        case 2: return (orb & ddrb) | (0x3Fu & ~ddrb);
        default: return ddrb;
      }
    }
    uint32_t timer, sub, shift, tflag;
    timer_sync(c + 1, timer, sub, shift, tflag);
    if ((a & 5u) == 4u) { timer_put(timer, sub, shift, 0); return timer; }   // INTIM clears the flag
    timer_put(timer, sub, shift, tflag);
    return tflag << 7;                                                        // TIMINT
  }
  DEV void riot_write(uint32_t a, uint32_t v, int32_t c) {
    if ((a & 4u) == 0) { S(S_PORTS) = set_byte(S(S_PORTS), a & 3u, v); return; }
    if ((a & 0x14u) == 0x14u) {
      const uint32_t k = a & 3u;
      const uint32_t shift = (k == 0) ? 0u : (k == 1) ? 3u : (k == 2) ? 6u : 10u;
      timer_put(v & 0xFFu, (1u << shift) - 1u, shift, 0); S(S_TTICKS) = (uint32_t)(c + 1);
    }
  }

  // side-effect-light read used for instruction bytes, zero-page pointers, JMP() vectors and stack
  // pulls: cartridge (incl. F8 hotspots) or RAM.  Anything else is outside the modelled set (status bit 2).
  DEV uint32_t lite_rd(uint32_t addr) {
    const uint32_t a = addr & 0x1FFFu;
    if (a & 0x1000u) return rom_rd(a);
    if ((a & 0x0280u) == 0x0080u) return ram_rd(a);
    status |= STATUS_UNMODELLED; return 0;
  }
  DEV void push(uint32_t v) {
    if (SP & 0x80u) ram_wr(SP, v); else status |= STATUS_UNMODELLED;
    SP = (SP - 1u) & 0xFFu;
  }
  DEV uint32_t pull() {
    SP = (SP + 1u) & 0xFFu;
    if (SP & 0x80u) return ram_rd(SP);
    status |= STATUS_UNMODELLED; return 0;
  }
  // dummy read of an indexed mode's uncorrected address in cycle cyc+k: only INTIM and F8 hotspots react
  DEV void dummy_rd(uint32_t addr, int k) {
    const uint32_t a = addr & 0x1FFFu;
    if (a & 0x1000u) hotspot(a);
    else if ((a & 0x0285u) == 0x0284u) { uint32_t t, s, sh, f; timer_sync(cyc + k + 1, t, s, sh, f); timer_put(t, s, sh, 0); }
  }
  DEV void tia_events(uint32_t ev, int k) {        // after a TIA access k cycles into the instruction
    n -= LINE_CYC * (int32_t)(ev >> 4);
    wsync = (ev & EV_WSYNC) != 0;
    if (ev & EV_FRAME) { fdone += 1; fstart = cyc + k + 1; }
  }
  // the generic operand read (C.3 decode), k cycles into the instruction
  DEV uint32_t bus_read(uint32_t addr, int k) {
    const uint32_t a = addr & 0x1FFFu;
    if ((a & 0x1280u) == 0x0080u) return ram_rd(a);
    if (a & 0x1000u) return rom_rd(a);
    if (a & 0x0080u) return riot_read(a, cyc + k);
    const uint32_t r = T::read(a & 0xFu, n + k);
    if (r >> 12) { n -= LINE_CYC * (int32_t)(r >> 12); wsync = false; }
    return r & 0xFFu;
  }
  DEV void bus_write(uint32_t addr, uint32_t v, int k) {
    const uint32_t a = addr & 0x1FFFu;
    if ((a & 0x1280u) == 0x0080u) { ram_wr(a, v); return; }
    if (a & 0x1000u) { hotspot(a); return; }
    if (a & 0x0080u) { riot_write(a, v, cyc + k); return; }
    const uint32_t r = a & 0x3Fu;
    if (r > 0x2Cu || (r >= 0x15u && r <= 0x1Au) || r == 0x03u) return;      // no effect (audio: PAPER.md L205)
    tia_events(T::write(r, v, n + k), k);
  }
  DEV uint32_t pack_p() const {
    return (nv & 0x80u) | (fV << 6) | 0x20u | (fD << 3) | (fI << 2) | (((zv & 0xFFu) == 0) ? 2u : 0u) | fC;
  }
  DEV void unpack_p(uint32_t p) {
    fC = p & 1u; zv = (p & 2u) ? 0u : 1u; fI = (p >> 2) & 1u; fD = (p >> 3) & 1u; fV = (p >> 6) & 1u; nv = p & 0x80u;
  }
  DEV void adc(uint32_t v) {                               // C.6, binary and NMOS decimal
    const uint32_t a = A, C = fC;
    if (!fD) {
      const uint32_t s = a + v + C;
      fC = s >> 8; fV = ((a ^ s) & (v ^ s) & 0x80u) >> 7; A = s & 0xFFu; zv = nv = A;
      return;
    }
    int al = (int)(a & 0x0Fu) + (int)(v & 0x0Fu) + (int)C;
    if (al >= 0x0A) al = ((al + 6) & 0x0F) + 0x10;
    int s = (int)(a & 0xF0u) + (int)(v & 0xF0u) + al;
    const int sv = (int)(int8_t)(a & 0xF0u) + (int)(int8_t)(v & 0xF0u) + al;
    nv = (uint32_t)s & 0x80u;
    fV = (sv < -128 || sv > 127) ? 1u : 0u;
    zv = (a + v + C) & 0xFFu;
    if (s >= 0xA0) s += 0x60;
    fC = (s >= 0x100) ? 1u : 0u;
    A = (uint32_t)s & 0xFFu;
  }
  DEV void sbc(uint32_t v) {
    const uint32_t a = A, C = fC;
    const uint32_t nb = v ^ 0xFFu, s = a + nb + C;         // flags exactly as binary
    const uint32_t bin = s & 0xFFu;
    fC = s >> 8; fV = ((a ^ s) & (nb ^ s) & 0x80u) >> 7; zv = nv = bin;
    if (!fD) { A = bin; return; }
    int al = (int)(a & 0x0Fu) - (int)(v & 0x0Fu) + (int)C - 1;
    if (al < 0) al = ((al - 6) & 0x0F) - 0x10;
    int d = (int)(a & 0xF0u) - (int)(v & 0xF0u) + al;
    if (d < 0) d -= 0x60;
    A = (uint32_t)d & 0xFFu;
  }

  // ---------------------------------------------------------------- one instruction (C.5)
  DEV void instruction(const uint16_t *optab) {
    const uint32_t pc = PC;
    const bool slow = (ib & IB_SLOW) != 0;
    const uint32_t opc = slow ? lite_rd(pc) : (ib & 0xFFu);
    const uint32_t ent = optab[opc];
    const uint32_t mode = ent & 15u, op = (ent >> 4) & 63u, kind = ent >> 10;
    if (op == OP_ILL) {                                    // C.12: halt for good, PC stays
      if (!(status & STATUS_UNMODELLED)) status |= STATUS_ILLEGAL;
      cyc += 1; n += 1; return;
    }
    const uint32_t b1 = slow ? lite_rd(pc + 1) : ((ib >> 8) & 0xFFu);    // operand byte, or the dummy read @PC+1
    const uint32_t b2f = (ib >> 16) & 0xFFu;
#define FETCH2() (slow ? lite_rd(pc + 2) : b2f)
    uint32_t ea = 0, v = 0, wv = 0;
    int k = 0;                                             // cycles before the operand access
    int total = 2;
    uint32_t npc = pc + 2;
    switch (mode) {
      case MD_IMP: case MD_ACC: npc = pc + 1; break;
      case MD_IMM: v = b1; k = 1; break;
      case MD_ZP:  ea = b1; k = 2; break;
      case MD_ZPX: ea = (b1 + X) & 0xFFu; k = 3; break;
      case MD_ZPY: ea = (b1 + Y) & 0xFFu; k = 3; break;
      case MD_ABS: ea = b1 | (FETCH2() << 8); k = 3; npc = pc + 3; break;
      case MD_ABX: case MD_ABY: case MD_IZY: {
        uint32_t lo, hi;
        if (mode == MD_IZY) { lo = lite_rd(b1); hi = lite_rd((b1 + 1u) & 0xFFu); k = 4; }
        else { lo = b1; hi = FETCH2(); k = 3; npc = pc + 3; }
        const uint32_t t = lo + ((mode == MD_ABX) ? X : Y);
        const uint32_t unc = (hi << 8) | (t & 0xFFu);
        ea = (unc + (t & 0x100u)) & 0xFFFFu;
        if (kind != K_READ || (t & 0x100u)) { dummy_rd(unc, k); k += 1; }
      } break;
      case MD_IZX: { const uint32_t z = (b1 + X) & 0xFFu; ea = lite_rd(z) | (lite_rd((z + 1u) & 0xFFu) << 8); k = 5; } break;
      default: break;                                      // MD_REL, MD_SPC: handled by op
    }
    if (kind & K_READ) {                                   // K_READ or K_RMW: the one generic read site
      if (mode != MD_IMM) v = bus_read(ea, k);
      total = k + 1;
    }
    switch (op) {
      case OP_LDA: A = v; zv = nv = v; break;
      case OP_LDX: X = v; zv = nv = v; break;
      case OP_LDY: Y = v; zv = nv = v; break;
      case OP_AND: A &= v; zv = nv = A; break;
      case OP_ORA: A |= v; zv = nv = A; break;
      case OP_EOR: A ^= v; zv = nv = A; break;
      case OP_ADC: adc(v); break;
      case OP_SBC: sbc(v); break;
      case OP_CMP: case OP_CPX: case OP_CPY: {
        const uint32_t r = (op == OP_CMP) ? A : (op == OP_CPX) ? X : Y;
        fC = (r >= v) ? 1u : 0u; zv = nv = (r - v) & 0xFFu; } break;
      case OP_BIT: zv = A & v; nv = v; fV = (v >> 6) & 1u; break;
      case OP_STA: wv = A; break;
      case OP_STX: wv = X; break;
      case OP_STY: wv = Y; break;
      case OP_ASL: case OP_LSR: case OP_ROL: case OP_ROR: case OP_INC: case OP_DEC: {
        const uint32_t s = (mode == MD_ACC) ? A : v; uint32_t r;
        if (op == OP_ASL)      { r = (s << 1) & 0xFFu; fC = s >> 7; }
        else if (op == OP_LSR) { r = s >> 1; fC = s & 1u; }
        else if (op == OP_ROL) { r = ((s << 1) | fC) & 0xFFu; fC = s >> 7; }
        else if (op == OP_ROR) { r = (s >> 1) | (fC << 7); fC = s & 1u; }
        else if (op == OP_INC) { r = (s + 1u) & 0xFFu; }
        else                   { r = (s - 1u) & 0xFFu; }
        zv = nv = r;
        if (mode == MD_ACC) A = r; else wv = r;
      } break;
      case OP_CLC: fC = 0; break;
      case OP_SEC: fC = 1; break;
      case OP_CLD: fD = 0; break;
      case OP_SED: fD = 1; break;
      case OP_CLI: fI = 0; break;
      case OP_SEI: fI = 1; break;
      case OP_CLV: fV = 0; break;
      case OP_NOP: break;
      case OP_DEX: X = (X - 1u) & 0xFFu; zv = nv = X; break;
      case OP_DEY: Y = (Y - 1u) & 0xFFu; zv = nv = Y; break;
      case OP_INX: X = (X + 1u) & 0xFFu; zv = nv = X; break;
      case OP_INY: Y = (Y + 1u) & 0xFFu; zv = nv = Y; break;
      case OP_TAX: X = A; zv = nv = X; break;
      case OP_TAY: Y = A; zv = nv = Y; break;
      case OP_TSX: X = SP; zv = nv = X; break;
      case OP_TXA: A = X; zv = nv = A; break;
      case OP_TYA: A = Y; zv = nv = A; break;
      case OP_TXS: SP = X; break;
      case OP_BPL: case OP_BMI: case OP_BVC: case OP_BVS: case OP_BCC: case OP_BCS: case OP_BNE: case OP_BEQ: {
        const uint32_t idx = op - OP_BPL; uint32_t f;
        switch (idx >> 1) { case 0: f = (nv >> 7) & 1u; break; case 1: f = fV; break; case 2: f = fC; break;
                            default: f = ((zv & 0xFFu) == 0) ? 1u : 0u; break; }
        if (f == (idx & 1u)) {
          const uint32_t next = (pc + 2u) & 0xFFFFu;
          const uint32_t target = (next + (uint32_t)(int32_t)(int8_t)b1) & 0xFFFFu;
          hotspot(next & 0x1FFFu);                         // dummy read @PC
          total = 3;
          if ((target ^ next) & 0xFF00u) { hotspot(((next & 0xFF00u) | (target & 0xFFu)) & 0x1FFFu); total = 4; }
          npc = target;
        }
      } break;
      case OP_JMP: npc = b1 | (FETCH2() << 8); total = 3; break;
      case OP_JMPI: { const uint32_t hi = FETCH2();
        const uint32_t l2 = lite_rd((hi << 8) | b1), h2 = lite_rd((hi << 8) | ((b1 + 1u) & 0xFFu));   // no carry into the page
        npc = l2 | (h2 << 8); total = 5; } break;
      case OP_JSR: { const uint32_t ret = (pc + 2u) & 0xFFFFu;     // address of the 3rd byte
        push(ret >> 8); push(ret & 0xFFu);
        npc = b1 | (FETCH2() << 8); total = 6; } break;
      case OP_RTS: { const uint32_t lo = pull(), hi = pull(); const uint32_t r = lo | (hi << 8);
        hotspot(r & 0x1FFFu); npc = (r + 1u) & 0xFFFFu; total = 6; } break;
      case OP_RTI: { unpack_p(pull()); const uint32_t lo = pull(), hi = pull(); npc = lo | (hi << 8); total = 6; } break;
      case OP_PHA: push(A); npc = pc + 1; total = 3; break;
      case OP_PHP: push(pack_p() | 0x30u); npc = pc + 1; total = 3; break;
      case OP_PLA: A = pull(); zv = nv = A; npc = pc + 1; total = 4; break;
      case OP_PLP: unpack_p(pull()); npc = pc + 1; total = 4; break;
      case OP_BRK: { const uint32_t ret = (pc + 2u) & 0xFFFFu;
        push(ret >> 8); push(ret & 0xFFu); push(pack_p() | 0x30u);
        npc = lite_rd(0xFFFEu) | (lite_rd(0xFFFFu) << 8); fI = 1; total = 7; } break;
      default: break;
    }
#undef FETCH2
    PC = npc & 0xFFFFu;
    if (kind & K_WRITE) {                                  // K_WRITE: one write; K_RMW: old value, then new
      const bool rmw = (kind == K_RMW);
      total = k + (rmw ? 3 : 1);
#pragma unroll 1
      for (int i = rmw ? 0 : 1; i < 2; ++i)               // the one generic write site
        bus_write(ea, i ? wv : v, k + (rmw ? 1 + i : 0));
    }
    cyc += total; n += total;
  }
};

// ---- TMA 1-D bulk copy helpers (cp.async.bulk + mbarrier; SASS: UBLKCP / SYNCS)
DEV uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
DEV void mbar_init(uint32_t bar, uint32_t count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count)); }
DEV void mbar_expect_tx(uint32_t bar, uint32_t bytes) { asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory"); }
DEV void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
DEV void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile("{\n .reg .pred p;\n WAIT_%=:\n mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n @!p bra WAIT_%=;\n}" ::"r"(bar), "r"(parity) : "memory");
}

template <int BLOCK, bool ROMS>
__global__ void __launch_bounds__(BLOCK, 512 / BLOCK) vcs_step_kernel(StepParams p) {
  using T = Tia<BLOCK>;
  __shared__ __align__(8) unsigned long long s_bar;
  uint32_t *s_ctx = smem + S_WORDS * BLOCK;
  uint16_t *s_optab = reinterpret_cast<uint16_t *>(s_ctx + C_WORDS);
  constexpr uint32_t ROM_OFF = (S_WORDS * BLOCK + C_WORDS + 128) * 4;     // byte offset of the ROM image in smem
  const int tid = threadIdx.x;
  const int e0 = blockIdx.x * BLOCK;
  const int e = e0 + tid;
  const int B = p.batch;
  const bool live = e < B;
  const RomMeta rm = p.rom_meta[p.env_rom[live ? e : e0]];

  if (tid == 0) {
    const unsigned long long scr = reinterpret_cast<unsigned long long>(p.screen);
    s_ctx[C_SCREEN_LO] = (uint32_t)scr; s_ctx[C_SCREEN_HI] = (uint32_t)(scr >> 32);
    s_ctx[C_Y0] = (uint32_t)p.y0; s_ctx[C_FRAMESKIP] = (uint32_t)p.frameskip; s_ctx[C_BATCH] = (uint32_t)B; s_ctx[C_ENV0] = (uint32_t)e0;
    if constexpr (ROMS) { mbar_init(smem_u32(&s_bar), 1); asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
  }
  for (int i = tid; i < 256; i += BLOCK) s_optab[i] = c_optab[i];
  __syncthreads();
  if constexpr (ROMS) {                                    // a3: stage the block's ROM (2 KB images twice: the mirror)
    if (tid == 0) {
      const uint32_t bar = smem_u32(&s_bar), dst = smem_u32(smem) + ROM_OFF;
      const uint8_t *src = p.rom_blob + rm.offset;
      mbar_expect_tx(bar, rm.size == 2048 ? 4096u : rm.size);
      bulk_g2s(dst, src, rm.size, bar);
      if (rm.size == 2048) bulk_g2s(dst + 2048, src, 2048, bar);
    }
  }

  Cpu<BLOCK, ROMS> s;
  // ---- a1 state load (coalesced SoA)
  uint32_t n0 = 0, fl = 0;
  if (live) {
    uint32_t w;
    w = p.st[W_AXYS * B + e]; s.A = w & 0xFF; s.X = (w >> 8) & 0xFF; s.Y = (w >> 16) & 0xFF; s.SP = w >> 24;
    w = p.st[W_PC * B + e]; s.PC = w & 0xFFFF; s.unpack_p((w >> 16) & 0xFF); s.status = w >> 24;
    w = p.st[W_BEAM * B + e]; n0 = w & 0xFF; T::S(S_LINE) = (w >> 8) & 0xFFFF; s.bank = w >> 24;
    s.fstart = -(int32_t)p.st[W_FCYC * B + e];
    T::S(S_TMR) = p.st[W_TIMER * B + e]; T::S(S_TTICKS) = 0;
    T::S(S_PORTS) = p.st[W_PORTS * B + e];
    T::S(S_COLU) = p.st[W_COLU * B + e]; T::S(S_PF) = p.st[W_PF * B + e]; T::S(S_GRP) = p.st[W_GRP * B + e]; T::S(S_NUSIZ) = p.st[W_NUSIZ * B + e];
    T::S(S_POS) = p.st[W_POS * B + e]; w = p.st[W_POS2 * B + e]; T::S(S_POS2) = w & 0xFFFF; T::S(S_RX) = w >> 16;
    fl = (p.st[W_FLAGS * B + e] & TF_ARCH_MASK) | TF_DIRTY_ALL; T::S(S_CX) = p.st[W_CX * B + e];
    T::S(S_PX) = 0; T::S(S_FDONE) = 0;
    for (int i = 0; i < 32; ++i) smem[(S_RAM + i) * BLOCK + tid] = p.ram[i * B + e];
    for (int i = 0; i < 10; ++i) smem[(S_PLANE + i) * BLOCK + tid] = 0;
    if (p.frameskip == 1) { fl |= TF_STORING; if ((T::S(S_LINE) - (uint32_t)p.y0) < (uint32_t)SCR_H) fl |= TF_ROWVIS; }
  } else {
    s.A = s.X = s.Y = s.SP = s.PC = 0; s.unpack_p(0x24); s.status = 0; s.bank = 0; s.fstart = 0;
  }
  s.cyc = 0; s.n = (int32_t)n0; s.fdone = live ? 0u : (uint32_t)p.frameskip;
  s.rom_mask = (rm.size == 2048 && !ROMS) ? 0x7FFu : 0xFFFu; s.is_f8 = (rm.size == 8192);
  s.rom_off = ROM_OFF; s.rom_g = p.rom_blob + rm.offset;
  // ---- a2 action latch (C.11)
  if (live) {
    uint32_t act = p.actions[e]; if (act >= 18u) act = 0;
    //            NOOP FIRE UP RIGHT LEFT DOWN UR UL DR DL UF RF LF DF URF ULF DRF DLF
    const uint32_t up = 0x0C4C4u, down = 0x32320u, left = 0x29290u, right = 0x14948u, fire = 0x3FC02u;
    uint32_t ina = 0xFFu;
    if ((up >> act) & 1u) ina &= ~0x10u;
    if ((down >> act) & 1u) ina &= ~0x20u;
    if ((left >> act) & 1u) ina &= ~0x40u;
    if ((right >> act) & 1u) ina &= ~0x80u;
    const uint32_t fire0 = (fire >> act) & 1u;
    T::S(S_INP) = ina | (fire0 << 8);
    if ((fl & TF_LATCHEN) && fire0) fl &= ~TF_INPT4_LATCH;
    T::S(S_FL) = fl;
  }
  s.wsync = (fl & TF_WSYNC) != 0;
  if constexpr (ROMS) mbar_wait(smem_u32(&s_bar), 0);
  const int32_t cap = p.max_lines * LINE_CYC;
  const uint32_t fskip = (uint32_t)p.frameskip;
  s.ib = IB_SLOW;
  if (live) s.prefetch();

  // ---- the hot loop: whole instructions until `frameskip` frame-end events (C.10), min-key lanes first.
  // Line bookkeeping mirrors C.4: the line counter advances with the FIRST cycle of a new line, so an
  // instruction that ends exactly on a line boundary leaves n == 76 pending (a frame end at that point
  // makes the finished line "line 0" and the next one line 1).
  for (;;) {
    const uint32_t key = (s.fdone >= fskip) ? 0xFFFFFFFFu
                       : (min(s.fdone, 63u) << 25) | (s.SP << 17) | (s.bank << 16) | s.PC;
    const uint32_t mk = __reduce_min_sync(0xFFFFFFFFu, key);
    if (mk == 0xFFFFFFFFu) break;
    if (key == mk) {
      if (s.cyc - s.fstart >= cap) {                       // frame cap at the instruction boundary
        s.status |= STATUS_CAP; T::frame_end(3u * (uint32_t)s.n); s.fdone += 1; s.fstart = s.cyc;
      } else {
        if (s.n >= LINE_CYC) { T::line_end(); s.n -= LINE_CYC; s.wsync = false; }     // n == 76 exactly (see above)
        if (s.status & (STATUS_ILLEGAL | STATUS_UNMODELLED)) {  // halted: idle cycles to the line end / the cap
          const int d = min(LINE_CYC - s.n, cap - (s.cyc - s.fstart));
          s.cyc += d; s.n += d;
        } else {
          if (s.wsync) {                                   // a12: RDY holds the CPU until the line ends
            s.cyc += LINE_CYC - s.n; T::line_end(); s.n = 0; s.wsync = false;
          }
          s.instruction(s_optab);
          if (s.n > LINE_CYC) { T::line_end(); s.n -= LINE_CYC; s.wsync = false; }
          s.prefetch();
        }
      }
    }
  }
  if (!live) return;
  // ---- a16 state store
  {
    uint32_t timer, sub, shift, tflag;
    s.timer_sync(s.cyc, timer, sub, shift, tflag);
    p.st[W_AXYS * B + e] = s.A | (s.X << 8) | (s.Y << 16) | (s.SP << 24);
    p.st[W_PC * B + e] = s.PC | (s.pack_p() << 16) | (s.status << 24);
    p.st[W_BEAM * B + e] = (uint32_t)s.n | (T::S(S_LINE) << 8) | (s.bank << 24);
    p.st[W_FRAME * B + e] += s.fdone;
    p.st[W_FCYC * B + e] = (uint32_t)(s.cyc - s.fstart);
    p.st[W_TIMER * B + e] = timer | (shift << 8) | (tflag << 12) | (sub << 16);
    p.st[W_PORTS * B + e] = T::S(S_PORTS);
    p.st[W_COLU * B + e] = T::S(S_COLU); p.st[W_PF * B + e] = T::S(S_PF); p.st[W_GRP * B + e] = T::S(S_GRP); p.st[W_NUSIZ * B + e] = T::S(S_NUSIZ);
    p.st[W_POS * B + e] = T::S(S_POS); p.st[W_POS2 * B + e] = (T::S(S_POS2) & 0xFFFF) | (T::S(S_RX) << 16);
    p.st[W_FLAGS * B + e] = T::S(S_FL) & TF_ARCH_MASK; p.st[W_CX * B + e] = T::S(S_CX);
    for (int i = 0; i < 32; ++i) p.ram[i * B + e] = smem[(S_RAM + i) * BLOCK + tid];
    p.cyc[e] += (unsigned long long)s.cyc;
  }
}

size_t step_smem_bytes(int block, bool roms, uint32_t max_rom) {
  return (size_t)(S_WORDS * block + C_WORDS + 128) * 4 + (roms ? (max_rom < 4096 ? 4096 : max_rom) + 16 : 0);
}

template <int BLOCK, bool ROMS>
static cudaError_t launch_one(const StepParams &p, cudaStream_t stream) {
  const size_t smem_bytes = step_smem_bytes(BLOCK, ROMS, p.max_rom);
  static size_t configured = 0;
  if (configured < smem_bytes) {
    cudaError_t e = cudaFuncSetAttribute(vcs_step_kernel<BLOCK, ROMS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
    if (e != cudaSuccess) return e;
    configured = smem_bytes;
  }
  const int grid = (p.batch + BLOCK - 1) / BLOCK;
  vcs_step_kernel<BLOCK, ROMS><<<grid, BLOCK, smem_bytes, stream>>>(p);
  return cudaGetLastError();
}

cudaError_t launch_step(const StepParams &p, cudaStream_t stream) {
  if (p.rom_smem) {
    switch (p.block) { case 64: return launch_one<64, true>(p, stream); case 256: return launch_one<256, true>(p, stream); default: return launch_one<128, true>(p, stream); }
  }
  switch (p.block) { case 64: return launch_one<64, false>(p, stream); case 256: return launch_one<256, false>(p, stream); default: return launch_one<128, false>(p, stream); }
}

}  // namespace vcs
