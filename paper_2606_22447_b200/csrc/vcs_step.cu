// vcs_step.cu — the persistent interpreter kernel behind vcs_step (SURVEY.md §8(a) a1–a16).
//
// One thread = one environment for the whole env-step (all `frameskip` frames): CPU registers, beam,
// RIOT and TIA latches stay in registers, the 128 RAM bytes and the scanline buffer in shared memory.
// Each loop iteration executes one 6507 instruction in four phases shared by all opcodes —
// addressing (switch on 13 modes) -> ONE generic operand-read site -> ALU (switch on op) -> ONE generic
// write site — so that lanes running different opcodes re-converge at the two bus sites, which are the
// only places the (large) lazy-TIA code is instantiated.  Cycle accounting is per bus access
// (C.4/C.5): an access `k` cycles into the instruction happens in cycle `cyc + k`, scanline slot `n + k`.
#include "vcs_env.cuh"
#include "vcs_optable.cuh"
#include "vcs_step.cuh"

namespace vcs {

__constant__ uint16_t c_optab[256];

void upload_optable() { cudaMemcpyToSymbol(c_optab, kOpTable, sizeof(kOpTable)); }
const uint16_t *host_optable() { return kOpTable; }

template <int BLOCK>
struct Cpu : Env<BLOCK> {
  using E = Env<BLOCK>;
  // side-effect-light read used for instruction bytes, zero-page pointers, JMP() vectors and stack
  // pulls: cartridge (incl. F8 hotspots) or RAM.  Anything else is outside the modelled set (status bit 2).
  DEV uint32_t lite_rd(uint32_t addr) {
    uint32_t a = addr & 0x1FFFu;
    if (a & 0x1000u) return E::rom_rd(a);
    if ((a & 0x0280u) == 0x0080u) return E::ram_rd(a);
    E::status |= STATUS_UNMODELLED; return 0;
  }
  DEV void push(uint32_t v) {
    if (E::SP & 0x80u) E::ram_wr(E::SP, v); else E::status |= STATUS_UNMODELLED;
    E::SP = (E::SP - 1u) & 0xFFu;
  }
  DEV uint32_t pull() {
    E::SP = (E::SP + 1u) & 0xFFu;
    if (E::SP & 0x80u) return E::ram_rd(E::SP);
    E::status |= STATUS_UNMODELLED; return 0;
  }
  // dummy read of an indexed mode's uncorrected address in cycle cyc+k: only INTIM and F8 hotspots react
  DEV void dummy_rd(uint32_t addr, int k) {
    uint32_t a = addr & 0x1FFFu;
    if (a & 0x1000u) E::hotspot(a);
    else if ((a & 0x0285u) == 0x0284u) { E::timer_sync(E::cyc + k + 1); E::tflag = 0; }
  }
  // the generic operand read (C.3 decode), k cycles into the instruction
  DEV uint32_t bus_read(uint32_t addr, int k) {
    uint32_t a = addr & 0x1FFFu;
    if ((a & 0x1280u) == 0x0080u) return E::ram_rd(a);
    if (a & 0x1000u) return E::rom_rd(a);
    if (a & 0x0080u) return E::riot_read(a, E::cyc + k);
    return E::tia_read(a, E::n + k);
  }
  DEV void bus_write(uint32_t addr, uint32_t v, int k) {
    uint32_t a = addr & 0x1FFFu;
    if ((a & 0x1280u) == 0x0080u) { E::ram_wr(a, v); return; }
    if (a & 0x1000u) { E::hotspot(a); return; }
    if (a & 0x0080u) { E::riot_write(a, v, E::cyc + k); return; }
    E::tia_write(a, v, E::cyc + k, E::n + k);
  }
  DEV uint32_t pack_p() const {
    return (E::nv & 0x80u) | (E::fV << 6) | 0x20u | (E::fD << 3) | (E::fI << 2) | (((E::zv & 0xFFu) == 0) ? 2u : 0u) | E::fC;
  }
  DEV void unpack_p(uint32_t p) {
    E::fC = p & 1u; E::zv = (p & 2u) ? 0u : 1u; E::fI = (p >> 2) & 1u; E::fD = (p >> 3) & 1u; E::fV = (p >> 6) & 1u; E::nv = p & 0x80u;
  }
  DEV void adc(uint32_t v) {                               // C.6, binary and NMOS decimal
    uint32_t A = E::A, C = E::fC;
    if (!E::fD) {
      uint32_t s = A + v + C;
      E::fC = s >> 8; E::fV = ((A ^ s) & (v ^ s) & 0x80u) >> 7; E::A = s & 0xFFu; E::zv = E::nv = E::A;
      return;
    }
    int al = (int)(A & 0x0Fu) + (int)(v & 0x0Fu) + (int)C;
    if (al >= 0x0A) al = ((al + 6) & 0x0F) + 0x10;
    int s = (int)(A & 0xF0u) + (int)(v & 0xF0u) + al;
    int sv = (int)(int8_t)(A & 0xF0u) + (int)(int8_t)(v & 0xF0u) + al;
    E::nv = (uint32_t)s & 0x80u;
    E::fV = (sv < -128 || sv > 127) ? 1u : 0u;
    E::zv = (A + v + C) & 0xFFu;
    if (s >= 0xA0) s += 0x60;
    E::fC = (s >= 0x100) ? 1u : 0u;
    E::A = (uint32_t)s & 0xFFu;
  }
  DEV void sbc(uint32_t v) {
    uint32_t A = E::A, C = E::fC;
    uint32_t nb = v ^ 0xFFu, s = A + nb + C;               // flags exactly as binary
    uint32_t bin = s & 0xFFu;
    E::fC = s >> 8; E::fV = ((A ^ s) & (nb ^ s) & 0x80u) >> 7; E::zv = E::nv = bin;
    if (!E::fD) { E::A = bin; return; }
    int al = (int)(A & 0x0Fu) - (int)(v & 0x0Fu) + (int)C - 1;
    if (al < 0) al = ((al - 6) & 0x0F) - 0x10;
    int d = (int)(A & 0xF0u) - (int)(v & 0xF0u) + al;
    if (d < 0) d -= 0x60;
    E::A = (uint32_t)d & 0xFFu;
  }

  // ---------------------------------------------------------------- one instruction (C.5)
  DEV void instruction(const uint16_t *optab) {
    const uint32_t pc = E::PC;
    const uint32_t opc = lite_rd(pc);
    const uint32_t ent = optab[opc];
    const uint32_t mode = ent & 15u, op = (ent >> 4) & 63u, kind = ent >> 10;
    if (op == OP_ILL) {                                    // C.12: halt for good, PC stays
      if (!(E::status & STATUS_UNMODELLED)) E::status |= STATUS_ILLEGAL;
      E::cyc += 1; E::n += 1; return;
    }
    const uint32_t b1 = lite_rd(pc + 1);                   // operand byte, or the dummy read @PC+1
    uint32_t ea = 0, v = 0, wv = 0;
    int k = 0;                                             // cycles before the operand access
    int total = 2;
    uint32_t npc = pc + 2;
    switch (mode) {
      case MD_IMP: case MD_ACC: npc = pc + 1; break;
      case MD_IMM: v = b1; k = 1; break;
      case MD_ZP:  ea = b1; k = 2; break;
      case MD_ZPX: ea = (b1 + E::X) & 0xFFu; k = 3; break;
      case MD_ZPY: ea = (b1 + E::Y) & 0xFFu; k = 3; break;
      case MD_ABS: ea = b1 | (lite_rd(pc + 2) << 8); k = 3; npc = pc + 3; break;
      case MD_ABX: case MD_ABY: case MD_IZY: {
        uint32_t lo, hi;
        if (mode == MD_IZY) { lo = lite_rd(b1); hi = lite_rd((b1 + 1u) & 0xFFu); k = 4; }
        else { lo = b1; hi = lite_rd(pc + 2); k = 3; npc = pc + 3; }
        uint32_t t = lo + ((mode == MD_ABX) ? E::X : E::Y);
        uint32_t unc = (hi << 8) | (t & 0xFFu);
        ea = (unc + (t & 0x100u)) & 0xFFFFu;
        if (kind != K_READ || (t & 0x100u)) { dummy_rd(unc, k); k += 1; }
      } break;
      case MD_IZX: { uint32_t z = (b1 + E::X) & 0xFFu; ea = lite_rd(z) | (lite_rd((z + 1u) & 0xFFu) << 8); k = 5; } break;
      default: break;                                      // MD_REL, MD_SPC: handled by op
    }
    if (kind & K_READ) {                                   // K_READ or K_RMW: the one generic read site
      if (mode != MD_IMM) v = bus_read(ea, k);
      total = k + 1;
    }
    switch (op) {
      case OP_LDA: E::A = v; E::zv = E::nv = v; break;
      case OP_LDX: E::X = v; E::zv = E::nv = v; break;
      case OP_LDY: E::Y = v; E::zv = E::nv = v; break;
      case OP_AND: E::A &= v; E::zv = E::nv = E::A; break;
      case OP_ORA: E::A |= v; E::zv = E::nv = E::A; break;
      case OP_EOR: E::A ^= v; E::zv = E::nv = E::A; break;
      case OP_ADC: adc(v); break;
      case OP_SBC: sbc(v); break;
      case OP_CMP: case OP_CPX: case OP_CPY: {
        uint32_t r = (op == OP_CMP) ? E::A : (op == OP_CPX) ? E::X : E::Y;
        E::fC = (r >= v) ? 1u : 0u; E::zv = E::nv = (r - v) & 0xFFu; } break;
      case OP_BIT: E::zv = E::A & v; E::nv = v; E::fV = (v >> 6) & 1u; break;
      case OP_STA: wv = E::A; break;
      case OP_STX: wv = E::X; break;
      case OP_STY: wv = E::Y; break;
      case OP_ASL: case OP_LSR: case OP_ROL: case OP_ROR: case OP_INC: case OP_DEC: {
        uint32_t s = (mode == MD_ACC) ? E::A : v, r;
        if (op == OP_ASL)      { r = (s << 1) & 0xFFu; E::fC = s >> 7; }
        else if (op == OP_LSR) { r = s >> 1; E::fC = s & 1u; }
        else if (op == OP_ROL) { r = ((s << 1) | E::fC) & 0xFFu; E::fC = s >> 7; }
        else if (op == OP_ROR) { r = (s >> 1) | (E::fC << 7); E::fC = s & 1u; }
        else if (op == OP_INC) { r = (s + 1u) & 0xFFu; }
        else                   { r = (s - 1u) & 0xFFu; }
        E::zv = E::nv = r;
        if (mode == MD_ACC) E::A = r; else wv = r;
      } break;
      case OP_CLC: E::fC = 0; break;
      case OP_SEC: E::fC = 1; break;
      case OP_CLD: E::fD = 0; break;
      case OP_SED: E::fD = 1; break;
      case OP_CLI: E::fI = 0; break;
      case OP_SEI: E::fI = 1; break;
      case OP_CLV: E::fV = 0; break;
      case OP_NOP: break;
      case OP_DEX: E::X = (E::X - 1u) & 0xFFu; E::zv = E::nv = E::X; break;
      case OP_DEY: E::Y = (E::Y - 1u) & 0xFFu; E::zv = E::nv = E::Y; break;
      case OP_INX: E::X = (E::X + 1u) & 0xFFu; E::zv = E::nv = E::X; break;
      case OP_INY: E::Y = (E::Y + 1u) & 0xFFu; E::zv = E::nv = E::Y; break;
      case OP_TAX: E::X = E::A; E::zv = E::nv = E::X; break;
      case OP_TAY: E::Y = E::A; E::zv = E::nv = E::Y; break;
      case OP_TSX: E::X = E::SP; E::zv = E::nv = E::X; break;
      case OP_TXA: E::A = E::X; E::zv = E::nv = E::A; break;
      case OP_TYA: E::A = E::Y; E::zv = E::nv = E::A; break;
      case OP_TXS: E::SP = E::X; break;
      case OP_BPL: case OP_BMI: case OP_BVC: case OP_BVS: case OP_BCC: case OP_BCS: case OP_BNE: case OP_BEQ: {
        uint32_t idx = op - OP_BPL, f;
        switch (idx >> 1) { case 0: f = (E::nv >> 7) & 1u; break; case 1: f = E::fV; break; case 2: f = E::fC; break;
                            default: f = ((E::zv & 0xFFu) == 0) ? 1u : 0u; break; }
        if (f == (idx & 1u)) {
          uint32_t next = (pc + 2u) & 0xFFFFu;
          uint32_t target = (next + (uint32_t)(int32_t)(int8_t)b1) & 0xFFFFu;
          E::hotspot(next & 0x1FFFu);                      // dummy read @PC
          total = 3;
          if ((target ^ next) & 0xFF00u) { E::hotspot(((next & 0xFF00u) | (target & 0xFFu)) & 0x1FFFu); total = 4; }
          npc = target;
        }
      } break;
      case OP_JMP: npc = b1 | (lite_rd(pc + 2) << 8); total = 3; break;
      case OP_JMPI: { uint32_t hi = lite_rd(pc + 2);
        uint32_t l2 = lite_rd((hi << 8) | b1), h2 = lite_rd((hi << 8) | ((b1 + 1u) & 0xFFu));   // no carry into the page
        npc = l2 | (h2 << 8); total = 5; } break;
      case OP_JSR: { uint32_t ret = (pc + 2u) & 0xFFFFu;     // address of the 3rd byte
        push(ret >> 8); push(ret & 0xFFu);
        npc = b1 | (lite_rd(ret) << 8); total = 6; } break;
      case OP_RTS: { uint32_t lo = pull(), hi = pull(); uint32_t r = lo | (hi << 8);
        E::hotspot(r & 0x1FFFu); npc = (r + 1u) & 0xFFFFu; total = 6; } break;
      case OP_RTI: { unpack_p(pull()); uint32_t lo = pull(), hi = pull(); npc = lo | (hi << 8); total = 6; } break;
      case OP_PHA: push(E::A); npc = pc + 1; total = 3; break;
      case OP_PHP: push(pack_p() | 0x30u); npc = pc + 1; total = 3; break;
      case OP_PLA: E::A = pull(); E::zv = E::nv = E::A; npc = pc + 1; total = 4; break;
      case OP_PLP: unpack_p(pull()); npc = pc + 1; total = 4; break;
      case OP_BRK: { uint32_t ret = (pc + 2u) & 0xFFFFu;
        push(ret >> 8); push(ret & 0xFFu); push(pack_p() | 0x30u);
        npc = lite_rd(0xFFFEu) | (lite_rd(0xFFFFu) << 8); E::fI = 1; total = 7; } break;
      default: break;
    }
    E::PC = npc & 0xFFFFu;
    if (kind & K_WRITE) {                                  // K_WRITE: one write; K_RMW: old value, then new
      const bool rmw = (kind == K_RMW);
      total = k + (rmw ? 3 : 1);
#pragma unroll 1
      for (int i = rmw ? 0 : 1; i < 2; ++i)               // the one generic write site
        bus_write(ea, i ? wv : v, k + (rmw ? 1 + i : 0));
    }
    E::cyc += total; E::n += total;
  }
};

template <int BLOCK>
__global__ void __launch_bounds__(BLOCK) vcs_step_kernel(StepParams p) {
  extern __shared__ uint32_t smem[];
  uint32_t *s_ram = smem;                                  // [32][BLOCK]
  uint32_t *s_lbuf = smem + 32 * BLOCK;                    // [40][BLOCK]
  uint16_t *s_optab = reinterpret_cast<uint16_t *>(smem + 72 * BLOCK);
  const int tid = threadIdx.x;
  const int e = blockIdx.x * BLOCK + tid;
  for (int i = tid; i < 256; i += BLOCK) s_optab[i] = c_optab[i];
  __syncthreads();
  if (e >= p.batch) return;
  const int B = p.batch;

  Cpu<BLOCK> s;
  // ---- a1 state load (coalesced SoA)
  {
    uint32_t w;
    w = p.st[W_AXYS * B + e]; s.A = w & 0xFF; s.X = (w >> 8) & 0xFF; s.Y = (w >> 16) & 0xFF; s.SP = w >> 24;
    w = p.st[W_PC * B + e]; s.PC = w & 0xFFFF; s.unpack_p((w >> 16) & 0xFF); s.status = w >> 24;
    w = p.st[W_BEAM * B + e]; s.n = w & 0xFF; s.line = (w >> 8) & 0xFFFF; s.bank = w >> 24;
    s.frame = p.st[W_FRAME * B + e];
    s.cyc = 0; s.fstart = -(int32_t)p.st[W_FCYC * B + e];
    w = p.st[W_TIMER * B + e]; s.timer = w & 0xFF; s.shift = (w >> 8) & 0xF; s.tflag = (w >> 12) & 1; s.sub = w >> 16; s.tticks = 0;
    s.ports = p.st[W_PORTS * B + e];
    s.colu = p.st[W_COLU * B + e]; s.pf = p.st[W_PF * B + e]; s.grp = p.st[W_GRP * B + e]; s.nusiz = p.st[W_NUSIZ * B + e];
    s.pos = p.st[W_POS * B + e]; w = p.st[W_POS2 * B + e]; s.pos2 = w & 0xFFFF; s.rx = w >> 16;
    s.fl = p.st[W_FLAGS * B + e]; s.cx = p.st[W_CX * B + e];
    for (int i = 0; i < 32; ++i) s_ram[i * BLOCK + tid] = p.ram[i * B + e];
  }
  s.ram = reinterpret_cast<uint8_t *>(s_ram) + 4 * tid;
  s.lbuf = s_lbuf + tid;
  s.screen = p.screen + (size_t)e * (SCR_W * SCR_H);
  s.y0 = p.y0; s.cap = p.max_lines * LINE_CYC;
  s.frames_done = 0; s.frameskip = p.frameskip; s.storing = (p.frameskip == 1);
  {
    const RomMeta rm = p.rom_meta[p.env_rom[e]];
    s.rom = p.rom_blob + rm.offset; s.rom_mask = (rm.size == 2048) ? 0x7FFu : 0xFFFu; s.is_f8 = (rm.size == 8192);
  }
  // ---- a2 action latch (C.11)
  {
    uint32_t act = p.actions[e]; if (act >= 18u) act = 0;
    //            NOOP FIRE UP RIGHT LEFT DOWN UR UL DR DL UF RF LF DF URF ULF DRF DLF
    const uint32_t up = 0x0C4C4u, down = 0x32320u, left = 0x29290u, right = 0x14948u, fire = 0x3FC02u;
    uint32_t ina = 0xFFu;
    if ((up >> act) & 1u) ina &= ~0x10u;
    if ((down >> act) & 1u) ina &= ~0x20u;
    if ((left >> act) & 1u) ina &= ~0x40u;
    if ((right >> act) & 1u) ina &= ~0x80u;
    s.ina = ina; s.fire0 = (fire >> act) & 1u;
    s.eval_fire_latch();
  }
  // ---- the hot loop: whole instructions until `frameskip` frame-end events (C.10)
  // Line bookkeeping mirrors C.4: the line counter advances with the FIRST cycle of a new line, so an
  // instruction that ends exactly on a line boundary leaves n == 76 pending (a frame end at that point
  // makes the finished line "line 0" and the next one line 1).
  while (s.frames_done < s.frameskip) {
    if (s.cyc - s.fstart >= s.cap) {                       // frame cap at the instruction boundary
      s.status |= STATUS_CAP; s.frame_end(3u * (uint32_t)s.n, s.cyc); continue;
    }
    if (s.n >= LINE_CYC) s.new_line();                     // n == 76 exactly (see above)
    if (s.status & (STATUS_ILLEGAL | STATUS_UNMODELLED)) {  // halted: idle cycles to the line end / the cap
      int d = min(LINE_CYC - s.n, s.cap - (s.cyc - s.fstart));
      s.cyc += d; s.n += d;
      continue;
    }
    if (s.fl & TF_WSYNC) {                                 // a12: RDY holds the CPU until the line ends
      s.cyc += LINE_CYC - s.n; s.n = LINE_CYC; s.new_line();
    }
    s.instruction(s_optab);
    if (s.n > LINE_CYC) s.new_line();
  }
  // ---- a16 state store
  s.timer_sync(s.cyc);
  {
    p.st[W_AXYS * B + e] = s.A | (s.X << 8) | (s.Y << 16) | (s.SP << 24);
    p.st[W_PC * B + e] = s.PC | (s.pack_p() << 16) | (s.status << 24);
    p.st[W_BEAM * B + e] = (uint32_t)s.n | (s.line << 8) | (s.bank << 24);
    p.st[W_FRAME * B + e] = s.frame;
    p.st[W_FCYC * B + e] = (uint32_t)(s.cyc - s.fstart);
    p.st[W_TIMER * B + e] = s.timer | (s.shift << 8) | (s.tflag << 12) | (s.sub << 16);
    p.st[W_PORTS * B + e] = s.ports;
    p.st[W_COLU * B + e] = s.colu; p.st[W_PF * B + e] = s.pf; p.st[W_GRP * B + e] = s.grp; p.st[W_NUSIZ * B + e] = s.nusiz;
    p.st[W_POS * B + e] = s.pos; p.st[W_POS2 * B + e] = (s.pos2 & 0xFFFF) | (s.rx << 16);
    p.st[W_FLAGS * B + e] = s.fl; p.st[W_CX * B + e] = s.cx;
    for (int i = 0; i < 32; ++i) p.ram[i * B + e] = s_ram[i * BLOCK + tid];
    p.cyc[e] += (unsigned long long)s.cyc;
  }
}

cudaError_t launch_step(const StepParams &p, cudaStream_t stream) {
  constexpr int BLOCK = STEP_BLOCK;
  const size_t smem = (size_t)72 * BLOCK * 4 + 512;
  static bool configured = false;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(vcs_step_kernel<BLOCK>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  const int grid = (p.batch + BLOCK - 1) / BLOCK;
  vcs_step_kernel<BLOCK><<<grid, BLOCK, smem, stream>>>(p);
  return cudaGetLastError();
}

}  // namespace vcs
