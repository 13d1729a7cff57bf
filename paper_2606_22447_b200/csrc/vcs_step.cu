// vcs_step.cu — the persistent interpreter kernel behind vcs_step (SURVEY.md §8(a) a1–a16).
//
// One thread = one environment for the whole env-step (all `frameskip` frames).  CPU registers and the beam
// position live in registers; RAM, the TIA/RIOT latches, the cached TIA object masks and the colour-index
// planes live in the thread's shared-memory file; the block's cartridge ROM is staged in shared memory with
// one bulk asynchronous copy (TMA 1-D, cp.async.bulk + mbarrier) when all of the block's envs share a ROM.
//
// Dispatch.  vcs_create pre-decodes every byte offset of every ROM bank into a 64-bit entry (vcs_decode.cuh):
// a fused handler id, the instruction's base cycles and length, a "leader" flag and a 32-bit operand (already
// turned into a shared-memory offset for RAM cells).  The hot loop loads that entry through the read-only
// path (L1), prefetches the sequentially next one before it dispatches, adds cycles and length straight from
// the entry and jumps ONCE (one BRX) into a handler that is specialised for opcode x address class; only
// indexed / indirect / absolute-I/O modes take a second-level operation switch and count their own bus
// accesses.  PCs outside cartridge space and the last 16 bytes of a bank decode at run time (H_SLOW).
//
// The program counter is kept as (di, pbase): di = bank<<12 | PC & 0xFFF indexes the decode entries and
// PC = (pbase + di) & 0xFFFF; straight-line code and in-window branches only touch di.
//
// Divergence (the measured choice north_star asks for): lanes of a warp are NOT run in lock-step.  At every
// scheduling point each lane forms the key (frames done, SP, bank, PC); a warp-wide REDUX.MIN picks the
// smallest and only the lanes holding it run — all at the same PC of the same ROM, hence the same handler,
// the same operand and (for stores) the same TIA register: dispatch, the TIA write switch and the lazy-TIA
// catch-up are warp-uniform.  Lower SP first returns lanes from subroutines, lower PC first re-joins forward
// branches, the frame count bounds how long a lane can wait.  A group keeps running straight-line code
// without re-forming until it executes a control transfer or reaches a leader (a static branch/JMP/JSR target
// or return point — the only places where another lane can be waiting), so the REDUX is paid per basic
// block, not per instruction.
//
// Cycle accounting is per bus access (C.4/C.5).  Specialised handlers add the entry's cycle count before
// they run (their one side-effecting access is the last cycle: cycle index cyc - 1 afterwards); generic
// handlers run with `cyc` at the instruction's first cycle, an access `k` cycles into the instruction
// happens in cycle `cyc + k`, scanline slot `cyc - lstart + k`, and add their total at the end.
#include "vcs_tia.cuh"
#include "vcs_decode.cuh"
#include "vcs_step.cuh"

#ifndef VCS_PAD
#define VCS_PAD 0
#endif
namespace vcs {

__constant__ uint32_t c_gen[256];       // generic decode per opcode (vcs_decode.cuh generic_entry) for H_SLOW

void upload_optable() {
  uint32_t g[256];
  for (int i = 0; i < 256; ++i) g[i] = generic_entry((uint32_t)i);
  cudaMemcpyToSymbol(c_gen, g, sizeof(g));
  uint32_t td[64]; tia_desc_table(td);
  cudaMemcpyToSymbol(c_tia_desc, td, sizeof(td));
}
const uint16_t *host_optable() { return kOpTable; }

constexpr int32_t LIM_NOW = (int32_t)0x80000000;     // `lim` value that forces the slow pre-check
constexpr uint32_t KEY_PARKED = 0xFFFE0000u;         // keys >= this: parked for a regroup / finished the step
constexpr uint32_t NOSLOT = 0xFFFFFFFFu;             // a thread of the spare warp that holds no environment right now
constexpr int32_t LIM_WSYNC = LIM_NOW + 1;            // `lim` while WSYNC holds the CPU (and nothing else is pending)

// ---- RIOT: interval timer in closed form and the two I/O ports (C.7).  All of its state lives in the thread's
// shared-memory file, so these are plain static functions of the file slot.
template <int BLOCK, int TAG = 0>
struct Riot {
  using T = Tia<BLOCK, TAG>;
  static DEV uint32_t &S(uint32_t sl, int i) { return T::S(sl, i); }
  // advance the (timer, sub, tflag) state in smem to "after `ticks` cycles of this step" and return it unpacked
  static DEV void timer_sync(uint32_t sl, int32_t ticks, uint32_t &timer, uint32_t &sub, uint32_t &shift, uint32_t &tflag) {
    const uint32_t tw = S(sl, S_TMR);
    timer = tw & 0xFFu; shift = (tw >> 8) & 0xFu; tflag = (tw >> 12) & 1u; sub = tw >> 16;
    const uint32_t d = (uint32_t)(ticks - (int32_t)S(sl, S_TTICKS));
    if ((int32_t)d <= 0) return;
    S(sl, S_TTICKS) = (uint32_t)ticks;
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
  static DEV void timer_put(uint32_t sl, uint32_t timer, uint32_t sub, uint32_t shift, uint32_t tflag) { S(sl, S_TMR) = timer | (shift << 8) | (tflag << 12) | (sub << 16); }
  // INTIM / TIMINT read in cycle index c (tick c happened first)
  static DEV uint32_t timer_read(uint32_t sl, uint32_t a, int32_t c) {
    const uint32_t tw = S(sl, S_TMR);
    const uint32_t d = (uint32_t)(c + 1 - (int32_t)S(sl, S_TTICKS));
    if (!(tw & 0x1000u) && (int32_t)d > 0) {          // before the underflow nothing has to be written back
      const uint32_t timer = tw & 0xFFu, k = ((tw >> 16) + d) >> ((tw >> 8) & 0xFu);
      if (k <= timer) return (a & 1u) ? 0u : timer - k;
    }
    uint32_t timer, sub, shift, tflag;
    timer_sync(sl, c + 1, timer, sub, shift, tflag);
    if (!(a & 1u)) { timer_put(sl, timer, sub, shift, 0); return timer; }     // INTIM clears the flag
    timer_put(sl, timer, sub, shift, tflag);
    return tflag << 7;                                                        // TIMINT
  }
  static DEV uint32_t read(uint32_t sl, uint32_t a, int32_t c) {     // access in cycle index c
    if ((a & 4u) == 0) {
      const uint32_t ports = S(sl, S_PORTS);
      const uint32_t ora = byte_of(ports, 0), ddra = byte_of(ports, 1), orb = byte_of(ports, 2), ddrb = byte_of(ports, 3);
      switch (a & 3u) {
        case 0: return (ora & ddra) | (S(sl, S_INP) & ~ddra & 0xFFu);
        case 1: return ddra;
        case 2: { const uint32_t k = S(sl, S_INP) >> 9;    // console switches (vcs_set_switches), pins 2, 4, 5 not connected
                  const uint32_t inb = 0x34u | (k & 3u) | ((k & 4u) << 1) | ((k & 0x18u) << 3);
                  return (orb & ddrb) | (inb & ~ddrb); }
        default: return ddrb;
      }
    }
    return timer_read(sl, a, c);
  }
  static DEV void write(uint32_t sl, uint32_t a, uint32_t v, int32_t c) {
    if ((a & 4u) == 0) { S(sl, S_PORTS) = set_byte(S(sl, S_PORTS), a & 3u, v); return; }
    if ((a & 0x14u) == 0x14u) {
      const uint32_t k = a & 3u;
      const uint32_t shift = (k == 0) ? 0u : (k == 1) ? 3u : (k == 2) ? 6u : 10u;
      timer_put(sl, v & 0xFFu, (1u << shift) - 1u, shift, 0); S(sl, S_TTICKS) = (uint32_t)(c + 1);
    }
  }
};
// Bus accesses that are neither RAM nor cartridge (a = addr & 0x1FFF without A12; c = cycle index in this step, m = cycle
// in the scanline).  Inline: a call level more on the way to the TIA functions costs them convergence-barrier registers
// (ptxas then saves / restores B registers with BMOV inside render_visible & co.: measured +20 % instructions there).
template <int BLOCK, int TAG>
DEV uint32_t io_read(uint32_t sl, uint32_t a, int32_t c, int m) {       // -> value | line ends performed << 12
  if (a & 0x0080u) return Riot<BLOCK, TAG>::read(sl, a, c);
  return Tia<BLOCK, TAG>::read(sl, a & 0xFu, m);
}
template <int BLOCK, int TAG>
DEV uint32_t io_write(uint32_t sl, uint32_t a, uint32_t v, int32_t c, int m) {   // -> TIA events (EV_*)
  if (a & 0x0080u) { Riot<BLOCK, TAG>::write(sl, a, v, c); return 0; }
  const uint32_t r = a & 0x3Fu;
  if (r > 0x2Cu || (r >= 0x15u && r <= 0x1Au) || r == 0x03u) return 0;      // no effect (audio: PAPER.md L205)
  return Tia<BLOCK, TAG>::write(sl, r, v, m);
}
template <int BLOCK, int TAG>
DEV void io_dummy_intim(uint32_t sl, int32_t ticks) {      // a discarded read of INTIM still clears the underflow flag
  uint32_t t, s, sh, f; Riot<BLOCK, TAG>::timer_sync(sl, ticks, t, s, sh, f); Riot<BLOCK, TAG>::timer_put(sl, t, s, sh, 0);
}

// ---- SOFT-STE mode (vcs_step_soft; eq. (8)-(10), reading R14): per-env sums in shared memory behind the block
// context (the soft kernel stages no ROM): word k of env slot sl at SOFT_ACC + k * BLOCK + sl, k = sum of soft ROM reads,
// of soft RAM reads, of branch gates, the three counts, STE/hard mismatches, max |soft - hard|.
template <int BLOCK> DEV float &soft_acc(uint32_t sl, int k) { return reinterpret_cast<float *>(smem)[S_WORDS * BLOCK + C_WORDS + k * BLOCK + sl]; }
template <int BLOCK> DEV void soft_note(uint32_t sl, int k, float soft_v, float hard, float ste) {
  soft_acc<BLOCK>(sl, k) += soft_v; soft_acc<BLOCK>(sl, 3 + k) += 1.f;
  if (rintf(ste) != hard) soft_acc<BLOCK>(sl, 6) += 1.f;
  if (k < 2) soft_acc<BLOCK>(sl, 7) = fmaxf(soft_acc<BLOCK>(sl, 7), fabsf(soft_v - hard));
}
// eq. (10) on the 128-cell RAM tape, window |k| <= K clipped to the tape, then STE + round (one copy: the inline loop and
// the out-of-line executor both read RAM through it in soft mode).  The weights are e^{-|k|/T} = q^|k|, so each side of
// the window is a Horner chain from its far end towards the cell, taken a RAM word (4 cells) at a time: the four cells
// of a word combine off the critical path and the running sum advances by one multiply-add (x q^4) per word; no weight
// loads.  The normaliser comes from the cumulative table cw[n] = sum_{j<=n} e^{-j/T} (host, in double): den = cw[nl] +
// cw[nr] - 1.  `hard` is ram[cell].
template <int BLOCK>
__device__ __noinline__ uint32_t soft_ram_read(uint32_t sl, uint32_t cell, uint32_t hard) {
  using T = Tia<BLOCK>;
  const int K = (int)(T::ctx(C_SOFT_K) & 0x7FFFFFFFu);
  const float *wt = reinterpret_cast<const float *>((unsigned long long)T::ctx(C_SOFT_W_LO) | ((unsigned long long)T::ctx(C_SOFT_W_HI) << 32));
  const uint32_t *ramw = smem + sl;                        // RAM word i of this env at ramw[i * BLOCK], cell 4 i + j in byte j
  const float q = __ldg(wt + 1), q4 = (q * q) * (q * q);
  const int c = (int)cell, nl = min(K, c), nr = min(K, 127 - c), a = c - nl, b = c + nr, wc = c >> 2, m = c & 3;
  const uint32_t keep_a = 0xFFFFFFFFu << (8 * (a & 3)), keep_b = 0xFFFFFFFFu >> (8 * (3 - (b & 3)));   // cells of the edge words inside [a, b]
  auto f = [](uint32_t x, int j) { return (float)((x >> (8 * j)) & 0xFFu); };
  float L = 0.f, R = 0.f;                                  // L: sum_{j < 4 wc} q^(4 wc - 1 - j) ram[j];  R: sum_{j >= 4 wc + 4} q^(j - 4 wc - 4) ram[j]
#pragma unroll 2
  for (int w = a >> 2; w < wc; ++w) {
    uint32_t x = ramw[w * BLOCK]; if (w == (a >> 2)) x &= keep_a;
    L = fmaf(L, q4, fmaf(fmaf(fmaf(f(x, 0), q, f(x, 1)), q, f(x, 2)), q, f(x, 3)));
  }
#pragma unroll 2
  for (int w = b >> 2; w > wc; --w) {
    uint32_t x = ramw[w * BLOCK]; if (w == (b >> 2)) x &= keep_b;
    R = fmaf(R, q4, fmaf(fmaf(fmaf(f(x, 3), q, f(x, 2)), q, f(x, 1)), q, f(x, 0)));
  }
  uint32_t x = ramw[wc * BLOCK];                           // the cell's own word: up to 3 more cells on either side
  if ((a >> 2) == wc) x &= keep_a;
  if ((b >> 2) == wc) x &= keep_b;
  if (m > 0) L = fmaf(L, q, f(x, 0));
  if (m > 1) L = fmaf(L, q, f(x, 1));
  if (m > 2) L = fmaf(L, q, f(x, 2));
  if (m < 3) R = fmaf(R, q, f(x, 3));
  if (m < 2) R = fmaf(R, q, f(x, 2));
  if (m < 1) R = fmaf(R, q, f(x, 1));
  const float h = (float)hard;
  const float sv = (h + (L + R) * q) / (__ldg(wt + SOFT_CW + nl) + __ldg(wt + SOFT_CW + nr) - 1.f), ste = sv + (h - sv);
  soft_note<BLOCK>(sl, 1, sv, h, ste);
  return (uint32_t)(int)rintf(ste) & 0xFFu;
}
// eq. (8) + STE for a conditional branch: f = the flag tested, sense = +1 branch-if-set / -1 branch-if-clear
template <int BLOCK>
__device__ __noinline__ void soft_branch_note(uint32_t sl, uint32_t f, float sense, float delta, bool taken, float pc_nb) {
  const float z = sense * (2.f * (float)f - 1.f), alpha = __uint_as_float(Tia<BLOCK>::ctx(C_SOFT_ALPHA));
  const float g = 1.f / (1.f + expf(-alpha * z));
  const float pc_soft = pc_nb + g * delta, pc_hard = pc_nb + (taken ? delta : 0.f);
  soft_note<BLOCK>(sl, 2, g, pc_hard, pc_soft + (pc_hard - pc_soft));
}

// What the inline interpreter loop keeps in registers.  A, X, Y, SP are the four bytes of `axys`, so that "which
// register" is a byte-permute selector from the decode entry; `fl` holds C, I, D, V at their P-register bits.
// Everything else of an environment (status, frame start, TIA/RIOT latches, RAM) lives in its shared-memory file
// and block-uniform values live in the block context; the out-of-line paths below rebuild a full Cpu from both.
#ifndef VCS_COLD_TAG
#define VCS_COLD_TAG 2
#endif
constexpr int COLD_TAG = VCS_COLD_TAG;               // the copy of the TIA code the compact out-of-line executor calls (vcs_tia.cuh)
constexpr uint32_t AUX_GENERIC = 2u;                 // Hot::aux after cold_exec: run the entry (wx, wy) on cold_exec_generic
struct Hot {
  uint32_t axys, fl, zn;               // Z <=> (zn & 0xFF) == 0 ; N <=> (zn & 0x180) != 0
  uint32_t di, pbase;                  // PC = (pbase + di) & 0xFFFF ; di = bank<<12 | PC & 0xFFF
  int32_t cyc, lstart, lim;
  uint32_t keyhi;                      // scheduling key without the PC
  uint32_t wx, wy;                     // decode entry at (bank, PC)
  uint32_t aux;                        // return flag of the out-of-line calls
};

template <int BLOCK, int ROMS, int THREADS, bool SOFT, int TAG = 0>      // TAG: which copy of the TIA code this Cpu calls (vcs_tia.cuh)
struct Cpu {
  using T = Tia<BLOCK, TAG>;
  // ---- CPU
  uint32_t A, X, Y, SP;
  uint32_t di, pbase;                  // PC = (pbase + di) & 0xFFFF ; di = bank<<12 | PC & 0xFFF
  uint32_t fC, fV, fDI, zn;            // fDI: bit3 D, bit2 I ; Z <=> (zn & 0xFF) == 0 ; N <=> (zn & 0x180) != 0
  uint32_t status, romid;
  // ---- beam / time (cycle counts are relative to the start of this vcs_step call)
  int32_t cyc;        // CPU cycles executed in this step
  int32_t lstart;     // value of `cyc` at which the current scanline began (cycle-in-line n = cyc - lstart, 0..76+)
  int32_t fstart;     // value of `cyc` at which the current frame began (frame_cyc = cyc - fstart)
  int32_t lim;        // fast path allowed while cyc < lim: min(line end, frame cap), LIM_NOW when WSYNC/halted
  int32_t cap;        // frame cap in cycles
  uint32_t fdone;     // frames completed in this step (mirror of S_FDONE)
  uint32_t fskip;     // frames to run
  uint32_t keyhi;     // scheduling key without the PC: frames done << 27 | SP << 19 | bank << 16 (or KEY_PARKED / ~0)
  bool wsync;         // mirror of TF_WSYNC
  // ---- cart
  uint32_t hs_lo, hs_n, rom_mask;      // bank hotspots: hs_n addresses from hs_lo (F8 $1FF8 x2, F6 $1FF6 x4, F4 $1FF4 x8); hs_n 0 = none
  uint32_t kind;      // MapKind of this env's cartridge
  uint32_t park;      // bit0: this block regroups its envs at bank-hotspot accesses; bit1: this lane is parked for a
                      // regroup; bit2: a bank hotspot was accessed by the instruction in flight
  uint32_t rom_off;   // ROMS == 1: byte offset of the ROM image inside smem
  const uint8_t *rom_g;    // ROMS != 1: the image in global memory
  const uint2 *dr;         // decode entries of this env's ROM (4096 per bank)
  uint2 w;            // decode entry at (bank, PC) — valid at every scheduling point
  uint32_t sl, sl4;   // this thread's file slot (word i of the file lives at smem[i*BLOCK + sl]) and 4*sl
  const float *soft_tab;   // SOFT-STE mode (vcs_step_soft): the relaxed read of every cell of this env's ROM (4096 per bank), else nullptr

  DEV uint32_t &S(int i) const { return T::S(sl, i); }

  // ---- Hot <-> Cpu (the out-of-line paths run on a full Cpu; see struct Hot)
  template <bool CART = true>
  DEV void load(const Hot &h, uint32_t slot) {
    sl = slot; sl4 = 4u * slot;
    A = h.axys & 0xFFu; X = (h.axys >> 8) & 0xFFu; Y = (h.axys >> 16) & 0xFFu; SP = h.axys >> 24;
    fC = h.fl & 1u; fDI = h.fl & 0x0Cu; fV = (h.fl >> 6) & 1u; zn = h.zn;
    di = h.di; pbase = h.pbase; cyc = h.cyc; lstart = h.lstart; lim = h.lim; keyhi = h.keyhi; w = make_uint2(h.wx, h.wy);
    const uint32_t sw = S(S_STATUS);
    status = sw & 0xFFu; romid = sw >> 8; fstart = (int32_t)S(S_FSTART); fdone = S(S_FDONE); wsync = (S(S_FL) & TF_WSYNC) != 0;
    cap = (int32_t)T::ctx(C_CAP); fskip = T::ctx(C_FRAMESKIP); rom_off = T::ctx(C_ROMOFF);
    if constexpr (CART) {                                  // (the line-end / event paths never touch the cartridge)
      auto ptr = [](int lo) { return (unsigned long long)T::ctx(lo) | ((unsigned long long)T::ctx(lo + 1) << 32); };
      const RomMeta rm = reinterpret_cast<const RomMeta *>(ptr(C_META_LO))[romid];
      hs_n = (rm.hs >> 16) & 0xFFu; hs_lo = rm.hs & 0xFFFFu; kind = rm.kind; rom_mask = (rm.size == 2048 && ROMS != 1) ? 0x7FFu : 0xFFFu;
      rom_g = reinterpret_cast<const uint8_t *>(ptr(C_BLOB_LO)) + rm.offset;
      dr = reinterpret_cast<const uint2 *>(ptr(C_DROM_LO)) + rm.doff;
      if constexpr (SOFT) soft_tab = reinterpret_cast<const float *>(ptr(C_SOFT_TAB_LO)) + rm.pad;
      else soft_tab = nullptr;
    } else { hs_n = 0; hs_lo = 0; kind = MK_4K; rom_mask = 0xFFFu; rom_g = nullptr; dr = nullptr; soft_tab = nullptr; }
    park = T::ctx(C_REGROUP) | ((keyhi == KEY_PARKED) ? 2u : 0u);
  }
  DEV Hot store() const {
    Hot h;
    h.axys = A | (X << 8) | (Y << 16) | (SP << 24); h.fl = fC | fDI | (fV << 6); h.zn = zn;
    h.di = di; h.pbase = pbase; h.cyc = cyc; h.lstart = lstart; h.lim = lim; h.keyhi = keyhi; h.wx = w.x; h.wy = w.y; h.aux = 0;
    S(S_STATUS) = status | (romid << 8); S(S_FSTART) = (uint32_t)fstart;
    return h;
  }

  DEV uint32_t pc() const { return (pbase + di) & 0xFFFFu; }
  DEV void set_pc(uint32_t p) { const uint32_t nd = (di & 0x7000u) | (p & 0xFFFu); pbase = p - nd; di = nd; }
  DEV void rekey() {
    keyhi = (fdone >= fskip) ? 0xFFFFFFFFu : (park & 2u) ? KEY_PARKED : (min(fdone, 30u) << 27) | (SP << 19) | ((di & 0x7000u) << 4);
  }

  // ------------------------------------------------------------------ RAM (smem, conflict-free)
  DEV uint32_t ram_rd_off(uint32_t off) const { return reinterpret_cast<const uint8_t *>(smem)[off + sl4]; }
  DEV void ram_wr_off(uint32_t off, uint32_t v) { reinterpret_cast<uint8_t *>(smem)[off + sl4] = (uint8_t)v; }
  DEV uint32_t ram_rd(uint32_t a, bool value = true) {
    const uint32_t v = ram_rd_off(((a & 0x7Cu) * BLOCK) | (a & 3u));
    if constexpr (SOFT) { if (value) return soft_ram(a & 0x7Fu, v); }
    return v;
  }
  DEV void ram_wr(uint32_t a, uint32_t v) { ram_wr_off(((a & 0x7Cu) * BLOCK) | (a & 3u), v); }

  // ------------------------------------------------------------------ ROM
  DEV uint32_t rom_byte(uint32_t off) const {
    if constexpr (ROMS == 1) return reinterpret_cast<const uint8_t *>(smem)[rom_off + off];
    else return __ldg(rom_g + off);
  }
  // any access to a hotspot ($1FF8/$1FF9 on F8 carts) selects the bank; in a block that regroups it also parks the lane (park bit 1)
  // --- formats only the generic executor (TAG 1) runs: Superchip RAM ports, E0's 1 KB windows, FE (include/vcs.h)
  DEV uint8_t *sc_cell(uint32_t cell) const {              // byte `cell` of this env's Superchip RAM ([32][batch] words in global memory)
    uint32_t *base = reinterpret_cast<uint32_t *>((unsigned long long)T::ctx(C_SCRAM_LO) | ((unsigned long long)T::ctx(C_SCRAM_HI) << 32));
    return reinterpret_cast<uint8_t *>(base + (size_t)(cell >> 2) * T::ctx(C_BATCH) + (T::ctx(C_ENV0) + (S(S_INP) >> 16))) + (cell & 3u);
  }
  DEV bool has_sc() const { return kind - MK_F8SC <= MK_F4SC - MK_F8SC; }
  DEV void fe_snoop(uint32_t a, uint32_t data) {           // FE: the access after one to $01FE selects the bank from bit 5 of its data
    if (kind != MK_FE) return;
    uint32_t c = S(S_CART);
    if (c & 0x200u) {
      const uint32_t nd = (di & 0xFFFu) | ((data & 0x20u) ? 0u : 0x1000u);
      pbase += di - nd; di = nd; rekey();
      c &= ~0x200u;
    }
    if (a == 0x01FEu) c |= 0x200u;
    S(S_CART) = c;
  }
  DEV void hotspot(uint32_t a) {
    if constexpr (TAG == 1) {
      if (kind == MK_E0) {                                 // $1FE0-7 / $1FE8-F / $1FF0-7: slice of the window at $1000 / $1400 / $1800
        if (a - 0x1FE0u < 0x18u) { const uint32_t sh = 3u * ((a - 0x1FE0u) >> 3); S(S_CART) = (S(S_CART) & ~(7u << sh)) | ((a & 7u) << sh); }
        return;
      }
    }
    if (a - hs_lo < hs_n) {
      const uint32_t nd = (di & 0xFFFu) | ((a - hs_lo) << 12);
      pbase += di - nd; di = nd;                     // PC is unchanged
      park |= 4u | ((park & 1u) << 1);
      rekey();
    }
  }
  DEV uint32_t rom_rd(uint32_t a, bool value = true) {   // a = addr & 0x1FFF with A12 set; value: the byte is used (not a dummy cycle)
    hotspot(a);
    if constexpr (TAG == 1) {
      if (has_sc() && (a & 0x0F00u) == 0) return *sc_cell(a & 0x7Fu);          // read port (a read of the write port sees the cell too)
      if (kind == MK_E0) { const uint32_t w = (a >> 10) & 3u, slice = (w == 3u) ? 7u : (S(S_CART) >> (3u * w)) & 7u; return rom_byte(slice * 1024u + (a & 0x3FFu)); }
    }
    const uint32_t v = rom_byte((di & 0x7000u) + (a & rom_mask));
    if constexpr (SOFT) { if (value) return soft_rom(a & 0xFFFu, v); }
    return v;
  }
  // decode entry at (bank, PC); H_SLOW outside cartridge space
  DEV uint2 fetch() const {
    if (!((pbase + di) & 0x1000u)) return make_uint2(HC_COLD + H_SLOW, 0);
    return __ldg(dr + di);
  }

  // ------------------------------------------------------------------ RIOT (struct Riot above)
  using R = Riot<BLOCK, TAG>;
  DEV void timer_sync(int32_t ticks, uint32_t &timer, uint32_t &sub, uint32_t &shift, uint32_t &tflag) { R::timer_sync(sl, ticks, timer, sub, shift, tflag); }
  DEV uint32_t timer_read(uint32_t a, int32_t c) { return R::timer_read(sl, a, c); }

  // stack accesses (C.3: $0100 | SP decodes like any other address — RAM for SP >= $80, TIA registers below) k cycles
  // into the instruction
  // GEN = false is the compact form of the common case (the whole access stays in RAM; exec_one<false> bails out to
  // exec_one<true> before it touches anything when that does not hold)
  template <bool GEN> DEV void push(uint32_t v, int k) {
    if constexpr (GEN) bus_write(0x0100u | SP, v, k); else ram_wr(SP, v);
    SP = (SP - 1u) & 0xFFu;
  }
  template <bool GEN> DEV uint32_t pull(int k) {
    SP = (SP + 1u) & 0xFFu;
    if constexpr (GEN) return bus_read(0x0100u | SP, k); else return ram_rd(SP);
  }
  // pointer / vector / instruction bytes: cartridge or RAM in the compact form, anything in the generic one
  template <bool GEN> DEV uint32_t rd8(uint32_t addr, int k, bool value = true) {
    if constexpr (GEN) return bus_read(addr, k, value);
    else { const uint32_t a = addr & 0x1FFFu; return (a & 0x1000u) ? rom_rd(a, value) : ram_rd(a, value); }
  }
  static DEV bool ram_or_rom(uint32_t addr) { return (addr & 0x1000u) || (addr & 0x0280u) == 0x0080u; }
  // a READ cycle k cycles into the instruction while WSYNC holds RDY (C.4: only read cycles are stalled, so the writes of
  // a JSR / BRK sequence run through a freshly set latch and the next read idles to the line end)
  DEV void rdy(int k) {
    if (!wsync) return;
    const int32_t n = cyc + k - lstart;
    if (n < LINE_CYC) cyc += LINE_CYC - n;
    T::line_end(sl); lstart += LINE_CYC; wsync = false; relim();
  }
  // a read whose value is discarded (C.5 "dummy") in cycle cyc+k: only INTIM and bank hotspots react
  DEV void dummy_rd(uint32_t addr, int k) {
    if constexpr (TAG == 1) { if (kind == MK_FE) { (void)bus_read(addr, k, false); return; } }     // (FE watches every cycle's address and data)
    const uint32_t a = addr & 0x1FFFu;
    if (a & 0x1000u) hotspot(a);
    else if ((a & 0x0285u) == 0x0284u) io_dummy_intim<BLOCK, TAG>(sl, cyc + k + 1);
  }
  // lim from (lstart, fstart, wsync, status)
  DEV void relim() {
    lim = (status & STATUS_ILLEGAL) ? LIM_NOW : wsync ? LIM_WSYNC : min(lstart + LINE_CYC, fstart + cap);
  }
  // after a TIA access that reported events; fc = cycle count at which a frame that just ended did so
  DEV void tia_events(uint32_t ev, int32_t fc) {
    lstart += LINE_CYC * (int32_t)(ev >> 4);
    wsync = (ev & EV_WSYNC) != 0;
    if (ev & EV_FRAME) { fdone += 1; fstart = fc; rekey(); }
    relim();
  }
  // the generic operand read (C.3 decode), k cycles into the instruction
  DEV uint32_t bus_read0(uint32_t a, int k, bool value) {
    if ((a & 0x1280u) == 0x0080u) return ram_rd(a, value);
    if (a & 0x1000u) return rom_rd(a, value);
    const uint32_t r = io_read<BLOCK, TAG>(sl, a, cyc + k, cyc - lstart + k);
    if (r >> 12) { lstart += LINE_CYC * (int32_t)(r >> 12); wsync = false; relim(); }
    return r & 0xFFu;
  }
  DEV uint32_t bus_read(uint32_t addr, int k, bool value = true) {     // value: the byte is used (soft reads skip discarded ones)
    const uint32_t a = addr & 0x1FFFu;
    const uint32_t v = bus_read0(a, k, value);
    if constexpr (TAG == 1) fe_snoop(a, v);
    return v;
  }
  DEV void bus_write(uint32_t addr, uint32_t v, int k) {
    const uint32_t a = addr & 0x1FFFu;
    if ((a & 0x1280u) == 0x0080u) ram_wr(a, v);
    else if (a & 0x1000u) { hotspot(a); if constexpr (TAG == 1) { if (has_sc() && (a & 0x0F80u) == 0) *sc_cell(a & 0x7Fu) = (uint8_t)v; } }   // Superchip write port
    else { const uint32_t ev = io_write<BLOCK, TAG>(sl, a, v, cyc + k, cyc - lstart + k); if (ev) tia_events(ev, cyc + k + 1); }
    if constexpr (TAG == 1) fe_snoop(a, v);
  }
  // ---------------------------------------------------------------- SOFT-STE mode (include/vcs.h vcs_step_soft; eq. 8-10)
  // FULL mode (appendix D; include/vcs.h vcs_step_instructions_soft): the cast of the soft value itself decides
  // what the machine reads, so it is taken exactly as the oracle takes it — eq. (10) tap by tap in double, k = -K .. K,
  // with the host's e^{-k/T} (no fused multiply-adds), then (float) and round.  Not a fast path and not meant to be.
  DEV bool soft_full() const { return (T::ctx(C_SOFT_K) >> 31) != 0; }
  DEV const double *soft_wd() const { return reinterpret_cast<const double *>((unsigned long long)T::ctx(C_SOFT_WD_LO) | ((unsigned long long)T::ctx(C_SOFT_WD_HI) << 32)); }
  DEV uint32_t full_rom(uint32_t o, uint32_t hard) {
    const int K = (int)(T::ctx(C_SOFT_K) & 0x7FFFFFFFu);
    const double *wd = soft_wd();
    double plane[8] = {0, 0, 0, 0, 0, 0, 0, 0}, den = 0.0;
#pragma unroll 1
    for (int k = -K; k <= K; ++k) {
      const int i = (int)o + k; if (i < 0 || i >= 4096) continue;
      const double w = wd[k < 0 ? -k : k];
      const uint32_t b = rom_byte((di & 0x7000u) + ((uint32_t)i & rom_mask));
#pragma unroll
      for (int j = 0; j < 8; ++j) plane[j] = __dadd_rn(plane[j], ((b >> j) & 1u) ? w : 0.0);
      den = __dadd_rn(den, w);
    }
    double soft = 0.0;
#pragma unroll
    for (int j = 0; j < 8; ++j) soft = __dadd_rn(soft, __dmul_rn((double)(1 << j), __ddiv_rn(plane[j], den)));
    const float sv = (float)soft;
    soft_note<BLOCK>(sl, 0, sv, (float)hard, sv);
    return (uint32_t)(int)rintf(sv) & 0xFFu;
  }
  DEV uint32_t full_ram(uint32_t cell, uint32_t hard) {
    const int K = (int)(T::ctx(C_SOFT_K) & 0x7FFFFFFFu);
    const double *wd = soft_wd();
    double num = 0.0, den = 0.0;
#pragma unroll 1
    for (int k = -K; k <= K; ++k) {
      const int i = (int)cell + k; if (i < 0 || i >= 128) continue;
      const double w = wd[k < 0 ? -k : k];
      num = __dadd_rn(num, __dmul_rn(w, (double)ram_rd_off((((uint32_t)i & 0x7Cu) * BLOCK) | ((uint32_t)i & 3u))));
      den = __dadd_rn(den, w);
    }
    const float sv = (float)__ddiv_rn(num, den);
    soft_note<BLOCK>(sl, 1, sv, (float)hard, sv);
    return (uint32_t)(int)rintf(sv) & 0xFFu;
  }
  DEV uint32_t full_branch(uint32_t f, bool set_sense, int32_t delta, bool taken) {        // -> PC = round(pc_nb + g delta)
    const double g = soft_wd()[SOFT_WD_GATE + ((f != 0) == set_sense ? 0 : 1)];            // z = s (2 f - 1) = +1 / -1
    const uint32_t pc_nb = pc();
    const float v = rintf((float)__dadd_rn((double)pc_nb, __dmul_rn(g, (double)delta)));
    const float pc_hard = (float)pc_nb + (taken ? (float)delta : 0.f);
    soft_note<BLOCK>(sl, 2, (float)g, pc_hard, v);
    return (uint32_t)(int)v & 0xFFFFu;
  }
  DEV uint32_t soft_rom(uint32_t o, uint32_t hard) {       // eq. (10) on the 4096 x 8 bit tensor of the visible bank, then STE + round
    if (soft_full()) return full_rom(o, hard);
    // the ROM is constant, so W(T) x ROM is computed once per temperature (soft_table_kernel): a fetch is one lookup
    const float sv = __ldg(soft_tab + (di & 0x7000u) + o);
    const float h = (float)hard, ste = sv + (h - sv);      // eq. (9), forward
    soft_note<BLOCK>(sl, 0, sv, h, ste);
    return (uint32_t)(int)rintf(ste) & 0xFFu;
  }
  DEV uint32_t soft_ram(uint32_t cell, uint32_t hard) { return soft_full() ? full_ram(cell, hard) : soft_ram_read<BLOCK>(sl, cell, hard); }
  // SOFT-STE: the PC itself is set by the hard path (R14), returns NO_PC; FULL: returns the PC the cast gives (R18)
  static constexpr uint32_t NO_PC = 0xFFFFFFFFu;
  DEV uint32_t soft_branch(uint32_t f, float sense, float delta, bool taken) {
    if (soft_full()) return full_branch(f, sense > 0.f, (int32_t)delta, taken);
    soft_branch_note<BLOCK>(sl, f, sense, delta, taken, (float)pc());
    return NO_PC;
  }
  DEV uint32_t pack_p() const {
    return ((zn & 0x180u) ? 0x80u : 0u) | (fV << 6) | 0x20u | fDI | (((zn & 0xFFu) == 0) ? 2u : 0u) | fC;
  }
  DEV void unpack_p(uint32_t p) {
    fC = p & 1u; zn = ((p & 0x80u) << 1) | ((p & 2u) ? 0u : 1u); fDI = p & 0x0Cu; fV = (p >> 6) & 1u;
  }
  DEV void adc(uint32_t v) {                               // C.6, binary and NMOS decimal
    const uint32_t a = A, C = fC;
    if (!(fDI & 8u)) {
      const uint32_t s = a + v + C;
      fC = s >> 8; fV = ((a ^ s) & (v ^ s) & 0x80u) >> 7; A = s & 0xFFu; zn = A;
      return;
    }
    int al = (int)(a & 0x0Fu) + (int)(v & 0x0Fu) + (int)C;
    if (al >= 0x0A) al = ((al + 6) & 0x0F) + 0x10;
    int s = (int)(a & 0xF0u) + (int)(v & 0xF0u) + al;
    const int sv = (int)(int8_t)(a & 0xF0u) + (int)(int8_t)(v & 0xF0u) + al;
    zn = (((a + v + C) & 0xFFu) ? 1u : 0u) | (((uint32_t)s & 0x80u) << 1);   // Z from the binary sum, N from the high-nibble sum
    fV = (sv < -128 || sv > 127) ? 1u : 0u;
    if (s >= 0xA0) s += 0x60;
    fC = (s >= 0x100) ? 1u : 0u;
    A = (uint32_t)s & 0xFFu;
  }
  DEV void sbc(uint32_t v) {
    const uint32_t a = A, C = fC;
    const uint32_t nb = v ^ 0xFFu, s = a + nb + C;         // flags exactly as binary
    const uint32_t bin = s & 0xFFu;
    fC = s >> 8; fV = ((a ^ s) & (nb ^ s) & 0x80u) >> 7; zn = bin;
    if (!(fDI & 8u)) { A = bin; return; }
    int al = (int)(a & 0x0Fu) - (int)(v & 0x0Fu) + (int)C - 1;
    if (al < 0) al = ((al - 6) & 0x0F) - 0x10;
    int d = (int)(a & 0xF0u) - (int)(v & 0xF0u) + al;
    if (d < 0) d -= 0x60;
    A = (uint32_t)d & 0xFFu;
  }
  DEV void cmp(uint32_t r, uint32_t v) { fC = (r >= v) ? 1u : 0u; zn = (r - v) & 0xFFu; }
  DEV void bit(uint32_t v) { zn = (A & v) | ((v & 0x80u) << 1); fV = (v >> 6) & 1u; }
  DEV void read_op(uint32_t o, uint32_t v) {               // o = op - OP_LDA
    switch (o) {
      case 0: A = v; zn = v; break;
      case 1: X = v; zn = v; break;
      case 2: Y = v; zn = v; break;
      case 3: A &= v; zn = A; break;
      case 4: A |= v; zn = A; break;
      case 5: A ^= v; zn = A; break;
      case 6: adc(v); break;
      case 7: sbc(v); break;
      case 8: cmp(A, v); break;
      case 9: cmp(X, v); break;
      case 10: cmp(Y, v); break;
      case 11: bit(v); break;
      case 12: A = v; X = v; zn = v; break;                // LAX
      default: break;                                      // NOP with an operand: the read happened, nothing is kept
    }
  }
  DEV uint32_t rmw_op(uint32_t o, uint32_t s) {            // o = op - OP_ASL
    uint32_t r;
    switch (o) {
      case 0: r = (s << 1) & 0xFFu; fC = s >> 7; break;
      case 1: r = s >> 1; fC = s & 1u; break;
      case 2: r = ((s << 1) | fC) & 0xFFu; fC = s >> 7; break;
      case 3: r = (s >> 1) | (fC << 7); fC = s & 1u; break;
      case 4: r = (s + 1u) & 0xFFu; break;
      default: r = (s - 1u) & 0xFFu; break;
    }
    zn = r;
    return r;
  }

  // ---------------------------------------------------------------- the checks ahead of an instruction (C.4, C.10)
  // entered when cyc >= lim.  Returns false when no instruction may run now (a frame ended at the cap, or
  // the CPU is halted and idled): the lane goes back to the scheduling point.
  // COUNT (vcs_step_instructions): the lane runs on an instruction budget (smem word S_BUDGET); a halted CPU spends one
  // idle cycle per unit of it, as the oracle's single-instruction step does.
  template <bool COUNT = false>
  DEV bool slow_pre() {
    if (cyc - lstart > LINE_CYC) { T::line_end(sl); lstart += LINE_CYC; wsync = false; }     // the previous instruction ran over the line end
    if (cyc - fstart >= cap) {                             // frame cap at the instruction boundary
      status |= STATUS_CAP; T::frame_end(sl, 3u * (uint32_t)(cyc - lstart)); fdone += 1; fstart = cyc;
      rekey(); relim(); return false;
    }
    if (cyc - lstart >= LINE_CYC) { T::line_end(sl); lstart += LINE_CYC; wsync = false; }     // n == 76 exactly
    if (status & STATUS_ILLEGAL) {                         // halted: idle cycles to the line end / the cap
      int32_t m = min(LINE_CYC - (cyc - lstart), cap - (cyc - fstart));
      if constexpr (COUNT) { m = min(m, (int32_t)S(S_BUDGET)); S(S_BUDGET) -= (uint32_t)m; }
      cyc += m;
      return false;
    }
    if (wsync) {                                           // a12: RDY holds the CPU until the line ends
      cyc = lstart + LINE_CYC; T::line_end(sl); lstart = cyc; wsync = false;
    }
    relim();
    return true;       // (when the cap falls on the line start reached by WSYNC the instruction still runs: the stall is part of
                       //  its first read cycle, C.4, and the cap is looked at on instruction boundaries only, C.10)
  }

  // ---------------------------------------------------------------- block-wide regroup (F8 divergence)
  // Called by every thread of the block, converged, when every lane is parked at a bank-hotspot access or has
  // finished the step.  The block's environments are sorted by (frames done, bank, SP, PC) and MOVED between
  // threads — shared-memory file words [0, S_MOVED) plus the CPU registers — so that each warp again holds
  // lanes of one bank at one PC.  Environments are independent, so which thread runs which one is free.
  DEV void regroup() {
    const bool has = sl != NOSLOT;
    uint32_t skey = 0xFFFFFFFFu;
    if (has) {
      const uint32_t bank = di >> 12, PC = pc();
      S(S_OBJ + 0) = A | (X << 8) | (Y << 16) | (SP << 24);
      S(S_OBJ + 1) = PC | (pack_p() << 16) | (status << 24);
      S(S_OBJ + 2) = (uint32_t)cyc; S(S_OBJ + 3) = (uint32_t)lstart; S(S_OBJ + 4) = (uint32_t)fstart;
      S(S_OBJ + 5) = fdone | (bank << 8) | ((wsync ? 1u : 0u) << 16);
      skey = (fdone >= fskip) ? 0xFFFFFFFFu : (min(fdone, 30u) << 27) | (bank << 24) | (SP << 16) | PC;    // (bank: 3 bits, F4 has eight)
      S(S_OBJ + 6) = skey;
    }
    __syncthreads();
    uint32_t rank = 0;
    const uint32_t *keys = smem + (S_OBJ + 6) * BLOCK;
    if (has) {
#pragma unroll 4
      for (int j = 0; j < BLOCK; ++j) { const uint32_t kj = keys[j]; rank += (kj < skey || (kj == skey && (uint32_t)j < sl)) ? 1u : 0u; }
    }
    constexpr int NB = 23;
    static_assert(S_MOVED % NB == 0, "batching");
#pragma unroll 1
    for (int base = 0; base < S_MOVED; base += NB) {
      uint32_t t[NB];
      if (has) {
#pragma unroll
        for (int i = 0; i < NB; ++i) t[i] = smem[(base + i) * BLOCK + sl];
      }
      __syncthreads();                                     // every file's words [base, base+NB) are in registers
      if (has) {
#pragma unroll
        for (int i = 0; i < NB; ++i) smem[(base + i) * BLOCK + rank] = t[i];
      }
    }
    __syncthreads();
    // which file this thread runs next.  With a spare warp the lowest (frames done, bank) class gets whole warps of
    // its own and everything else is packed behind it from the next warp boundary on, so that no warp mixes the two
    // banks; slots inside a warp stay consecutive, hence bank-conflict free.
    uint32_t ns = threadIdx.x;
    if constexpr (THREADS != BLOCK && ROMS == 2) {
      // F6 / F4 (four / eight banks): files stay in sorted order, and every (frames done, bank) class starts at a warp
      // boundary for as long as the spare warp's 32 lanes of padding last
      uint32_t pos = 0, slack = THREADS - BLOCK, prev = keys[0] >> 24;
      ns = NOSLOT;
#pragma unroll 4
      for (int j = 0; j < BLOCK; ++j) {
        const uint32_t c = keys[j] >> 24;
        if (c != prev) { const uint32_t pad = (32u - (pos & 31u)) & 31u; if (pad <= slack) { pos += pad; slack -= pad; } prev = c; }
        if (pos == threadIdx.x) ns = (uint32_t)j;
        ++pos;
      }
      __syncthreads();                                     // (as below)
    } else if constexpr (THREADS != BLOCK) {
      const uint32_t c0 = keys[0] >> 24;
      uint32_t n0 = 0;
#pragma unroll 4
      for (int j = 0; j < BLOCK; ++j) n0 += ((keys[j] >> 24) == c0) ? 1u : 0u;
      // both groups spread evenly over the warps they get (in proportion to their sizes): no nearly empty warp
      // beside full ones, and fewer lanes per warp means fewer divergent groups to run one after the other
      constexpr uint32_t NW = THREADS / 32;
      const uint32_t n1 = (uint32_t)BLOCK - n0;
      uint32_t w0 = (n0 * NW + (uint32_t)BLOCK / 2u) / (uint32_t)BLOCK;
      w0 = max(w0, (n0 + 31u) >> 5); w0 = min(w0, NW - ((n1 + 31u) >> 5));          // each group fits its warps
      const uint32_t w1 = NW - w0, wid = threadIdx.x >> 5, lane = threadIdx.x & 31u;
      if (wid < w0) { const uint32_t per = (n0 + w0 - 1u) / w0, sidx = wid * per + lane; ns = (lane < per && sidx < n0) ? sidx : NOSLOT; }
      else if (n1) { const uint32_t per = (n1 + w1 - 1u) / w1, sidx = (wid - w0) * per + lane; ns = (lane < per && sidx < n1) ? n0 + sidx : NOSLOT; }
      else ns = NOSLOT;
      __syncthreads();                                     // the keys sit in the object-mask cache: nobody resumes before all have read them
    }
    sl = ns; sl4 = 4u * ns;
    park &= 1u;
    if (sl != NOSLOT) {
      uint32_t r;
      r = S(S_OBJ + 0); A = r & 0xFFu; X = (r >> 8) & 0xFFu; Y = (r >> 16) & 0xFFu; SP = r >> 24;
      r = S(S_OBJ + 1); const uint32_t npc = r & 0xFFFFu; unpack_p((r >> 16) & 0xFFu); status = r >> 24;
      cyc = (int32_t)S(S_OBJ + 2); lstart = (int32_t)S(S_OBJ + 3); fstart = (int32_t)S(S_OBJ + 4);
      r = S(S_OBJ + 5); fdone = r & 0xFFu; wsync = ((r >> 16) & 1u) != 0;
      di = (((r >> 8) & 7u) << 12) | (npc & 0xFFFu); pbase = npc - di;
      S(S_FL) |= TF_DIRTY_ALL;                             // the object-mask cache was the scratch area
      rekey(); relim();
      w = fetch();
    } else {
      fdone = fskip; wsync = false; status = 0; di = 0; pbase = 0;
      rekey();
    }
  }

  // ---------------------------------------------------------------- the out-of-line executor: ONE instruction
  // Runs the entry (cx, pl) in the vcs_decode.cuh Hid numbering; di and cyc have already been advanced by the
  // entry's length and base cycles.  Leaves w = the entry at the new (bank, PC): the caller re-schedules.
  // GEN = false: the compact executor for the common case — code in cartridge space, stack and pointer cells in RAM.
  // It returns true, having changed nothing but this Cpu's registers, when the instruction needs an access outside that
  // (stack on TIA registers, pointer / vector bytes or code in TIA / RIOT / RAM space): the caller then drops this Cpu
  // and runs the instruction again on exec_one<true>, where every access goes through the generic bus code.
  template <bool GEN>
  DEV bool exec_one(uint32_t cx, uint32_t pl) {
    {
      bool slow = false;                                   // run-time decoded
      uint32_t ea = 0, v = 0, wv = 0, op2 = 0, hid, cast_pc = 0xFFFFFFFFu;     // cast_pc: FULL mode, the PC a branch's cast gives
      int k = 0, i0 = 0, total = 0, kb = 0;
      if constexpr (!GEN) { if (kind >= MK_F8SC) return true; }          // Superchip / E0 / FE carts: the generic executor knows their ports
    dispatch:
      hid = cx & 0x7Fu;
      kb = -(int)((cx >> DW_CY_SHIFT) & 0xFFu);            // cyc + kb = the instruction's first cycle (cy is already added; 0 for the generic handlers)
      switch (hid) {
        case H_SLOW: {                                     // byte-wise fetch with side effects, run-time decode
          // the instruction bytes are ordinary bus reads in cycles 0, 1, 2 of the instruction (C.3 / C.5): cartridge,
          // RAM, TIA (collision latches) or RIOT (an INTIM read clears the underflow flag), whatever PC decodes to
          const uint32_t pc0 = pc();
          if constexpr (!GEN) { if (((pc0 & 0x1000u) == 0) | (((pc0 + 2u) & 0x1000u) == 0)) return true; }
          const uint32_t opc = rd8<GEN>(pc0, 0);
          uint32_t g = c_gen[opc];
          const uint32_t ln = (g >> DW_LEN_SHIFT) & 0xFFu, gh = g & 0x7Fu;
          uint32_t b1 = 0, b2 = 0;
          if (gh != H_ILL) {
            if (ln == 1 || gh == H_BRK) dummy_rd(pc0 + 1u, 1);             // "R dummy@PC" of the one-byte instructions and of BRK
            else b1 = rd8<GEN>(pc0 + 1u, 1);
            if (ln == 3 && !(GEN && gh == H_JSR)) b2 = rd8<GEN>(pc0 + 2u, 2);   // (a generic JSR reads its high byte after the pushes)
          }
          pl = b1 | (b2 << 8);
          if ((g & 0x7Fu) >= H_BR0 && (g & 0x7Fu) < H_BR0 + 8) {
            const uint32_t next = (pc0 + 2u) & 0xFFFFu, target = (next + (uint32_t)(int32_t)(int8_t)b1) & 0xFFFFu;
            pl = (uint32_t)(int32_t)(int8_t)b1;
            g = (g & 0x00FFFFFFu) | ((((target ^ next) & 0xFF00u) ? 2u : 1u) << DW_OP2_SHIFT);
          }
          set_pc((pc0 + ln) & 0xFFFFu);
          cyc += (int32_t)((g >> DW_CY_SHIFT) & 0xFFu);
          cx = g; slow = true;
          goto dispatch;
        }
        // ---- immediate (or a fixed ROM byte)
        case H_IMM0 + 0: A = pl; zn = pl; break;
        case H_IMM0 + 1: X = pl; zn = pl; break;
        case H_IMM0 + 2: Y = pl; zn = pl; break;
        case H_IMM0 + 3: A &= pl; zn = A; break;
        case H_IMM0 + 4: A |= pl; zn = A; break;
        case H_IMM0 + 5: A ^= pl; zn = A; break;
        case H_IMM0 + 6: adc(pl); break;
        case H_IMM0 + 7: sbc(pl); break;
        case H_IMM0 + 8: cmp(A, pl); break;
        case H_IMM0 + 9: cmp(X, pl); break;
        case H_IMM0 + 10: cmp(Y, pl); break;
        // ---- RAM cell reads
        case H_ZR0 + 0: A = ram_rd_off(pl); zn = A; break;
        case H_ZR0 + 1: X = ram_rd_off(pl); zn = X; break;
        case H_ZR0 + 2: Y = ram_rd_off(pl); zn = Y; break;
        case H_ZR0 + 3: A &= ram_rd_off(pl); zn = A; break;
        case H_ZR0 + 4: A |= ram_rd_off(pl); zn = A; break;
        case H_ZR0 + 5: A ^= ram_rd_off(pl); zn = A; break;
        case H_ZR0 + 6: adc(ram_rd_off(pl)); break;
        case H_ZR0 + 7: sbc(ram_rd_off(pl)); break;
        case H_ZR0 + 8: cmp(A, ram_rd_off(pl)); break;
        case H_ZR0 + 9: cmp(X, ram_rd_off(pl)); break;
        case H_ZR0 + 10: cmp(Y, ram_rd_off(pl)); break;
        case H_ZR0 + 11: bit(ram_rd_off(pl)); break;
        // ---- RAM cell stores
        case H_STZR0 + 0: ram_wr_off(pl, A); break;
        case H_STZR0 + 1: ram_wr_off(pl, X); break;
        case H_STZR0 + 2: ram_wr_off(pl, Y); break;
        // ---- TIA register stores (the write is the instruction's last cycle)
        case H_STZT0 + 0: v = A; goto tia_store;
        case H_STZT0 + 1: v = X; goto tia_store;
        case H_STZT0 + 2: v = Y; goto tia_store;
        case H_NOP: break;
        // ---- RAM cell read-modify-write
        case H_MZR0 + 0: case H_MZR0 + 1: case H_MZR0 + 2: case H_MZR0 + 3: case H_MZR0 + 4: case H_MZR0 + 5:
          ram_wr_off(pl, rmw_op(hid - H_MZR0, ram_rd_off(pl))); break;
        case H_ACC0 + 0: case H_ACC0 + 1: case H_ACC0 + 2: case H_ACC0 + 3: A = rmw_op(hid - H_ACC0, A); break;
        // ---- implied
        case H_IMP0 + 0: fC = 0; break;
        case H_IMP0 + 1: fC = 1; break;
        case H_IMP0 + 2: fDI &= ~8u; break;
        case H_IMP0 + 3: fDI |= 8u; break;
        case H_IMP0 + 4: fDI &= ~4u; break;
        case H_IMP0 + 5: fDI |= 4u; break;
        case H_IMP0 + 6: fV = 0; break;
        case H_IMP0 + 7: break;
        case H_IMP0 + 8: X = (X - 1u) & 0xFFu; zn = X; break;
        case H_IMP0 + 9: Y = (Y - 1u) & 0xFFu; zn = Y; break;
        case H_IMP0 + 10: X = (X + 1u) & 0xFFu; zn = X; break;
        case H_IMP0 + 11: Y = (Y + 1u) & 0xFFu; zn = Y; break;
        case H_IMP0 + 12: X = A; zn = X; break;
        case H_IMP0 + 13: Y = A; zn = Y; break;
        case H_IMP0 + 14: X = SP; zn = X; break;
        case H_IMP0 + 15: A = X; zn = A; break;
        case H_IMP0 + 16: A = Y; zn = A; break;
        case H_IMP0 + 17: SP = X; rekey(); break;
        // ---- branches: payload = signed displacement, op2 = extra cycles when taken
        case H_BR0 + 0: case H_BR0 + 1: case H_BR0 + 2: case H_BR0 + 3: case H_BR0 + 4: case H_BR0 + 5: case H_BR0 + 6: case H_BR0 + 7: {
          const uint32_t kk = hid - H_BR0;                 // BPL BMI BVC BVS BCC BCS BNE BEQ: flag N V C Z, taken when flag == kk & 1
          uint32_t f;
          switch (kk >> 1) { case 0: f = (zn & 0x180u) ? 1u : 0u; break; case 1: f = fV; break; case 2: f = fC; break;
                             default: f = (zn & 0xFFu) ? 0u : 1u; break; }
          const bool taken = f == (kk & 1u);
          if constexpr (SOFT) cast_pc = soft_branch(f, (kk & 1u) ? 1.f : -1.f, (float)(int32_t)pl, taken);
          if (!taken) { if constexpr (SOFT) { if (cast_pc != 0xFFFFFFFFu) set_pc(cast_pc); } break; }
        } goto br_taken;
        // ---- control transfers and stack
        case H_JMP: set_pc(pl); goto ctl;
        // (C.5 sequences; the dummy stack read of JSR / RTS / RTI / PLA / PLP lands in RAM or on a TIA read address: no effect)
        case H_JSR: { const uint32_t ret = (pc() - 1u) & 0xFFFFu;     // address of the 3rd byte
          if constexpr (!GEN) { if (SP < 0x81u) return true; }
          if constexpr (GEN) dummy_rd(0x0100u | SP, kb + 2);
          push<GEN>(ret >> 8, kb + 3); push<GEN>(ret & 0xFFu, kb + 4); rekey();
          if constexpr (GEN) {
            rdy(kb + 5);                                                      // R hi@PC comes after the pushes:
            if (slow) pl |= bus_read(ret, kb + 5) << 8;                        // they may have set WSYNC, or rewritten that byte
          }
          set_pc(pl); } goto ctl;
        case H_RTS: { if constexpr (!GEN) { if (SP - 0x7Fu > 0xFDu - 0x7Fu) return true; }      // pulls from SP+1, SP+2
          if constexpr (GEN) dummy_rd(0x0100u | SP, kb + 2);
          const uint32_t lo = pull<GEN>(kb + 3), hi = pull<GEN>(kb + 4); const uint32_t r = lo | (hi << 8);
          rekey(); dummy_rd(r, kb + 5); set_pc((r + 1u) & 0xFFFFu); } goto ctl;
        case H_PHA: if constexpr (!GEN) { if (SP < 0x80u) return true; } push<GEN>(A, kb + 2); rekey(); break;
        case H_PHP: if constexpr (!GEN) { if (SP < 0x80u) return true; } push<GEN>(pack_p() | 0x30u, kb + 2); rekey(); break;
        case H_PLA: if constexpr (!GEN) { if (SP - 0x7Fu > 0xFEu - 0x7Fu) return true; } if constexpr (GEN) dummy_rd(0x0100u | SP, kb + 2);
                    A = pull<GEN>(kb + 3); zn = A; rekey(); break;
        case H_PLP: if constexpr (!GEN) { if (SP - 0x7Fu > 0xFEu - 0x7Fu) return true; } if constexpr (GEN) dummy_rd(0x0100u | SP, kb + 2);
                    unpack_p(pull<GEN>(kb + 3)); rekey(); break;
        // ---- absolute read of INTIM / TIMINT (4th cycle)
        case H_RTIM: read_op(cx >> DW_OP2_SHIFT, timer_read(pl, cyc - 1)); break;
        // ---- generic addressing: reads (cyc = first cycle of the instruction; they add `total` themselves)
        case H_R0 + 0: v = pl & 0xFFu; total = 2; goto do_read_op;
        case H_R0 + 1: ea = pl & 0xFFu; k = 2; goto do_read;
        case H_R0 + 2: if constexpr (GEN) dummy_rd(pl & 0xFFu, 2); ea = (pl + X) & 0xFFu; k = 3; goto do_read;      // (R dummy@zp)
        case H_R0 + 3: if constexpr (GEN) dummy_rd(pl & 0xFFu, 2); ea = (pl + Y) & 0xFFu; k = 3; goto do_read;
        case H_R0 + 4: ea = pl; k = 3; goto do_read;
        case H_R0 + 5: case H_R0 + 6: case H_R0 + 8: {
          uint32_t lo, hi;
          if (hid == H_R0 + 8) { if constexpr (!GEN) { if ((pl & 0xFFu) - 0x80u > 0x7Eu) return true; }       // pointer cells pl, pl+1 in RAM
                                 lo = rd8<GEN>(pl & 0xFFu, 2); hi = rd8<GEN>((pl + 1u) & 0xFFu, 3); k = 4; }
          else { lo = pl & 0xFFu; hi = pl >> 8; k = 3; }
          const uint32_t t = lo + ((hid == H_R0 + 5) ? X : Y);
          const uint32_t unc = (hi << 8) | (t & 0xFFu);
          ea = (unc + (t & 0x100u)) & 0xFFFFu;
          if (t & 0x100u) { dummy_rd(unc, k); k += 1; }
        } goto do_read;
        case H_R0 + 7: { const uint32_t z = (pl + X) & 0xFFu; if constexpr (!GEN) { if (z - 0x80u > 0x7Eu) return true; }
          if constexpr (GEN) dummy_rd(pl & 0xFFu, 2);
          ea = rd8<GEN>(z, 3); ea |= rd8<GEN>((z + 1u) & 0xFFu, 4) << 8; k = 5; } goto do_read;
        // ---- generic addressing: stores
        case H_W0 + 0: ea = pl & 0xFFu; k = 2; goto do_write;
        case H_W0 + 1: if constexpr (GEN) dummy_rd(pl & 0xFFu, 2); ea = (pl + X) & 0xFFu; k = 3; goto do_write;
        case H_W0 + 2: if constexpr (GEN) dummy_rd(pl & 0xFFu, 2); ea = (pl + Y) & 0xFFu; k = 3; goto do_write;
        case H_W0 + 3: ea = pl; k = 3; goto do_write;
        case H_W0 + 4: case H_W0 + 5: case H_W0 + 7: {
          uint32_t lo, hi;
          if (hid == H_W0 + 7) { if constexpr (!GEN) { if ((pl & 0xFFu) - 0x80u > 0x7Eu) return true; }
                                 lo = rd8<GEN>(pl & 0xFFu, 2); hi = rd8<GEN>((pl + 1u) & 0xFFu, 3); k = 4; }
          else { lo = pl & 0xFFu; hi = pl >> 8; k = 3; }
          const uint32_t t = lo + ((hid == H_W0 + 4) ? X : Y);
          const uint32_t unc = (hi << 8) | (t & 0xFFu);
          ea = (unc + (t & 0x100u)) & 0xFFFFu;
          dummy_rd(unc, k); k += 1;
        } goto do_write;
        case H_W0 + 6: { const uint32_t z = (pl + X) & 0xFFu; if constexpr (!GEN) { if (z - 0x80u > 0x7Eu) return true; }
          if constexpr (GEN) dummy_rd(pl & 0xFFu, 2);
          ea = rd8<GEN>(z, 3); ea |= rd8<GEN>((z + 1u) & 0xFFu, 4) << 8; k = 5; } goto do_write;
        // ---- generic addressing: read-modify-write
        case H_M0 + 0: ea = pl & 0xFFu; k = 2; goto do_rmw;
        case H_M0 + 1: if constexpr (GEN) dummy_rd(pl & 0xFFu, 2); ea = (pl + X) & 0xFFu; k = 3; goto do_rmw;
        case H_M0 + 2: ea = pl; k = 3; goto do_rmw;
        case H_M0 + 3: { const uint32_t t = (pl & 0xFFu) + X; const uint32_t unc = (pl & 0xFF00u) | (t & 0xFFu);
          ea = (unc + (t & 0x100u)) & 0xFFFFu; dummy_rd(unc, 3); k = 4; } goto do_rmw;
        // ---- rare
        case H_JMPI: { const uint32_t p2 = (pl & 0xFF00u) | ((pl + 1u) & 0xFFu);                  // no carry into the page
          if constexpr (!GEN) { if (!ram_or_rom(pl) || !ram_or_rom(p2)) return true; }
          const uint32_t l2 = rd8<GEN>(pl, kb + 3), h2 = rd8<GEN>(p2, kb + 4);
          set_pc(l2 | (h2 << 8)); } goto ctl;
        case H_RTI: { if constexpr (!GEN) { if (SP - 0x7Fu > 0xFCu - 0x7Fu) return true; }       // pulls from SP+1 .. SP+3
          if constexpr (GEN) dummy_rd(0x0100u | SP, kb + 2);
          unpack_p(pull<GEN>(kb + 3)); const uint32_t lo = pull<GEN>(kb + 4), hi = pull<GEN>(kb + 5); rekey(); set_pc(lo | (hi << 8)); } goto ctl;
        case H_BRK: { const uint32_t ret = pc();             // address of the opcode + 2
          if constexpr (!GEN) { if (SP < 0x82u) return true; }
          push<GEN>(ret >> 8, kb + 2); push<GEN>(ret & 0xFFu, kb + 3); push<GEN>(pack_p() | 0x30u, kb + 4); rekey();
          if constexpr (GEN) rdy(kb + 5);
          const uint32_t l2 = rd8<GEN>(0xFFFEu, kb + 5), h2 = rd8<GEN>(0xFFFFu, kb + 6);       // ($FFFE / $FFFF: always the cartridge)
          set_pc(l2 | (h2 << 8)); fDI |= 4u; } goto ctl;
        default:                                           // H_ILL — C.12: halt for good, PC stays
          status |= STATUS_ILLEGAL;
          lim = LIM_NOW; goto ctl;
        do_read:
          v = bus_read(ea, k); total = k + 1;
        do_read_op:
          read_op(cx >> DW_OP2_SHIFT, v); goto gen_end;
        do_write:
          op2 = cx >> DW_OP2_SHIFT;
          wv = (op2 == 0) ? A : (op2 == 1) ? X : (op2 == 2) ? Y : (A & X);      // STA STX STY SAX
          i0 = 1; k -= 1; goto do_store;
        do_rmw:
          v = bus_read(ea, k);
          wv = rmw_op(cx >> DW_OP2_SHIFT, v);
          i0 = 0; k += 1;
        do_store:                                          // the one generic write site: [old value,] new value (C.5)
#pragma unroll 1
          for (int i = i0; i < 2; ++i) bus_write(ea, i ? wv : v, k + i);
          total = k + 2;
        gen_end:
          cyc += total;
          if ((park & 4u) || fdone >= fskip) goto ctl;     // a bank hotspot was touched (the prefetched entry may be the other bank's)
          break;
        br_taken:
          if (slow) {                                      // the dummy reads @PC and @(old PCH : new PCL), any target
            const uint32_t next = pc(), target = (next + pl) & 0xFFFFu;
            dummy_rd(next, 0);                             // (cyc already counts the two base cycles: this is the third)
            if ((cx >> DW_OP2_SHIFT) == 2u) dummy_rd((next & 0xFF00u) | (target & 0xFFu), 1);
            set_pc(target);
          } else di += pl;
          if constexpr (SOFT) { if (cast_pc != 0xFFFFFFFFu) set_pc(cast_pc); }     // (cycles and discarded reads are the hard decision's)
          cyc += (int32_t)(cx >> DW_OP2_SHIFT);
          goto ctl;
        tia_store: {
          const uint32_t ev = T::write(sl, pl, v, cyc - 1 - lstart);
          if (ev) { tia_events(ev, cyc); if (ev & EV_FRAME) goto ctl; }
        } break;
      }
    }
    ctl:                                                   // every path ends here: refetch at the new (bank, PC)
      park &= ~4u;
      w = fetch();
      return false;
  }
};

// ---- ALU on the packed registers (C.6).  op = read op (vcs_optable.cuh: LDA LDX LDY AND ORA EOR ADC SBC CMP CPX CPY BIT)
DEV void hot_adc(Hot &h, uint32_t v) {
  const uint32_t a = h.axys & 0xFFu, C = h.fl & 1u;
  uint32_t r, c, ov;
  if (!(h.fl & 8u)) {
    const uint32_t s = a + v + C;
    c = s >> 8; ov = ((a ^ s) & (v ^ s) & 0x80u) >> 1; r = s & 0xFFu; h.zn = r;
  } else {                                                  // NMOS decimal mode
    int al = (int)(a & 0x0Fu) + (int)(v & 0x0Fu) + (int)C;
    if (al >= 0x0A) al = ((al + 6) & 0x0F) + 0x10;
    int s = (int)(a & 0xF0u) + (int)(v & 0xF0u) + al;
    const int sv = (int)(int8_t)(a & 0xF0u) + (int)(int8_t)(v & 0xF0u) + al;
    h.zn = (((a + v + C) & 0xFFu) ? 1u : 0u) | (((uint32_t)s & 0x80u) << 1);
    ov = (sv < -128 || sv > 127) ? 0x40u : 0u;
    if (s >= 0xA0) s += 0x60;
    c = (s >= 0x100) ? 1u : 0u;
    r = (uint32_t)s & 0xFFu;
  }
  h.fl = (h.fl & ~0x41u) | c | ov;
  h.axys = __byte_perm(h.axys, r, 0x3214u);
}
DEV void hot_sbc(Hot &h, uint32_t v) {
  const uint32_t a = h.axys & 0xFFu, C = h.fl & 1u;
  const uint32_t nb = v ^ 0xFFu, s = a + nb + C;            // flags exactly as binary
  uint32_t r = s & 0xFFu;
  h.zn = r;
  const uint32_t fl = (h.fl & ~0x41u) | (s >> 8) | (((a ^ s) & (nb ^ s) & 0x80u) >> 1);
  if (h.fl & 8u) {
    int al = (int)(a & 0x0Fu) - (int)(v & 0x0Fu) + (int)C - 1;
    if (al < 0) al = ((al - 6) & 0x0F) - 0x10;
    int d = (int)(a & 0xF0u) - (int)(v & 0xF0u) + al;
    if (d < 0) d -= 0x60;
    r = (uint32_t)d & 0xFFu;
  }
  h.fl = fl;
  h.axys = __byte_perm(h.axys, r, 0x3214u);
}
DEV void hot_cmp(Hot &h, uint32_t r, uint32_t v) { h.fl = (h.fl & ~1u) | ((r >= v) ? 1u : 0u); h.zn = (r - v) & 0xFFu; }
DEV void alu(Hot &h, uint32_t op, uint32_t v) {
  if (op == 0) { h.axys = __byte_perm(h.axys, v, 0x3214u); h.zn = v; return; }                 // LDA (INTIM polls)
  if (op == 11) { h.zn = (((h.axys & v) & 0xFFu) ? 1u : 0u) | ((v & 0x80u) << 1); h.fl = (h.fl & ~0x40u) | (v & 0x40u); return; }   // BIT
  uint32_t a = h.axys & 0xFFu;
  switch (op) {
    case 1: h.axys = __byte_perm(h.axys, v, 0x3240u); h.zn = v; break;
    case 2: h.axys = __byte_perm(h.axys, v, 0x3410u); h.zn = v; break;
    case 3: a &= v; h.axys = __byte_perm(h.axys, a, 0x3214u); h.zn = a; break;
    case 4: a |= v; h.axys = __byte_perm(h.axys, a, 0x3214u); h.zn = a; break;
    case 5: a ^= v; h.axys = __byte_perm(h.axys, a, 0x3214u); h.zn = a; break;
    case 6: hot_adc(h, v); break;
    case 7: hot_sbc(h, v); break;
    case 8: hot_cmp(h, a, v); break;
    case 9: hot_cmp(h, (h.axys >> 8) & 0xFFu, v); break;
    default: hot_cmp(h, (h.axys >> 16) & 0xFFu, v); break;
  }
}
// RMW ops (ASL LSR ROL ROR INC DEC) on the value s
DEV uint32_t rmw(Hot &h, uint32_t o, uint32_t s) {
  const uint32_t C = h.fl & 1u;
  uint32_t r, c = C;
  switch (o) {
    case 0: r = (s << 1) & 0xFFu; c = s >> 7; break;
    case 1: r = s >> 1; c = s & 1u; break;
    case 2: r = ((s << 1) | C) & 0xFFu; c = s >> 7; break;
    case 3: r = (s >> 1) | (C << 7); c = s & 1u; break;
    case 4: r = (s + 1u) & 0xFFu; break;
    default: r = (s - 1u) & 0xFFu; break;
  }
  h.fl = (h.fl & ~1u) | c;
  h.zn = r;
  return r;
}

// ---------------------------------------------------------------------------------------------------------------
// Out-of-line paths.  Each takes the Hot registers by value, rebuilds a Cpu, does its work and hands the registers
// back: the struct copy through the stack is only paid on these (rare) calls, and the instruction cache keeps the
// inline loop below to itself.
template <int BLOCK, int ROMS, int THREADS, bool SOFT>
__device__ __noinline__ Hot cold_exec_generic(Hot h, uint32_t sl, uint32_t cx, uint32_t pl) {   // one instruction, any bus pattern
  Cpu<BLOCK, ROMS, THREADS, SOFT, SOFT ? 0 : 1> c; c.load(h, sl);     // (its own copy of the TIA code: see vcs_tia.cuh, TAG)
  c.template exec_one<true>((cx & 0xFFFFFF80u) | ((cx & 0x7Fu) - HC_COLD), pl);
  return c.store();
}
template <int BLOCK, int ROMS, int THREADS, bool SOFT>
__device__ __noinline__ Hot cold_exec(Hot h, uint32_t sl, uint32_t cx, uint32_t pl) {       // one instruction
  if constexpr (SOFT) return cold_exec_generic<BLOCK, ROMS, THREADS, SOFT>(h, sl, cx, pl);   // (soft reads are counted: no second try)
  Cpu<BLOCK, ROMS, THREADS, SOFT, COLD_TAG> c; c.load(h, sl);
  // a bus pattern outside the compact executor's: nothing of `c` is stored; the kernel's scheduling loop runs the
  // instruction again on cold_exec_generic (from there, not from here: the generic code calls into the TIA too, and the
  // TIA functions pay for every call level above them)
  if (c.template exec_one<false>((cx & 0xFFFFFF80u) | ((cx & 0x7Fu) - HC_COLD), pl)) { h.aux = AUX_GENERIC; return h; }
  return c.store();
}
template <int BLOCK, int ROMS, int THREADS, bool SOFT, bool COUNT = false>
__device__ __noinline__ Hot cold_pre(Hot h, uint32_t sl) {                                   // cyc >= lim: line end, WSYNC, cap, halt
  Cpu<BLOCK, ROMS, THREADS, SOFT> c; c.template load<false>(h, sl);
  const bool ok = c.template slow_pre<COUNT>();
  Hot r = c.store(); r.aux = ok ? 1u : 0u;
  return r;
}
template <int BLOCK, int ROMS, int THREADS, bool SOFT>
__device__ __noinline__ Hot cold_events(Hot h, uint32_t sl, uint32_t ev) {                   // a TIA write crossed a line / ended a frame
  Cpu<BLOCK, ROMS, THREADS, SOFT> c; c.template load<false>(h, sl);
  if (ev & EV_FRAME) c.fdone -= 1;                          // (S_FDONE, loaded above, already counts the frame that just ended)
  c.tia_events(ev, c.cyc);
  Hot r = c.store(); r.aux = (ev & EV_FRAME) ? 1u : 0u;
  return r;
}
template <int BLOCK, int ROMS, int THREADS, bool SOFT>
__device__ __noinline__ uint32_t cold_timer_read(uint32_t sl, uint32_t a, int32_t c) {       // INTIM / TIMINT around the underflow
  return Riot<BLOCK, 0>::timer_read(sl, a, c);
}

// The common ways a line ends — WSYNC released at the end of the line (a12: ws), or the code simply ran into the next
// line: returns the new `lim`, or LIM_NOW when the case is not the plain one (a stalled instruction that had already
// run over the line end, the frame cap in reach or reached) and cold_pre must decide.
template <int BLOCK>
__device__ __noinline__ int32_t line_step(uint32_t sl, int32_t cyc, int32_t lstart, bool ws) {
  using T = Tia<BLOCK>;
  const int32_t fcap = (int32_t)T::S(sl, S_FSTART) + (int32_t)T::ctx(C_CAP);
  if (ws ? (cyc - lstart > LINE_CYC || lstart + 2 * LINE_CYC >= fcap) : (cyc - lstart < LINE_CYC || cyc >= fcap)) return LIM_NOW;
  T::line_end(sl);
  return min(lstart + 2 * LINE_CYC, fcap);
}

// is `addr` a RAM cell or a plain byte of the (shared-memory staged) cartridge?  hs = first hotspot | count << 16
template <int ROMS>
DEV bool plain_addr(uint32_t addr, uint32_t hs) {
  const uint32_t a = addr & 0x1FFFu;
  if ((a & 0x1280u) == 0x0080u) return true;
  if constexpr (ROMS) return (a & 0x1000u) && (a - (hs & 0xFFFFu)) >= ((hs >> 16) & 0xFFu) && !((hs & HS_SC) && (a & 0x0F00u) == 0);
  else return false;                                       // (ROM in global memory: left to the out-of-line executor)
}
template <int BLOCK> DEV uint32_t cell_of(uint32_t off) { return ((off / BLOCK) & 0x7Cu) | (off & 3u); }   // RAM cell of a smem byte offset
template <int BLOCK, int ROMS>
DEV uint32_t rom_byte_hot(uint32_t off) {                  // byte `off` (bank << 12 | offset) of the block's ROM: staged, or (ROMS == 2) in global memory
  if constexpr (ROMS == 1) return reinterpret_cast<const uint8_t *>(smem)[(S_WORDS * BLOCK + C_WORDS) * 4 + off];
  else if constexpr (ROMS == 2)                            // (C_ROMOFF then holds the mask of the image's byte offsets: a 2 KB image has no mirror there)
    return __ldg(reinterpret_cast<const uint8_t *>((unsigned long long)Tia<BLOCK>::ctx(C_ROMG_LO) | ((unsigned long long)Tia<BLOCK>::ctx(C_ROMG_HI) << 32)) + (off & Tia<BLOCK>::ctx(C_ROMOFF)));
  else return 0;
}

// ---------------------------------------------------------------------------------------------------------------
// The inline interpreter loop: instructions of this lane's min-key group until the next scheduling point.
// SOFT: `se` = per decode entry {sum of the soft values of the instruction's own bytes, their count, their largest
// |soft - hard|, STE mismatches among them} (soft_entry_kernel); data reads of RAM and branches are noted where they run.
template <int BLOCK, int ROMS, int THREADS, bool SOFT, bool COUNT = false>
DEV void run_block(Hot &h, const uint2 *dr, const uint32_t sl, const uint32_t live, const float4 *se = nullptr, const float *stab = nullptr) {
  using T = Tia<BLOCK>;
  uint8_t *const ramb = reinterpret_cast<uint8_t *>(smem) + 4u * sl;
  auto soft_cell = [&](uint32_t a, uint32_t hard) -> uint32_t {          // SOFT: a value read of RAM cell a & 0x7F (else the byte as it is)
    if constexpr (SOFT) return soft_ram_read<BLOCK>(sl, a & 0x7Fu, hard); else return hard; };
  for (;;) {
    if constexpr (COUNT) { if (T::S(sl, S_BUDGET) == 0) { h.keyhi = 0xFFFFFFFFu; return; } }   // the budget is spent: this lane is done
    if (h.cyc >= h.lim) {
      int32_t nl = LIM_NOW;
      const bool ws = h.lim == LIM_WSYNC;
      if (h.lim != LIM_NOW) nl = line_step<BLOCK>(sl, h.cyc, h.lstart, ws);
      if (nl != LIM_NOW) { h.lstart += LINE_CYC; if (ws) h.cyc = h.lstart; h.lim = nl; }
      else { h = cold_pre<BLOCK, ROMS, THREADS, SOFT, COUNT>(h, sl); if (!h.aux) return; }
    }
    if constexpr (COUNT) T::S(sl, S_BUDGET) -= 1u;         // (a frame end at the cap or an idle cycle above is not an instruction)
    uint32_t cx = h.wx, pl = h.wy;                         // the entry being executed
    const int32_t cyc0 = h.cyc;                            // its first cycle
    if constexpr (SOFT) { if ((cx & 0x7Fu) != HC_COLD + H_SLOW) {     // the instruction's own bytes, pre-summed (one decoded at run time — code in RAM
      const float4 e = __ldg(se + h.di);                             // included, whose di aliases a ROM entry — notes its bytes as it fetches them)
      soft_acc<BLOCK>(sl, 0) += e.x; soft_acc<BLOCK>(sl, 3) += e.y; soft_acc<BLOCK>(sl, 6) += e.w;
      soft_acc<BLOCK>(sl, 7) = fmaxf(soft_acc<BLOCK>(sl, 7), e.z);
    } }
    h.di += (cx >> DW_LEN_SHIFT) & 0xFFu;
    uint2 wn = __ldg(dr + h.di);                           // sequential prefetch
    // (the entry moves into h.wx / h.wy through an OR with a zero the compiler cannot see through — di < 2^15 — so that
    // the move stays where it is written, after the instruction's own work, instead of right behind the load, where it
    // would wait out every L1 miss of the decode table: 5 % of the warps' time)
    const uint32_t late0 = h.di & 0x80000000u;
    h.cyc += (int32_t)((cx >> DW_CY_SHIFT) & 0xFu);
    uint32_t cls = cx & 0x7Fu, aux = cx >> DW_OP2_SHIFT;
    uint32_t v;
    if (cx & (DW_F_LDST | DW_F_STTIA)) {
      uint32_t reg = pl & 0xFFu;
      if (cx & DW_F_LDST) {                                // LDx #imm ; STx reg in one entry
        h.axys = __byte_perm(h.axys, pl, pl >> 16); h.zn = pl & 0xFFu;
        if (h.cyc - 3 - (int32_t)aux >= h.lim) {           // boundary work pending between the two: the store runs as its own entry
          h.di -= 2u + aux; h.cyc -= 3 + (int32_t)aux;
          goto ctl;
        }
        reg = (pl >> 8) & 0x3Fu;
        v = __byte_perm(h.axys, 0u, 0x4440u | ((pl >> 14) & 3u));
      } else v = __byte_perm(h.axys, 0u, pl >> 16);
      if (reg == 0x02u && h.cyc - 1 - h.lstart < LINE_CYC) {                 // STx WSYNC inside the line: only the latch changes
        T::S(sl, S_FL) |= TF_WSYNC; h.lim = LIM_WSYNC;
        goto seq;
      }
      const uint32_t ev = T::write(sl, reg, v, h.cyc - 1 - h.lstart);
      if (ev) {
        if (ev == EV_WSYNC) h.lim = LIM_WSYNC;
        else { h.wx = wn.x | late0; h.wy = wn.y | late0; h = cold_events<BLOCK, ROMS, THREADS, SOFT>(h, sl, ev); if (h.aux) return; continue; }
      }
    }
    else if (cx & DW_F_LDIMM) { h.axys = __byte_perm(h.axys, pl, pl >> 16); h.zn = pl & 0xFFu; }
    else if (cx & DW_F_BR) {
      const uint32_t t = (h.fl & 0x41u) | ((h.zn & 0x180u) ? 0x80u : 0u) | ((h.zn & 0xFFu) ? 0u : 2u);
      const bool taken = ((t >> (aux & 7u)) & 1u) == ((aux >> 3) & 1u);
      if constexpr (SOFT) soft_branch_note<BLOCK>(sl, (t >> (aux & 7u)) & 1u, (aux & 8u) ? 1.f : -1.f, (float)(int32_t)pl, taken, (float)((h.pbase + h.di) & 0xFFFFu));
      if (taken) { h.di += pl; h.cyc += (int32_t)(aux >> 4); goto ctl; }
    }
    else if (cls == HC_RTIM) {                             // absolute read of INTIM / TIMINT in the 4th cycle
    do_rtim:
      const uint32_t tw = T::S(sl, S_TMR);
      const uint32_t d = (uint32_t)(h.cyc - (int32_t)T::S(sl, S_TTICKS));
      const uint32_t timer = tw & 0xFFu, kk = ((tw >> 16) + d) >> ((tw >> 8) & 0xFu);
      if (!(tw & 0x1000u) && (int32_t)d > 0 && kk <= timer) v = (pl & 1u) ? 0u : timer - kk;      // before the underflow
      else v = cold_timer_read<BLOCK, ROMS, THREADS, SOFT>(sl, pl, h.cyc - 1);
      goto do_alu;
    }
    else if (cls == HC_INCDEC) {
      v = (__byte_perm(h.axys, 0u, pl) + aux) & 0xFFu;
      h.axys = __byte_perm(h.axys, v, pl >> 16); h.zn = v;
    }
    else if (cls == HC_LD_RAM) { v = ramb[pl & 0xFFFFu]; if constexpr (SOFT) v = soft_ram_read<BLOCK>(sl, cell_of<BLOCK>(pl & 0xFFFFu), v);
                                 h.axys = __byte_perm(h.axys, v, pl >> 16); h.zn = v; }
    else {
      switch (cls) {
        case HC_ST_RAM: ramb[pl & 0xFFFFu] = (uint8_t)__byte_perm(h.axys, 0u, pl >> 16); break;
        case HC_XFER:
          v = __byte_perm(h.axys, 0u, pl); h.axys = __byte_perm(h.axys, v, pl >> 16);
          if (aux) h.zn = v;
          else if (h.keyhi < KEY_PARKED) h.keyhi = (h.keyhi & ~(0xFFu << 19)) | (v << 19);      // TXS: SP is part of the key
          break;
        case HC_ALU_IMM: v = pl; goto do_alu;
        case HC_ALU_RAM: v = ramb[pl]; if constexpr (SOFT) v = soft_ram_read<BLOCK>(sl, cell_of<BLOCK>(pl), v); goto do_alu;
        case HC_RMW_RAM: v = ramb[pl]; if constexpr (SOFT) v = soft_ram_read<BLOCK>(sl, cell_of<BLOCK>(pl), v);
                         v = rmw(h, aux, v); ramb[pl] = (uint8_t)v; break;
        case HC_ACC: v = rmw(h, aux, h.axys & 0xFFu); h.axys = __byte_perm(h.axys, v, 0x3214u); break;
        case HC_FLAG: h.fl = (h.fl & ~pl) | (pl >> 16); break;
        case HC_NOP: break;
        case HC_SPIN: {
      // The timer wait loop in closed form.  Poll i reads the timer in tick cyc + 7 i + 4 (4th cycle of LDA / BIT abs;
      // a taken branch back is 3 cycles); the loop leaves with the first poll that reads INTIM == 0 (aux 0) or TIMINT
      // bit 7 set (aux 1), 2 cycles later.  Covered: no underflow flag set yet, the deciding poll lands while the
      // value is 0 / right after the underflow, no frame cap on the way.  Nothing in the loop touches the TIA, so
      // the line ends on the way are all it owes the beam.
      const uint32_t tw = T::S(sl, S_TMR);
      const uint32_t shift = (tw >> 8) & 0xFu, sub0 = tw >> 16, tv = tw & 0xFFu;
      const int32_t dfirst = h.cyc + 4 - (int32_t)T::S(sl, S_TTICKS);
      const int32_t dz = (int32_t)((tv << shift) - sub0), du = (int32_t)(((tv + 1u) << shift) - sub0);   // ticks until the value is 0 / underflows
      const int32_t need = aux ? du : dz;
      const int32_t k = (need > dfirst) ? (need - dfirst + 6) / 7 : 0;
      const int32_t cend = h.cyc + 7 * k + 6;
      const int32_t fcap = (int32_t)T::S(sl, S_FSTART) + (int32_t)T::ctx(C_CAP);
      if (!(tw & 0x1000u) && dfirst > 0 && (aux || dfirst + 7 * k < du) && cend - 2 < fcap) {
        if (aux) { h.zn = ((h.axys & 0x80u) ? 1u : 0u) | 0x100u; h.fl &= ~0x40u; }      // BIT with v = $80
        else { h.axys &= ~0xFFu; h.zn = 0; }                                             // LDA with v = 0
        h.cyc = cend; h.di += 5u;
        while (h.lstart + LINE_CYC <= cend - 2) { T::line_end(sl); h.lstart += LINE_CYC; }
        h.lim = min(h.lstart + LINE_CYC, fcap);
        goto ctl;
      }
      cx = pl; pl = 0x0284u | aux;                         // not covered: run the poll itself
      h.di += 3u; h.cyc += 4; wn = __ldg(dr + h.di);
      aux = cx >> DW_OP2_SHIFT;
        } goto do_rtim;
        case HC_JMP: { const uint32_t nd = (h.di & 0x7000u) | (pl & 0xFFFu); h.pbase = pl - nd; h.di = nd; } goto ctl;
        // ---- indexed / indirect accesses and the stack, as long as every bus access of the instruction is a RAM cell
        // or a plain cartridge byte (C.5 sequences; their dummy cycles then have no effect).  Anything else — TIA / RIOT
        // registers, bank hotspots, stack or pointer cells outside RAM — goes to the out-of-line executor untouched.
        case HC_IDX_RD: case HC_IDX_ST: case HC_IZY_RD: case HC_IZY_ST: case HC_IZX_RD: case HC_IZX_ST: {
          const bool store = cls >= HC_IDX_ST;
          const uint32_t hs = T::ctx(C_HS);
          uint32_t ea, gid;                                // effective address ; the generic handler id of this instruction
          bool ok = true;
          if (cls == HC_IDX_RD || cls == HC_IDX_ST) {
            const uint32_t idx = __byte_perm(h.axys, 0u, pl >> 16), base = pl & 0xFFFFu, useX = ((pl >> 16) & 3u) == 1u;
            if (aux & 0x80u) { ea = (base + idx) & 0xFFu; gid = (store ? H_W0 + 2u : H_R0 + 3u) - useX; }
            else {
              const uint32_t t = (base & 0xFFu) + idx, unc = (base & 0xFF00u) | (t & 0xFFu);
              ea = (unc + (t & 0x100u)) & 0xFFFFu; gid = (store ? H_W0 + 5u : H_R0 + 6u) - useX;
              if (store || (t & 0x100u)) ok = plain_addr<ROMS>(unc, hs);        // the discarded read at the uncorrected address
              if (!store) h.cyc += (int32_t)(t >> 8);                            // page crossed: one more cycle
            }
            aux &= 0x7Fu;
          } else {
            const bool izy = cls == HC_IZY_RD || cls == HC_IZY_ST;
            uint32_t lo, hi, iy = 0;
            if (izy) { lo = ramb[pl & 0x7FFFu]; hi = ramb[pl >> 15]; iy = (h.axys >> 16) & 0xFFu; gid = store ? H_W0 + 7u : H_R0 + 8u; }
            else {
              const uint32_t z = (pl + ((h.axys >> 8) & 0xFFu)) & 0xFFu; gid = store ? H_W0 + 6u : H_R0 + 7u;
              ok = z - 0x80u <= 0x7Eu;                                           // both pointer cells in RAM
              lo = ramb[((z & 0x7Cu) * BLOCK) | (z & 3u)]; hi = ramb[(((z + 1u) & 0x7Cu) * BLOCK) | ((z + 1u) & 3u)];
            }
            const uint32_t t = lo + iy, unc = (hi << 8) | (t & 0xFFu);
            ea = (unc + (t & 0x100u)) & 0xFFFFu;
            if (izy && (store || (t & 0x100u))) ok = ok && plain_addr<ROMS>(unc, hs);     // (zp),Y: the discarded read at the uncorrected address
            if (izy && !store) h.cyc += (int32_t)(t >> 8);                                 // page crossed: one more cycle
          }
          const bool in_ram = (ea & 0x1280u) == 0x0080u;
          ok = ok && (store ? in_ram : plain_addr<ROMS>(ea, hs));
          if (!ok) {                                       // not this simple: the generic handler, from the instruction's first cycle
            h.cyc = cyc0;
            uint32_t gpl = pl & 0xFFFFu;
            if (cls == HC_IZY_RD || cls == HC_IZY_ST) { const uint32_t o = pl & 0x7FFFu; gpl = 0x80u | ((o / BLOCK) & 0x7Cu) | (o & 3u); }
            else if (cls == HC_IZX_RD || cls == HC_IZX_ST) gpl = pl & 0xFFu;
            h.wx = (HC_COLD + gid) | (cx & 0x00FF0000u) | (aux << DW_OP2_SHIFT); h.wy = gpl;   // (kept in h: cold_exec may pass it on, AUX_GENERIC)
            h = cold_exec<BLOCK, ROMS, THREADS, SOFT>(h, sl, h.wx, h.wy);
            return;
          }
          const uint32_t ro = ((ea & 0x7Cu) * BLOCK) | (ea & 3u);
          if constexpr (SOFT) {                            // the pointer bytes are value reads of RAM (their hard values formed ea)
            if (cls == HC_IZY_RD || cls == HC_IZY_ST) { const uint32_t o = pl & 0x7FFFu, z = ((o / BLOCK) & 0x7Cu) | (o & 3u);
                                                        soft_cell(z, ramb[o]); soft_cell(z + 1u, ramb[pl >> 15]); }
            else if (cls == HC_IZX_RD || cls == HC_IZX_ST) { const uint32_t z = (pl + ((h.axys >> 8) & 0xFFu)) & 0xFFu;
                                                             soft_cell(z, ramb[((z & 0x7Cu) * BLOCK) | (z & 3u)]); soft_cell(z + 1u, ramb[(((z + 1u) & 0x7Cu) * BLOCK) | ((z + 1u) & 3u)]); }
          }
          if (store) { ramb[ro] = (uint8_t)__byte_perm(h.axys, 0u, 0x4440u | aux); break; }
          if (in_ram) v = soft_cell(ea, ramb[ro]);
          else {
            v = rom_byte_hot<BLOCK, ROMS>((h.di & 0x7000u) + (ea & 0xFFFu));
            if constexpr (SOFT) { const float sv = __ldg(stab + (h.di & 0x7000u) + (ea & 0xFFFu)), hv = (float)v, ste = sv + (hv - sv);
                                  soft_note<BLOCK>(sl, 0, sv, hv, ste); v = (uint32_t)(int)rintf(ste) & 0xFFu; }
          }
        } goto do_alu;
        case HC_JSR: case HC_RTS: case HC_STACK: {
          const uint32_t sp = h.axys >> 24;
          uint32_t nsp, target;
          auto cell = [&](uint32_t a) -> uint8_t & { return ramb[((a & 0x7Cu) * BLOCK) | (a & 3u)]; };
          if (cls == HC_JSR) {
            if (sp < 0x81u) goto generic_stack;
            const uint32_t ret = (h.pbase + h.di - 1u) & 0xFFFFu;               // address of the instruction's third byte
            cell(sp) = (uint8_t)(ret >> 8); cell(sp - 1u) = (uint8_t)ret; nsp = sp - 2u; target = pl;
          } else if (cls == HC_RTS) {
            if (sp - 0x7Fu > 0xFDu - 0x7Fu) goto generic_stack;
            const uint32_t r = (uint32_t)cell(sp + 1u) | ((uint32_t)cell(sp + 2u) << 8);
            if (!((r & 0x1000u) && plain_addr<ROMS>(r, T::ctx(C_HS)))) goto generic_stack;   // the discarded read at the pulled address
            if constexpr (SOFT) { soft_cell(sp + 1u, r & 0xFFu); soft_cell(sp + 2u, r >> 8); }
            nsp = sp + 2u; target = (r + 1u) & 0xFFFFu;
          } else if (aux < 2u) {                           // PHA / PHP
            if (sp < 0x80u) goto generic_stack;
            cell(sp) = aux ? (uint8_t)((h.fl & 0x4Du) | 0x30u | ((h.zn & 0x180u) ? 0x80u : 0u) | ((h.zn & 0xFFu) ? 0u : 2u)) : (uint8_t)h.axys;
            nsp = (sp - 1u) & 0xFFu; target = 0x10000u;
          } else {                                         // PLA / PLP
            if (sp - 0x7Fu > 0xFEu - 0x7Fu) goto generic_stack;
            v = soft_cell(sp + 1u, cell(sp + 1u)); nsp = sp + 1u; target = 0x10000u;
            if (aux == 2u) { h.axys = __byte_perm(h.axys, v, 0x3214u); h.zn = v; }
            else { h.fl = v & 0x4Du; h.zn = ((v & 0x80u) << 1) | ((v & 2u) ? 0u : 1u); }
          }
          h.axys = (h.axys & 0x00FFFFFFu) | (nsp << 24);
          if (h.keyhi < KEY_PARKED) h.keyhi = (h.keyhi & ~(0xFFu << 19)) | (nsp << 19);          // SP is part of the scheduling key
          if (target < 0x10000u) { const uint32_t nd = (h.di & 0x7000u) | (target & 0xFFFu); h.pbase = target - nd; h.di = nd; goto ctl; }
          break;
        generic_stack:
          h.wx = (HC_COLD + (cls == HC_JSR ? (uint32_t)H_JSR : cls == HC_RTS ? (uint32_t)H_RTS : H_PHA + aux)) | (cx & 0x00FFFF00u);
          h = cold_exec<BLOCK, ROMS, THREADS, SOFT>(h, sl, h.wx, pl);
          return;
        }
        case HC_ST_RIOT: {                                 // STx abs to a RIOT register: the write is the instruction's 4th cycle
          v = __byte_perm(h.axys, 0u, pl >> 16);
          if ((pl & 4u) == 0) { const uint32_t sh = 8u * (pl & 3u); T::S(sl, S_PORTS) = (T::S(sl, S_PORTS) & ~(0xFFu << sh)) | (v << sh); }
          else if ((pl & 0x14u) == 0x14u) {
            const uint32_t k = pl & 3u, shift = (0x0A630u >> (4u * k)) & 0xFu;                 // 0, 3, 6, 10
            T::S(sl, S_TMR) = v | (shift << 8) | (((1u << shift) - 1u) << 16); T::S(sl, S_TTICKS) = (uint32_t)h.cyc;
          }
        } break;
        default:                                           // everything else: out of line, then re-schedule
          h = cold_exec<BLOCK, ROMS, THREADS, SOFT>(h, sl, cx, pl);
          return;
      }
    }
    goto seq;
  do_alu:
    alu(h, aux, v);
  seq:                                                     // sequential successor
    h.wx = wn.x | late0; h.wy = wn.y | late0;
    // a leader is where another lane of the warp may be waiting: re-form the group — unless every lane of the warp that
    // can run at all (`live`: holds an env, not parked, not done — as of the last scheduling pass; a lane can only
    // leave that set before the next pass) is in this group already: nobody can be waiting, and which lanes run
    // together never changes results, only the time they take
    if (!(h.wx & DW_LEADER) || __activemask() == live) continue;
    return;
  ctl:                                                     // taken branch / jump: fetch at the new PC, re-schedule
    if (!((h.pbase + h.di) & 0x1000u)) { h.wx = HC_COLD + H_SLOW; h.wy = 0; }
    else { const uint2 t = __ldg(dr + h.di); h.wx = t.x; h.wy = t.y; }
    if (__activemask() == live) continue;                  // (every runnable lane of the warp took it together)
    return;
  }
}

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

template <int BLOCK, int ROMS, int THREADS, bool SOFT, bool COUNT = false>
__global__ void __launch_bounds__(THREADS, 512 / BLOCK) vcs_step_kernel(StepParams p) {
  using T = Tia<BLOCK>;
  __shared__ __align__(8) unsigned long long s_bar;
  uint32_t *s_ctx = smem + S_WORDS * BLOCK;
  constexpr uint32_t ROM_OFF = (S_WORDS * BLOCK + C_WORDS) * 4;          // byte offset of the ROM image in smem
  const int tid = threadIdx.x;
  // Code placement.  The kernel is instruction-cache bound and its hot device functions follow the kernel body in the
  // image, so where their 128-byte lines begin moves with the body's size (+-4 % from placement alone).
  // VCS_PAD filler instructions (one clock read each, executed once per thread) in the headline variant's prologue
  // put that offset where it measured best; 0..7 cover every placement modulo 128 bytes.
  if constexpr (BLOCK == 256 && ROMS == 1 && THREADS == 288 && !SOFT && !COUNT) {
#pragma unroll
    for (int i = 0; i < VCS_PAD; ++i) { uint32_t t; asm volatile("mov.u32 %0, %%clock;" : "=r"(t)); }
  }
  if (p.blk_time && tid == 0) {                            // placement bookkeeping: when and where this block ran
    unsigned long long t; uint32_t sm;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); asm volatile("mov.u32 %0, %%smid;" : "=r"(sm));
    p.blk_time[3 * blockIdx.x] = t; p.blk_time[3 * blockIdx.x + 1] = 0; p.blk_time[3 * blockIdx.x + 2] = sm;
  }
  const int e0 = (p.perm ? p.perm[blockIdx.x] : (int)blockIdx.x) * BLOCK;   // which group of BLOCK envs this block runs
  const int B = p.batch;
  const int ei = e0 + tid;                                 // the env this thread starts with
  const bool filed = tid < BLOCK;                          // threads of the spare warp start without a file
  const bool live0 = filed && ei < B && (!p.mask || p.mask[ei]);   // vcs_step_masked: envs with mask 0 stay frozen
  const uint32_t romid = (uint32_t)p.env_rom[live0 ? ei : e0];
  const RomMeta rm = p.rom_meta[romid];

  if (tid == 0) {
    const unsigned long long scr = reinterpret_cast<unsigned long long>(p.screen);
    s_ctx[C_SCREEN_LO] = (uint32_t)scr; s_ctx[C_SCREEN_HI] = (uint32_t)(scr >> 32);
    s_ctx[C_Y0] = (uint32_t)p.y0; s_ctx[C_FRAMESKIP] = (uint32_t)p.frameskip; s_ctx[C_BATCH] = (uint32_t)B; s_ctx[C_ENV0] = (uint32_t)e0;
    s_ctx[C_CAP] = (uint32_t)(p.max_lines * LINE_CYC); s_ctx[C_ROMOFF] = (ROMS == 2) ? ((rm.size == 2048) ? 0x7FFu : 0xFFFFFFFFu) : ROM_OFF;
    s_ctx[C_REGROUP] = (ROMS && rm.kind >= MK_F8 && rm.kind <= MK_F4SC && p.regroup) ? 1u : 0u;
    s_ctx[C_HS] = rm.hs;
    { const unsigned long long v = reinterpret_cast<unsigned long long>(p.sc_ram); s_ctx[C_SCRAM_LO] = (uint32_t)v; s_ctx[C_SCRAM_HI] = (uint32_t)(v >> 32); }
    auto put = [&](int lo, const void *q) { const unsigned long long v = reinterpret_cast<unsigned long long>(q); s_ctx[lo] = (uint32_t)v; s_ctx[lo + 1] = (uint32_t)(v >> 32); };
    put(C_META_LO, p.rom_meta); put(C_BLOB_LO, p.rom_blob); put(C_DROM_LO, p.drom); put(C_ROMG_LO, p.rom_blob + rm.offset);
    put(C_SOFT_WD_LO, p.soft_wd); put(C_SOFT_W_LO, p.soft_w); put(C_SOFT_TAB_LO, p.soft_tab); s_ctx[C_SOFT_K] = (uint32_t)p.soft_K | (p.soft_full ? 0x80000000u : 0u); s_ctx[C_SOFT_ALPHA] = __float_as_uint(p.soft_alpha);
    if constexpr (ROMS == 1) { mbar_init(smem_u32(&s_bar), 1); asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
  }
  __syncthreads();
  if constexpr (ROMS == 1) {                               // a3: stage the block's ROM (2 KB images twice: the mirror)
    if (tid == 0) {
      const uint32_t bar = smem_u32(&s_bar), dst = smem_u32(smem) + ROM_OFF;
      const uint8_t *src = p.rom_blob + rm.offset;
      mbar_expect_tx(bar, rm.size == 2048 ? 4096u : rm.size);
      bulk_g2s(dst, src, rm.size, bar);
      if (rm.size == 2048) bulk_g2s(dst + 2048, src, 2048, bar);
    }
  }

  Cpu<BLOCK, ROMS, THREADS, SOFT> s;
  s.sl = filed ? (uint32_t)tid : NOSLOT; s.sl4 = 4u * s.sl;
  const uint32_t sl = s.sl;
  // ---- a1 state load (coalesced SoA)
  uint32_t n0 = 0, fl = 0, pc0 = 0, bank0 = 0;
  if (live0) {
    uint32_t w;
    w = p.st[W_AXYS * B + ei]; s.A = w & 0xFF; s.X = (w >> 8) & 0xFF; s.Y = (w >> 16) & 0xFF; s.SP = w >> 24;
    w = p.st[W_PC * B + ei]; pc0 = w & 0xFFFF; s.unpack_p((w >> 16) & 0xFF); s.status = w >> 24;
    w = p.st[W_BEAM * B + ei]; n0 = w & 0xFF; T::S(sl, S_LINE) = (w >> 8) & 0xFFFF; bank0 = (w >> 24) & 7u;
    s.fstart = -(int32_t)p.st[W_FCYC * B + ei];
    T::S(sl, S_TMR) = p.st[W_TIMER * B + ei]; T::S(sl, S_TTICKS) = 0;
    T::S(sl, S_PORTS) = p.st[W_PORTS * B + ei];
    T::S(sl, S_COLU) = p.st[W_COLU * B + ei]; T::S(sl, S_PF) = p.st[W_PF * B + ei]; T::S(sl, S_GRP) = p.st[W_GRP * B + ei]; T::S(sl, S_NUSIZ) = p.st[W_NUSIZ * B + ei];
    T::S(sl, S_POS) = p.st[W_POS * B + ei]; w = p.st[W_POS2 * B + ei]; T::S(sl, S_POS2) = w & 0xFFFF; T::S(sl, S_RX) = w >> 16;
    fl = (p.st[W_FLAGS * B + ei] & TF_ARCH_MASK) | TF_DIRTY_ALL; T::S(sl, S_CX) = p.st[W_CX * B + ei]; T::S(sl, S_CART) = p.st[W_CART * B + ei];
    T::S(sl, S_PX) = 0; T::S(sl, S_FDONE) = 0;
    for (int i = 0; i < 32; ++i) smem[(S_RAM + i) * BLOCK + tid] = p.ram[i * B + ei];
    for (int i = 0; i < 10; ++i) smem[(S_PLANE + i) * BLOCK + tid] = 0;
    if constexpr (COUNT) T::S(sl, S_BUDGET) = (uint32_t)p.n_instr;        // (no row is kept in this mode: the planes are free)
    if (p.frameskip == 1) { fl |= TF_STORING; if ((T::S(sl, S_LINE) - (uint32_t)p.y0) < (uint32_t)SCR_H) fl |= TF_ROWVIS; }
  } else {
    s.A = s.X = s.Y = s.SP = 0; s.unpack_p(0x24); s.status = 0; s.fstart = 0;
    if (filed) { T::S(sl, S_INP) = (uint32_t)tid << 16; T::S(sl, S_FL) = 0; T::S(sl, S_TMR) = 0; T::S(sl, S_TTICKS) = 0; }
  }
  s.di = (bank0 << 12) | (pc0 & 0xFFFu); s.pbase = pc0 - s.di;
  s.fskip = (uint32_t)p.frameskip;
  s.cyc = 0; s.lstart = -(int32_t)n0; s.fdone = live0 ? 0u : s.fskip; s.romid = romid;
  s.cap = p.max_lines * LINE_CYC;
  s.hs_n = (rm.hs >> 16) & 0xFFu; s.hs_lo = rm.hs & 0xFFFFu; s.kind = rm.kind;
  const bool regroups = ROMS && rm.kind >= MK_F8 && rm.kind <= MK_F4SC && p.regroup;    // block-uniform
  s.park = regroups ? 1u : 0u;
  s.rom_off = ROM_OFF; s.rom_g = p.rom_blob + rm.offset; s.dr = p.drom + rm.doff; 
  s.rom_mask = (rm.size == 2048 && ROMS != 1) ? 0x7FFu : 0xFFFu;
  // ---- a2 action latch (C.11)
  if (live0) {
    uint32_t act = p.actions[ei]; if (act >= 18u) act = 0;
    uint32_t inb = p.switches[ei];                         // SWCHB input pins
    {                                                      // vcs_auto_reset: an env that is still booting ignores the agent
      const uint32_t b = p.boot[ei], c = b & 0xFFu, k = (b >> 8) & 0xFFu, R = b >> 16;     // steps left | NOOP starts | RESET steps
      if (c) { act = 0; if (c > k && c <= k + R) inb &= ~1u; p.boot[ei] = b - 1u; }
    }
    //            NOOP FIRE UP RIGHT LEFT DOWN UR UL DR DL UF RF LF DF URF ULF DRF DLF
    const uint32_t up = 0x0C4C4u, down = 0x32320u, left = 0x29290u, right = 0x14948u, fire = 0x3FC02u;
    uint32_t ina = 0xFFu;
    if ((up >> act) & 1u) ina &= ~0x10u;
    if ((down >> act) & 1u) ina &= ~0x20u;
    if ((left >> act) & 1u) ina &= ~0x40u;
    if ((right >> act) & 1u) ina &= ~0x80u;
    const uint32_t fire0 = (fire >> act) & 1u;
    // the live SWCHB pins (bits 0, 1, 3, 6, 7) travel in S_INP bits 9..13
    T::S(sl, S_INP) = ina | (fire0 << 8) | (((inb & 3u) | ((inb >> 1) & 4u) | ((inb >> 3) & 0x18u)) << 9) | ((uint32_t)tid << 16);
    if ((fl & TF_LATCHEN) && fire0) fl &= ~TF_INPT4_LATCH;
    T::S(sl, S_FL) = fl;
  }
  s.wsync = (fl & TF_WSYNC) != 0;
  s.relim(); s.rekey();
  if constexpr (ROMS == 1) mbar_wait(smem_u32(&s_bar), 0);
  s.w = live0 ? s.fetch() : make_uint2(HC_COLD + H_SLOW, 0);
  Hot h;
  if (filed) { if (!live0) T::S(sl, S_FDONE) = s.fskip; h = s.store(); }
  else { h.axys = h.fl = h.zn = h.di = h.pbase = 0; h.cyc = h.lstart = 0; h.lim = LIM_NOW; h.wx = HC_COLD + H_SLOW; h.wy = 0; h.aux = 0; }
  h.keyhi = s.keyhi;
  const uint2 *const dr = s.dr;
  const float4 *const se = SOFT ? p.soft_ent + rm.doff : nullptr;
  const float *const stab = SOFT ? p.soft_tab + rm.pad : nullptr;
  if constexpr (SOFT) { if (filed) { for (int k = 0; k < 8; ++k) soft_acc<BLOCK>(sl, k) = 0.f; } }
  uint32_t cur = sl;                                       // the file this thread runs (changes at a regroup)

  // ---- the hot loop: whole instructions until `frameskip` frame-end events (C.10), min-key lanes first.
  // Line bookkeeping mirrors C.4: the line counter advances with the FIRST cycle of a new line, so an
  // instruction that ends exactly on a line boundary leaves n == 76 pending (a frame end at that point
  // makes the finished line "line 0" and the next one line 1).
  for (;;) {
    for (;;) {
      const uint32_t key = h.keyhi | ((h.pbase + h.di) & 0xFFFFu);
      const uint32_t mk = __reduce_min_sync(0xFFFFFFFFu, key);
      if (mk >= KEY_PARKED) break;                         // every lane is parked or has finished the step
      const uint32_t live = __ballot_sync(0xFFFFFFFFu, key < KEY_PARKED);      // the lanes that can run
      if (key == mk) run_block<BLOCK, ROMS, THREADS, SOFT, COUNT>(h, dr, cur, live, se, stab);
      if (h.aux == AUX_GENERIC) h = cold_exec_generic<BLOCK, ROMS, THREADS, SOFT>(h, cur, h.wx, h.wy);   // (a rare bus pattern: see cold_exec)
    }
    if (!regroups) break;
    if (!__syncthreads_or(h.keyhi == KEY_PARKED)) break;   // nobody left to run in this block
    if (cur != NOSLOT) s.load(h, cur); else { s.sl = NOSLOT; s.fskip = (uint32_t)p.frameskip; s.park = 1u; }
    s.regroup();
    cur = s.sl;
    if (cur != NOSLOT) h = s.store(); else h.keyhi = 0xFFFFFFFFu;
  }
  if (cur == NOSLOT) return;
  const uint32_t fs = cur;                                 // the file (and env) this thread ends up holding
  const int e = e0 + (int)(T::S(fs, S_INP) >> 16);
  const bool live = e < B && (!p.mask || p.mask[e]);
  if (!live) return;
  s.load(h, fs);
  if (s.cyc - s.lstart > LINE_CYC) { T::line_end(fs); s.lstart += LINE_CYC; }      // the last instruction ran over the line end
  // ---- a16 state store
  {
    uint32_t timer, sub, shift, tflag;
    s.timer_sync(s.cyc, timer, sub, shift, tflag);
    p.st[W_AXYS * B + e] = s.A | (s.X << 8) | (s.Y << 16) | (s.SP << 24);
    p.st[W_PC * B + e] = s.pc() | (s.pack_p() << 16) | (s.status << 24);
    p.st[W_BEAM * B + e] = (uint32_t)(s.cyc - s.lstart) | (T::S(fs, S_LINE) << 8) | ((s.di >> 12) << 24);
    p.st[W_FRAME * B + e] += s.fdone;
    p.st[W_FCYC * B + e] = (uint32_t)(s.cyc - s.fstart);
    p.st[W_TIMER * B + e] = timer | (shift << 8) | (tflag << 12) | (sub << 16);
    p.st[W_PORTS * B + e] = T::S(fs, S_PORTS);
    p.st[W_COLU * B + e] = T::S(fs, S_COLU); p.st[W_PF * B + e] = T::S(fs, S_PF); p.st[W_GRP * B + e] = T::S(fs, S_GRP); p.st[W_NUSIZ * B + e] = T::S(fs, S_NUSIZ);
    p.st[W_POS * B + e] = T::S(fs, S_POS); p.st[W_POS2 * B + e] = (T::S(fs, S_POS2) & 0xFFFF) | (T::S(fs, S_RX) << 16);
    p.st[W_FLAGS * B + e] = T::S(fs, S_FL) & TF_ARCH_MASK; p.st[W_CX * B + e] = T::S(fs, S_CX); p.st[W_CART * B + e] = T::S(fs, S_CART);
    for (int i = 0; i < 32; ++i) p.ram[i * B + e] = smem[(S_RAM + i) * BLOCK + fs];
    p.cyc[e] += (unsigned long long)s.cyc;
    if constexpr (SOFT) { for (int k = 0; k < 8; ++k) p.soft_out[8 * (size_t)e + k] = soft_acc<BLOCK>(fs, k); }
  }
  if (p.blk_time) { unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); atomicMax(&p.blk_time[3 * blockIdx.x + 1], t); }
}

// W(T) x ROM: for every cell o of every bank of every cartridge the relaxed read of eq. (10) on the 4096 x 8 bit
// tensor (byte = sum_j 2^j * bit plane j), window |k| <= K clipped to the bank, normalised over the cells kept.
// A banded [4096 x 4096] x [4096 x 8] contraction per bank, done once per temperature instead of once per fetch.
__global__ void soft_table_kernel(const uint8_t *rom_blob, const RomMeta *meta, const float *wt, int K, float *tab) {
  const RomMeta rm = meta[blockIdx.y];
  const int nb = max(1, (int)(rm.size >> 12));
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;            // bank * 4096 + o
  if (idx >= nb * 4096) return;
  const int bank = idx >> 12, o = idx & 0xFFF;
  const uint32_t mask = (rm.size == 2048) ? 0x7FFu : 0xFFFu;
  const uint8_t *img = rom_blob + rm.offset + bank * 4096;
  float pl0 = 0, pl1 = 0, pl2 = 0, pl3 = 0, pl4 = 0, pl5 = 0, pl6 = 0, pl7 = 0, den = 0;
  const int lo = max(-K, -o), hi = min(K, 4095 - o);
  for (int k = lo; k <= hi; ++k) {
    const float w = __ldg(wt + abs(k));
    const uint32_t b = img[(uint32_t)(o + k) & mask];
    pl0 += w * (float)(b & 1u); pl1 += w * (float)((b >> 1) & 1u); pl2 += w * (float)((b >> 2) & 1u); pl3 += w * (float)((b >> 3) & 1u);
    pl4 += w * (float)((b >> 4) & 1u); pl5 += w * (float)((b >> 5) & 1u); pl6 += w * (float)((b >> 6) & 1u); pl7 += w * (float)((b >> 7) & 1u);
    den += w;
  }
  const float inv = 1.f / den;
  tab[rm.pad + idx] = pl0 * inv + 2.f * (pl1 * inv) + 4.f * (pl2 * inv) + 8.f * (pl3 * inv) + 16.f * (pl4 * inv) + 32.f * (pl5 * inv) + 64.f * (pl6 * inv) + 128.f * (pl7 * inv);
}
cudaError_t launch_soft_table(const uint8_t *rom_blob, const RomMeta *meta, int n_roms, const float *w, int K, float *tab, cudaStream_t stream) {
  soft_table_kernel<<<dim3(32768 / 256, n_roms), 256, 0, stream>>>(rom_blob, meta, w, K, tab);
  return cudaGetLastError();
}

// Per decode entry of the soft table: what fetching that instruction's own bytes adds to the soft sums (each byte is a
// value read of the ROM tensor: eq. (10) from W(T) x ROM, then STE + round) — {sum, count, max |soft - hard|, mismatches}.
// One-byte instructions and BRK read their second byte as a discarded cycle; an absolute load folded into an immediate
// also reads its ROM operand; entries decoded at run time fetch (and note) their bytes themselves.
__global__ void soft_entry_kernel(const uint8_t *rom_blob, const RomMeta *meta, const uint2 *drom, const float *tab, float4 *ent) {
  const RomMeta rm = meta[blockIdx.y];
  const int nb = max(1, (int)(rm.size >> 12));
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;            // bank * 4096 + o
  if (idx >= nb * 4096) return;
  const uint32_t bank = (uint32_t)idx >> 12, o = idx & 0xFFF, mask = (rm.size == 2048) ? 0x7FFu : 0xFFFu;
  const uint8_t *img = rom_blob + rm.offset + bank * 4096;
  const float *t = tab + rm.pad + bank * 4096;
  const uint2 e = drom[rm.doff + idx];
  const uint32_t cls = e.x & 0x7Fu, len = (e.x >> DW_LEN_SHIFT) & 0xFFu;
  float4 r = make_float4(0.f, 0.f, 0.f, 0.f);
  auto add = [&](uint32_t off) { const float sv = t[off & 0xFFFu], h = (float)img[off & mask];
                                 r.x += sv; r.y += 1.f; r.z = fmaxf(r.z, fabsf(sv - h)); if (rintf(sv + (h - sv)) != h) r.w += 1.f; };
  if (cls != HC_COLD + H_SLOW) {
    const uint32_t n = (cls == HC_COLD + H_ILL) ? 1u : (cls == HC_COLD + H_BRK) ? 1u : len;
    for (uint32_t i = 0; i < n; ++i) add(o + i);
    if ((cls == HC_LD_IMM || cls == HC_ALU_IMM) && len == 3u) add((uint32_t)img[(o + 1) & mask] | ((uint32_t)img[(o + 2) & mask] << 8));   // folded ROM operand
  }
  ent[rm.doff + idx] = r;
}
cudaError_t launch_soft_entries(const uint8_t *rom_blob, const RomMeta *meta, int n_roms, const uint2 *drom, const float *tab, float4 *ent, cudaStream_t stream) {
  soft_entry_kernel<<<dim3(32768 / 256, n_roms), 256, 0, stream>>>(rom_blob, meta, drom, tab, ent);
  return cudaGetLastError();
}

// Block placement.  All blocks of a step are resident at once (one wave), two 256-env blocks per SM at most, and 256
// blocks on 148 SMs leave 108 SMs with two blocks and 40 with one; a block is a ROM's envs, and ROMs differ in work per
// frame, so with blocks placed in env order the step waits for the unluckiest SM (measured: slowest SM 9.3 ms, mean
// 7.4 ms).  Every plain vcs_step records when and on which SM each block ran; from that, this kernel estimates each
// group's stand-alone time W (a block that shares its SM runs A = 1.27x slower while its partner is still there:
// measured 6.3 -> 7.9 ms on 4K carts, 7.4 -> 9.6 ms on F8 carts) and re-assigns groups to block indices for the next
// launches — the hardware places block indices on SMs the same way every launch: the heaviest groups get the SMs that
// hold one block, the others are paired heaviest with lightest.  Results do not depend on the placement (envs are
// independent); only the step time does.  n <= 1024 blocks; with more than two blocks per SM: longest first (below).
__global__ void rebalance_kernel(int32_t *perm, const unsigned long long *blk, int n, float A, float *w_avg) {
  __shared__ float W[1024]; __shared__ int partner[1024]; __shared__ int grp[1024]; __shared__ int slot_of_rank[1024];
  __shared__ int bad, n_single, crowded;
  if (threadIdx.x == 0) { bad = 0; n_single = 0; crowded = 0; }
  __syncthreads();
  for (int s = threadIdx.x; s < n; s += blockDim.x) {
    grp[s] = perm[s];
    const unsigned long long sm = blk[3 * s + 2];
    int p = -1, cnt = 0;
    for (int j = 0; j < n; ++j) if (j != s && blk[3 * j + 2] == sm) { p = j; ++cnt; }
    partner[s] = p;
    if (blk[3 * s + 1] <= blk[3 * s]) bad = 1;                        // no measurement
    else if (cnt > 1) atomicOr(&crowded, 1);                          // more than two blocks ran on that SM
  }
  __syncthreads();
  if (bad) return;
  if (crowded) {
    __shared__ unsigned long long t_first, t_last, d_max;
    if (threadIdx.x == 0) { t_first = ~0ull; t_last = 0; d_max = 0; }
    __syncthreads();
    for (int s = threadIdx.x; s < n; s += blockDim.x) {
      atomicMin(&t_first, blk[3 * s]); atomicMax(&t_last, blk[3 * s]); atomicMax(&d_max, blk[3 * s + 1] - blk[3 * s]);
    }
    __syncthreads();
    if (t_last - t_first < d_max / 4) return;             // one wave of small blocks: every block started at once, leave it alone
    // More blocks than the SMs hold at once (batches beyond one wave) or small blocks: the hardware hands out block
    // indices in order as SMs free up, so run the longest blocks first and let the short ones fill the tail.
    for (int s = threadIdx.x; s < n; s += blockDim.x) {
      float &avg = w_avg[grp[s]];
      const float d = (float)(blk[3 * s + 1] - blk[3 * s]);
      W[s] = avg = (avg > 0.f) ? 0.7f * avg + 0.3f * d : d;
    }
    __syncthreads();
    for (int s = threadIdx.x; s < n; s += blockDim.x) {
      int r = 0; const float w = W[s];
      for (int j = 0; j < n; ++j) r += (W[j] > w || (W[j] == w && j < s)) ? 1 : 0;
      perm[r] = grp[s];
    }
    return;
  }
  for (int s = threadIdx.x; s < n; s += blockDim.x) {                  // stand-alone time of the group in slot s
    const float d = (float)(blk[3 * s + 1] - blk[3 * s]);
    const int p = partner[s];
    if (p < 0) W[s] = d;
    else {
      const float dp = (float)(blk[3 * p + 1] - blk[3 * p]);
      const bool lighter = d < dp || (d == dp && s < p);
      W[s] = lighter ? d / A : d - (A - 1.f) * (dp / A);
    }
    float &avg = w_avg[grp[s]];                                        // per group, smoothed over the steps measured so far:
    W[s] = avg = (avg > 0.f) ? 0.7f * avg + 0.3f * W[s] : W[s];        // one step's inputs move a ROM's time by a few per cent
  }
  __syncthreads();
  // slots in placement order: single-SM slots first, then the pairs (first slot = lower index)
  for (int s = threadIdx.x; s < n; s += blockDim.x) {
    if (partner[s] < 0) { int r = 0; for (int j = 0; j < s; ++j) r += partner[j] < 0; slot_of_rank[r] = s; atomicAdd(&n_single, 1); }
  }
  __syncthreads();
  const int ns = n_single, np = (n - ns) / 2;
  for (int s = threadIdx.x; s < n; s += blockDim.x) {
    const int p = partner[s];
    if (p > s) { int r = 0; for (int j = 0; j < s; ++j) r += partner[j] > j; slot_of_rank[ns + r] = s; slot_of_rank[ns + 2 * np - 1 - r] = p; }
  }
  __syncthreads();
  for (int s = threadIdx.x; s < n; s += blockDim.x) {                  // rank of the group in slot s by W, heaviest first
    int r = 0; const float w = W[s];
    for (int j = 0; j < n; ++j) r += (W[j] > w || (W[j] == w && j < s)) ? 1 : 0;
    perm[slot_of_rank[r]] = grp[s];       // ranks 0..ns-1: alone; rank ns+q pairs with rank ns+2np-1-q
  }
}
cudaError_t launch_rebalance(int32_t *perm, const unsigned long long *blk_time, int n, float slowdown, float *w_avg, cudaStream_t stream) {
  if (n < 2 || n > 1024) return cudaSuccess;
  rebalance_kernel<<<1, 256, 0, stream>>>(perm, blk_time, n, slowdown, w_avg);
  return cudaGetLastError();
}

size_t step_smem_bytes(int block, bool roms, uint32_t max_rom, bool soft) {
  return (size_t)(S_WORDS * block + C_WORDS) * 4 + (roms ? (max_rom < 4096 ? 4096 : max_rom) + 16 : 0) + (soft ? (size_t)8 * block * 4 : 0);
}

template <int BLOCK, int ROMS, int THREADS, bool SOFT, bool COUNT = false>
static cudaError_t launch_one(const StepParams &p, cudaStream_t stream) {
  const size_t smem_bytes = step_smem_bytes(BLOCK, ROMS == 1, p.max_rom, SOFT);
  static size_t configured[64] = {0};                   // per device: the attribute belongs to the (function, device) pair
  int dev = 0; cudaGetDevice(&dev);
  if (dev < 0 || dev >= 64 || configured[dev] < smem_bytes) {
    cudaError_t e = cudaFuncSetAttribute(vcs_step_kernel<BLOCK, ROMS, THREADS, SOFT, COUNT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes);
    if (e != cudaSuccess) return e;
    if (dev >= 0 && dev < 64) configured[dev] = smem_bytes;
  }
  const int grid = (p.batch + BLOCK - 1) / BLOCK;
  vcs_step_kernel<BLOCK, ROMS, THREADS, SOFT, COUNT><<<grid, THREADS, smem_bytes, stream>>>(p);
  return cudaGetLastError();
}

cudaError_t launch_step(const StepParams &p, cudaStream_t stream) {
  if (p.n_instr > 0 && p.soft_out)                         // vcs_step_instructions_soft (SOFT-STE or FULL, per instruction)
    return launch_one<128, 0, 128, true, true>(p, stream);
  if (p.n_instr > 0)                                       // vcs_step_instructions: one variant (128 envs per block, ROM through the read-only path)
    return launch_one<128, 0, 128, false, true>(p, stream);
  if (p.soft_out)                                          // SOFT-STE mode: one variant (ROM through the read-only path, no regroup)
    return launch_one<128, 0, 128, true>(p, stream);
  if (p.rom_smem && !p.rom_staged)                         // one ROM per block, 16 / 32 KB images: read through the read-only path (ROMS = 2); they are
    switch (p.block) { case 64: return launch_one<64, 2, 96, false>(p, stream); case 256: return launch_one<256, 2, 288, false>(p, stream); default: return launch_one<128, 2, 160, false>(p, stream); }   // banked: spare warp
  if (p.rom_smem && p.regroup && p.banked) {               // F8 carts present: one spare warp per block for the regroup
    switch (p.block) { case 64: return launch_one<64, 1, 96, false>(p, stream); case 256: return launch_one<256, 1, 288, false>(p, stream); default: return launch_one<128, 1, 160, false>(p, stream); }
  }
  if (p.rom_smem) {
    switch (p.block) { case 64: return launch_one<64, 1, 64, false>(p, stream); case 256: return launch_one<256, 1, 256, false>(p, stream); default: return launch_one<128, 1, 128, false>(p, stream); }
  }
  switch (p.block) { case 64: return launch_one<64, 0, 64, false>(p, stream); case 256: return launch_one<256, 0, 256, false>(p, stream); default: return launch_one<128, 0, 128, false>(p, stream); }
}

}  // namespace vcs
