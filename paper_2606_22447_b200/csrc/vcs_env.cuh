// vcs_env.cuh — one environment's live state inside the interpreter kernel, with the lazy TIA and the
// closed-form RIOT timer.  Everything here is force-inlined into the single persistent step kernel and
// lives in registers; RAM and the scanline buffer live in shared memory (word-interleaved per thread, so
// a warp's accesses never bank-conflict whatever addresses its lanes use).
//
// Lazy TIA (SURVEY.md §0.3, §8(a) a10–a12): instead of rendering 3 colour clocks per CPU cycle, the
// kernel keeps `rx` = colour clocks of the current line already rendered and catches up only when a TIA
// register is written, a collision latch is read, a line ends or a frame ends.  A segment is rendered
// 32 pixels at a time from bit masks of the six objects (PF, BL, P0, P1, M0, M1).  Pixel bytes are only
// produced during the last frame of a step; collision latches always.
#pragma once
#include "vcs_state.cuh"

namespace vcs {

#define DEV __device__ __forceinline__

DEV uint32_t bfe(uint32_t v, int pos, int len) { return (v >> pos) & ((1u << len) - 1u); }
DEV uint32_t byte_of(uint32_t w, int i) { return (w >> (8 * i)) & 0xFFu; }
DEV uint32_t set_byte(uint32_t w, int i, uint32_t v) { return (w & ~(0xFFu << (8 * i))) | ((v & 0xFFu) << (8 * i)); }
DEV uint32_t brev8(uint32_t v) { return __brev(v) >> 24; }
// each of the low 8 bits -> 4 consecutive bits
DEV uint32_t expand4(uint32_t b) {
  uint32_t x = b & 0xFFu;
  x = (x | (x << 12)) & 0x000F000Fu;
  x = (x | (x << 6)) & 0x03030303u;
  x = (x | (x << 3)) & 0x11111111u;
  return x * 15u;
}
// each of the low 8 bits -> 2 consecutive bits
DEV uint32_t expand2(uint32_t b) {
  uint32_t x = b & 0xFFu;
  x = (x | (x << 4)) & 0x0F0Fu;
  x = (x | (x << 2)) & 0x3333u;
  x = (x | (x << 1)) & 0x5555u;
  return x * 3u;
}
// 4 mask bits -> 4 byte masks (0x00 / 0xFF)
DEV uint32_t nib_to_bytes(uint32_t nib) { return (((nib & 0xFu) * 0x00204081u) & 0x01010101u) * 0xFFu; }
DEV uint32_t rep4(uint32_t c) { return (c & 0xFFu) * 0x01010101u; }

template <int BLOCK>
struct Env {
  // ---- CPU
  uint32_t A, X, Y, SP, PC;
  uint32_t fC, fV, fD, fI, zv, nv;     // Z <=> (zv & 0xFF) == 0 ; N <=> nv & 0x80
  uint32_t status;
  // ---- beam / time (cycle counts are relative to the start of this vcs_step call)
  int32_t cyc;        // CPU cycles executed in this step
  int32_t n;          // cycle-in-line of `cyc` (0..75; transiently negative inside an instruction
                      // whose early accesses already crossed into the next line)
  uint32_t line, frame;
  int32_t fstart;     // value of `cyc` at which the current frame began (frame_cyc = cyc - fstart)
  int32_t frames_done, frameskip;
  bool storing;       // pixels of the frame in progress go to the screen
  // ---- RIOT
  uint32_t timer, sub, shift, tflag; int32_t tticks;   // timer state after `tticks` cycles of this step
  uint32_t ports;     // ora | ddra<<8 | orb<<16 | ddrb<<24
  uint32_t ina, fire0;
  // ---- TIA
  uint32_t colu, pf, grp, nusiz, pos, pos2, fl, cx;
  uint32_t rx;        // colour clocks of the current line already rendered
  // ---- cart
  const uint8_t *rom; uint32_t rom_mask, is_f8, bank;
  // ---- memory
  uint8_t *ram;       // this thread's slice base in shared memory (byte pointer, word-interleaved)
  uint32_t *lbuf;     // this thread's scanline buffer (40 words, stride BLOCK)
  uint8_t *screen;    // this env's front screen in HBM
  int32_t y0, cap;

  // ------------------------------------------------------------------ RAM (smem, conflict-free)
  DEV uint32_t ram_rd(uint32_t a) const { return ram[((a & 0x7Cu) * BLOCK) | (a & 3u)]; }
  DEV void ram_wr(uint32_t a, uint32_t v) { ram[((a & 0x7Cu) * BLOCK) | (a & 3u)] = (uint8_t)v; }

  // ------------------------------------------------------------------ ROM
  DEV uint32_t rom_rd(uint32_t a) {            // a = addr & 0x1FFF with A12 set
    if (is_f8 && (a | 1u) == 0x1FF9u) bank = a & 1u;
    return __ldg(rom + (bank << 12) + (a & rom_mask));
  }
  DEV void hotspot(uint32_t a) { if (is_f8 && (a | 1u) == 0x1FF9u) bank = a & 1u; }

  // ------------------------------------------------------------------ RIOT timer, closed form (C.7)
  // advance the (timer, sub, tflag) state to "after `ticks` cycles of this step"
  DEV void timer_sync(int32_t ticks) {
    uint32_t d = (uint32_t)(ticks - tticks);
    if ((int32_t)d <= 0) return;
    tticks = ticks;
    uint32_t mask = (1u << shift) - 1u;
    if (tflag) { timer = (timer - d) & 0xFFu; sub = (sub + d) & mask; return; }
    uint32_t k = (sub + d) >> shift;                  // prescaler wraps (decrement events) in d ticks
    if (k <= timer) { timer -= k; }
    else {                                            // event number timer+1 is the underflow
      uint32_t iu = ((timer + 1u) << shift) - sub;    // tick index (1-based) of the underflow
      timer = (0xFFu - (d - iu)) & 0xFFu; tflag = 1;
    }
    sub = (sub + d) & mask;
  }
  DEV uint32_t riot_read(uint32_t a, int32_t c) {     // access in cycle index c (tick c happened first)
    if ((a & 4u) == 0) {
      uint32_t ora = byte_of(ports, 0), ddra = byte_of(ports, 1), orb = byte_of(ports, 2), ddrb = byte_of(ports, 3);
      switch (a & 3u) {
        case 0: return (ora & ddra) | (ina & ~ddra & 0xFFu);
        case 1: return ddra;
        case 2: return (orb & ddrb) | (0x3Fu & ~ddrb);
        default: return ddrb;
      }
    }
    timer_sync(c + 1);
    if ((a & 5u) == 4u) { tflag = 0; return timer; }   // INTIM
    return tflag << 7;                                  // TIMINT
  }
  DEV void riot_write(uint32_t a, uint32_t v, int32_t c) {
    if ((a & 4u) == 0) { ports = set_byte(ports, a & 3u, v); return; }
    if ((a & 0x14u) == 0x14u) {
      uint32_t k = a & 3u;
      shift = (k == 0) ? 0u : (k == 1) ? 3u : (k == 2) ? 6u : 10u;
      timer = v & 0xFFu; sub = (1u << shift) - 1u; tflag = 0; tticks = c + 1;
    }
  }

  // ------------------------------------------------------------------ TIA object masks for one 32-px word
  // place a pattern that starts at pixel c (0..159) into the word covering pixels [32w, 32w+32)
  DEV uint32_t place(uint32_t pat, uint32_t c, int w) const {
    int r = (int)c - 32 * w; if (r < 0) r += 160;
    return (r < 32) ? (pat << r) : (r > 128) ? (pat >> (160 - r)) : 0u;
  }
  DEV uint32_t copies(uint32_t pat, uint32_t p, uint32_t m, bool fresh, int w) const {
    // copy offsets O(m): {0:[0],1:[0,16],2:[0,32],3:[0,16,32],4:[0,64],5:[0],6:[0,32,64],7:[0]}
    uint32_t o1 = (uint32_t)(0x0020004010201000ull >> (8 * m)) & 0xFFu;   // second copy offset (0 = none)
    uint32_t o2 = (m == 3) ? 32u : (m == 6) ? 64u : 0u;
    uint32_t r = fresh ? 0u : place(pat, p, w);
    if (o1) { uint32_t c = p + o1; if (c >= 160) c -= 160; r |= place(pat, c, w); }
    if (o2) { uint32_t c = p + o2; if (c >= 160) c -= 160; r |= place(pat, c, w); }
    return r;
  }
  DEV uint32_t player_word(int p, int w) const {
    uint32_t g = byte_of(grp, 2 * p + ((fl & (p ? TF_VDELP1 : TF_VDELP0)) ? 1 : 0));
    if (g == 0) return 0;
    uint32_t m = byte_of(nusiz, p) & 7u;
    uint32_t gg = (fl & (p ? TF_REFP1 : TF_REFP0)) ? g : brev8(g);      // bit d = pixel d of the sprite
    uint32_t pat = (m == 5) ? expand2(gg) : (m == 7) ? expand4(gg) : gg;
    return copies(pat, byte_of(pos, p), m, fl & (p ? TF_FRESH_P1 : TF_FRESH_P0), w);
  }
  DEV uint32_t missile_word(int p, int w) const {
    if (!(fl & (p ? TF_ENAM1 : TF_ENAM0)) || (fl & (p ? TF_RESMP1 : TF_RESMP0))) return 0;
    uint32_t ns = byte_of(nusiz, p);
    uint32_t pat = (1u << (1u << ((ns >> 4) & 3u))) - 1u;
    return copies(pat, byte_of(pos, 2 + p), ns & 7u, fl & (p ? TF_FRESH_M1 : TF_FRESH_M0), w);
  }
  DEV uint32_t ball_word(int w) const {
    if (!(fl & ((fl & TF_VDELBL) ? TF_ENABL_OLD : TF_ENABL_NEW))) return 0;
    uint32_t pat = (1u << (1u << ((byte_of(pf, 3) >> 4) & 3u))) - 1u;
    return place(pat, byte_of(pos2, 0), w);
  }
  DEV uint32_t pf_word(int w) const {
    uint32_t pf20 = (byte_of(pf, 0) >> 4) | (brev8(byte_of(pf, 1)) << 4) | (byte_of(pf, 2) << 12);
    if (pf20 == 0) return 0;
    uint32_t right = (byte_of(pf, 3) & 1u) ? (__brev(pf20) >> 12) : pf20;
    unsigned long long p40 = (unsigned long long)pf20 | ((unsigned long long)right << 20);
    return expand4((uint32_t)(p40 >> (8 * w)));
  }

  // render visible pixels [x0, x1) of the current line with the registers in force (C.8 pixel function)
  DEV void render_visible(int x0, int x1) {
    const bool store = storing && (int)line >= y0 && (int)line < y0 + SCR_H;
    if (fl & TF_VBLANK) {
      if (store) fill_zero(x0, x1);
      return;
    }
    const uint32_t ctrl = byte_of(pf, 3);
    for (int w = x0 >> 5; w <= (x1 - 1) >> 5; ++w) {
      int lo = max(x0 - 32 * w, 0), hi = min(x1 - 32 * w, 32);
      uint32_t rm = (hi >= 32 ? 0xFFFFFFFFu : ((1u << hi) - 1u)) & ~((1u << lo) - 1u);
      uint32_t act = rm;
      if ((fl & TF_HMBLANK) && w == 0) act &= ~0xFFu;            // HMOVE comb: x 0..7 black, no collisions
      uint32_t PF = pf_word(w) & act, BL = ball_word(w) & act;
      uint32_t P0 = player_word(0, w) & act, P1 = player_word(1, w) & act;
      uint32_t M0 = missile_word(0, w) & act, M1 = missile_word(1, w) & act;
      uint32_t c = 0;
      if (M0) { c |= (M0 & P1 ? 1u << CX_M0P1 : 0) | (M0 & P0 ? 1u << CX_M0P0 : 0) | (M0 & PF ? 1u << CX_M0PF : 0) |
                     (M0 & BL ? 1u << CX_M0BL : 0) | (M0 & M1 ? 1u << CX_M0M1 : 0); }
      if (M1) { c |= (M1 & P0 ? 1u << CX_M1P0 : 0) | (M1 & P1 ? 1u << CX_M1P1 : 0) | (M1 & PF ? 1u << CX_M1PF : 0) |
                     (M1 & BL ? 1u << CX_M1BL : 0); }
      if (P0) { c |= (P0 & PF ? 1u << CX_P0PF : 0) | (P0 & BL ? 1u << CX_P0BL : 0) | (P0 & P1 ? 1u << CX_P0P1 : 0); }
      if (P1) { c |= (P1 & PF ? 1u << CX_P1PF : 0) | (P1 & BL ? 1u << CX_P1BL : 0); }
      if (BL & PF) c |= 1u << CX_BLPF;
      cx |= c;
      if (!store) continue;
      // priority -> four disjoint masks (C.8 colour rule)
      uint32_t e0, e1, ef;
      uint32_t o0 = P0 | M0, o1 = P1 | M1, of = PF | BL;
      if (ctrl & 4u) { ef = of; e0 = o0 & ~ef; e1 = o1 & ~(ef | e0); }                // PFP (SCORE ignored)
      else {
        if (ctrl & 2u) {                                                               // SCORE
          uint32_t left = (w < 2) ? 0xFFFFFFFFu : (w == 2) ? 0x0000FFFFu : 0u;         // x < 80
          o0 |= PF & left; o1 |= PF & ~left;
        }
        e0 = o0; e1 = o1 & ~e0; ef = of & ~(e0 | e1);
      }
      uint32_t eb = act & ~(e0 | e1 | ef);
      uint32_t c0 = rep4(byte_of(colu, 0)), c1 = rep4(byte_of(colu, 1)), cf = rep4(byte_of(colu, 2)), cb = rep4(byte_of(colu, 3));
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        uint32_t nib = (rm >> (4 * j)) & 0xFu;
        if (nib == 0) continue;
        uint32_t px = (c0 & nib_to_bytes(e0 >> (4 * j))) | (c1 & nib_to_bytes(e1 >> (4 * j))) |
                      (cf & nib_to_bytes(ef >> (4 * j))) | (cb & nib_to_bytes(eb >> (4 * j)));
        uint32_t bm = nib_to_bytes(nib);
        uint32_t *dst = lbuf + (8 * w + j) * BLOCK;
        *dst = (*dst & ~bm) | (px & bm);
      }
    }
  }
  DEV void fill_zero(int x0, int x1) {                 // zero pixels [x0,x1) of the scanline buffer
    for (int q = x0 >> 2; q <= (x1 - 1) >> 2; ++q) {
      int lo = max(x0 - 4 * q, 0), hi = min(x1 - 4 * q, 4);
      uint32_t bm = (hi >= 4 ? 0xFFFFFFFFu : ((1u << (8 * hi)) - 1u)) & ~((1u << (8 * lo)) - 1u);
      lbuf[q * BLOCK] &= ~bm;
    }
  }
  // catch the beam up to colour clock `clk` (0..228) of the current line
  DEV void render_to(uint32_t clk) {
    if (clk <= rx) return;
    int x0 = (int)max(rx, (uint32_t)HBLANK) - HBLANK, x1 = (int)max(clk, (uint32_t)HBLANK) - HBLANK;
    rx = clk;
    if (x1 > x0) render_visible(x0, x1);
  }
  DEV void flush_row() {                                // scanline buffer -> screen row (16-byte stores)
    int r = (int)line - y0;
    if (!storing || r < 0 || r >= SCR_H) return;
    uint4 *dst = reinterpret_cast<uint4 *>(screen + r * SCR_W);
#pragma unroll
    for (int q = 0; q < 10; ++q)
      dst[q] = make_uint4(lbuf[(4 * q) * BLOCK], lbuf[(4 * q + 1) * BLOCK], lbuf[(4 * q + 2) * BLOCK], lbuf[(4 * q + 3) * BLOCK]);
  }
  // the scanline in progress ends: finish it, store it, start the next one (C.4 new-line bookkeeping)
  DEV void new_line() {
    render_to(LINE_CLK);
    flush_row();
    line++; rx = 0; n -= LINE_CYC;
    fl &= ~(TF_WSYNC | TF_HMBLANK | TF_FRESH_ALL);
  }
  // C.10 frame end at colour clock `clk` of the current line; `next_cyc` = first cycle of the new frame
  DEV void frame_end(uint32_t clk, int32_t next_cyc) {
    render_to(clk);
    if (storing) {
      int r = (int)line - y0;
      if (r >= 0 && r < SCR_H) {
        int x = (int)max(clk, (uint32_t)HBLANK) - HBLANK;
        if (x < SCR_W) fill_zero(x, SCR_W);
        flush_row();
      }
      const uint4 z = make_uint4(0, 0, 0, 0);            // rows the beam never reached in this frame
      for (int rr = max(r + 1, 0); rr < SCR_H; ++rr) {
        uint4 *dst = reinterpret_cast<uint4 *>(screen + rr * SCR_W);
#pragma unroll
        for (int q = 0; q < 10; ++q) dst[q] = z;
      }
    }
    frames_done++; frame++; line = 0; fstart = next_cyc;
    storing = (frames_done == frameskip - 1);
  }

  // ------------------------------------------------------------------ TIA bus access (C.8)
  // m = cycle-in-line of the access (may be >= 76 when the instruction ran over the line end)
  DEV int32_t tia_catch_up(int32_t m) {
    while (m >= LINE_CYC) { new_line(); m -= LINE_CYC; }
    render_to(3u * (uint32_t)(m + 1));
    return m;
  }
  DEV uint32_t tia_read(uint32_t a, int32_t m) {
    uint32_t r = a & 0xFu;
    if (r < 8) {
      tia_catch_up(m);
      uint32_t b7, b6;
      switch (r) {
        case 0: b7 = cx >> CX_M0P1; b6 = cx >> CX_M0P0; break;
        case 1: b7 = cx >> CX_M1P0; b6 = cx >> CX_M1P1; break;
        case 2: b7 = cx >> CX_P0PF; b6 = cx >> CX_P0BL; break;
        case 3: b7 = cx >> CX_P1PF; b6 = cx >> CX_P1BL; break;
        case 4: b7 = cx >> CX_M0PF; b6 = cx >> CX_M0BL; break;
        case 5: b7 = cx >> CX_M1PF; b6 = cx >> CX_M1BL; break;
        case 6: b7 = cx >> CX_BLPF; b6 = 0; break;
        default: b7 = cx >> CX_P0P1; b6 = cx >> CX_M0M1; break;
      }
      return ((b7 & 1u) << 7) | ((b6 & 1u) << 6);
    }
    if (r == 0xC) { bool lat = (fl & TF_LATCHEN) ? (fl & TF_INPT4_LATCH) != 0 : true; return (!fire0 && lat) ? 0x80u : 0u; }
    if (r == 0xD) { bool lat = (fl & TF_LATCHEN) ? (fl & TF_INPT5_LATCH) != 0 : true; return lat ? 0x80u : 0u; }
    return 0;
  }
  DEV void set_flag(uint32_t bit, bool on) { fl = on ? (fl | bit) : (fl & ~bit); }
  DEV void eval_fire_latch() { if ((fl & TF_LATCHEN) && fire0) fl &= ~TF_INPT4_LATCH; }
  // c = cycle index of the write within this step, m = its cycle-in-line
  DEV void tia_write(uint32_t a, uint32_t v, int32_t c, int32_t m) {
    uint32_t r = a & 0x3Fu;
    if (r > 0x2C || (r >= 0x15 && r <= 0x1A) || r == 0x03) return;      // no effect (audio: PAPER.md L205)
    m = tia_catch_up(m);
    int x_now = 3 * (m + 1) - HBLANK;
    switch (r) {
      case 0x00: { bool nv2 = (v >> 1) & 1u;
                   if ((fl & TF_VSYNC) && !nv2) frame_end(3u * (uint32_t)(m + 1), c + 1);
                   set_flag(TF_VSYNC, nv2); } break;
      case 0x01: set_flag(TF_VBLANK, (v >> 1) & 1u); set_flag(TF_LATCHEN, (v >> 6) & 1u);
                 if (!(fl & TF_LATCHEN)) fl |= TF_INPT4_LATCH | TF_INPT5_LATCH;
                 eval_fire_latch(); break;
      case 0x02: fl |= TF_WSYNC; break;
      case 0x04: nusiz = set_byte(nusiz, 0, v & 0x37u); break;
      case 0x05: nusiz = set_byte(nusiz, 1, v & 0x37u); break;
      case 0x06: case 0x07: case 0x08: case 0x09: colu = set_byte(colu, r - 6, v & 0xFEu); break;
      case 0x0A: pf = set_byte(pf, 3, v & 0x37u); break;
      case 0x0B: set_flag(TF_REFP0, (v >> 3) & 1u); break;
      case 0x0C: set_flag(TF_REFP1, (v >> 3) & 1u); break;
      case 0x0D: pf = set_byte(pf, 0, v & 0xF0u); break;
      case 0x0E: pf = set_byte(pf, 1, v); break;
      case 0x0F: pf = set_byte(pf, 2, v); break;
      case 0x10: case 0x11: pos = set_byte(pos, r - 0x10, x_now < 0 ? 3 : (x_now + 5) % 160);
                 fl |= (r == 0x10) ? TF_FRESH_P0 : TF_FRESH_P1; break;
      case 0x12: case 0x13: pos = set_byte(pos, r - 0x10, x_now < 0 ? 2 : (x_now + 4) % 160);
                 fl |= (r == 0x12) ? TF_FRESH_M0 : TF_FRESH_M1; break;
      case 0x14: pos2 = set_byte(pos2, 0, x_now < 0 ? 2 : (x_now + 4) % 160); break;
      case 0x1B: grp = set_byte(set_byte(grp, 0, v), 3, byte_of(grp, 2)); break;               // GRP0; GRP1_old := GRP1_new
      case 0x1C: grp = set_byte(set_byte(grp, 2, v), 1, byte_of(grp, 0));                      // GRP1; GRP0_old := GRP0_new
                 set_flag(TF_ENABL_OLD, fl & TF_ENABL_NEW); break;
      case 0x1D: set_flag(TF_ENAM0, (v >> 1) & 1u); break;
      case 0x1E: set_flag(TF_ENAM1, (v >> 1) & 1u); break;
      case 0x1F: set_flag(TF_ENABL_NEW, (v >> 1) & 1u); break;
      case 0x20: case 0x21: case 0x22: case 0x23: { int sh = 16 + 4 * (r - 0x20); nusiz = (nusiz & ~(0xFu << sh)) | ((v >> 4) << sh); } break;
      case 0x24: pos2 = set_byte(pos2, 1, v >> 4); break;
      case 0x25: set_flag(TF_VDELP0, v & 1u); break;
      case 0x26: set_flag(TF_VDELP1, v & 1u); break;
      case 0x27: set_flag(TF_VDELBL, v & 1u); break;
      case 0x28: case 0x29: { int p = r - 0x28; uint32_t bit = p ? TF_RESMP1 : TF_RESMP0; bool nv2 = (v >> 1) & 1u;
                 if ((fl & bit) && !nv2) {
                   uint32_t mm = byte_of(nusiz, p) & 7u, mid = (mm == 5) ? 8u : (mm == 7) ? 16u : 4u;
                   pos = set_byte(pos, 2 + p, (byte_of(pos, p) + mid) % 160u);
                 }
                 set_flag(bit, nv2); } break;
      case 0x2A: {                                                                              // HMOVE
#pragma unroll
                 for (int k = 0; k < 5; ++k) {
                   uint32_t h = (k < 4) ? (nusiz >> (16 + 4 * k)) & 0xFu : byte_of(pos2, 1) & 0xFu;
                   int s = (h < 8) ? (int)h : (int)h - 16;
                   int p = (int)((k < 4) ? byte_of(pos, k) : byte_of(pos2, 0)) - s;
                   if (p < 0) p += 160; if (p >= 160) p -= 160;
                   if (k < 4) pos = set_byte(pos, k, p); else pos2 = set_byte(pos2, 0, p);
                 }
                 if (x_now < 0) fl |= TF_HMBLANK; } break;
      case 0x2B: nusiz &= 0x0000FFFFu; pos2 = set_byte(pos2, 1, 0); break;                    // HMCLR
      case 0x2C: cx = 0; break;                                                                 // CXCLR
      default: break;
    }
  }
};

}  // namespace vcs
