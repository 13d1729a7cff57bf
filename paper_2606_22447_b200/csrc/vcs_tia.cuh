// vcs_tia.cuh — the lazy TIA of the interpreter kernel (SURVEY.md §0.3, §8(a) a10–a12, a14; machine model C.8).
//
// All TIA state of an environment lives in that thread's shared-memory file (vcs_state.cuh, S_*), so the
// functions below are plain out-of-line device functions (one copy each in the kernel image: the
// interpreter is instruction-cache bound) that need no per-call state in registers.
//
// Instead of rendering 3 colour clocks per CPU cycle the kernel keeps S_RX = colour clocks of the current
// line already rendered and catches up only when a TIA register is written, a collision latch is read, a
// line ends or a frame ends.  A catch-up works on bit masks:
//   * each of the six objects (PF, BL, P0, P1, M0, M1) has a cached 160-bit line mask (5 words) that is
//     rebuilt lazily, only after a write that changes that object (TF_DIRTY*);
//   * a segment [x0,x1) is 1..5 word visits: 6 mask loads, 15 AND/OR accumulations for the collision
//     latches and, in the one frame of a step whose pixels are kept, the priority rule evaluated on whole
//     words into two colour-index bit planes;
//   * bytes are produced only when a scanline is complete (or a colour register / VBLANK changes mid-line):
//     8 pixels per byte-permute pair from the planes and the four colour registers, written straight to
//     the row in HBM with 16-byte stores.
#pragma once
#include "vcs_state.cuh"

namespace vcs {

#define DEV __device__ __forceinline__
#define DEVNI __device__ __noinline__

extern __shared__ __align__(128) uint32_t smem[];

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
// bit k of the low 8 bits -> bit 4k
DEV uint32_t spread8(uint32_t b) {
  uint32_t x = b & 0xFFu;
  x = (x | (x << 12)) & 0x000F000Fu;
  x = (x | (x << 6)) & 0x03030303u;
  x = (x | (x << 3)) & 0x11111111u;
  return x;
}

enum : uint32_t { EV_FRAME = 1u, EV_WSYNC = 2u, EV_CROSS = 16u };   // EV_CROSS * (line ends performed)

// 16 bytes of a screen row -> HBM: one st.global.v4 (SASS STG.E.128), streaming (.cs: the kernel never reads a row
// back and a step's 2.2 GB of rows would only evict what it does re-use from L2).  Rows are 160 B = 10 such stores;
// 33,600 B per env and 160 B per row keep every row 16-byte aligned (the screen base comes from cudaMalloc).
DEV void st_row16(uint4 *p, uint4 v) {
  asm volatile("st.global.cs.v4.b32 [%0], {%1, %2, %3, %4};" ::"l"(__cvta_generic_to_global(p)), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

// ---- descriptors of the plain VALUE registers (SURVEY C.8 write effects that are "store a masked field"): the write
// path handles them with one piece of code instead of one switch case each (the hot code must stay small: icache).
//   bits 2:0 kind (0 special, 1 field store into a packed word, 2 flag) ; 5:3 word - S_COLU ; 10:6 bit shift of the
//   field (kind 2: flag bit number) ; 18:11 value mask ; 21:19 right shift applied to the written value first ;
//   27:22 objects whose line mask the register feeds ; 28 lazy (no catch-up outside kept rows) ; 29 colour (the
//   pixels before the write are painted with the old value in a kept row) ; 30 the field is a nibble
constexpr uint32_t tia_field(int word, int shift, uint32_t mask, int pre, uint32_t dirty, bool lazy, bool paint, bool nib) {
  return 1u | ((uint32_t)(word - S_COLU) << 3) | ((uint32_t)shift << 6) | (mask << 11) | ((uint32_t)pre << 19) | (dirty << 22) |
         (lazy ? 1u << 28 : 0u) | (paint ? 1u << 29 : 0u) | (nib ? 1u << 30 : 0u);
}
constexpr uint32_t tia_flagd(int bit, int pre, uint32_t dirty) { return 2u | ((uint32_t)bit << 6) | ((uint32_t)pre << 19) | (dirty << 22); }
constexpr int ctz32(uint32_t v) { int n = 0; while (!(v & 1u)) { v >>= 1; ++n; } return n; }
inline void tia_desc_table(uint32_t *t) {
  for (int i = 0; i < 64; ++i) t[i] = 0;
  const uint32_t PF = 1u << OB_PF, BL = 1u << OB_BL, P0 = 1u << OB_P0, P1 = 1u << OB_P1, M0 = 1u << OB_M0, M1 = 1u << OB_M1;
  t[0x04] = tia_field(S_NUSIZ, 0, 0x37, 0, P0 | M0, false, false, false);
  t[0x05] = tia_field(S_NUSIZ, 8, 0x37, 0, P1 | M1, false, false, false);
  for (int k = 0; k < 4; ++k) t[0x06 + k] = tia_field(S_COLU, 8 * k, 0xFE, 0, 0, true, true, false);
  t[0x0A] = tia_field(S_PF, 24, 0x37, 0, PF | BL, false, false, false);
  t[0x0D] = tia_field(S_PF, 0, 0xF0, 0, PF, false, false, false);
  t[0x0E] = tia_field(S_PF, 8, 0xFF, 0, PF, false, false, false);
  t[0x0F] = tia_field(S_PF, 16, 0xFF, 0, PF, false, false, false);
  for (int k = 0; k < 4; ++k) t[0x20 + k] = tia_field(S_NUSIZ, 16 + 4 * k, 0x0F, 4, 0, true, false, true);    // HMP0 HMP1 HMM0 HMM1
  t[0x24] = tia_field(S_POS2, 8, 0x0F, 4, 0, true, false, false);                                            // HMBL
  t[0x0B] = tia_flagd(ctz32(TF_REFP0), 3, P0); t[0x0C] = tia_flagd(ctz32(TF_REFP1), 3, P1);
  t[0x1D] = tia_flagd(ctz32(TF_ENAM0), 1, M0); t[0x1E] = tia_flagd(ctz32(TF_ENAM1), 1, M1);
  t[0x1F] = tia_flagd(ctz32(TF_ENABL_NEW), 1, BL);
  t[0x25] = tia_flagd(ctz32(TF_VDELP0), 0, P0); t[0x26] = tia_flagd(ctz32(TF_VDELP1), 0, P1); t[0x27] = tia_flagd(ctz32(TF_VDELBL), 0, BL);
}
__constant__ uint32_t c_tia_desc[64];

// TAG tells copies of this code apart: the kernel's inline interpreter loop uses TAG 0, the out-of-line executors their
// own (vcs_step.cu).  Same source, same results — but ptxas hands out convergence-barrier registers over the whole call
// graph, and a hot function that is also reachable from a deeply nested rare path pays for it on every call (BMOV
// saves / restores inside render_visible & co.); with a copy per caller the hot copy is compiled for the hot path alone.
template <int BLOCK, int TAG = 0>
struct Tia {
  static DEV uint32_t &S(uint32_t sl, int i) { return smem[i * BLOCK + sl]; }
  static DEV uint32_t ctx(int i) { return smem[S_WORDS * BLOCK + i]; }
  static DEV uint8_t *row_ptr(uint32_t sl, uint32_t r) {
    unsigned long long base = (unsigned long long)ctx(C_SCREEN_LO) | ((unsigned long long)ctx(C_SCREEN_HI) << 32);
    return reinterpret_cast<uint8_t *>(base) + ((size_t)(ctx(C_ENV0) + (S(sl, S_INP) >> 16)) * SCR_H + r) * SCR_W;
  }

  // ------------------------------------------------------------------ cached object line masks
  static DEV void obj_clear(uint32_t sl, int o) {
#pragma unroll
    for (int w = 0; w < 5; ++w) S(sl, S_OBJ + 5 * o + w) = 0;
  }
  // OR a pattern (<= 32 px) whose first pixel is at c (0..159) into object o's line mask, wrapping at 160
  static DEV void obj_or(uint32_t sl, int o, uint32_t pat, uint32_t c) {
    const uint32_t q = c >> 5, s = c & 31u;
    const uint32_t lo = pat << s, hi = __funnelshift_l(pat, 0u, s);
    uint32_t *p = &smem[(S_OBJ + 5 * o) * BLOCK + sl];
    p[q * BLOCK] |= lo;
    if (hi) p[(q == 4 ? 0 : q + 1) * BLOCK] |= hi;
  }
  // copy offsets O(m): {0:[0],1:[0,16],2:[0,32],3:[0,16,32],4:[0,64],5:[0],6:[0,32,64],7:[0]} (C.8)
  static DEV void obj_copies(uint32_t sl, int o, uint32_t pat, uint32_t p, uint32_t m, bool fresh) {
    const uint32_t o1 = ((0x02041210u >> (4 * m)) & 0xFu) << 4;        // second copy offset (0 = none)
    const uint32_t o2 = (m == 3) ? 32u : (m == 6) ? 64u : 0u;
    if (!fresh) obj_or(sl, o, pat, p);
    if (o1) { uint32_t c = p + o1; if (c >= 160) c -= 160; obj_or(sl, o, pat, c); }
    if (o2) { uint32_t c = p + o2; if (c >= 160) c -= 160; obj_or(sl, o, pat, c); }
  }
  static DEVNI void rebuild_player(uint32_t sl, int p, uint32_t fl) {      // out of line, one copy: the hot code must stay small (icache)
    obj_clear(sl, OB_P0 + p);
    const uint32_t g = byte_of(S(sl, S_GRP), 2 * p + ((fl & (p ? TF_VDELP1 : TF_VDELP0)) ? 1 : 0));
    if (g == 0) return;
    const uint32_t m = byte_of(S(sl, S_NUSIZ), p) & 7u;
    const uint32_t gg = (fl & (p ? TF_REFP1 : TF_REFP0)) ? g : brev8(g);      // bit d = pixel d of the sprite
    const uint32_t pat = (m == 5) ? expand2(gg) : (m == 7) ? expand4(gg) : gg;
    obj_copies(sl, OB_P0 + p, pat, byte_of(S(sl, S_POS), p), m, fl & (p ? TF_FRESH_P1 : TF_FRESH_P0));
  }
  static DEVNI void rebuild_missile(uint32_t sl, int p, uint32_t fl) {
    obj_clear(sl, OB_M0 + p);
    if (!(fl & (p ? TF_ENAM1 : TF_ENAM0)) || (fl & (p ? TF_RESMP1 : TF_RESMP0))) return;
    const uint32_t ns = byte_of(S(sl, S_NUSIZ), p);
    const uint32_t pat = (1u << (1u << ((ns >> 4) & 3u))) - 1u;
    obj_copies(sl, OB_M0 + p, pat, byte_of(S(sl, S_POS), 2 + p), ns & 7u, fl & (p ? TF_FRESH_M1 : TF_FRESH_M0));
  }
  static DEVNI void rebuild(uint32_t sl, uint32_t fl) {
    if (fl & (TF_DIRTY0 << OB_PF)) {
      const uint32_t pf = S(sl, S_PF);
      const uint32_t pf20 = (byte_of(pf, 0) >> 4) | (brev8(byte_of(pf, 1)) << 4) | (byte_of(pf, 2) << 12);
      const uint32_t right = (pf & (1u << 24)) ? (__brev(pf20) >> 12) : pf20;      // CTRLPF.REF
      const uint32_t lo = pf20 | (right << 20), hi = right >> 12;                  // 40 playfield bits, 4 px each
      S(sl, S_OBJ + 0) = expand4(lo); S(sl, S_OBJ + 1) = expand4(lo >> 8); S(sl, S_OBJ + 2) = expand4(lo >> 16);
      S(sl, S_OBJ + 3) = expand4(lo >> 24); S(sl, S_OBJ + 4) = expand4(hi);
    }
    if (fl & (TF_DIRTY0 << OB_BL)) {
      obj_clear(sl, OB_BL);
      if (fl & ((fl & TF_VDELBL) ? TF_ENABL_OLD : TF_ENABL_NEW))
        obj_or(sl, OB_BL, (1u << (1u << ((S(sl, S_PF) >> 28) & 3u))) - 1u, byte_of(S(sl, S_POS2), 0));
    }
    if (fl & (TF_DIRTY0 << OB_P0)) rebuild_player(sl, 0, fl);
    if (fl & (TF_DIRTY0 << OB_P1)) rebuild_player(sl, 1, fl);
    if (fl & (TF_DIRTY0 << OB_M0)) rebuild_missile(sl, 0, fl);
    if (fl & (TF_DIRTY0 << OB_M1)) rebuild_missile(sl, 1, fl);
  }

  // ------------------------------------------------------------------ segment rendering (C.8 pixel function)
  // visible pixels [x0, x1) of the current line with the registers in force; VBLANK is off
  static DEVNI void render_visible(uint32_t sl, int x0, int x1) {
    uint32_t fl = S(sl, S_FL);
    if (fl & TF_DIRTY_ALL) { rebuild(sl, fl); fl &= ~TF_DIRTY_ALL; S(sl, S_FL) = fl; }
    const bool vis = (fl & TF_ROWVIS) != 0;
    const uint32_t ctrl = S(sl, S_PF) >> 24;
    uint32_t a0 = 0, a1 = 0, a2 = 0, a3 = 0, a4 = 0, a5 = 0, a6 = 0, a7 = 0, a8 = 0, a9 = 0, a10 = 0, a11 = 0, a12 = 0, a13 = 0, a14 = 0, any2 = 0;
    const int w1 = (x1 - 1) >> 5;
    const uint32_t m_last = 0xFFFFFFFFu >> (31 - ((x1 - 1) & 31));           // pixels of the last word before x1
    uint32_t m = 0xFFFFFFFFu << (x0 & 31);                                     // pixels of the word in hand inside [x0, x1): the first word starts at x0
    uint32_t comb = ((fl & TF_HMBLANK) && x0 < 32) ? ~0xFFu : 0xFFFFFFFFu;     // HMOVE comb: x 0..7 black, no collisions (word 0 only)
#pragma unroll 1
    for (int w = x0 >> 5; w <= w1; ++w) {
      const uint32_t rm = (w == w1) ? (m & m_last) : m;
      const uint32_t act = rm & comb;
      m = 0xFFFFFFFFu; comb = 0xFFFFFFFFu;
      const uint32_t *o = &smem[(S_OBJ + w) * BLOCK + sl];
      const uint32_t PF = o[0] & act, BL = o[5 * BLOCK] & act, P0 = o[10 * BLOCK] & act, P1 = o[15 * BLOCK] & act,
                     M0 = o[20 * BLOCK] & act, M1 = o[25 * BLOCK] & act;
      // pixels where two or more objects are lit (no such pixel in the word: no pair to look at): two carry-save adders
      // over three masks each (sum = xor, carry = majority), then carry | carry | sum & sum
      const uint32_t s1 = PF ^ BL ^ P0, c1 = (PF & BL) | (P0 & (PF | BL)), s2 = P1 ^ M0 ^ M1, c2 = (P1 & M0) | (M1 & (P1 | M0));
      if (c1 | c2 | (s1 & s2)) {
        any2 = 1;
        a0 |= M0 & P1; a1 |= M0 & P0; a2 |= M1 & P0; a3 |= M1 & P1; a4 |= P0 & PF; a5 |= P0 & BL; a6 |= P1 & PF; a7 |= P1 & BL;
        a8 |= M0 & PF; a9 |= M0 & BL; a10 |= M1 & PF; a11 |= M1 & BL; a12 |= BL & PF; a13 |= P0 & P1; a14 |= M0 & M1;
      }
      if (vis) {                                                   // priority -> colour index 0 P0, 1 P1, 2 PF, 3 BK
        uint32_t o0 = P0 | M0, o1 = P1 | M1, e0, e1, ef;
        const uint32_t of = PF | BL;
        if (ctrl & 4u) { ef = of; e0 = o0 & ~ef; e1 = o1 & ~(ef | e0); }              // PFP (SCORE ignored)
        else {
          if (ctrl & 2u) {                                                            // SCORE
            const uint32_t left = (w < 2) ? 0xFFFFFFFFu : (w == 2) ? 0x0000FFFFu : 0u; // x < 80
            o0 |= PF & left; o1 |= PF & ~left;
          }
          e0 = o0; e1 = o1 & ~e0; ef = of & ~(e0 | e1);
        }
        const uint32_t eb = ~(e0 | e1 | ef);
        uint32_t *pl = &smem[(S_PLANE + w) * BLOCK + sl];
        pl[0] = (pl[0] & ~rm) | ((e1 | eb) & rm);
        pl[5 * BLOCK] = (pl[5 * BLOCK] & ~rm) | ((ef | eb) & rm);
      }
    }
    if (!any2) return;
    uint32_t c = 0;
    c |= a0 ? 1u << CX_M0P1 : 0; c |= a1 ? 1u << CX_M0P0 : 0; c |= a2 ? 1u << CX_M1P0 : 0; c |= a3 ? 1u << CX_M1P1 : 0;
    c |= a4 ? 1u << CX_P0PF : 0; c |= a5 ? 1u << CX_P0BL : 0; c |= a6 ? 1u << CX_P1PF : 0; c |= a7 ? 1u << CX_P1BL : 0;
    c |= a8 ? 1u << CX_M0PF : 0; c |= a9 ? 1u << CX_M0BL : 0; c |= a10 ? 1u << CX_M1PF : 0; c |= a11 ? 1u << CX_M1BL : 0;
    c |= a12 ? 1u << CX_BLPF : 0; c |= a13 ? 1u << CX_P0P1 : 0; c |= a14 ? 1u << CX_M0M1 : 0;
    if (c) S(sl, S_CX) |= c;
  }
  // catch the beam up to colour clock `clk` (0..228) of the current line
  static DEV void render_to(uint32_t sl, uint32_t clk) {
    const uint32_t rx = S(sl, S_RX);
    if (clk <= rx) return;
    S(sl, S_RX) = clk;
    const int x0 = (int)max(rx, (uint32_t)HBLANK) - HBLANK, x1 = (int)max(clk, (uint32_t)HBLANK) - HBLANK;
    if (x1 <= x0 || (S(sl, S_FL) & TF_VBLANK)) return;               // VBLANK: no collisions, painted black
    render_visible(sl, x0, x1);
  }

  // ------------------------------------------------------------------ painting: planes + colours -> bytes in HBM
  // the whole row r from pixel 0 (the common case: no colour change inside the visible line)
  static DEVNI void paint_row_full(uint32_t sl, uint32_t r, uint32_t fl) {
    uint4 *dst = reinterpret_cast<uint4 *>(row_ptr(sl, r));
    if (fl & TF_VBLANK) {
#pragma unroll
      for (int q = 0; q < 10; ++q) st_row16(dst + q, make_uint4(0, 0, 0, 0));
      return;
    }
    const uint32_t colu = S(sl, S_COLU);
#pragma unroll 1
    for (int w = 0; w < 5; ++w) {
      const uint32_t i0 = S(sl, S_PLANE + w), i1 = S(sl, S_PLANE + 5 + w);
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const uint32_t a = i0 >> (16 * h), b = i1 >> (16 * h);
        const uint32_t s0 = spread8(a) | (spread8(b) << 1), s1 = spread8(a >> 8) | (spread8(b >> 8) << 1);
        uint4 v = make_uint4(__byte_perm(colu, 0, s0), __byte_perm(colu, 0, s0 >> 16), __byte_perm(colu, 0, s1), __byte_perm(colu, 0, s1 >> 16));
        if (w == 0 && h == 0 && (fl & TF_HMBLANK)) { v.x = 0; v.y = 0; }
        st_row16(dst + 2 * w + h, v);
      }
    }
  }
  // pixels [a, b) of row r: from the planes with the colours in force, or zeros
  static DEVNI void paint_range(uint32_t sl, uint32_t r, int a, int b, uint32_t fl, bool zero) {
    uint8_t *row = row_ptr(sl, r);
    const uint32_t colu = (zero || (fl & TF_VBLANK)) ? 0u : S(sl, S_COLU);
    const bool comb = (fl & TF_HMBLANK) != 0;
#pragma unroll 1
    for (int x = a; x < b;) {
      const int w = x >> 5, s = x & 31;
      const uint32_t i0 = S(sl, S_PLANE + w) >> s, i1 = S(sl, S_PLANE + 5 + w) >> s;
      if ((x & 3) == 0 && x + 4 <= b) {
        uint32_t n0 = i0 & 0xFu, n1 = i1 & 0xFu;
        n0 = (n0 | (n0 << 6)) & 0x0303u; n0 = (n0 | (n0 << 3)) & 0x1111u;
        n1 = (n1 | (n1 << 6)) & 0x0303u; n1 = (n1 | (n1 << 3)) & 0x1111u;
        uint32_t v = __byte_perm(colu, 0, n0 | (n1 << 1));
        if (comb && x < 8) v = 0;
        *reinterpret_cast<uint32_t *>(row + x) = v; x += 4;
      } else {
        uint32_t v = (colu >> (8 * ((i0 & 1u) | ((i1 & 1u) << 1)))) & 0xFFu;
        if (comb && x < 8) v = 0;
        row[x] = (uint8_t)v; x += 1;
      }
    }
  }
  // before a colour register / VBLANK changes at visible pixel x_now: fix the pixels before it
  static DEV void paint_upto(uint32_t sl, int x_now, uint32_t fl) {
    const int xe = min(max(x_now, 0), SCR_W), px = (int)S(sl, S_PX);
    if (xe > px) { paint_range(sl, S(sl, S_LINE) - ctx(C_Y0), px, xe, fl, false); S(sl, S_PX) = (uint32_t)xe; }
  }

  // ------------------------------------------------------------------ line / frame ends
  // the scanline in progress ends: finish it, store its row, start the next one (C.4 new-line bookkeeping)
  static DEVNI void line_end(uint32_t sl) {
    render_to(sl, LINE_CLK);
    uint32_t fl = S(sl, S_FL);
    uint32_t line = S(sl, S_LINE);
    if (fl & TF_ROWVIS) {
      const int px = (int)S(sl, S_PX);
      if (px == 0) paint_row_full(sl, line - ctx(C_Y0), fl);
      else if (px < SCR_W) paint_range(sl, line - ctx(C_Y0), px, SCR_W, fl, false);
    }
    line += 1; S(sl, S_LINE) = line; S(sl, S_RX) = 0; S(sl, S_PX) = 0;
    const uint32_t fresh = (fl >> 15) & 0xFu;                      // objects whose main copy re-appears
    fl = (fl & ~(TF_WSYNC | TF_HMBLANK | TF_FRESH_ALL | TF_ROWVIS)) | (fresh << (22 + OB_P0));
    if ((fl & TF_STORING) && (line - ctx(C_Y0)) < (uint32_t)SCR_H) fl |= TF_ROWVIS;
    S(sl, S_FL) = fl;
  }
  // C.10 frame end at colour clock `clk` of the current line (which becomes line 0 of the next frame)
  static DEVNI void frame_end(uint32_t sl, uint32_t clk) {
    render_to(sl, clk);
    uint32_t fl = S(sl, S_FL);
    if (fl & TF_STORING) {
      const int r = (int)S(sl, S_LINE) - (int)ctx(C_Y0);
      if (fl & TF_ROWVIS) {
        const int x = (int)max(clk, (uint32_t)HBLANK) - HBLANK, px = (int)S(sl, S_PX);
        if (x > px) paint_range(sl, r, px, x, fl, false);
        if (max(x, px) < SCR_W) paint_range(sl, r, max(x, px), SCR_W, fl, true);
      }
      const uint4 z = make_uint4(0, 0, 0, 0);                      // rows the beam never reached in this frame
#pragma unroll 1
      for (int rr = max(r + 1, 0); rr < SCR_H; ++rr) {
        uint4 *dst = reinterpret_cast<uint4 *>(row_ptr(sl, rr));
#pragma unroll
        for (int q = 0; q < 10; ++q) st_row16(dst + q, z);
      }
    }
    const uint32_t fd = S(sl, S_FDONE) + 1;
    S(sl, S_FDONE) = fd; S(sl, S_LINE) = 0; S(sl, S_PX) = 0;
    fl &= ~(TF_ROWVIS | TF_STORING);
    if (fd + 1 == ctx(C_FRAMESKIP)) fl |= TF_STORING;
    S(sl, S_FL) = fl;
  }

  // ------------------------------------------------------------------ TIA bus accesses (C.8)
  // m = cycle-in-line of the access (>= 76 when the instruction ran over the line end)
  static DEV uint32_t catch_up(uint32_t sl, int &m) {
    uint32_t ev = 0;
    while (m >= LINE_CYC) { line_end(sl); m -= LINE_CYC; ev += EV_CROSS; }
    render_to(sl, 3u * (uint32_t)(m + 1));
    return ev;
  }
  // read of register a&15 -> value | events<<8
  static DEVNI uint32_t read(uint32_t sl, uint32_t r, int m) {
    if (r < 8) {
      const uint32_t ev = catch_up(sl, m);
      const uint32_t cx = S(sl, S_CX);
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
      return ((b7 & 1u) << 7) | ((b6 & 1u) << 6) | (ev << 8);
    }
    const uint32_t fl = S(sl, S_FL);
    if (r == 0xC) { const bool lat = (fl & TF_LATCHEN) ? (fl & TF_INPT4_LATCH) != 0 : true; return (!(S(sl, S_INP) & 0x100u) && lat) ? 0x80u : 0u; }
    if (r == 0xD) { const bool lat = (fl & TF_LATCHEN) ? (fl & TF_INPT5_LATCH) != 0 : true; return lat ? 0x80u : 0u; }
    return 0;
  }
  static DEV uint32_t flag(uint32_t fl, uint32_t bit, bool on) { return on ? (fl | bit) : (fl & ~bit); }
  static DEV uint32_t dirty(int o) { return TF_DIRTY0 << o; }
  // does writing v to the VALUE register r leave every TIA latch as it is?  (display kernels re-write the same
  // playfield / graphics / colour bytes line after line: such a write needs no catch-up and dirties no mask)
  static DEV bool same(uint32_t sl, uint32_t r, uint32_t v, uint32_t fl) {
    switch (r) {
      case 0x1B: { const uint32_t g = S(sl, S_GRP); return byte_of(g, 0) == (v & 0xFFu) && byte_of(g, 3) == byte_of(g, 2); }
      case 0x1C: { const uint32_t g = S(sl, S_GRP);
                   return byte_of(g, 2) == (v & 0xFFu) && byte_of(g, 1) == byte_of(g, 0) && ((fl & TF_ENABL_OLD) != 0) == ((fl & TF_ENABL_NEW) != 0); }
      case 0x28: return ((fl & TF_RESMP0) != 0) == (((v >> 1) & 1u) != 0);
      case 0x29: return ((fl & TF_RESMP1) != 0) == (((v >> 1) & 1u) != 0);
      default: return false;
    }
  }
  // write of v to register r (= a & 0x3F, one with an effect) in cycle-in-line m -> events
  static DEVNI uint32_t write(uint32_t sl, uint32_t r, uint32_t v, int m) {
    uint32_t ev = 0;
    while (m >= LINE_CYC) { line_end(sl); m -= LINE_CYC; ev += EV_CROSS; }
    const int x_now = 3 * (m + 1) - HBLANK;
    uint32_t fl = S(sl, S_FL);
    const uint32_t d = c_tia_desc[r];
    if (d & 3u) {                                          // a plain value register: field store or flag
      const uint32_t pv = v >> ((d >> 19) & 7u);
      uint32_t nfl = fl;
      uint32_t old = 0, neu = 0; int wi = 0;
      if (d & 1u) {
        wi = S_COLU + (int)((d >> 3) & 7u);
        const uint32_t sh = (d >> 6) & 31u, fm = ((d >> 30) & 1u) ? 0xFu : 0xFFu;
        old = S(sl, wi); neu = (old & ~(fm << sh)) | ((pv & ((d >> 11) & 0xFFu)) << sh);
        if (neu == old) return ev | ((fl & TF_WSYNC) ? EV_WSYNC : 0u);        // re-written with the value it holds: nothing changes
      } else {
        const uint32_t bit = 1u << ((d >> 6) & 31u);
        nfl = (pv & 1u) ? (fl | bit) : (fl & ~bit);
        if (nfl == fl) return ev | ((fl & TF_WSYNC) ? EV_WSYNC : 0u);
      }
      // colour, HMxx: neither an object mask nor a collision changes, so outside the kept rows the catch-up can wait
      if ((fl & TF_ROWVIS) || !((d >> 28) & 1u)) {
        render_to(sl, 3u * (uint32_t)(m + 1));
        const uint32_t fl2 = S(sl, S_FL); nfl = (nfl & ~(TF_DIRTY_ALL | 0u)) | (fl2 & (TF_DIRTY_ALL | 0u)); fl = fl2;
        if (((d >> 29) & 1u) && (fl & TF_ROWVIS)) paint_upto(sl, x_now, fl);
      }
      if (d & 1u) S(sl, wi) = neu;
      nfl |= ((d >> 22) & 63u) << 22;
      S(sl, S_FL) = nfl;
      return ev | ((nfl & TF_WSYNC) ? EV_WSYNC : 0u);
    }
    if (same(sl, r, v, fl)) return ev | ((fl & TF_WSYNC) ? EV_WSYNC : 0u);    // GRPx / RESMPx re-written with what they hold
    // WSYNC and HMCLR change neither an object's line mask nor a collision: lazy as above
    if ((fl & TF_ROWVIS) || !(r == 0x02u || r == 0x2Bu)) { render_to(sl, 3u * (uint32_t)(m + 1)); fl = S(sl, S_FL); }
    switch (r) {
      case 0x00: { const bool nv = (v >> 1) & 1u;
                   if ((fl & TF_VSYNC) && !nv) { frame_end(sl, 3u * (uint32_t)(m + 1)); ev |= EV_FRAME; fl = S(sl, S_FL); }
                   fl = flag(fl, TF_VSYNC, nv); } break;
      case 0x01: if (fl & TF_ROWVIS) paint_upto(sl, x_now, fl);
                 fl = flag(fl, TF_VBLANK, (v >> 1) & 1u); fl = flag(fl, TF_LATCHEN, (v >> 6) & 1u);
                 if (!(fl & TF_LATCHEN)) fl |= TF_INPT4_LATCH | TF_INPT5_LATCH;
                 if ((fl & TF_LATCHEN) && (S(sl, S_INP) & 0x100u)) fl &= ~TF_INPT4_LATCH;
                 break;
      case 0x02: fl |= TF_WSYNC; break;
      case 0x10: case 0x11: S(sl, S_POS) = set_byte(S(sl, S_POS), r - 0x10, x_now < 0 ? 3 : (x_now + 5) % 160);
                 fl |= (r == 0x10) ? (TF_FRESH_P0 | dirty(OB_P0)) : (TF_FRESH_P1 | dirty(OB_P1)); break;
      case 0x12: case 0x13: S(sl, S_POS) = set_byte(S(sl, S_POS), r - 0x10, x_now < 0 ? 2 : (x_now + 4) % 160);
                 fl |= (r == 0x12) ? (TF_FRESH_M0 | dirty(OB_M0)) : (TF_FRESH_M1 | dirty(OB_M1)); break;
      case 0x14: S(sl, S_POS2) = set_byte(S(sl, S_POS2), 0, x_now < 0 ? 2 : (x_now + 4) % 160); fl |= dirty(OB_BL); break;
      case 0x1B: { const uint32_t g = S(sl, S_GRP); S(sl, S_GRP) = set_byte(set_byte(g, 0, v), 3, byte_of(g, 2)); }   // GRP0; GRP1_old := GRP1_new
                 fl |= dirty(OB_P0) | dirty(OB_P1); break;
      case 0x1C: { const uint32_t g = S(sl, S_GRP); S(sl, S_GRP) = set_byte(set_byte(g, 2, v), 1, byte_of(g, 0)); }   // GRP1; GRP0_old := GRP0_new
                 fl = flag(fl, TF_ENABL_OLD, fl & TF_ENABL_NEW) | dirty(OB_P0) | dirty(OB_P1) | dirty(OB_BL); break;
      case 0x28: case 0x29: { const int p = r - 0x28; const uint32_t bit = p ? TF_RESMP1 : TF_RESMP0; const bool nv = (v >> 1) & 1u;
                 if ((fl & bit) && !nv) {
                   const uint32_t mm = byte_of(S(sl, S_NUSIZ), p) & 7u, mid = (mm == 5) ? 8u : (mm == 7) ? 16u : 4u;
                   S(sl, S_POS) = set_byte(S(sl, S_POS), 2 + p, (byte_of(S(sl, S_POS), p) + mid) % 160u);
                 }
                 fl = flag(fl, bit, nv) | dirty(OB_M0 + p); } break;
      case 0x2A: {                                                                              // HMOVE
                 uint32_t pos = S(sl, S_POS), pos2 = S(sl, S_POS2); const uint32_t nus = S(sl, S_NUSIZ);
#pragma unroll 1
                 for (int k = 0; k < 5; ++k) {
                   const uint32_t h = (k < 4) ? (nus >> (16 + 4 * k)) & 0xFu : byte_of(pos2, 1) & 0xFu;
                   const int s = (h < 8) ? (int)h : (int)h - 16;
                   int p = (int)((k < 4) ? byte_of(pos, k) : byte_of(pos2, 0)) - s;
                   if (p < 0) p += 160;
                   if (p >= 160) p -= 160;
                   if (k < 4) pos = set_byte(pos, k, p); else pos2 = set_byte(pos2, 0, p);
                 }
                 S(sl, S_POS) = pos; S(sl, S_POS2) = pos2;
                 fl |= dirty(OB_BL) | dirty(OB_P0) | dirty(OB_P1) | dirty(OB_M0) | dirty(OB_M1);
                 if (x_now < 0) fl |= TF_HMBLANK; } break;
      case 0x2B: S(sl, S_NUSIZ) &= 0x0000FFFFu; S(sl, S_POS2) = set_byte(S(sl, S_POS2), 1, 0); break;      // HMCLR
      case 0x2C: S(sl, S_CX) = 0; break;                                                            // CXCLR

      default: break;
    }
    S(sl, S_FL) = fl;
    return ev | ((fl & TF_WSYNC) ? EV_WSYNC : 0u);
  }
};

}  // namespace vcs
