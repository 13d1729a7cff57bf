/* oracle/ovcs.c — plain per-cycle CPU oracle.  TEST INFRASTRUCTURE (see ovcs.h).
 *
 * One CPU cycle = one bus access = 3 colour clocks ("cycle
 * by cycle").  Nothing here is blocked, fused, lazy or closed-form: the timer is ticked,
 * every colour clock is rendered pixel by pixel, WSYNC stalls one cycle at a time.
 * Clause numbers C.x refer to SURVEY.md §8(c); L-numbers to /root/reference/PAPER.md.
 */
#include "ovcs.h"
#include <stdlib.h>
#include <string.h>

enum { SCR_W = 160, SCR_H = 210, LINE_CYC = 76, HBLANK = 68 };

/* ---------------------------------------------------------------- C.1 state */
typedef struct {
  /* CPU */
  uint8_t A, X, Y, SP, P; uint16_t PC; uint64_t cyc; uint8_t halted, status;
  /* beam */
  uint32_t line, frame, frame_cyc; uint64_t events; uint64_t clocks;
  /* RIOT */
  uint8_t ram[128]; uint8_t timer; uint16_t sub; uint8_t shift, tflag;
  uint8_t ora, ddra, orb, ddrb, ina, inb, switches_set;
  /* TIA */
  uint8_t vsync, vblank, latch_en, wsync;
  uint8_t nusiz[2], colup[2], colupf, colubk, ctrlpf, refp[2], pf0, pf1, pf2;
  uint8_t grp_new[2], grp_old[2], enam[2], enabl_new, enabl_old;
  uint8_t hm[5];                 /* P0 P1 M0 M1 BL, 4-bit */
  uint8_t vdelp[2], vdelbl, resmp[2];
  uint8_t pos[5];                /* P0 P1 M0 M1 BL in [0,160) */
  uint8_t fresh;                 /* bit0 P0, bit1 P1, bit2 M0, bit3 M1 */
  uint8_t hmove_blank; uint16_t cx;
  uint8_t inpt4_latch, inpt5_latch, fire0;
  /* cart */
  const uint8_t *rom; uint32_t rom_size; uint8_t bank;
  uint8_t kind;                  /* OVCS_MAP_* (never BY_SIZE) */
  uint8_t sc_ram[128];           /* Superchip RAM */
  uint8_t seg[3];                /* E0: slices shown at $1000, $1400, $1800 */
  uint8_t fe_pending;            /* FE: the previous access was to $01FE */
  uint64_t seed;
  uint64_t n_instr, n_tia_writes;    /* instrumentation only (bench work model); never read by the model */
  uint8_t *back, *front;
} env_t;

struct ovcs_s {
  int32_t batch, n_roms; ovcs_config cfg;
  uint8_t **rom_data; uint32_t *rom_size;
  env_t *env;
};

/* ------------------------------------------------------------ G.0 splitmix64 */
uint64_t ovcs_splitmix64(uint64_t *s) {
  uint64_t z = (*s += 0x9E3779B97F4A7C15ULL);
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  return z ^ (z >> 31);
}

/* ------------------------------------------------------------- C.9 cartridge */
static int cart_banks(const env_t *e) {          /* 4 KB banks switched by hotspots (0 = none) */
  switch (e->kind) { case OVCS_MAP_F8: case OVCS_MAP_F8SC: return 2; case OVCS_MAP_F6: case OVCS_MAP_F6SC: return 4;
                     case OVCS_MAP_F4: case OVCS_MAP_F4SC: return 8; default: return 0; }
}
static int cart_has_sc(const env_t *e) { return e->kind == OVCS_MAP_F8SC || e->kind == OVCS_MAP_F6SC || e->kind == OVCS_MAP_F4SC; }
static void cart_hotspot(env_t *e, uint16_t a) {          /* any bus access, a = addr&0x1FFF with A12 set */
  /* F8: $1FF8/9 -> bank 0/1 [D]; F6 (16 KB): $1FF6..$1FF9 -> banks 0..3; F4 (32 KB): $1FF4..$1FFB -> banks 0..7
   * (PAPER.md L61, L69, L469); the Superchip variants switch the same way */
  int nb = cart_banks(e);
  if (nb) { uint16_t lo = (uint16_t)(nb == 8 ? 0x1FF4 : 0x1FFA - nb); if (a >= lo && a < lo + nb) e->bank = (uint8_t)(a - lo); }
  /* E0 [D]: $1FE0-7 choose the slice of the $1000 window, $1FE8-F of $1400, $1FF0-7 of $1800 */
  if (e->kind == OVCS_MAP_E0 && a >= 0x1FE0 && a <= 0x1FF7) e->seg[(a - 0x1FE0) >> 3] = (uint8_t)(a & 7);
}
static uint8_t cart_peek(const env_t *e, uint16_t a) {
  uint32_t o = a & 0x0FFF;
  if (cart_has_sc(e) && o < 0x100) return e->sc_ram[o & 0x7F];   /* read port $1080-$10FF; a read of the write port sees the cell too, unchanged [R] */
  if (e->kind == OVCS_MAP_2K) return e->rom[o & 0x7FF];
  if (e->kind == OVCS_MAP_4K) return e->rom[o];
  if (e->kind == OVCS_MAP_E0) { uint32_t w = o >> 10, slice = (w == 3) ? 7u : e->seg[w]; return e->rom[slice * 1024u + (o & 0x3FF)]; }
  return e->rom[(uint32_t)e->bank * 4096u + o];                   /* F8 / F6 / F4 (+SC), FE */
}
static void cart_poke(env_t *e, uint16_t a, uint8_t v) {          /* a write cycle in cartridge space (after the hotspot check) */
  if (cart_has_sc(e) && (a & 0x0F80) == 0) e->sc_ram[a & 0x7F] = v;   /* write port $1000-$107F [D] */
}
/* FE [D]: the board watches the bus for $01FE (the stack cell JSR / RTS touch last / first); the data of the access that
 * FOLLOWS it carries the high byte of the new PC, and its bit 5 tells the $F000 page (bank 0) from the $D000 page (bank 1) */
static void fe_snoop(env_t *e, uint16_t a, uint8_t data) {
  if (e->kind != OVCS_MAP_FE) return;
  if (e->fe_pending) { e->bank = (data & 0x20) ? 0 : 1; e->fe_pending = 0; }
  if (a == 0x01FE) e->fe_pending = 1;
}

/* ------------------------------------------------------------------ C.7 RIOT */
static void riot_tick(env_t *e) {
  e->sub = (uint16_t)((e->sub + 1) & ((1u << e->shift) - 1u));
  if (e->tflag) e->timer = (uint8_t)(e->timer - 1);
  else if (e->sub == 0) {
    if (e->timer == 0) { e->timer = 0xFF; e->tflag = 1; }
    else e->timer--;
  }
}
static uint8_t riot_read(env_t *e, uint16_t a) {
  if ((a & 0x04) == 0) {
    switch (a & 3) {
      case 0: return (uint8_t)((e->ora & e->ddra) | (e->ina & ~e->ddra));
      case 1: return e->ddra;
      case 2: return (uint8_t)((e->orb & e->ddrb) | (e->inb & ~e->ddrb));
      default: return e->ddrb;
    }
  }
  if ((a & 0x05) == 0x04) { uint8_t v = e->timer; e->tflag = 0; return v; }   /* INTIM  */
  return (uint8_t)(e->tflag << 7);                                             /* TIMINT */
}
static void riot_write(env_t *e, uint16_t a, uint8_t v) {
  static const uint8_t shifts[4] = {0, 3, 6, 10};
  if ((a & 0x04) == 0) {
    switch (a & 3) { case 0: e->ora = v; break; case 1: e->ddra = v; break;
                     case 2: e->orb = v; break; default: e->ddrb = v; }
  } else if ((a & 0x14) == 0x14) {
    e->timer = v; e->shift = shifts[a & 3]; e->sub = (uint16_t)((1u << e->shift) - 1u); e->tflag = 0;
  } /* (a&0x14)==0x04: edge-detect control, ignored [R] */
}

/* ------------------------------------------------------------------- C.8 TIA */
static const int8_t COPY_OFF[8][3] = {            /* O(m), -1 = none  [D] */
  {0,-1,-1}, {0,16,-1}, {0,32,-1}, {0,16,32}, {0,64,-1}, {0,-1,-1}, {0,32,64}, {0,-1,-1} };

static int mod160(int v) { v %= 160; if (v < 0) v += 160; return v; }

static int pf_bit(const env_t *e, int x) {
  int i = (x < 80) ? (x >> 2) : ((e->ctrlpf & 1) ? 19 - ((x - 80) >> 2) : ((x - 80) >> 2));
  if (i < 4)  return (e->pf0 >> (4 + i)) & 1;
  if (i < 12) return (e->pf1 >> (7 - (i - 4))) & 1;
  return (e->pf2 >> (i - 12)) & 1;
}
static int player_lit(const env_t *e, int p, int x) {
  uint8_t g = e->vdelp[p] ? e->grp_old[p] : e->grp_new[p];
  int m = e->nusiz[p] & 7, s = (m == 5) ? 2 : (m == 7) ? 4 : 1, lit = 0;
  for (int k = 0; k < 3; k++) {
    int o = COPY_OFF[m][k]; if (o < 0) continue;
    if (o == 0 && ((e->fresh >> p) & 1)) continue;
    int d = mod160(x - e->pos[p] - o);
    if (d < 8 * s) { int b = e->refp[p] ? d / s : 7 - d / s; if ((g >> b) & 1) lit = 1; }
  }
  return lit;
}
static int missile_lit(const env_t *e, int p, int x) {
  if (!e->enam[p] || e->resmp[p]) return 0;
  int m = e->nusiz[p] & 7, w = 1 << ((e->nusiz[p] >> 4) & 3), lit = 0;
  for (int k = 0; k < 3; k++) {
    int o = COPY_OFF[m][k]; if (o < 0) continue;
    if (o == 0 && ((e->fresh >> (2 + p)) & 1)) continue;
    if (mod160(x - e->pos[2 + p] - o) < w) lit = 1;
  }
  return lit;
}
static int ball_lit(const env_t *e, int x) {
  int en = e->vdelbl ? e->enabl_old : e->enabl_new, w = 1 << ((e->ctrlpf >> 4) & 3);
  return en && mod160(x - e->pos[4]) < w;
}

/* one colour clock hc in [0,228) of the current line */
static void tia_clock(env_t *e, int hc, int y0) {
  e->clocks++;
  if (hc < HBLANK) return;
  int x = hc - HBLANK; uint8_t colour;
  if (e->vblank || (e->hmove_blank && x < 8)) colour = 0;
  else {
    int PF = pf_bit(e, x), BL = ball_lit(e, x);
    int P0 = player_lit(e, 0, x), P1 = player_lit(e, 1, x);
    int M0 = missile_lit(e, 0, x), M1 = missile_lit(e, 1, x);
    uint16_t c = 0;                         /* bit layout: see cx_read() */
    if (M0 && P1) c |= 1u << 0;
    if (M0 && P0) c |= 1u << 1;
    if (M1 && P0) c |= 1u << 2;
    if (M1 && P1) c |= 1u << 3;
    if (P0 && PF) c |= 1u << 4;
    if (P0 && BL) c |= 1u << 5;
    if (P1 && PF) c |= 1u << 6;
    if (P1 && BL) c |= 1u << 7;
    if (M0 && PF) c |= 1u << 8;
    if (M0 && BL) c |= 1u << 9;
    if (M1 && PF) c |= 1u << 10;
    if (M1 && BL) c |= 1u << 11;
    if (BL && PF) c |= 1u << 12;
    if (P0 && P1) c |= 1u << 13;
    if (M0 && M1) c |= 1u << 14;
    e->cx |= c;
    if (e->ctrlpf & 4)                       /* PFP: playfield/ball on top; SCORE ignored [R] */
      colour = (PF || BL) ? e->colupf : (P0 || M0) ? e->colup[0] : (P1 || M1) ? e->colup[1] : e->colubk;
    else {
      int score = (e->ctrlpf >> 1) & 1, pfl = score && PF && x < 80, pfr = score && PF && x >= 80;
      colour = (P0 || M0 || pfl) ? e->colup[0] : (P1 || M1 || pfr) ? e->colup[1]
             : (PF || BL) ? e->colupf : e->colubk;
    }
  }
  int r = (int)e->line - y0;
  if (r >= 0 && r < SCR_H) e->back[r * SCR_W + x] = colour;
}

static uint8_t tia_read(env_t *e, uint16_t a) {
  uint16_t c = e->cx; int b7 = 0, b6 = 0;
  switch (a & 0x0F) {
    case 0x0: b7 = c >> 0;  b6 = c >> 1;  break;   /* CXM0P : M0.P1, M0.P0 */
    case 0x1: b7 = c >> 2;  b6 = c >> 3;  break;   /* CXM1P : M1.P0, M1.P1 */
    case 0x2: b7 = c >> 4;  b6 = c >> 5;  break;   /* CXP0FB: P0.PF, P0.BL */
    case 0x3: b7 = c >> 6;  b6 = c >> 7;  break;   /* CXP1FB: P1.PF, P1.BL */
    case 0x4: b7 = c >> 8;  b6 = c >> 9;  break;   /* CXM0FB: M0.PF, M0.BL */
    case 0x5: b7 = c >> 10; b6 = c >> 11; break;   /* CXM1FB: M1.PF, M1.BL */
    case 0x6: b7 = c >> 12; b6 = 0;       break;   /* CXBLPF: BL.PF        */
    case 0x7: b7 = c >> 13; b6 = c >> 14; break;   /* CXPPMM: P0.P1, M0.M1 */
    case 0xC: b7 = (!e->fire0) && (e->latch_en ? e->inpt4_latch : 1); break;     /* INPT4 */
    case 0xD: b7 = e->latch_en ? e->inpt5_latch : 1; break;      /* INPT5: never pressed  */
    default: break;                                /* INPT0-3 no paddles [R]; E,F -> 0      */
  }
  return (uint8_t)(((b7 & 1) << 7) | ((b6 & 1) << 6));   /* low 6 bits read 0 [R] */
}

/* C.10 frame end: front = back; back = 0; the scanline in progress becomes line 0 */
static void frame_end(env_t *e) {
  memcpy(e->front, e->back, SCR_W * SCR_H);
  memset(e->back, 0, SCR_W * SCR_H);
  e->frame++; e->line = 0; e->frame_cyc = 0; e->events++;
}

/* C.11: the fire latch drops whenever latch_en && fire pressed holds (evaluated when the
 * action is latched and at every VBLANK write) */
static void eval_fire_latch(env_t *e) { if (e->latch_en && e->fire0) e->inpt4_latch = 0; }

/* C.8 write effects.  n = index in the line of the cycle doing the write. */
static void tia_write(env_t *e, uint16_t a, uint8_t v, int n) {
  int x_now = 3 * (n + 1) - HBLANK;
  switch (a & 0x3F) {
    case 0x00: { uint8_t nv = (v >> 1) & 1; if (e->vsync == 1 && nv == 0) frame_end(e); e->vsync = nv; } break;
    case 0x01: e->vblank = (v >> 1) & 1; e->latch_en = (v >> 6) & 1;
               if (!e->latch_en) { e->inpt4_latch = 1; e->inpt5_latch = 1; }
               eval_fire_latch(e); break;
    case 0x02: e->wsync = 1; break;
    case 0x03: break;                                              /* RSYNC: no effect [R] */
    case 0x04: e->nusiz[0] = v & 0x37; break;
    case 0x05: e->nusiz[1] = v & 0x37; break;
    case 0x06: e->colup[0] = v & 0xFE; break;
    case 0x07: e->colup[1] = v & 0xFE; break;
    case 0x08: e->colupf = v & 0xFE; break;
    case 0x09: e->colubk = v & 0xFE; break;
    case 0x0A: e->ctrlpf = v & 0x37; break;
    case 0x0B: e->refp[0] = (v >> 3) & 1; break;
    case 0x0C: e->refp[1] = (v >> 3) & 1; break;
    case 0x0D: e->pf0 = v & 0xF0; break;
    case 0x0E: e->pf1 = v; break;
    case 0x0F: e->pf2 = v; break;
    case 0x10: case 0x11: { int p = (a & 0x3F) - 0x10;                        /* RESP0/1 */
               e->pos[p] = (uint8_t)((x_now < 0) ? 3 : (x_now + 5) % 160); e->fresh |= (uint8_t)(1u << p); } break;
    case 0x12: case 0x13: { int p = (a & 0x3F) - 0x12;                        /* RESM0/1 */
               e->pos[2 + p] = (uint8_t)((x_now < 0) ? 2 : (x_now + 4) % 160); e->fresh |= (uint8_t)(4u << p); } break;
    case 0x14: e->pos[4] = (uint8_t)((x_now < 0) ? 2 : (x_now + 4) % 160); break;   /* RESBL */
    case 0x1B: e->grp_new[0] = v; e->grp_old[1] = e->grp_new[1]; break;        /* GRP0 */
    case 0x1C: e->grp_new[1] = v; e->grp_old[0] = e->grp_new[0]; e->enabl_old = e->enabl_new; break;
    case 0x1D: e->enam[0] = (v >> 1) & 1; break;
    case 0x1E: e->enam[1] = (v >> 1) & 1; break;
    case 0x1F: e->enabl_new = (v >> 1) & 1; break;
    case 0x20: case 0x21: case 0x22: case 0x23: case 0x24: e->hm[(a & 0x3F) - 0x20] = v >> 4; break;
    case 0x25: e->vdelp[0] = v & 1; break;
    case 0x26: e->vdelp[1] = v & 1; break;
    case 0x27: e->vdelbl = v & 1; break;
    case 0x28: case 0x29: { int p = (a & 0x3F) - 0x28; uint8_t nv = (v >> 1) & 1;   /* RESMPp */
               if (e->resmp[p] == 1 && nv == 0) {
                 int m = e->nusiz[p] & 7, mid = (m == 5) ? 8 : (m == 7) ? 16 : 4;
                 e->pos[2 + p] = (uint8_t)((e->pos[p] + mid) % 160);
               }
               e->resmp[p] = nv; } break;
    case 0x2A: for (int k = 0; k < 5; k++) {                                   /* HMOVE */
                 int h = e->hm[k], s = (h < 8) ? h : h - 16;
                 e->pos[k] = (uint8_t)mod160((int)e->pos[k] - s);
               }
               if (x_now < 0) e->hmove_blank = 1;
               break;
    case 0x2B: memset(e->hm, 0, 5); break;                                     /* HMCLR */
    case 0x2C: e->cx = 0; break;                                               /* CXCLR */
    default: break;                             /* AUDxx (L205: no audio), 2D-3F: no effect */
  }
}

/* ------------------------------------------------------- C.4 the cycle protocol */
struct osoft_cfg_s; struct osoft_acc_s;
typedef struct { env_t *e; const ovcs_config *cfg; const void *soft; void *acc; int dummy; } ctx_t;   /* soft != NULL: SOFT-STE mode (ovcs_soft.inc) */

static void tick(ctx_t *c) {
  env_t *e = c->e;
  int n = (int)(e->cyc % LINE_CYC);
  if (n == 0 && e->cyc > 0) {            /* a new scanline starts with this cycle */
    e->line++; e->wsync = 0; e->hmove_blank = 0; e->fresh = 0;
  }
  e->cyc++; e->frame_cyc++;
  riot_tick(e);
  for (int k = 0; k < 3; k++) tia_clock(e, 3 * n + k, c->cfg->y0);   /* state before the access */
}

#include "ovcs_soft.inc"   /* SOFT-STE mode primitives (config 5) */
static uint8_t soft_rom(ctx_t *c, uint16_t a, uint8_t v) { return osoft_rom_read((const osoft_cfg *)c->soft, (osoft_acc *)c->acc, c->e, a, v); }
static uint8_t soft_ram(ctx_t *c, int cell, uint8_t v) { return osoft_ram_read((const osoft_cfg *)c->soft, (osoft_acc *)c->acc, c->e, cell, v); }

/* C.3 address decode + the access itself (post-tick) */
static uint8_t bus_read(ctx_t *c, uint16_t addr) {
  env_t *e = c->e; uint16_t a = addr & 0x1FFF; uint8_t v;
  while (e->wsync && (e->cyc % LINE_CYC) != 0) tick(c);   /* RDY halts read cycles only [D] */
  tick(c);
  const int dummy = c->dummy; c->dummy = 0;                /* set by DUMMY_READ: a cycle whose value is discarded */
  if (a & 0x1000) { cart_hotspot(e, a); v = cart_peek(e, a); if (c->soft && !dummy && !(cart_has_sc(e) && (a & 0xF00) == 0)) v = soft_rom(c, a, v); }
  else if ((a & 0x0080) == 0) v = tia_read(e, a);
  else if ((a & 0x0200) == 0) { v = e->ram[a & 0x7F]; if (c->soft && !dummy) v = soft_ram(c, a & 0x7F, v); }
  else v = riot_read(e, a);
  fe_snoop(e, a, v);
  return v;
}
#define DUMMY_READ(c, addr) ((c)->dummy = 1, (void)bus_read((c), (addr)))
static void bus_write(ctx_t *c, uint16_t addr, uint8_t v) {
  env_t *e = c->e; uint16_t a = addr & 0x1FFF;
  tick(c);
  int n = (int)((e->cyc - 1) % LINE_CYC);
  if (a & 0x1000) { cart_hotspot(e, a); cart_poke(e, a, v); }
  else if ((a & 0x0080) == 0) { e->n_tia_writes++; tia_write(e, a, v, n); }
  else if ((a & 0x0200) == 0) e->ram[a & 0x7F] = v;
  else riot_write(e, a, v);
  fe_snoop(e, a, v);
}

#include "ovcs_cpu.inc"   /* C.5/C.6: the 6507 */
#include "ovcs_api.inc"   /* C.2/C.10/C.11 + the C ABI mirror */
