/* oracle/ovcs.h — CPU ORACLE for the batched Atari 2600 VCS hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header, table or helper with the CUDA path (paper_2606_22447_b200/csrc) and neither
 * includes the other.
 *
 * What it is: a plain, slow, single-threaded, one-CPU-cycle-at-a-time model of the
 * machine the paper re-implements (§1, L55 Fig. 1, L61 "Why the Atari VCS
 * Is Good Ground Truth": 6507 CPU + TIA + RIOT + bank-switched cartridge), in hard mode
 * (§3: "opcode bytes index an integer dispatch table, the ALU is integer
 * arithmetic, and flags are bits").  The paper does not define the chips at register
 * level; the register-level machine model is SURVEY.md §8(c) C.1–C.12 (tags [P] paper,
 * [D] public 6502/6532/TIA documentation, [R] reading).  Every function in ovcs.c cites
 * the clause it follows.  All readings are listed in DESIGN.md §3.
 *
 * Parity status: pinned by tests/test_oracle_*.py (-m "not gpu") against the opcode
 * matrices (151 documented + the paper's 38 undocumented bytes, tests/golden/), wide-integer ADC/SBC definitions, base-100 BCD arithmetic, the RIOT closed
 * form, hand-assembled programs with hand-derived RAM/screens.  PARITY UNPINNED (no
 * source other than the [R] readings exists in this container): per-register TIA write
 * latencies, mid-line HMOVE, RSYNC, double/quad-size player 1-clock shift, bus residue
 * in TIA reads, same-cycle INTIM/underflow, F8 start bank, power-on timer/RAM state, y0,
 * the Superchip / E0 / FE power-up states and the read of a Superchip write port (R16),
 * and the format guess of ovcs_detect_mapper against the paper's (xitari's) signatures (R17).
 * FULL mode (R18) is pinned by the paper's closed forms; its Table 3 N_div values need a ROM that is not here.
 * Decimal-mode results for invalid BCD operands are pinned against the digit-wise
 * definition since round 2 (tests/test_oracle_pins_cpu.py).
 */
#ifndef OVCS_H
#define OVCS_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct ovcs_s ovcs_t;

/* Cartridge formats ("cartridge mappers", L469: 2K, 4K, F8, F6, F4, F8SC, F6SC, F4SC, E0, FE; SURVEY C.9 and
 * §8(f) NEXT-3; behaviour per the public documentation of these boards [D], power-up states [R], R15-R17):
 *   2K / 4K        no switching (2K mirrored)
 *   F8 / F6 / F4   2 / 4 / 8 banks of 4 KB; any access to $1FF8-9 / $1FF6-9 / $1FF4-B selects the bank before data returns
 *   ..SC           the same plus 128 bytes of cartridge RAM in every bank: write port $1000-$107F, read port $1080-$10FF
 *   E0             eight 1 KB slices; windows $1000 / $1400 / $1800 show the slice chosen by any access to
 *                  $1FE0-7 / $1FE8-F / $1FF0-7, window $1C00 always shows slice 7
 *   FE             two 4 KB banks; the access after one to $01FE selects the bank from bit 5 of its data (1: bank 0)
 * OVCS_MAP_BY_SIZE picks 2K / 4K / F8 / F6 / F4 from the image size. */
enum { OVCS_MAP_BY_SIZE = 0, OVCS_MAP_2K, OVCS_MAP_4K, OVCS_MAP_F8, OVCS_MAP_F6, OVCS_MAP_F4, OVCS_MAP_F8SC, OVCS_MAP_F6SC, OVCS_MAP_F4SC,
       OVCS_MAP_E0, OVCS_MAP_FE, OVCS_MAP_COUNT };
typedef struct { const uint8_t *data; uint32_t size; /* 2048 | 4096 | 8192 | 16384 | 32768 */ uint32_t mapper; /* OVCS_MAP_* */ } ovcs_rom;
/* content-based format guess from size and image bytes (PAPER.md L69 / L469 "mapper auto-detected"; the rules are this
 * build's reading R17 in DESIGN.md): returns OVCS_MAP_2K .. OVCS_MAP_FE, or -1 for a size no format has */
int  ovcs_detect_mapper(const uint8_t *data, uint32_t size);
typedef struct { int32_t y0, max_lines, f8_start_bank; uint32_t flags; } ovcs_config;

/* Same 32-byte record as include/vcs.h's vcs_regs; retyped, not shared. */
typedef struct {
  uint64_t cycles;
  uint32_t frame;
  uint16_t pc; uint8_t a, x, y, sp, p;
  uint8_t bank;
  uint16_t line; uint8_t cyc_in_line;
  uint8_t status;            /* bit0 illegal-opcode halt, bit1 frame cap was hit */
  uint8_t intim, timint, pad[6];   /* pad[0]: E0 — slice in the $1800 window (bank = slice@$1000 | slice@$1400 << 3); FE — 1 while an access to $01FE awaits its successor */
} ovcs_regs;

/* Debug view of the TIA/RIOT latches, for the hand-program pins (tests only). */
typedef struct {
  uint8_t posP0, posP1, posM0, posM1, posBL;
  uint8_t fresh, hmove_blank, vsync, vblank, latch_en, wsync;
  uint8_t inpt4_latch, grp0_new, grp0_old, grp1_new, grp1_old;
  uint16_t cx;
  uint8_t timer, tflag, shift; uint16_t sub;
  uint64_t clocks_rendered;      /* colour clocks rendered since reset: must equal 3*cycles */
  uint64_t n_instr, n_tia_writes; /* instrumentation: instructions executed / TIA register writes since reset */
} ovcs_debug;

enum { OVCS_OK = 0, OVCS_EINVAL = -1, OVCS_ENOMEM = -3, OVCS_EROM = -4 };

/* All pointers are HOST pointers.  roms/env_rom/seeds are copied. */
int  ovcs_create(ovcs_t **out, int32_t batch, const ovcs_rom *roms, int32_t n_roms,
                 const int32_t *env_rom, const uint64_t *seeds, const ovcs_config *cfg);
int  ovcs_reset(ovcs_t *h, const uint8_t *mask /* [batch] or NULL = all */);
int  ovcs_step(ovcs_t *h, const uint8_t *actions /* [batch] */, int32_t frameskip);
/* Same as ovcs_step restricted to envs [lo,hi): lets a test fan independent envs over
 * OS threads; the oracle code itself stays single-threaded per env. */
int  ovcs_step_range(ovcs_t *h, const uint8_t *actions, int32_t frameskip, int32_t lo, int32_t hi);
/* SURVEY §8(f) NEXT-4 (Table 8): masked step, console switches, the ALE episode start. */
int  ovcs_step_masked(ovcs_t *h, const uint8_t *actions, int32_t frameskip, const uint8_t *mask /* [batch] or NULL */);
int  ovcs_step_masked_range(ovcs_t *h, const uint8_t *actions, int32_t frameskip, const uint8_t *mask, int32_t lo, int32_t hi);
int  ovcs_set_switches(ovcs_t *h, const uint8_t *switches /* [batch] SWCHB pins, NULL = 0x3F */);
int  ovcs_boot(ovcs_t *h, const uint8_t *mask, int32_t noop_frames, int32_t reset_frames, const uint8_t *noop_starts,
               int32_t max_noop_starts, int32_t frameskip);
/* the paper's step unit: latch the actions, then n_instr single-instruction steps (ovcs_step_instruction) per env of [lo,hi) */
int  ovcs_step_instructions_range(ovcs_t *h, const uint8_t *actions, int32_t n_instr, int32_t lo, int32_t hi);
int  ovcs_get_ram(ovcs_t *h, uint8_t *out /* [batch][128] */);
int  ovcs_get_cart_ram(ovcs_t *h, uint8_t *out /* [batch][128]: the Superchip RAM (zeros for carts without) */);
int  ovcs_get_regs(ovcs_t *h, ovcs_regs *out /* [batch] */);
int  ovcs_get_screen(ovcs_t *h, uint8_t *out /* [batch][210][160] */);
int  ovcs_destroy(ovcs_t *h);

/* SOFT-STE forward mode (BASELINE config 5; reading R14 in DESIGN.md §2):
 * ovcs_step_range with every value-carrying ROM/RAM read returned as round(STE(relaxed read at temperature T, hard))
 * and every branch as round(STE(pc_soft(alpha), pc_hard)), float32.  out: HOST [batch][8] doubles per env for this
 * call: sum of soft ROM reads, of soft RAM reads, of branch gates, the three counts, STE/hard mismatches (Theorem 1:
 * always 0) and the largest |soft - hard|. */
int  ovcs_step_soft_range(ovcs_t *h, const uint8_t *actions, int32_t frameskip, double T, double alpha,
                          double *out, int32_t lo, int32_t hi);
/* n single-instruction steps per env in SOFT-STE (full = 0) or FULL mode (full = 1: PAPER.md appendix D, the fully
 * relaxed forward whose casts act on the executed values; ovcs_soft.inc); out as above. */
int  ovcs_step_instructions_soft_range(ovcs_t *h, const uint8_t *actions, int32_t n_instr, double T, double alpha, int full,
                                       double *out, int32_t lo, int32_t hi);
/* the soft primitives themselves, for the pins: eq. (6), eq. (10) with window K, eq. (8), eq. (9) in float32 */
double ovcs_soft_peek(const double *r, int M, int a);
double ovcs_soft_peek_relaxed(const double *r, int M, int a, double T, int K);
double ovcs_soft_gate(double alpha, int s, double f);
float  ovcs_soft_ste(float soft, float hard);

/* Test hooks: one env at a time. */
int  ovcs_set_action(ovcs_t *h, int32_t env, int32_t action);  /* latch pins only (C.11)  */
int  ovcs_step_instruction(ovcs_t *h, int32_t env);             /* returns frame-end events */
int  ovcs_tick(ovcs_t *h, int32_t env);                         /* one idle CPU cycle       */
int  ovcs_tick_trace(ovcs_t *h, int32_t env, int32_t n, uint8_t *timer_out, uint8_t *tflag_out); /* n idle cycles, timer / flag after each */
int  ovcs_get_debug(ovcs_t *h, int32_t env, ovcs_debug *out);
int  ovcs_get_back(ovcs_t *h, int32_t env, uint8_t *out /* [210][160] */);
int  ovcs_set_cpu(ovcs_t *h, int32_t env, int a, int x, int y, int sp, int p, int pc); /* <0 = keep */
int  ovcs_poke_ram(ovcs_t *h, int32_t env, int idx, int value);

/* Bare ALU entry points for the brute-force pins (C.6).  flags in/out use the P layout. */
void ovcs_alu_adc(int a, int m, int p_in, int *a_out, int *p_out);
void ovcs_alu_sbc(int a, int m, int p_in, int *a_out, int *p_out);
/* splitmix64: advances *state, returns the draw. */
uint64_t ovcs_splitmix64(uint64_t *state);

#ifdef __cplusplus
}
#endif
#endif
