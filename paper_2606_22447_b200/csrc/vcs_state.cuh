// vcs_state.cuh — state layout of libvcsb200 (the CUDA path; shares nothing with oracle/).
//
// In HBM, per environment, structure-of-arrays so that a warp's loads/stores coalesce:
//   st   [ST_WORDS][batch] u32   packed CPU / beam / RIOT / TIA latches (word index below)
//   ram  [32][batch]       u32   the 128 RIOT RAM bytes, little-endian words
//   cyc  [batch]           u64   CPU cycles since reset
//   screen [batch][210][160] u8  front frame, palette indices
// In shared memory, while vcs_step runs: one "file" of S_WORDS words per thread, word i of thread t at
// smem[i * BLOCK + t] (word-interleaved, so a warp's accesses never bank-conflict whatever per-lane
// addresses are used), followed by a per-block context, the 256-entry decode table and the block's ROM.
// Machine model: SURVEY.md §8(c) C.1 (state), restated in DESIGN.md §2.
#pragma once
#include <stdint.h>
#include <cuda_runtime.h>

namespace vcs {

constexpr int SCR_W = 160, SCR_H = 210, LINE_CYC = 76, HBLANK = 68, LINE_CLK = 228;

enum StWord {
  W_AXYS = 0,   // A | X<<8 | Y<<16 | SP<<24
  W_PC,         // PC | P<<16 | status<<24
  W_BEAM,       // n (cycle in line, 0..76) | line<<8 (16 bit) | bank<<24
  W_FRAME,      // completed frames since reset
  W_FCYC,       // cycles since the current frame began
  W_TIMER,      // timer | shift<<8 | tflag<<12 | sub<<16
  W_PORTS,      // ora | ddra<<8 | orb<<16 | ddrb<<24
  W_COLU,       // COLUP0 | COLUP1<<8 | COLUPF<<16 | COLUBK<<24
  W_PF,         // PF0 | PF1<<8 | PF2<<16 | CTRLPF<<24
  W_GRP,        // GRP0_new | GRP0_old<<8 | GRP1_new<<16 | GRP1_old<<24
  W_NUSIZ,      // NUSIZ0 | NUSIZ1<<8 | HMP0<<16 | HMP1<<20 | HMM0<<24 | HMM1<<28
  W_POS,        // posP0 | posP1<<8 | posM0<<16 | posM1<<24
  W_POS2,       // posBL | HMBL<<8 | rx<<16 (colour clocks of the current line already rendered, 0..228)
  W_FLAGS,      // TIA / input flag bits, see TF_* (only the bits below TF_DIRTY0 are architectural)
  W_CX,         // 15 collision latches
  W_CART,       // E0: slice shown at $1000 | at $1400 << 3 | at $1800 << 6 ; FE: bit 9 = the previous access was to $01FE
  ST_WORDS
};
// cartridge formats (the numbers are include/vcs.h's VCS_MAP_*)
enum MapKind : uint32_t { MK_2K = 1, MK_4K, MK_F8, MK_F6, MK_F4, MK_F8SC, MK_F6SC, MK_F4SC, MK_E0, MK_FE };
constexpr uint32_t HS_SC = 1u << 31;       // RomMeta::hs / C_HS: the first 256 bytes of every bank are the Superchip RAM ports

// W_FLAGS bits
enum : uint32_t {
  TF_VSYNC = 1u << 0, TF_VBLANK = 1u << 1, TF_LATCHEN = 1u << 2, TF_WSYNC = 1u << 3,
  TF_REFP0 = 1u << 4, TF_REFP1 = 1u << 5, TF_ENAM0 = 1u << 6, TF_ENAM1 = 1u << 7,
  TF_ENABL_NEW = 1u << 8, TF_ENABL_OLD = 1u << 9, TF_VDELP0 = 1u << 10, TF_VDELP1 = 1u << 11,
  TF_VDELBL = 1u << 12, TF_RESMP0 = 1u << 13, TF_RESMP1 = 1u << 14,
  TF_FRESH_P0 = 1u << 15, TF_FRESH_P1 = 1u << 16, TF_FRESH_M0 = 1u << 17, TF_FRESH_M1 = 1u << 18,
  TF_HMBLANK = 1u << 19, TF_INPT4_LATCH = 1u << 20, TF_INPT5_LATCH = 1u << 21,
  TF_FRESH_ALL = TF_FRESH_P0 | TF_FRESH_P1 | TF_FRESH_M0 | TF_FRESH_M1,
  TF_ARCH_MASK = (1u << 22) - 1u,
  // kernel-only, derived (never stored to HBM): cached object line masks that must be rebuilt, row visibility
  TF_DIRTY0 = 1u << 22,            // << object index: PF, BL, P0, P1, M0, M1
  TF_DIRTY_ALL = 63u << 22,
  TF_ROWVIS = 1u << 28,            // the scanline in progress is a screen row of a frame whose pixels are kept
  TF_STORING = 1u << 29,           // the frame in progress is the last one of this vcs_step: its pixels are kept
};
enum { OB_PF = 0, OB_BL, OB_P0, OB_P1, OB_M0, OB_M1 };

// collision latch bit numbers inside W_CX (read map: SURVEY C.8)
enum { CX_M0P1 = 0, CX_M0P0, CX_M1P0, CX_M1P1, CX_P0PF, CX_P0BL, CX_P1PF, CX_P1BL,
       CX_M0PF, CX_M0BL, CX_M1PF, CX_M1BL, CX_BLPF, CX_P0P1, CX_M0M1 };

enum : uint32_t { STATUS_ILLEGAL = 1, STATUS_CAP = 2 };

// per-thread shared-memory file (word index; word i of thread t lives at smem[i*BLOCK + t])
enum SmWord {
  S_RAM = 0,                       // 32 words: the 128 RAM bytes
  S_PLANE = 32,                    // 10 words: colour-index bit planes of the scanline in progress (i0[5], i1[5])
  S_BUDGET = 32,                   // vcs_step_instructions only (it keeps no rows, so the planes are free): instructions left to run
  S_COLU = 42, S_PF, S_GRP, S_NUSIZ, S_POS, S_POS2,   // TIA registers, packed as the W_* words (S_POS2 without rx)
  S_CX, S_FL, S_RX, S_PX,          // collision latches, flags, clocks rendered, pixels painted of the current line
  S_LINE, S_FDONE,                 // scanline in frame, frames completed in this step
  S_PORTS, S_INP,                  // RIOT port latches; ina | fire0<<8 | switches (5 pins)<<9 | (env index inside the block)<<16
  S_TMR, S_TTICKS,                 // timer state packed as W_TIMER, valid after S_TTICKS cycles of this step
  S_STATUS, S_FSTART,              // status bits | ROM index << 8; value of the step's cycle count at which the current frame began
  S_CART,                          // W_CART: E0 window slices, FE's pending bit
  S_OBJ = 61,                      // 30 words: cached 160-bit line masks of PF, BL, P0, P1, M0, M1 (5 words each);
                                   //           a derived cache — also the scratch area of a regroup (vcs_step.cu)
  S_WORDS = 91,
  S_MOVED = S_OBJ + 8              // a regroup moves words [0, S_MOVED): the state proper + 8 words of saved CPU registers
};
static_assert(S_STATUS == 58 && S_CART == 60, "file layout");
// per-block context, in words after the thread files (block-uniform values the out-of-line paths need)
enum CtxWord { C_SCREEN_LO = 0, C_SCREEN_HI, C_Y0, C_FRAMESKIP, C_BATCH, C_ENV0, C_CAP, C_ROMOFF, C_REGROUP,
               C_META_LO, C_META_HI, C_BLOB_LO, C_BLOB_HI, C_DROM_LO, C_DROM_HI,
               C_SOFT_WD_LO, C_SOFT_WD_HI,     // FULL mode: e^{-k/T} (k <= K) and the two branch gates in double, as the host computed them
               C_SOFT_W_LO, C_SOFT_W_HI, C_SOFT_K, C_SOFT_ALPHA, C_SOFT_TAB_LO, C_SOFT_TAB_HI,
               C_HS,           // bank hotspots of the block's ROM (ROM staged in smem: one ROM per block): first address | count << 16 | HS_SC
               C_SCRAM_LO, C_SCRAM_HI,     // Superchip RAM of all envs, [32][batch] words like `ram` (nullptr when no cart has it)
               C_ROMG_LO, C_ROMG_HI,       // the block's ROM image in global memory (one ROM per block; read there when it is not staged, C_ROMOFF then = offset mask)
               C_WORDS = 28 };         // (a multiple of 4: the ROM image staged behind the context is a 16-byte aligned bulk-copy target)
static_assert(C_WORDS % 4 == 0 && C_ROMG_HI < C_WORDS, "context layout");
static_assert(C_HS < C_WORDS, "context layout");

struct RomMeta { uint32_t offset; uint32_t size; uint32_t doff; uint32_t pad;      // byte offset into the ROM blob, size, word offset into the decode blob
                 uint32_t kind; uint32_t hs; };                                      // MapKind ; first hotspot | count << 16 | HS_SC (F8 / F6 / F4 families)

struct Handle {                 // host-side bookkeeping behind vcs_t
  int32_t batch, n_roms;
  int32_t y0, max_lines, f8_start_bank;
  uint32_t *d_st; uint32_t *d_ram; unsigned long long *d_cyc; uint8_t *d_screen;
  uint32_t *d_sc_ram;           // Superchip RAM [32][batch] (only when a cart has it)
  uint8_t *d_rom_blob; uint2 *d_drom; RomMeta *d_rom_meta; int32_t *d_env_rom; unsigned long long *d_seeds;
  int device;                   // the CUDA device every pointer below belongs to
  float *h_soft_w; cudaEvent_t soft_w_done; int soft_K;            // soft mode: pinned e^{-k/T} staging buffer, its upload, window of the cached temperature
  double *d_soft_wd, *h_soft_wd; float soft_wd_T, soft_wd_alpha;   // FULL mode: weights and gates in double (SOFT_WD_WORDS), what they were built for
  uint2 *d_drom_slow;           // FULL mode: a decode table whose every entry says "decode at run time" (allocated on first use)
  float4 *d_soft_ent;           // soft mode: per decode entry of d_drom_soft, the soft sums of the instruction's own bytes at the cached temperature
  float *d_soft_tab; float soft_tab_T; size_t soft_tab_n;          // W(T) x ROM: the relaxed read of every ROM cell at the cached temperature
  uint2 *d_drom_plain;          // vcs_step_instructions: a decode table for 128-env blocks without fused / closed-form entries (one entry = one instruction)
  uint2 *d_drom_soft; RomMeta *d_rom_meta_soft; float *d_soft_w;   // soft mode: a decode table for 128-env blocks, one entry per instruction, indexed / stack instructions out of line; metas with pad = doff; e^{-k/T}
  uint8_t *d_actions_stage;     // for vcs_step_host
  uint8_t *d_switches;          // SWCHB input pins per env (vcs_set_switches; 0x3F after vcs_create)
  int32_t *d_perm; unsigned long long *d_blk_time; long long plain_steps; int balance; float balance_a; float *d_w_avg;   // block placement (rebalance_kernel in vcs_step.cu)
  uint32_t *d_boot_ctr;         // per env: boot steps left | NOOP starts << 8 | RESET steps << 16 (vcs_auto_reset; 0 = playing)
  uint8_t *d_boot;              // vcs_boot scratch: [batch] NOOP actions, [batch] per-iteration mask, [batch] switches with RESET held
  uint8_t *h_pinned; size_t h_pinned_bytes;
  int special_carts;            // some cart is Superchip / E0 / FE (hard mode only)
  int block;                    // threads (= envs) per block of the interpreter kernel
  int regroup;                  // F8 blocks re-sort their envs across threads at bank-hotspot accesses
  int rom_smem;                 // every block maps to a single ROM (the ROMS kernel variants: hot-path ROM reads, regroup)
  int rom_staged;               // ... and the images are small enough (<= 8 KB) to be staged in shared memory
  int banked;                   // some cartridge is an F8 / F6 / F4 (with or without Superchip RAM): its blocks regroup at bank switches (spare warp)
  uint32_t max_rom;             // largest ROM image
  long long launches;
  char err[256];
};

}  // namespace vcs
