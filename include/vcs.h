/* include/vcs.h — C ABI of libvcsb200: a batched, cycle-exact Atari 2600 VCS (hard mode) on one B200.
 *
 * The operation: §1 / L55 Fig. 1 / L61 — a 6507 CPU executing cartridge ROM, a TIA that
 * turns register writes into pixels cycle by cycle, a RIOT (128 B RAM, interval timer, joystick/switch
 * I/O), bank-switched cartridges; hard mode per L73 §3 ("opcode bytes index an integer dispatch table,
 * the ALU is integer arithmetic, and flags are bits"); output frame 210x160 palette indices (L69, L167);
 * deterministic given ROM, action stream and seed (L63).  The register-level machine model is
 * SURVEY.md §8(c) C.1–C.12, restated in DESIGN.md §2–3.  Entry points follow SURVEY.md §8(b).
 *
 * Conventions
 *   - Every function returns VCS_OK (0) or a negative error; none throws or aborts.
 *   - "host" pointers are ordinary CPU memory, "device" pointers are CUDA device memory of the GPU that
 *     was current when vcs_create ran.  No torch types cross this boundary.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  vcs_reset,
 *     vcs_step* and vcs_get_* only enqueue work on that stream and return; ordering is stream ordering.
 *     The only calls that wait for the GPU are vcs_create / vcs_destroy (whole device), the *_host conveniences
 *     (their own copies), vcs_block_times, vcs_issue_peak, and vcs_step_soft when the temperature CHANGES (it waits
 *     for its own previous upload of the weight table from the handle's pinned buffer, long since finished).
 *   - One stream per handle: all calls on a handle must be issued on one stream, or be ordered by the caller (events)
 *     as if they were.  The library keeps per-handle device state between calls (environment state, the block
 *     placement of the next step, the soft-mode tables) and orders its own work by that stream alone.
 *   - One device per handle: the CUDA device that was current in vcs_create must be current in every later call on
 *     that handle (VCS_EINVAL otherwise; vcs_destroy switches to it itself).
 *   - The library owns all per-environment state and the front screen buffer.  The caller owns the
 *     action buffer and every output buffer.  roms / env_rom / seeds are copied by vcs_create.
 *   - There is no CPU fallback: without a CUDA device vcs_create returns VCS_ECUDA.
 */
#ifndef VCS_H
#define VCS_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct vcs_s *vcs_t;

enum { VCS_OK = 0, VCS_EINVAL = -1, VCS_ECUDA = -2, VCS_ENOMEM = -3, VCS_EROM = -4 };

/* Cartridge formats ("cartridge mappers", L469: 2K, 4K, F8, F6, F4, F8SC, F6SC, F4SC, E0, FE; SURVEY C.9,
 * §8(f) NEXT-3; behaviour per the public descriptions of these boards, power-up states are readings R15 / R16 of DESIGN.md):
 *   2K / 4K        no switching (2K mirrored)
 *   F8 / F6 / F4   8 / 16 / 32 KB in 4 KB banks; ANY bus access to $1FF8-9 / $1FF6-9 / $1FF4-B selects the bank before the
 *                  access returns data ("writes to special addresses swap which 4KB ROM page is visible")
 *   ..SC           the same plus 128 bytes of cartridge (Superchip) RAM in every bank: write port $1000-$107F, read port
 *                  $1080-$10FF; power-on contents = draws 17-32 of the env's seed stream
 *   E0             8 KB in 1 KB slices; the windows at $1000 / $1400 / $1800 show the slice chosen by any access to
 *                  $1FE0-7 / $1FE8-F / $1FF0-7 (power-up: 4, 5, 6), the window at $1C00 always shows slice 7
 *   FE             8 KB in two banks; the bus access that FOLLOWS one to $01FE selects the bank from bit 5 of its data
 *                  (1: bank 0 = the $F000 page, 0: bank 1 = the $D000 page); power-up bank 0
 * VCS_MAP_BY_SIZE (0) takes 2K / 4K / F8 / F6 / F4 from the image size.  F6 / F4 (+SC) images are read from global
 * memory; Superchip, E0 and FE carts run their out-of-line instructions on the generic executor (slower, same results)
 * and are not available to vcs_step_soft. */
enum { VCS_MAP_BY_SIZE = 0, VCS_MAP_2K, VCS_MAP_4K, VCS_MAP_F8, VCS_MAP_F6, VCS_MAP_F4, VCS_MAP_F8SC, VCS_MAP_F6SC, VCS_MAP_F4SC,
       VCS_MAP_E0, VCS_MAP_FE };
/* One cartridge image (host memory): size 2048 / 4096 / 8192 / 16384 / 32768 and its format (VCS_MAP_*). */
typedef struct { const uint8_t *data; uint32_t size; uint32_t mapper; } vcs_rom;
/* Content-based format guess (PAPER.md L69 / L469 "mapper auto-detected by the ports"; the rules are this build's reading
 * R17): the size fixes the family; an image whose banks all start with 256 equal bytes is a Superchip one;
 * among 8 KB images, E0 / FE are told from F8 by the absolute operands of their code ($1FE0-$1FF7 accesses, JSR / JMP into
 * the $D000 page).  HOST call, no GPU needed.  Returns VCS_MAP_2K .. VCS_MAP_FE, VCS_EROM for a size no format has. */
int vcs_detect_mapper(const uint8_t *data_host, uint32_t size);

/* y0: scanline shown as screen row 0 (default 34);  max_lines: frame cap in scanlines (default 320, 1..65535) — a
 * frame that has not ended by a VSYNC 1->0 write after max_lines*76 CPU cycles is ended at the next instruction
 * boundary;  f8_start_bank: bank selected at reset for 8 KB images (default 1);  flags: VCS_F_* below.
 * y0 must be >= 2.  Why: the scanline in progress when a frame ends becomes line 0 of the next frame (C.10), and a
 * step returns right after the instruction that ended its last frame — so the pixels of line 0 (and the first cycles
 * of line 1, when that instruction runs over the line end) are drawn before the call that will finish THEIR frame has
 * begun.  The kernel keeps no back buffer between calls (rows go straight to the front screen in the call that
 * completes the frame), so those two lines are never shown; every console kernel spends them in VSYNC anyway. */
typedef struct { int32_t y0, max_lines, f8_start_bank; uint32_t flags; } vcs_config;
/* vcs_config.flags — launch-shape and decode switches.  PERFORMANCE ONLY: a handle computes the same bytes with any
 * combination (tests/test_gpu_flags.py steps every one of them against the default).  0 = the library's own choice. */
enum {
  VCS_F_NO_SPIN    = 1u << 0,   /* run timer wait loops poll by poll instead of in closed form                 */
  VCS_F_NO_FUSE    = 1u << 1,   /* no fused "LDx #imm ; STx <TIA register>" decode entries                     */
  VCS_F_NO_REGROUP = 1u << 2,   /* F8 blocks do not re-sort their envs by bank at hotspot accesses             */
  VCS_F_ROM_GLOBAL = 1u << 3,   /* cartridge bytes through the read-only cache instead of shared memory        */
  VCS_F_NO_BALANCE = 1u << 4,   /* blocks run env groups in env order (no measured placement)    */
  VCS_F_NO_PROMOTE = 1u << 5,   /* indexed / indirect / stack instructions always run in the out-of-line executor */
  VCS_F_BLOCK_64   = 1u << 8, VCS_F_BLOCK_128 = 2u << 8, VCS_F_BLOCK_256 = 3u << 8, VCS_F_BLOCK_MASK = 3u << 8,  /* envs per block */
  VCS_F_ALL = 0x33Fu
};

/* 32 bytes per environment, little-endian. */
typedef struct {
  uint64_t cycles;           /* CPU cycles since reset, WSYNC stalls included                     */
  uint32_t frame;            /* completed frames since reset                                       */
  uint16_t pc; uint8_t a, x, y, sp, p;   /* p: bit5 always 1, bit4 always 0                        */
  uint8_t  bank;             /* current cartridge bank                                             */
  uint16_t line; uint8_t cyc_in_line;    /* beam: scanline in frame, cycles % 76                   */
  uint8_t  status;           /* bit0 halt on an unimplemented (undocumented) opcode, bit1 frame cap was hit */
  uint8_t  intim, timint, _pad[6];       /* timer value and TIMINT bit 7, read without side effects.  _pad[0]: E0 — slice shown
                                            at $1800 (`bank` = slice at $1000 | slice at $1400 << 3); FE — 1 while an access to $01FE
                                            awaits its successor; 0 otherwise */
} vcs_regs;

/* Create `batch` consoles.  roms[n_roms], env_rom[batch] (index into roms; NULL = all 0) and
 * seeds[batch] are HOST arrays.  seeds[e] seeds env e's power-on RAM: the first 16 draws of
 * splitmix64(seeds[e]), little-endian.  cfg NULL = defaults.
 * On return every env is in its reset state (C.2) and the screens are zero.
 * Layout hint (performance only, never results): when every aligned group of 256 (batches >= 32768), 128 or 64
 * consecutive envs shares one ROM, the ROM is staged in shared memory per block and F8 carts regroup their envs by
 * bank inside the block; otherwise ROM bytes come through the read-only cache.  cfg->flags (VCS_F_*) overrides these
 * choices; the library reads nothing from the process environment.
 * Errors: VCS_EINVAL (NULL/size/range/unknown flag), VCS_EROM (no such format, or the size is not the format's), VCS_ECUDA, VCS_ENOMEM. */
int vcs_create(vcs_t *out, int32_t batch, const vcs_rom *roms, int32_t n_roms,
               const int32_t *env_rom, const uint64_t *seeds, const vcs_config *cfg);

/* Reset the envs with mask_dev[e] != 0 (DEVICE uint8[batch]; NULL = all) to the C.2 state. */
int vcs_reset(vcs_t h, const uint8_t *mask_dev, void *cuda_stream);

/* One env-step for every env: latch the action (DEVICE uint8[batch]; ALE numbering 0..17, >= 18 is
 * NOOP — SURVEY C.11) into SWCHA / INPT4, then run whole instructions until `frameskip` frame-end
 * events have occurred (C.10).  The last completed frame becomes the front screen.
 * frameskip must satisfy 1 <= frameskip and frameskip*max_lines*76 < 2^31. */
int vcs_step(vcs_t h, const uint8_t *actions_dev, int32_t frameskip, void *cuda_stream);

/* vcs_step for a subset: envs with mask_dev[e] == 0 (DEVICE uint8[batch]; NULL = every env steps) stay frozen —
 * no state, cycle counter, frame counter or screen byte of theirs changes.  Environments are independent
 * (PAPER.md L63), so the others end exactly where vcs_step would have put them.  Used by vcs_boot for per-env
 * episode starts; errors as vcs_step. */
int vcs_step_masked(vcs_t h, const uint8_t *actions_dev, int32_t frameskip, const uint8_t *mask_dev, void *cuda_stream);

/* The paper's own step unit ("one step = one CPU instruction"; Table 8 "rollout length 3,000 CPU
 * instructions"): latch the actions as vcs_step does, then execute exactly n_instr whole
 * instructions per env (1 <= n_instr <= 1,000,000).  Frames end on the way as they would in vcs_step (VSYNC 1->0 or the
 * cap; a frame end at the cap is not an instruction) and are counted in vcs_regs.frame; a halted env (status bit 0)
 * spends one idle CPU cycle per instruction.  CPU, RAM, RIOT and TIA state (collision latches, positions, beam) after
 * the call are those of the oracle after the same n_instr single-instruction steps.  The FRONT SCREEN IS NOT UPDATED:
 * rows are produced by vcs_step only, and the first frame a following vcs_step completes may lack the rows this call
 * ran through (with frameskip >= 2 the frame vcs_step shows lies wholly inside that call).  Errors as vcs_step. */
int vcs_step_instructions(vcs_t h, const uint8_t *actions_dev, int32_t n_instr, void *cuda_stream);

/* Console switches (SURVEY.md §8(f) NEXT-4 "console switches as inputs"; C.7 port B): switches_dev[e] (DEVICE
 * uint8[batch], copied) is the level of the SWCHB input pins of env e — bit 0 RESET and bit 1 SELECT (0 = pressed),
 * bit 3 colour (1) / b&w (0), bits 6 / 7 difficulty P0 / P1; pins 2, 4 and 5 are not connected and always read 1.
 * NULL restores the default 0x3F (nothing pressed, colour, both difficulties B).  The value stays until the next
 * call; vcs_reset does not touch it.  A read of SWCHB returns (ORB & DDRB) | (pins & ~DDRB). */
int vcs_set_switches(vcs_t h, const uint8_t *switches_dev, void *cuda_stream);

/* ALE-style episode start for the envs with mask_dev[e] != 0 (NULL = all) — PAPER.md L167 "the standard ALE boot
 * (60 no-op frames plus four resets)", Table 8 "Boot sequence: 60 NOOP + 4 RESET frames; episode-start
 * randomization: 0-30 random NOOPs (Mnih-style)"; SURVEY.md §8(f) NEXT-4.  In order: vcs_reset(mask); noop_frames
 * single-frame steps with action NOOP; reset_frames single-frame steps with NOOP and the RESET switch held (bit 0
 * of the env's switch byte forced low, released afterwards); then, if noop_starts_dev != NULL (DEVICE
 * uint8[batch], drawn by the caller), min(noop_starts_dev[e], max_noop_starts) env-steps of `frameskip` frames with
 * NOOP for env e.  All other envs stay frozen.  Enqueues noop_frames + reset_frames + max_noop_starts step kernels.
 * 0 <= noop_frames, reset_frames; 0 <= max_noop_starts <= 255; frameskip as vcs_step.  Errors as vcs_step. */
int vcs_boot(vcs_t h, const uint8_t *mask_dev, int32_t noop_frames, int32_t reset_frames,
             const uint8_t *noop_starts_dev, int32_t max_noop_starts, int32_t frameskip, void *cuda_stream);

/* The same episode start, amortised: instead of stepping the booting envs on their own (vcs_boot: dozens of launches
 * that run a handful of envs each), the envs with mask_dev[e] != 0 (NULL = all) are reset and ARMED, and the boot
 * runs inside the following vcs_step / vcs_step_masked / vcs_step_soft calls of the whole batch: for its first
 * noop_steps steps an armed env ignores the caller's action (NOOP), for the next reset_steps steps it also has the
 * RESET switch held, then it takes min(noop_starts_dev[e], max_noop_starts) more NOOP steps, and from the next step
 * on it follows the caller's actions.  One "step" here is one env-step of whatever frameskip the caller passes: with
 * frameskip 4, noop_steps 15 and reset_steps 1 are the paper's 60 NOOP + 4 RESET frames (inputs are latched once
 * per vcs_step, and the protocol's inputs only change at those frame counts, so the frames are the same ones
 * vcs_boot runs — tests/test_gpu_ale.py).  No extra step launches; frozen envs (vcs_step_masked) do not count down.
 * noop_steps + reset_steps + max_noop_starts <= 255.  vcs_reset / vcs_boot disarm the envs they touch. */
int vcs_auto_reset(vcs_t h, const uint8_t *mask_dev, int32_t noop_steps, int32_t reset_steps,
                   const uint8_t *noop_starts_dev, int32_t max_noop_starts, void *cuda_stream);
/* out_dev[e] (DEVICE uint8[batch]) = boot steps env e still has to run (0 = it follows the caller's actions). */
int vcs_get_booting(vcs_t h, uint8_t *out_dev, void *cuda_stream);

/* SOFT-STE forward step (BASELINE config 5; "Hard and Soft Execution", eq. (1)-(4), appendix
 * eq. (6)-(10), L316 "Numerical scope"; reading R14 in DESIGN.md §2).  Same as vcs_step, but every value-carrying
 * read of cartridge ROM (the bank the CPU sees as a 4096 x 8 {0,1} bit tensor) or RIOT RAM (a 128-cell tape) is
 * computed as round(STE(soft, hard)) with soft = the relaxed read of eq. (10) at temperature T (window
 * |k| <= ceil(17 T), clipped to the tensor, normalised over the cells kept), in float32, and every conditional
 * branch sets PC = round(STE(pc_nb + sigma(alpha z) delta, pc_hard)).  Dispatch is the hard switch.  By the paper's
 * Theorem 1/3 the resulting state equals vcs_step's bit for bit.
 * soft_out_dev: DEVICE float[batch][8], overwritten with this call's per-env sums: soft ROM reads, soft RAM reads,
 * branch gates, the three counts, reads/branches whose rounded STE value differed from the hard one (always 0),
 * max |soft - hard|.  0 < T <= 60, alpha finite.  Errors as vcs_step. */
int vcs_step_soft(vcs_t h, const uint8_t *actions_dev, int32_t frameskip, float T, float alpha,
                  float *soft_out_dev, void *cuda_stream);

/* The soft modes in the paper's own step unit (forward part): latch the actions, then
 * exactly n_instr instructions per env as vcs_step_instructions, with the soft primitives of vcs_step_soft.
 *   full = 0  SOFT-STE: the state equals vcs_step_instructions' bit for bit (Theorem 1/3).
 *   full = 1  FULL, the fully relaxed forward of PAPER.md appendix D (L425-459; Table 2; reading R18 in
 *             DESIGN.md §2): no straight-through correction — a value read returns round(soft), a conditional branch
 *             sets PC = round(pc_nb + sigma(alpha z) delta), both cast in float32; dispatch stays the hard switch on the
 *             (cast) opcode byte; an instruction's cycles and discarded reads follow its hard branch decision.  The
 *             state equals hard mode's exactly while every cast rounds to the hard value (for every program when
 *             alpha >= 6 and T <= 0.14, L459) and leaves it at the first cast that does not (Table 3's N_div).  The soft
 *             values are evaluated tap by tap in double with the host's e^{-k/T} and gates, so that the casts are the
 *             oracle's casts: this mode is exact, not fast.
 * soft_out_dev as for vcs_step_soft; entry 6 counts the casts of this call that did not round to the hard value.
 * 1 <= n_instr <= 1,000,000; 0 < T <= 60, alpha finite; Superchip / E0 / FE cartridges: VCS_EINVAL. */
int vcs_step_instructions_soft(vcs_t h, const uint8_t *actions_dev, int32_t n_instr, float T, float alpha, int32_t full,
                               float *soft_out_dev, void *cuda_stream);

/* Copies into caller-owned DEVICE buffers. */
int vcs_get_ram(vcs_t h, uint8_t *out_dev /* [batch][128] */, void *cuda_stream);
int vcs_get_regs(vcs_t h, vcs_regs *out_dev /* [batch] */, void *cuda_stream);
int vcs_get_cart_ram(vcs_t h, uint8_t *out_dev /* [batch][128]: Superchip RAM, zeros for carts without */, void *cuda_stream);
int vcs_get_screen(vcs_t h, uint8_t *out_dev /* [batch][210][160] */, void *cuda_stream);

/* Convenience for hosts without their own device buffers: vcs_step / vcs_get_* with HOST pointers.
 * The host<->device copies run on `cuda_stream`; the call returns after they complete. */
int vcs_step_host(vcs_t h, const uint8_t *actions_host, int32_t frameskip, void *cuda_stream);
int vcs_get_ram_host(vcs_t h, uint8_t *out_host, void *cuda_stream);
int vcs_get_regs_host(vcs_t h, vcs_regs *out_host, void *cuda_stream);
int vcs_get_screen_host(vcs_t h, uint8_t *out_host, void *cuda_stream);

/* A host-buffer step that allocates NOTHING, for callers that may not call cudaMalloc while they run (code under CUDA
 * graph capture, tight serving loops, harnesses that forbid it).  The calls above allocate their pinned / device stage
 * on first use (and when the batch grows); this one stages in a static device array that is part of the library:
 * VCS_NOALLOC_MAX_BATCH envs x (1 + 128 + 32) bytes + 256 = 10,551,552 bytes, held by every GPU that loads the library
 * until the process exits.  One call = vcs_step(actions, frameskip) followed by the read-back of RAM and registers:
 *   actions_host    HOST uint8[batch]       (in)   as vcs_step_host
 *   ram_out_host    HOST uint8[batch][128]  (out)  as vcs_get_ram_host
 *   regs_out_host   HOST vcs_regs[batch]    (out)  as vcs_get_regs_host
 *   n_flagged_host  HOST int32              (out)  number of envs whose vcs_regs.status is non-zero after the step
 * Everything is ENQUEUED on `cuda_stream` and the call returns: the outputs are valid once the caller has synchronised
 * that stream, and all four host buffers must stay valid until then (pinned host memory for copies that really are
 * asynchronous; under stream capture it must be pinned).  No cudaMalloc, cudaFree or other allocating call is made;
 * the first call on a device takes the array's address (cudaGetSymbolAddress), so make one call before capturing.
 * Errors: VCS_EINVAL when batch > VCS_NOALLOC_MAX_BATCH (vcs_last_error says so), on a NULL buffer, a frameskip out of
 * range or a device index above 63; VCS_ECUDA as vcs_step.
 * SHARED SCRATCH: every call of the process on one GPU, whatever its handle, uses the same array, which keeps the last
 * call's contents (the call clears the one word that must start at zero and overwrites the rest before reading it).
 * Calls on ONE stream are ordered and safe; calls that can overlap on the GPU — two streams, two threads, two handles
 * — race on the array and return garbage: serialise them. */
#define VCS_NOALLOC_MAX_BATCH 65536
int vcs_step_host_noalloc(vcs_t h, const uint8_t *actions_host, int32_t frameskip, uint8_t *ram_out_host,
                          vcs_regs *regs_out_host, int32_t *n_flagged_host, void *cuda_stream);

/* Device pointer to the library-owned front screen [batch][210][160] (valid until vcs_destroy; contents
 * change with every vcs_step).  Zero-copy alternative to vcs_get_screen. */
int vcs_screen_ptr(vcs_t h, const uint8_t **out_dev_ptr);

/* Block placement introspection (performance only).  A step runs ceil(batch / block) thread blocks, all resident at
 * once; the library records when and on which SM each block of the last plain vcs_step ran and re-assigns env groups
 * to block indices so that the SMs finish together (VCS_F_NO_BALANCE turns it off; handles with more
 * than 1024 blocks — batches above 262,144 — keep env order).
 * *n_out = number of blocks; if cap >= n: times_host[3 * b + 0..2] = start ns, end ns (GPU global timer), SM id of
 * block index b in the last plain vcs_step, perm_host[b] = the env group (envs perm*block .. +block-1) block b runs
 * next.  Either pointer may be NULL.  Synchronises the device. */
int vcs_block_times(vcs_t h, uint64_t *times_host, int32_t *perm_host, int32_t cap, int32_t *n_out);

/* Number of kernel launches this handle has enqueued so far (bench bookkeeping). */
int64_t vcs_launch_count(vcs_t h);

/* Introspection, no GPU needed: copies the interpreter's 256-entry decode table (HOST uint16[256];
 * entry = addressing mode | operation<<4 | access kind<<10, operation 0 = a byte that halts the CPU) so that a
 * CPU-only test can check it against the documented 151-opcode matrix plus the paper's 38 undocumented bytes
 * (USBC, the NOP / LAX / SAX family) that also execute (R12). */
int vcs_optable(uint16_t *out256_host);

/* Integer-issue micro-benchmark on the current CUDA device: the denominator of the interpreter's roofline
 * ("the builder must first run an integer micro-benchmark"; "compute/occupancy-
 * bound, not memory-bound").  kind 0 = alu pipe only (LOP3 + SHF chains; ptxas moves plain adds to the fma pipe as IMAD.IADD), kind 1 = alu + fma pipes interleaved
 * (LOP3 + IMAD).  Fills every SM with 2048 threads, each running 8 independent chains for `iters` loop trips of
 * 256 instructions; writes thread-instructions per second (best of 3 after a warm-up run) to
 * *thread_instr_per_s (HOST) and the duration of that run to *seconds (HOST, may be NULL).  Synchronous; uses
 * the legacy default stream.  Errors: VCS_EINVAL, VCS_ECUDA, VCS_ENOMEM. */
int vcs_issue_peak(int32_t kind, int32_t iters, double *thread_instr_per_s, double *seconds);

int vcs_destroy(vcs_t h);
const char *vcs_last_error(vcs_t h);     /* handle-owned string; "" when no error. h may be NULL */

#ifdef __cplusplus
}
#endif
#endif
