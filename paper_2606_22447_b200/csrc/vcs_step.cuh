// vcs_step.cuh — launch interface between the host API (vcs_api.cu) and the kernels.
#pragma once
#include <cuda_runtime.h>
#include "vcs_state.cuh"

namespace vcs {


constexpr int SOFT_WD_GATE = 1024, SOFT_WD_WORDS = 1026;     // soft_wd: e^{-k/T} in double, k < 1024; then sigma(alpha), sigma(-alpha)
constexpr int SOFT_W_N = 1024, SOFT_CW = SOFT_W_N, SOFT_W_WORDS = SOFT_W_N + 128;   // soft_w: e^{-k/T}, k < 1024; then cw[n] = sum_{j<=n} e^{-j/T}, n < 128
struct StepParams {
  uint32_t *st; uint32_t *ram; unsigned long long *cyc; uint8_t *screen; uint32_t *sc_ram;
  const uint8_t *rom_blob; const uint2 *drom; const RomMeta *rom_meta; const int32_t *env_rom;
  const uint8_t *actions; const uint8_t *switches; const uint8_t *mask; uint32_t *boot;
  const int32_t *perm; unsigned long long *blk_time;       // block placement (vcs_step.cu, rebalance_kernel): perm[blockIdx] = env group; blk_time[3 * blockIdx] = start ns, end ns, SM id   // switches: SWCHB input pins per env; mask: nullptr = every env steps; boot: per-env boot countdown (vcs_auto_reset)
  int32_t batch, frameskip, y0, max_lines;
  const float *soft_w; const float *soft_tab; float *soft_out; float soft_alpha; int32_t soft_K;   // soft_out != nullptr: SOFT-STE mode (vcs_step_soft)
  const double *soft_wd; int32_t soft_full;               // FULL mode (vcs_step_instructions_soft, full = 1): casts of the soft values themselves
  const float4 *soft_ent;                                 // ... per decode entry: the soft sums of the instruction's own bytes
  int32_t block, rom_smem, regroup; uint32_t max_rom;     // launch shape: envs per block (64/128/256), one ROM per block, regroups allowed, largest image
  int32_t rom_staged, banked;                             // the block's ROM is staged in smem (images <= 8 KB); some cartridge is a plain F8 / F6 / F4
  int32_t n_instr;                                        // > 0: vcs_step_instructions — run this many instructions per env instead of `frameskip` frames
};

void upload_optable();
const uint16_t *host_optable();
cudaError_t launch_step(const StepParams &p, cudaStream_t stream);
cudaError_t launch_soft_table(const uint8_t *rom_blob, const RomMeta *meta, int n_roms, const float *w, int K, float *tab, cudaStream_t stream);
cudaError_t launch_rebalance(int32_t *perm, const unsigned long long *blk_time, int n, float slowdown, float *w_avg, cudaStream_t stream);
cudaError_t launch_soft_entries(const uint8_t *rom_blob, const RomMeta *meta, int n_roms, const uint2 *drom, const float *tab, float4 *ent, cudaStream_t stream);
size_t step_smem_bytes(int block, bool roms, uint32_t max_rom, bool soft);

}  // namespace vcs
