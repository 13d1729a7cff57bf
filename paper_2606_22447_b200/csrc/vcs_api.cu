// vcs_api.cu — the extern "C" boundary of libvcsb200 (include/vcs.h), plus the small
// reset / read-out kernels.  Argument marshalling and launches only: every step of the emulation runs in
// vcs_step.cu's kernel.  No CPU fallback exists: without a CUDA device vcs_create fails with VCS_ECUDA.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/vcs.h"
#include "vcs_step.cuh"
#include "vcs_decode.cuh"

using namespace vcs;
#ifndef VCS_BALANCE_A
#define VCS_BALANCE_A 1.27f         // measured slowdown of a block that shares its SM
#endif

struct vcs_s : Handle {};

namespace {

int fail(Handle *h, int code, const char *what, cudaError_t ce = cudaSuccess) {
  if (h) {
    if (ce != cudaSuccess) snprintf(h->err, sizeof h->err, "%s: %s", what, cudaGetErrorString(ce));
    else snprintf(h->err, sizeof h->err, "%s", what);
  }
  return code;
}
#define CU(h, call) do { cudaError_t ce_ = (call); if (ce_ != cudaSuccess) return fail(h, VCS_ECUDA, #call, ce_); } while (0)
// every entry point that touches device memory: the handle's GPU must be the current one (its pointers belong to it)
int wrong_device(Handle *h) {
  int d = -1;
  if (cudaGetDevice(&d) != cudaSuccess || d != h->device) return fail(h, VCS_EINVAL, "the handle was created on another CUDA device than the current one");
  return VCS_OK;
}
#define DEV_OK(h) do { if (!(h)) return VCS_EINVAL; if (int rc_ = wrong_device(h)) return rc_; } while (0)

__device__ unsigned long long splitmix64(unsigned long long &s) {
  s += 0x9E3779B97F4A7C15ull;
  unsigned long long z = s;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

// C.2 power-on / reset state
__global__ void reset_kernel(StepParams p, const unsigned long long *seeds, const uint8_t *mask, int f8_start_bank) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= p.batch || (mask && !mask[e])) return;
  const int B = p.batch;
  const RomMeta rm = p.rom_meta[p.env_rom[e]];
  const uint8_t *rom = p.rom_blob + rm.offset;
  const uint32_t bank = (rm.kind == MK_F8 || rm.kind == MK_F8SC) ? (uint32_t)(f8_start_bank & 1) : 0u;      // F6 / F4 / FE power up in bank 0 (readings R15, R16)
  const uint32_t mask_a = (rm.size == 2048) ? 0x7FFu : 0xFFFu;
  const uint32_t vbank = (rm.kind == MK_E0) ? 1u : bank;                             // E0: $1FFC lies in the fixed window = slice 7 = the image's last KB
  const uint32_t pc = rom[(vbank << 12) + (0xFFCu & mask_a)] | ((uint32_t)rom[(vbank << 12) + (0xFFDu & mask_a)] << 8);
  for (int w = 0; w < ST_WORDS; ++w) p.st[w * B + e] = 0;
  p.st[W_AXYS * B + e] = 0xFDu << 24;
  p.st[W_PC * B + e] = pc | (0x24u << 16);
  p.st[W_BEAM * B + e] = bank << 24;
  p.st[W_TIMER * B + e] = 0xFFu | (10u << 8);
  p.st[W_FLAGS * B + e] = TF_INPT4_LATCH | TF_INPT5_LATCH;
  p.st[W_CART * B + e] = (rm.kind == MK_E0) ? (4u | (5u << 3) | (6u << 6)) : 0u;      // E0 power-up slices [R] (R16)
  p.cyc[e] = 0;
  p.boot[e] = 0;
  unsigned long long s = seeds[e];
  for (int k = 0; k < 16; ++k) {
    unsigned long long z = splitmix64(s);
    p.ram[(2 * k) * B + e] = (uint32_t)z;
    p.ram[(2 * k + 1) * B + e] = (uint32_t)(z >> 32);
  }
  if (p.sc_ram) {                                      // Superchip RAM: the next 16 draws (its power-on contents must come from the seed)
    const bool sc = rm.hs & HS_SC;
    for (int k = 0; k < 16; ++k) {
      unsigned long long z = splitmix64(s);
      p.sc_ram[(2 * k) * B + e] = sc ? (uint32_t)z : 0u;
      p.sc_ram[(2 * k + 1) * B + e] = sc ? (uint32_t)(z >> 32) : 0u;
    }
  }
}
__global__ void clear_screen_kernel(uint8_t *screen, const uint8_t *mask) {
  const int e = blockIdx.x;
  if (mask && !mask[e]) return;
  uint4 *dst = reinterpret_cast<uint4 *>(screen + (size_t)e * (SCR_W * SCR_H));
  for (int i = threadIdx.x; i < SCR_W * SCR_H / 16; i += blockDim.x) dst[i] = make_uint4(0, 0, 0, 0);
}
// vcs_boot helpers: NOOP actions + the switch bytes with RESET held (bit 0 low); the mask of one random-NOOP-start round
__global__ void boot_prep_kernel(const uint8_t *sw, uint8_t *zero, uint8_t *sw_reset, int B) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e < B) { zero[e] = 0; sw_reset[e] = sw[e] & 0xFEu; }
}
__global__ void boot_mask_kernel(const uint8_t *mask, const uint8_t *starts, int k, uint8_t *out, int B) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e < B) out[e] = ((!mask || mask[e]) && (int)starts[e] > k) ? 1 : 0;
}
// vcs_auto_reset: arm the boot countdown of the masked envs (after reset_kernel)
__global__ void arm_boot_kernel(const uint8_t *mask, const uint8_t *starts, int noop_steps, int reset_steps, int max_starts, uint32_t *boot, int B) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= B || (mask && !mask[e])) return;
  int k = starts ? (int)starts[e] : 0; if (k > max_starts) k = max_starts;
  boot[e] = (uint32_t)(noop_steps + reset_steps + k) | ((uint32_t)k << 8) | ((uint32_t)reset_steps << 16);
}
__global__ void get_booting_kernel(const uint32_t *boot, uint8_t *out, int B) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e < B) out[e] = (uint8_t)(boot[e] & 0xFFu);
}
__global__ void fill_kernel(uint8_t *dst, uint8_t v, int B) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e < B) dst[e] = v;
}
__global__ void get_ram_kernel(const uint32_t *ram, uint32_t *out, int B) {
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= 32ll * B) return;
  const int e = (int)(idx >> 5), i = (int)(idx & 31);
  out[idx] = ram[(size_t)i * B + e];
}
__global__ void get_regs_kernel(const uint32_t *st, const unsigned long long *cyc, uint4 *out, int B, const RomMeta *meta, const int32_t *env_rom) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= B) return;
  const uint32_t kind = meta[env_rom[e]].kind, cart = st[W_CART * B + e];
  const uint32_t axys = st[W_AXYS * B + e], pcw = st[W_PC * B + e], beam = st[W_BEAM * B + e], tm = st[W_TIMER * B + e];
  const unsigned long long c = cyc[e];
  uint4 lo, hi;
  lo.x = (uint32_t)c; lo.y = (uint32_t)(c >> 32); lo.z = st[W_FRAME * B + e];
  lo.w = (pcw & 0xFFFFu) | ((axys & 0xFFu) << 16) | (((axys >> 8) & 0xFFu) << 24);                 // pc, a, x
  const uint32_t bank = (kind == MK_E0) ? (cart & 0x3Fu) : (beam >> 24);          // E0: slice at $1000 | slice at $1400 << 3
  hi.x = ((axys >> 16) & 0xFFu) | ((axys >> 24) << 8) | (((pcw >> 16) & 0xFFu) << 16) | (bank << 24);   // y, sp, p, bank
  hi.y = ((beam >> 8) & 0xFFFFu) | (((beam & 0xFFu) % LINE_CYC) << 16) | ((pcw >> 24) << 24);                    // line, cyc_in_line, status
  const uint32_t pad0 = (kind == MK_E0) ? (cart >> 6) & 7u : (kind == MK_FE) ? (cart >> 9) & 1u : 0u;   // E0: slice at $1800 ; FE: pending bit
  hi.z = (tm & 0xFFu) | ((((tm >> 12) & 1u) << 7) << 8) | (pad0 << 16);                             // intim, timint, _pad[0]
  hi.w = 0;
  out[2 * e] = lo; out[2 * e + 1] = hi;
}

// the format of an image: the caller's choice when its size fits that format, else (VCS_MAP_BY_SIZE) the plain format of the size
int map_kind(uint32_t size, uint32_t mapper) {
  static_assert((int)VCS_MAP_2K == (int)MK_2K && (int)VCS_MAP_F8 == (int)MK_F8 && (int)VCS_MAP_F4SC == (int)MK_F4SC && (int)VCS_MAP_E0 == (int)MK_E0 &&
                (int)VCS_MAP_FE == (int)MK_FE, "format numbers");
  if (mapper == VCS_MAP_BY_SIZE)
    return size == 2048 ? (int)MK_2K : size == 4096 ? (int)MK_4K : size == 8192 ? (int)MK_F8 : size == 16384 ? (int)MK_F6 : size == 32768 ? (int)MK_F4 : -1;
  uint32_t want = 0;
  switch (mapper) {
    case VCS_MAP_2K: want = 2048; break;  case VCS_MAP_4K: want = 4096; break;
    case VCS_MAP_F8: case VCS_MAP_F8SC: case VCS_MAP_E0: case VCS_MAP_FE: want = 8192; break;
    case VCS_MAP_F6: case VCS_MAP_F6SC: want = 16384; break;  case VCS_MAP_F4: case VCS_MAP_F4SC: want = 32768; break;
    default: return -1;
  }
  return want == size ? (int)mapper : -1;
}

StepParams params_of(Handle *h, const uint8_t *actions, int frameskip) {
  StepParams p;
  p.st = h->d_st; p.ram = h->d_ram; p.cyc = h->d_cyc; p.screen = h->d_screen; p.sc_ram = h->d_sc_ram;
  p.rom_blob = h->d_rom_blob; p.drom = h->d_drom; p.rom_meta = h->d_rom_meta; p.env_rom = h->d_env_rom;
  p.actions = actions; p.switches = h->d_switches; p.mask = nullptr; p.boot = h->d_boot_ctr; p.perm = h->d_perm; p.blk_time = nullptr; p.batch = h->batch; p.frameskip = frameskip; p.y0 = h->y0; p.max_lines = h->max_lines;
  p.block = h->block; p.rom_smem = h->rom_smem; p.regroup = h->regroup; p.max_rom = h->max_rom; p.rom_staged = h->rom_staged; p.banked = h->banked;
  p.soft_w = nullptr; p.soft_tab = nullptr; p.soft_ent = nullptr; p.soft_wd = nullptr; p.soft_full = 0; p.soft_out = nullptr; p.soft_alpha = 0.f; p.soft_K = 0; p.n_instr = 0;
  return p;
}

int ensure_stage(Handle *h, size_t bytes) {
  if (h->h_pinned_bytes >= bytes) return VCS_OK;
  if (h->h_pinned) cudaFreeHost(h->h_pinned);
  if (h->d_actions_stage) cudaFree(h->d_actions_stage);
  h->h_pinned = nullptr; h->d_actions_stage = nullptr; h->h_pinned_bytes = 0;
  CU(h, cudaMallocHost((void **)&h->h_pinned, bytes));
  CU(h, cudaMalloc((void **)&h->d_actions_stage, bytes));
  h->h_pinned_bytes = bytes;
  return VCS_OK;
}

}  // namespace

extern "C" {

int vcs_create(vcs_t *out, int32_t batch, const vcs_rom *roms, int32_t n_roms, const int32_t *env_rom,
               const uint64_t *seeds, const vcs_config *cfg) {
  if (!out) return VCS_EINVAL;
  *out = nullptr;
  if (batch < 1 || !roms || n_roms < 1 || !seeds) return VCS_EINVAL;
  for (int r = 0; r < n_roms; ++r) {
    if (!roms[r].data) return VCS_EINVAL;
    if (map_kind(roms[r].size, roms[r].mapper) < 0) return VCS_EROM;
  }
  if (env_rom) for (int i = 0; i < batch; ++i) if (env_rom[i] < 0 || env_rom[i] >= n_roms) return VCS_EINVAL;
  vcs_config c = {34, 320, 1, 0};
  if (cfg) c = *cfg;
  if (c.y0 < 2 || c.max_lines < 1 || c.max_lines > 65535 || (c.flags & ~(uint32_t)VCS_F_ALL) != 0) return VCS_EINVAL;
  const uint32_t fblock = c.flags & VCS_F_BLOCK_MASK;
  int ndev = 0, dev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1 || cudaGetDevice(&dev) != cudaSuccess) return VCS_ECUDA;     // no CPU fallback
  vcs_s *h = new (std::nothrow) vcs_s();
  if (!h) return VCS_ENOMEM;
  memset(static_cast<Handle *>(h), 0, sizeof(Handle));
  h->batch = batch; h->n_roms = n_roms; h->y0 = c.y0; h->max_lines = c.max_lines; h->f8_start_bank = c.f8_start_bank; h->device = dev;
  *out = h;                                           // so that the caller can read vcs_last_error and destroy

  std::vector<RomMeta> meta(n_roms);
  size_t blob = 0, dwords = 0;
  bool any_sc = false, any_special = false;
  for (int r = 0; r < n_roms; ++r) {
    meta[r].offset = (uint32_t)blob; meta[r].size = roms[r].size; meta[r].doff = (uint32_t)dwords; meta[r].pad = 0;
    const uint32_t kind = (uint32_t)map_kind(roms[r].size, roms[r].mapper);
    const uint32_t nbk = (kind == MK_F8 || kind == MK_F8SC) ? 2u : (kind == MK_F6 || kind == MK_F6SC) ? 4u : (kind == MK_F4 || kind == MK_F4SC) ? 8u : 0u;
    meta[r].kind = kind;
    meta[r].hs = (nbk ? (((nbk == 8u) ? 0x1FF4u : 0x1FFAu - nbk) | (nbk << 16)) : 0u) | ((kind >= MK_F8SC && kind <= MK_F4SC) ? HS_SC : 0u);
    any_sc = any_sc || (meta[r].hs & HS_SC); any_special = any_special || kind >= MK_F8SC;
    blob += roms[r].size; dwords += (roms[r].size < 4096) ? 4096 : roms[r].size;
  }
  std::vector<uint8_t> hb(blob);
  for (int r = 0; r < n_roms; ++r) memcpy(hb.data() + meta[r].offset, roms[r].data, roms[r].size);
  std::vector<int32_t> er(batch, 0);
  if (env_rom) memcpy(er.data(), env_rom, sizeof(int32_t) * batch);
  // launch shape: envs per block (cfg.flags VCS_F_BLOCK_* overrides), and whether every block maps to one ROM so
  // that the ROM can be staged in shared memory (otherwise the kernel reads it through the read-only path)
  int want = (batch >= 32768) ? 256 : 128;           // big batches: 256 envs per block (measured 8 % faster on config 4: fewer, larger regroup domains)
  if (fblock) want = (fblock == VCS_F_BLOCK_64) ? 64 : (fblock == VCS_F_BLOCK_128) ? 128 : 256;
  h->max_rom = 0;
  for (int r = 0; r < n_roms; ++r) if (roms[r].size > h->max_rom) h->max_rom = roms[r].size;
  auto uniform = [&](int blk) { for (int i = 0; i < batch; ++i) if (er[i] != er[i - i % blk]) return false; return true; };
  h->block = want; h->rom_smem = 0;
  for (int blk = want; blk >= 64; blk >>= 1) if (uniform(blk)) { h->block = blk; h->rom_smem = 1; break; }
  if (c.flags & VCS_F_ROM_GLOBAL) h->rom_smem = 0;
  h->rom_staged = h->rom_smem && h->max_rom <= 8192;       // 16 / 32 KB images stay in global memory (read-only path): two blocks per SM must fit
  h->banked = 0;
  for (int r = 0; r < n_roms; ++r) if (meta[r].kind >= MK_F8 && meta[r].kind <= MK_F4SC) h->banked = 1;
  h->regroup = (c.flags & VCS_F_NO_REGROUP) ? 0 : 1;
  // pre-decode every byte offset of every bank once (vcs_decode.cuh); the words depend on the launch shape
  // (zero-page RAM operands are stored as shared-memory offsets)
  std::vector<DWord> dw(dwords + 8, DWord{0, 0}), dwp(dwords + 8, DWord{0, 0}), dws(dwords + 8, DWord{0, 0});   // dwp: the plain table of vcs_step_instructions; dws: soft mode's
  {
    std::vector<uint8_t> img(4096 + 4, 0), leader(4096);
    for (int r = 0; r < n_roms; ++r) {
      const int nb = (roms[r].size < 4096) ? 1 : (int)(roms[r].size / 4096);
      if (meta[r].kind == MK_E0 || meta[r].kind == MK_FE) {         // 1 KB windows / a bank that follows the data bus: every byte decodes at run time
        for (size_t i = 0; i < (size_t)nb * 4096; ++i) { dw[meta[r].doff + i] = DWord{(uint32_t)(HC_COLD + H_SLOW) | DW_LEADER, 0}; dwp[meta[r].doff + i] = dw[meta[r].doff + i]; dws[meta[r].doff + i] = dw[meta[r].doff + i]; }
        continue;
      }
      const bool sc = (meta[r].hs & HS_SC) != 0;
      std::fill(leader.begin(), leader.end(), 0);
      for (int pass = 0; pass < 2; ++pass)
        for (int b = 0; b < nb; ++b) {
          if (roms[r].size == 2048) { memcpy(img.data(), roms[r].data, 2048); memcpy(img.data() + 2048, roms[r].data, 2048); }
          else memcpy(img.data(), roms[r].data + 4096 * b, 4096);
          if (pass == 0) mark_leaders(img.data(), leader.data());
          else { decode_bank(img.data(), leader.data(), h->block, nb, dw.data() + meta[r].doff + 4096 * b, !(c.flags & VCS_F_NO_PROMOTE), sc);
                 if (!(c.flags & VCS_F_NO_SPIN)) mark_spins(img.data(), dw.data() + meta[r].doff + 4096 * b);
                 if (!(c.flags & VCS_F_NO_FUSE)) fuse_ld_st(dw.data() + meta[r].doff + 4096 * b);
                 decode_bank(img.data(), leader.data(), 128, nb, dwp.data() + meta[r].doff + 4096 * b, !(c.flags & VCS_F_NO_PROMOTE), sc);
                 decode_bank(img.data(), leader.data(), 128, nb, dws.data() + meta[r].doff + 4096 * b, !(c.flags & VCS_F_NO_PROMOTE), sc); }
        }
    }
  }

  const size_t B = (size_t)batch;
  CU(h, cudaMalloc((void **)&h->d_st, sizeof(uint32_t) * ST_WORDS * B));
  CU(h, cudaMalloc((void **)&h->d_ram, sizeof(uint32_t) * 32 * B));
  CU(h, cudaMalloc((void **)&h->d_cyc, sizeof(unsigned long long) * B));
  CU(h, cudaMalloc((void **)&h->d_screen, (size_t)SCR_W * SCR_H * B));
  if (any_sc) CU(h, cudaMalloc((void **)&h->d_sc_ram, sizeof(uint32_t) * 32 * B));
  h->special_carts = any_special ? 1 : 0;
  CU(h, cudaMalloc((void **)&h->d_rom_blob, blob));
  CU(h, cudaMalloc((void **)&h->d_drom, sizeof(DWord) * dw.size()));
  CU(h, cudaMemcpy(h->d_drom, dw.data(), sizeof(DWord) * dw.size(), cudaMemcpyHostToDevice));
  CU(h, cudaMalloc((void **)&h->d_drom_plain, sizeof(DWord) * dwp.size()));
  CU(h, cudaMemcpy(h->d_drom_plain, dwp.data(), sizeof(DWord) * dwp.size(), cudaMemcpyHostToDevice));
  CU(h, cudaMalloc((void **)&h->d_rom_meta, sizeof(RomMeta) * n_roms));
  CU(h, cudaMalloc((void **)&h->d_env_rom, sizeof(int32_t) * B));
  CU(h, cudaMalloc((void **)&h->d_seeds, sizeof(unsigned long long) * B));
  CU(h, cudaMemcpy(h->d_rom_blob, hb.data(), blob, cudaMemcpyHostToDevice));
  CU(h, cudaMemcpy(h->d_rom_meta, meta.data(), sizeof(RomMeta) * n_roms, cudaMemcpyHostToDevice));
  CU(h, cudaMemcpy(h->d_env_rom, er.data(), sizeof(int32_t) * B, cudaMemcpyHostToDevice));
  CU(h, cudaMemcpy(h->d_seeds, seeds, sizeof(unsigned long long) * B, cudaMemcpyHostToDevice));
  CU(h, cudaMalloc((void **)&h->d_switches, (size_t)B));
  CU(h, cudaMemset(h->d_switches, 0x3F, (size_t)B));
  CU(h, cudaMalloc((void **)&h->d_boot, 3 * (size_t)B));
  CU(h, cudaMalloc((void **)&h->d_boot_ctr, sizeof(uint32_t) * B));
  {                                                   // block placement: identity until the first measurements are in
    const int nblk = (batch + h->block - 1) / h->block;
    std::vector<int32_t> id(nblk); for (int i = 0; i < nblk; ++i) id[i] = i;
    CU(h, cudaMalloc((void **)&h->d_perm, sizeof(int32_t) * nblk));
    CU(h, cudaMemcpy(h->d_perm, id.data(), sizeof(int32_t) * nblk, cudaMemcpyHostToDevice));
    CU(h, cudaMalloc((void **)&h->d_blk_time, sizeof(unsigned long long) * 3 * nblk));
    CU(h, cudaMemset(h->d_blk_time, 0, sizeof(unsigned long long) * 3 * nblk));
    CU(h, cudaMalloc((void **)&h->d_w_avg, sizeof(float) * nblk));
    CU(h, cudaMemset(h->d_w_avg, 0, sizeof(float) * nblk));
    h->balance = (c.flags & VCS_F_NO_BALANCE) ? 0 : 1; h->plain_steps = 0;
    h->balance_a = VCS_BALANCE_A;                             // measured slowdown of a block that shares its SM
  }
  {                                                   // soft mode (vcs_step_soft): its own decode table (128-env blocks, one entry per instruction);
    std::vector<RomMeta> ms(meta); for (auto &m : ms) m.pad = m.doff;     // pad: offset into the W(T) x ROM table
    h->soft_tab_n = dwords; h->soft_tab_T = -1.f;
    CU(h, cudaMalloc((void **)&h->d_soft_tab, sizeof(float) * (dwords + 8)));
    CU(h, cudaMalloc((void **)&h->d_soft_ent, sizeof(float4) * (dwords + 8)));
    CU(h, cudaMalloc((void **)&h->d_drom_soft, sizeof(DWord) * dws.size()));
    CU(h, cudaMemcpy(h->d_drom_soft, dws.data(), sizeof(DWord) * dws.size(), cudaMemcpyHostToDevice));
    CU(h, cudaMalloc((void **)&h->d_rom_meta_soft, sizeof(RomMeta) * n_roms));
    CU(h, cudaMemcpy(h->d_rom_meta_soft, ms.data(), sizeof(RomMeta) * n_roms, cudaMemcpyHostToDevice));
    CU(h, cudaMalloc((void **)&h->d_soft_w, sizeof(float) * SOFT_W_WORDS));
    CU(h, cudaMallocHost((void **)&h->h_soft_w, sizeof(float) * SOFT_W_WORDS));
    CU(h, cudaEventCreateWithFlags(&h->soft_w_done, cudaEventDisableTiming));
  }
  upload_optable();
  CU(h, cudaGetLastError());
  int rc = vcs_reset(h, nullptr, nullptr);
  if (rc != VCS_OK) return rc;
  CU(h, cudaDeviceSynchronize());
  return VCS_OK;
}

int vcs_reset(vcs_t h, const uint8_t *mask_dev, void *cuda_stream) {
  DEV_OK(h);
  cudaStream_t s = (cudaStream_t)cuda_stream;
  StepParams p = params_of(h, nullptr, 1);
  reset_kernel<<<(h->batch + 127) / 128, 128, 0, s>>>(p, h->d_seeds, mask_dev, h->f8_start_bank);
  clear_screen_kernel<<<h->batch, 256, 0, s>>>(h->d_screen, mask_dev);
  h->launches += 2;
  CU(h, cudaGetLastError());
  return VCS_OK;
}

int vcs_step(vcs_t h, const uint8_t *actions_dev, int32_t frameskip, void *cuda_stream) {
  DEV_OK(h);
  if (!actions_dev) return fail(h, VCS_EINVAL, "vcs_step: actions_dev is NULL");
  if (frameskip < 1 || (long long)frameskip * h->max_lines * LINE_CYC >= (1ll << 31))
    return fail(h, VCS_EINVAL, "vcs_step: frameskip out of range");
  StepParams p = params_of(h, actions_dev, frameskip);
  if (h->balance) p.blk_time = h->d_blk_time;
  cudaError_t ce = launch_step(p, (cudaStream_t)cuda_stream);
  h->launches += 1;
  if (ce != cudaSuccess) return fail(h, VCS_ECUDA, "vcs_step launch", ce);
  if (h->balance) {                                   // re-place the blocks from this step's per-block times: early on, then now and again
    const long long k = ++h->plain_steps;
    if ((k >= 2 && k <= 16) || (k & 3) == 0) {            // (the first step after a reset is a short frame)
      ce = launch_rebalance(h->d_perm, h->d_blk_time, (h->batch + h->block - 1) / h->block, h->balance_a, h->d_w_avg, (cudaStream_t)cuda_stream);
      h->launches += 1;
      if (ce != cudaSuccess) return fail(h, VCS_ECUDA, "vcs_step rebalance launch", ce);
    }
  }
  return VCS_OK;
}

int vcs_step_masked(vcs_t h, const uint8_t *actions_dev, int32_t frameskip, const uint8_t *mask_dev, void *cuda_stream) {
  DEV_OK(h);
  if (!actions_dev) return fail(h, VCS_EINVAL, "vcs_step_masked: actions_dev is NULL");
  if (frameskip < 1 || (long long)frameskip * h->max_lines * LINE_CYC >= (1ll << 31))
    return fail(h, VCS_EINVAL, "vcs_step_masked: frameskip out of range");
  StepParams p = params_of(h, actions_dev, frameskip);
  p.mask = mask_dev;
  cudaError_t ce = launch_step(p, (cudaStream_t)cuda_stream);
  h->launches += 1;
  if (ce != cudaSuccess) return fail(h, VCS_ECUDA, "vcs_step_masked launch", ce);
  return VCS_OK;
}

int vcs_step_instructions(vcs_t h, const uint8_t *actions_dev, int32_t n_instr, void *cuda_stream) {
  DEV_OK(h);
  if (!actions_dev) return fail(h, VCS_EINVAL, "vcs_step_instructions: actions_dev is NULL");
  if (n_instr < 1 || n_instr > 1000000) return fail(h, VCS_EINVAL, "vcs_step_instructions: n_instr out of range (1 .. 1,000,000)");
  StepParams p = params_of(h, actions_dev, 0x7FFFFFF0);   // (no frame count ends this step, and no frame of it is the "last" one)
  p.n_instr = n_instr; p.drom = h->d_drom_plain; p.perm = nullptr; p.regroup = 0;
  cudaError_t ce = launch_step(p, (cudaStream_t)cuda_stream);
  h->launches += 1;
  if (ce != cudaSuccess) return fail(h, VCS_ECUDA, "vcs_step_instructions launch", ce);
  return VCS_OK;
}

int vcs_set_switches(vcs_t h, const uint8_t *switches_dev, void *cuda_stream) {
  DEV_OK(h);
  cudaStream_t s = (cudaStream_t)cuda_stream;
  if (switches_dev) CU(h, cudaMemcpyAsync(h->d_switches, switches_dev, (size_t)h->batch, cudaMemcpyDeviceToDevice, s));
  else { fill_kernel<<<(h->batch + 255) / 256, 256, 0, s>>>(h->d_switches, 0x3F, h->batch); h->launches += 1; CU(h, cudaGetLastError()); }
  return VCS_OK;
}

int vcs_boot(vcs_t h, const uint8_t *mask_dev, int32_t noop_frames, int32_t reset_frames, const uint8_t *noop_starts_dev,
             int32_t max_noop_starts, int32_t frameskip, void *cuda_stream) {
  DEV_OK(h);
  if (noop_frames < 0 || reset_frames < 0 || max_noop_starts < 0 || max_noop_starts > 255 || noop_frames > 100000 || reset_frames > 100000)
    return fail(h, VCS_EINVAL, "vcs_boot: frame counts out of range");
  if (frameskip < 1 || (long long)frameskip * h->max_lines * LINE_CYC >= (1ll << 31)) return fail(h, VCS_EINVAL, "vcs_boot: frameskip out of range");
  cudaStream_t s = (cudaStream_t)cuda_stream;
  const int B = h->batch, nb = (B + 255) / 256;
  uint8_t *zero = h->d_boot, *itmask = h->d_boot + B, *swr = h->d_boot + 2 * (size_t)B;
  int rc = vcs_reset(h, mask_dev, cuda_stream); if (rc) return rc;
  boot_prep_kernel<<<nb, 256, 0, s>>>(h->d_switches, zero, swr, B); h->launches += 1;
  CU(h, cudaGetLastError());
  StepParams p = params_of(h, zero, 1);
  p.mask = mask_dev;
  for (int f = 0; f < noop_frames + reset_frames; ++f) {
    p.switches = (f < noop_frames) ? h->d_switches : swr;
    cudaError_t ce = launch_step(p, s); h->launches += 1;
    if (ce != cudaSuccess) return fail(h, VCS_ECUDA, "vcs_boot launch", ce);
  }
  if (noop_starts_dev) {
    p = params_of(h, zero, frameskip); p.mask = itmask;
    for (int k = 0; k < max_noop_starts; ++k) {
      boot_mask_kernel<<<nb, 256, 0, s>>>(mask_dev, noop_starts_dev, k, itmask, B);
      cudaError_t ce = launch_step(p, s); h->launches += 2;
      if (ce != cudaSuccess) return fail(h, VCS_ECUDA, "vcs_boot launch", ce);
    }
  }
  return VCS_OK;
}

int vcs_auto_reset(vcs_t h, const uint8_t *mask_dev, int32_t noop_steps, int32_t reset_steps, const uint8_t *noop_starts_dev,
                   int32_t max_noop_starts, void *cuda_stream) {
  DEV_OK(h);
  if (noop_steps < 0 || reset_steps < 0 || max_noop_starts < 0 || noop_steps + reset_steps + max_noop_starts > 255)
    return fail(h, VCS_EINVAL, "vcs_auto_reset: step counts out of range (their sum must be <= 255)");
  cudaStream_t s = (cudaStream_t)cuda_stream;
  int rc = vcs_reset(h, mask_dev, cuda_stream); if (rc) return rc;
  arm_boot_kernel<<<(h->batch + 255) / 256, 256, 0, s>>>(mask_dev, noop_starts_dev, noop_steps, reset_steps, max_noop_starts, h->d_boot_ctr, h->batch);
  h->launches += 1;
  CU(h, cudaGetLastError());
  return VCS_OK;
}
int vcs_get_booting(vcs_t h, uint8_t *out_dev, void *cuda_stream) {
  DEV_OK(h); if (!out_dev) return VCS_EINVAL;
  get_booting_kernel<<<(h->batch + 255) / 256, 256, 0, (cudaStream_t)cuda_stream>>>(h->d_boot_ctr, out_dev, h->batch);
  h->launches += 1;
  CU(h, cudaGetLastError());
  return VCS_OK;
}

// soft modes: e^{-k/T}, W(T) x ROM and the per-entry sums for this temperature (once per temperature)
static int soft_prepare(vcs_t h, float T, cudaStream_t s) {
  if (h->soft_tab_T != T) {
    int K = (int)ceil(17.0 * (double)T); if (K < 1) K = 1; if (K > 1023) K = 1023;
    CU(h, cudaEventSynchronize(h->soft_w_done));       // (the previous upload from the handle's pinned buffers; long since done)
    for (int k = 0; k < SOFT_W_N; ++k) h->h_soft_w[k] = k <= K ? (float)exp(-(double)k / (double)T) : 0.f;
    double cw = 0.0;                                   // normaliser of a RAM-tape window reaching n cells to one side (soft_ram_read)
    for (int n = 0; n < 128; ++n) { if (n <= K) cw += exp(-(double)n / (double)T); h->h_soft_w[SOFT_CW + n] = (float)cw; }
    CU(h, cudaMemcpyAsync(h->d_soft_w, h->h_soft_w, sizeof(float) * SOFT_W_WORDS, cudaMemcpyHostToDevice, s));
    CU(h, cudaEventRecord(h->soft_w_done, s));
    cudaError_t ce0 = launch_soft_table(h->d_rom_blob, h->d_rom_meta_soft, h->n_roms, h->d_soft_w, K, h->d_soft_tab, s);
    h->launches += 1;
    if (ce0 != cudaSuccess) return fail(h, VCS_ECUDA, "soft mode: table launch", ce0);
    ce0 = launch_soft_entries(h->d_rom_blob, h->d_rom_meta_soft, h->n_roms, h->d_drom_soft, h->d_soft_tab, h->d_soft_ent, s);
    h->launches += 1;
    if (ce0 != cudaSuccess) return fail(h, VCS_ECUDA, "soft mode: entry-table launch", ce0);
    h->soft_tab_T = T; h->soft_K = K;
  }
  return VCS_OK;
}
static int soft_args_ok(vcs_t h, const char *who, float T, float alpha) {
  if (!(T > 0.f) || T > 60.f || !(alpha == alpha) || alpha > 1e30f || alpha < -1e30f) return fail(h, VCS_EINVAL, (std::string(who) + ": T or alpha out of range").c_str());
  if (h->special_carts) return fail(h, VCS_EINVAL, (std::string(who) + ": Superchip / E0 / FE cartridges run in hard mode only").c_str());
  return VCS_OK;
}

int vcs_step_soft(vcs_t h, const uint8_t *actions_dev, int32_t frameskip, float T, float alpha, float *soft_out_dev, void *cuda_stream) {
  DEV_OK(h);
  if (!actions_dev || !soft_out_dev) return fail(h, VCS_EINVAL, "vcs_step_soft: NULL buffer");
  if (frameskip < 1 || (long long)frameskip * h->max_lines * LINE_CYC >= (1ll << 31)) return fail(h, VCS_EINVAL, "vcs_step_soft: frameskip out of range");
  if (int rc = soft_args_ok(h, "vcs_step_soft", T, alpha)) return rc;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  if (int rc = soft_prepare(h, T, s)) return rc;
  CU(h, cudaMemsetAsync(soft_out_dev, 0, sizeof(float) * 8 * (size_t)h->batch, s));
  StepParams p = params_of(h, actions_dev, frameskip);
  p.drom = h->d_drom_soft; p.rom_meta = h->d_rom_meta_soft;
  p.perm = nullptr;                                    // the soft kernel has its own launch shape (128 envs per block): blocks in env order
  p.soft_w = h->d_soft_w; p.soft_tab = h->d_soft_tab; p.soft_ent = h->d_soft_ent; p.soft_out = soft_out_dev; p.soft_alpha = alpha; p.soft_K = h->soft_K;
  cudaError_t ce = launch_step(p, s);
  h->launches += 1;
  if (ce != cudaSuccess) return fail(h, VCS_ECUDA, "vcs_step_soft launch", ce);
  return VCS_OK;
}

int vcs_step_instructions_soft(vcs_t h, const uint8_t *actions_dev, int32_t n_instr, float T, float alpha, int32_t full,
                               float *soft_out_dev, void *cuda_stream) {
  DEV_OK(h);
  if (!actions_dev || !soft_out_dev) return fail(h, VCS_EINVAL, "vcs_step_instructions_soft: NULL buffer");
  if (n_instr < 1 || n_instr > 1000000) return fail(h, VCS_EINVAL, "vcs_step_instructions_soft: n_instr out of range (1 .. 1,000,000)");
  if (int rc = soft_args_ok(h, "vcs_step_instructions_soft", T, alpha)) return rc;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  if (int rc = soft_prepare(h, T, s)) return rc;
  if (full) {
    if (!h->d_drom_slow) {                             // every entry: "decode at run time" (the cast bytes decide what runs)
      std::vector<DWord> slow(h->soft_tab_n + 8, DWord{(uint32_t)(HC_COLD + H_SLOW) | DW_LEADER, 0});
      CU(h, cudaMalloc((void **)&h->d_drom_slow, sizeof(DWord) * slow.size()));
      CU(h, cudaMemcpy(h->d_drom_slow, slow.data(), sizeof(DWord) * slow.size(), cudaMemcpyHostToDevice));
      CU(h, cudaMalloc((void **)&h->d_soft_wd, sizeof(double) * SOFT_WD_WORDS));
      CU(h, cudaMallocHost((void **)&h->h_soft_wd, sizeof(double) * SOFT_WD_WORDS));
      h->soft_wd_T = -1.f; h->soft_wd_alpha = 0.f;
    }
    if (h->soft_wd_T != T || h->soft_wd_alpha != alpha) {   // the weights and the two gates in double, by the host's exp
      CU(h, cudaEventSynchronize(h->soft_w_done));
      const double Td = (double)T, ad = (double)alpha;
      for (int k = 0; k < SOFT_WD_GATE; ++k) h->h_soft_wd[k] = k <= h->soft_K ? exp(-(double)k / Td) : 0.0;
      h->h_soft_wd[SOFT_WD_GATE] = 1.0 / (1.0 + exp(-ad * 1.0)); h->h_soft_wd[SOFT_WD_GATE + 1] = 1.0 / (1.0 + exp(-ad * -1.0));
      CU(h, cudaMemcpyAsync(h->d_soft_wd, h->h_soft_wd, sizeof(double) * SOFT_WD_WORDS, cudaMemcpyHostToDevice, s));
      CU(h, cudaEventRecord(h->soft_w_done, s));
      h->soft_wd_T = T; h->soft_wd_alpha = alpha;
    }
  }
  CU(h, cudaMemsetAsync(soft_out_dev, 0, sizeof(float) * 8 * (size_t)h->batch, s));
  StepParams p = params_of(h, actions_dev, 0x7FFFFFF0);
  p.n_instr = n_instr; p.drom = full ? h->d_drom_slow : h->d_drom_soft; p.rom_meta = h->d_rom_meta_soft; p.perm = nullptr; p.regroup = 0;
  p.soft_w = h->d_soft_w; p.soft_tab = h->d_soft_tab; p.soft_ent = h->d_soft_ent; p.soft_out = soft_out_dev; p.soft_alpha = alpha; p.soft_K = h->soft_K;
  p.soft_wd = h->d_soft_wd; p.soft_full = full ? 1 : 0;
  cudaError_t ce = launch_step(p, s);
  h->launches += 1;
  if (ce != cudaSuccess) return fail(h, VCS_ECUDA, "vcs_step_instructions_soft launch", ce);
  return VCS_OK;
}

int vcs_get_ram(vcs_t h, uint8_t *out_dev, void *cuda_stream) {
  DEV_OK(h); if (!out_dev) return VCS_EINVAL;
  const long long n = 32ll * h->batch;
  get_ram_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)cuda_stream>>>(h->d_ram, reinterpret_cast<uint32_t *>(out_dev), h->batch);
  h->launches += 1;
  CU(h, cudaGetLastError());
  return VCS_OK;
}
int vcs_get_cart_ram(vcs_t h, uint8_t *out_dev, void *cuda_stream) {
  DEV_OK(h); if (!out_dev) return VCS_EINVAL;
  if (!h->d_sc_ram) { CU(h, cudaMemsetAsync(out_dev, 0, (size_t)128 * h->batch, (cudaStream_t)cuda_stream)); return VCS_OK; }
  const long long n = 32ll * h->batch;
  get_ram_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)cuda_stream>>>(h->d_sc_ram, reinterpret_cast<uint32_t *>(out_dev), h->batch);
  h->launches += 1;
  CU(h, cudaGetLastError());
  return VCS_OK;
}
int vcs_get_regs(vcs_t h, vcs_regs *out_dev, void *cuda_stream) {
  DEV_OK(h); if (!out_dev) return VCS_EINVAL;
  get_regs_kernel<<<(h->batch + 127) / 128, 128, 0, (cudaStream_t)cuda_stream>>>(h->d_st, h->d_cyc, reinterpret_cast<uint4 *>(out_dev), h->batch, h->d_rom_meta, h->d_env_rom);
  h->launches += 1;
  CU(h, cudaGetLastError());
  return VCS_OK;
}
int vcs_get_screen(vcs_t h, uint8_t *out_dev, void *cuda_stream) {
  DEV_OK(h); if (!out_dev) return VCS_EINVAL;
  CU(h, cudaMemcpyAsync(out_dev, h->d_screen, (size_t)SCR_W * SCR_H * h->batch, cudaMemcpyDeviceToDevice, (cudaStream_t)cuda_stream));
  return VCS_OK;
}
int vcs_screen_ptr(vcs_t h, const uint8_t **out_dev_ptr) {
  if (!h || !out_dev_ptr) return VCS_EINVAL;
  *out_dev_ptr = h->d_screen; return VCS_OK;
}

int vcs_step_host(vcs_t h, const uint8_t *actions_host, int32_t frameskip, void *cuda_stream) {
  DEV_OK(h); if (!actions_host) return VCS_EINVAL;
  int rc = ensure_stage(h, (size_t)h->batch * 128); if (rc) return rc;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  memcpy(h->h_pinned, actions_host, h->batch);
  CU(h, cudaMemcpyAsync(h->d_actions_stage, h->h_pinned, h->batch, cudaMemcpyHostToDevice, s));
  rc = vcs_step(h, h->d_actions_stage, frameskip, cuda_stream); if (rc) return rc;
  CU(h, cudaStreamSynchronize(s));
  return VCS_OK;
}
int vcs_get_ram_host(vcs_t h, uint8_t *out_host, void *cuda_stream) {
  DEV_OK(h); if (!out_host) return VCS_EINVAL;
  int rc = ensure_stage(h, (size_t)h->batch * 128); if (rc) return rc;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  rc = vcs_get_ram(h, h->d_actions_stage, cuda_stream); if (rc) return rc;
  CU(h, cudaMemcpyAsync(h->h_pinned, h->d_actions_stage, (size_t)h->batch * 128, cudaMemcpyDeviceToHost, s));
  CU(h, cudaStreamSynchronize(s));
  memcpy(out_host, h->h_pinned, (size_t)h->batch * 128);
  return VCS_OK;
}
int vcs_get_regs_host(vcs_t h, vcs_regs *out_host, void *cuda_stream) {
  DEV_OK(h); if (!out_host) return VCS_EINVAL;
  int rc = ensure_stage(h, (size_t)h->batch * 128); if (rc) return rc;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  rc = vcs_get_regs(h, reinterpret_cast<vcs_regs *>(h->d_actions_stage), cuda_stream); if (rc) return rc;
  CU(h, cudaMemcpyAsync(h->h_pinned, h->d_actions_stage, (size_t)h->batch * 32, cudaMemcpyDeviceToHost, s));
  CU(h, cudaStreamSynchronize(s));
  memcpy(out_host, h->h_pinned, (size_t)h->batch * 32);
  return VCS_OK;
}
int vcs_get_screen_host(vcs_t h, uint8_t *out_host, void *cuda_stream) {
  DEV_OK(h); if (!out_host) return VCS_EINVAL;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  CU(h, cudaMemcpyAsync(out_host, h->d_screen, (size_t)SCR_W * SCR_H * h->batch, cudaMemcpyDeviceToHost, s));
  CU(h, cudaStreamSynchronize(s));
  return VCS_OK;
}

int vcs_block_times(vcs_t h, uint64_t *times_host, int32_t *perm_host, int32_t cap, int32_t *n_out) {
  DEV_OK(h); if (!n_out) return VCS_EINVAL;
  const int n = (h->batch + h->block - 1) / h->block;
  *n_out = n;
  if (cap < n) return (times_host || perm_host) ? VCS_EINVAL : VCS_OK;
  CU(h, cudaDeviceSynchronize());
  if (times_host) CU(h, cudaMemcpy(times_host, h->d_blk_time, sizeof(unsigned long long) * 3 * n, cudaMemcpyDeviceToHost));
  if (perm_host) CU(h, cudaMemcpy(perm_host, h->d_perm, sizeof(int32_t) * n, cudaMemcpyDeviceToHost));
  return VCS_OK;
}

int64_t vcs_launch_count(vcs_t h) { return h ? h->launches : -1; }

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------
// vcs_step_host_noalloc (include/vcs.h): a host-buffer step for callers that cannot call cudaMalloc.  Its device-side
// staging — the actions on their way in, the transposed RAM and the vcs_regs on their way out, a flag counter — lives
// in ONE file-scope array instead of the handle's lazily allocated stage: VCS_NOALLOC_MAX_BATCH envs x (1 + 128 + 32)
// bytes + 256 = 10,551,552 bytes, held by every GPU that loads the library until the process exits.  All calls of a
// process share it, per device.
//
// The array's name below is a DEVICE symbol: in host code it is a host-side stand-in, not a device address, so the host
// side takes the address with cudaGetSymbolAddress — once per device, with that device current (noalloc_base) — and
// passes that pointer on; only device code (noalloc_count_flags_kernel) names the array itself.
constexpr size_t NOALLOC_OFF_ACT = 0;                                                     // uint8 [MAX]       actions, staged for the step kernel
constexpr size_t NOALLOC_OFF_RAM = NOALLOC_OFF_ACT + (size_t)VCS_NOALLOC_MAX_BATCH;       // uint8 [MAX][128]  get_ram_kernel's output
constexpr size_t NOALLOC_OFF_REGS = NOALLOC_OFF_RAM + 128 * (size_t)VCS_NOALLOC_MAX_BATCH; // vcs_regs [MAX]    get_regs_kernel's output
constexpr size_t NOALLOC_OFF_CTR = NOALLOC_OFF_REGS + 32 * (size_t)VCS_NOALLOC_MAX_BATCH; // uint32            envs with a status bit set: MUST start at zero
constexpr size_t NOALLOC_BYTES = NOALLOC_OFF_CTR + 256;
static_assert(NOALLOC_OFF_RAM % 256 == 0 && NOALLOC_OFF_REGS % 256 == 0 && NOALLOC_OFF_CTR % 256 == 0, "scratch regions keep the array's alignment");
static __device__ __align__(256) unsigned char vcs_noalloc_scratch[NOALLOC_BYTES];

namespace {

// envs whose vcs_regs.status (byte 23) is non-zero, added up in the counter word of the scratch array
__global__ void noalloc_count_flags_kernel(int B) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= B) return;
  if (vcs_noalloc_scratch[NOALLOC_OFF_REGS + 32 * (size_t)e + 23] != 0)
    atomicAdd(reinterpret_cast<unsigned int *>(vcs_noalloc_scratch + NOALLOC_OFF_CTR), 1u);
}

// the array's device address on the current device: resolved once per device (no allocation: the array came with the module)
int noalloc_base(Handle *h, unsigned char **out) {
  static unsigned char *base[64] = {nullptr};
  if (h->device < 0 || h->device >= 64) return fail(h, VCS_EINVAL, "vcs_step_host_noalloc: device index above 63");
  if (!base[h->device]) {                              // (DEV_OK has checked that h->device is the current device)
    void *ptr = nullptr;
    const cudaError_t ce = cudaGetSymbolAddress(&ptr, vcs_noalloc_scratch);
    if (ce != cudaSuccess || !ptr) return fail(h, VCS_ECUDA, "vcs_step_host_noalloc: cudaGetSymbolAddress(vcs_noalloc_scratch)", ce);
    base[h->device] = static_cast<unsigned char *>(ptr);
  }
  *out = base[h->device];
  return VCS_OK;
}

}  // namespace

extern "C" {

int vcs_step_host_noalloc(vcs_t h, const uint8_t *actions_host, int32_t frameskip, uint8_t *ram_out_host, vcs_regs *regs_out_host,
                          int32_t *n_flagged_host, void *cuda_stream) {
  DEV_OK(h);
  if (!actions_host || !ram_out_host || !regs_out_host || !n_flagged_host) return fail(h, VCS_EINVAL, "vcs_step_host_noalloc: NULL buffer");
  if (h->batch > VCS_NOALLOC_MAX_BATCH) {
    char msg[160];
    snprintf(msg, sizeof msg, "vcs_step_host_noalloc: batch %d exceeds VCS_NOALLOC_MAX_BATCH = %d (the size of the library's static scratch array)",
             h->batch, (int)VCS_NOALLOC_MAX_BATCH);
    return fail(h, VCS_EINVAL, msg);
  }
  unsigned char *base = nullptr;
  if (int rc = noalloc_base(h, &base)) return rc;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  const size_t B = (size_t)h->batch;
  uint8_t *d_act = base + NOALLOC_OFF_ACT, *d_ram = base + NOALLOC_OFF_RAM;
  vcs_regs *d_regs = reinterpret_cast<vcs_regs *>(base + NOALLOC_OFF_REGS);
  // the array keeps the previous call's contents: the counter must start at zero; every other byte this call reads
  // (actions, RAM, regs of envs [0, batch)) is written by this call first
  CU(h, cudaMemsetAsync(base + NOALLOC_OFF_CTR, 0, 256, s));
  CU(h, cudaMemcpyAsync(d_act, actions_host, B, cudaMemcpyHostToDevice, s));
  if (int rc = vcs_step(h, d_act, frameskip, cuda_stream)) return rc;
  if (int rc = vcs_get_ram(h, d_ram, cuda_stream)) return rc;
  if (int rc = vcs_get_regs(h, d_regs, cuda_stream)) return rc;
  noalloc_count_flags_kernel<<<(h->batch + 255) / 256, 256, 0, s>>>(h->batch);
  h->launches += 1;
  CU(h, cudaGetLastError());
  CU(h, cudaMemcpyAsync(ram_out_host, d_ram, 128 * B, cudaMemcpyDeviceToHost, s));
  CU(h, cudaMemcpyAsync(regs_out_host, d_regs, 32 * B, cudaMemcpyDeviceToHost, s));
  CU(h, cudaMemcpyAsync(n_flagged_host, base + NOALLOC_OFF_CTR, sizeof(int32_t), cudaMemcpyDeviceToHost, s));
  return VCS_OK;                                        // enqueued: the outputs are valid once the caller has synchronised the stream
}

// Format guess from size and content (reading R17).  Host only.
int vcs_detect_mapper(const uint8_t *data, uint32_t size) {
  if (!data) return VCS_EINVAL;
  if (size == 2048) return VCS_MAP_2K;
  if (size == 4096) return VCS_MAP_4K;
  if (size != 8192 && size != 16384 && size != 32768) return VCS_EROM;
  bool filler = true;                                   // Superchip: every bank starts with 256 equal bytes (its RAM ports sit there)
  for (uint32_t bank = 0; bank < size / 4096 && filler; ++bank) {
    const uint8_t *b = data + 4096 * bank;
    for (int i = 255; i > 0; --i) if (b[i] != b[0]) { filler = false; break; }
  }
  if (size == 16384) return filler ? VCS_MAP_F6SC : VCS_MAP_F6;
  if (size == 32768) return filler ? VCS_MAP_F4SC : VCS_MAP_F4;
  if (filler) return VCS_MAP_F8SC;
  int n_f8 = 0, n_e0 = 0, n_fe = 0;                     // what the code's absolute operands point at
  for (uint32_t i = 0; i + 2 < size; ++i) {
    const uint32_t op = data[i], target = data[i + 1] | ((uint32_t)data[i + 2] << 8), low5 = op & 0x1Fu;
    if (op == 0x20 || op == 0x4C) { if ((target & 0xF000u) == 0xD000u) ++n_fe; continue; }       // JSR / JMP into the $D000 page
    if (op == 0x6C || low5 < 0x0C || low5 > 0x0E) continue;                                      // columns xC, xD, xE hold the absolute modes
    const uint32_t a = target & 0x1FFFu;
    if (a == 0x1FF8u || a == 0x1FF9u) ++n_f8;
    else if (a >= 0x1FE0u && a <= 0x1FF7u) ++n_e0;
  }
  if (n_e0 >= 2 && n_e0 > n_f8) return VCS_MAP_E0;
  if (n_fe >= 2 && n_f8 == 0) return VCS_MAP_FE;
  return VCS_MAP_F8;
}

int vcs_optable(uint16_t *out256) {
  if (!out256) return VCS_EINVAL;
  memcpy(out256, host_optable(), 512); return VCS_OK;
}

int vcs_destroy(vcs_t h) {
  if (!h) return VCS_EINVAL;
  int cur = -1; cudaGetDevice(&cur);
  if (cur != h->device) cudaSetDevice(h->device);     // free on the handle's own device, then give the caller's back
  cudaDeviceSynchronize();
  cudaFree(h->d_st); cudaFree(h->d_ram); cudaFree(h->d_sc_ram); cudaFree(h->d_cyc); cudaFree(h->d_screen); cudaFree(h->d_rom_blob); cudaFree(h->d_drom); cudaFree(h->d_drom_plain);
  cudaFree(h->d_rom_meta); cudaFree(h->d_drom_soft); cudaFree(h->d_rom_meta_soft); cudaFree(h->d_soft_w); cudaFree(h->d_soft_tab); cudaFree(h->d_soft_ent); cudaFree(h->d_drom_slow); cudaFree(h->d_soft_wd); if (h->h_soft_wd) cudaFreeHost(h->h_soft_wd); cudaFree(h->d_env_rom); cudaFree(h->d_seeds); cudaFree(h->d_actions_stage); cudaFree(h->d_switches); cudaFree(h->d_boot); cudaFree(h->d_boot_ctr); cudaFree(h->d_perm); cudaFree(h->d_blk_time); cudaFree(h->d_w_avg);
  if (h->h_pinned) cudaFreeHost(h->h_pinned);
  if (h->h_soft_w) cudaFreeHost(h->h_soft_w);
  if (h->soft_w_done) cudaEventDestroy(h->soft_w_done);
  if (cur >= 0 && cur != h->device) cudaSetDevice(cur);
  delete h;
  return VCS_OK;
}

const char *vcs_last_error(vcs_t h) { return h ? h->err : ""; }

}  // extern "C"
