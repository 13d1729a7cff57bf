// vcs_peak.cu — integer-issue micro-benchmark behind vcs_issue_peak (include/vcs.h; SURVEY.md §8(d) "Roofline":
// the B200's integer-issue peak is not in MEASURED_PEAKS.json, so the library measures the denominator of the
// interpreter's roofline itself, on the same GPU, right beside the number it qualifies).
//
// Every thread runs CHAINS independent dependency chains of plain integer instructions for `iters` loop trips;
// the grid fills every SM with 2048 resident threads.  kind 0 = alu pipe only (LOP3 + SHF alternating: the
// pipe the interpreter's logic/shift/add work runs on), kind 1 = alu + fma pipes interleaved (LOP3 + IMAD: the
// most the four schedulers can issue, one warp-instruction per scheduler per clock).  The instruction count
// is by construction (OPS_PER_TRIP per thread per trip, checked against the SASS with cuobjdump);
// loop overhead is not counted, so the figure is a slight under-estimate of the true peak.
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/vcs.h"

namespace {

constexpr int CHAINS = 8, UNROLL = 16;
constexpr int OPS_PER_TRIP = CHAINS * UNROLL * 2;

template <int KIND>
__global__ void __launch_bounds__(256) issue_peak_kernel(uint32_t *out, int iters, uint32_t k1, uint32_t k2) {
  uint32_t c[CHAINS];
#pragma unroll
  for (int i = 0; i < CHAINS; ++i) c[i] = threadIdx.x * 2654435761u + i * 40503u + blockIdx.x;
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < UNROLL; ++u) {
#pragma unroll
      for (int i = 0; i < CHAINS; ++i) {
        uint32_t x = c[i];
        asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x) : "r"(k1), "r"(k2));          // alu pipe
        if (KIND == 0) asm volatile("shf.l.wrap.b32 %0, %0, %0, 5;" : "+r"(x));                 // alu pipe (SHF rotate)
        else asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(x) : "r"(k1), "r"(k2));         // fma pipe (IMAD)
        c[i] = x;
      }
    }
  }
  uint32_t s = 0;
#pragma unroll
  for (int i = 0; i < CHAINS; ++i) s ^= c[i];
  if (s == 0x12345u) out[0] = s;          // keeps the chains alive; practically never true
}

}  // namespace

extern "C" int vcs_issue_peak(int32_t kind, int32_t iters, double *thread_instr_per_s, double *seconds) {
  if ((kind != 0 && kind != 1) || iters < 1 || !thread_instr_per_s) return VCS_EINVAL;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return VCS_ECUDA;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return VCS_ECUDA;
  uint32_t *d = nullptr;
  if (cudaMalloc(&d, 4) != cudaSuccess) return VCS_ENOMEM;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int grid = sms * 8, block = 256;                      // 2048 threads per SM
  float best = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {                         // rep 0 warms up
    cudaEventRecord(e0, 0);
    if (kind == 0) issue_peak_kernel<0><<<grid, block>>>(d, iters, 0x9E3779B9u + rep, 0x7F4A7C15u);
    else issue_peak_kernel<1><<<grid, block>>>(d, iters, 0x9E3779B9u + rep, 0x7F4A7C15u);
    cudaEventRecord(e1, 0);
    if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(d); return VCS_ECUDA; }
    float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best) best = ms;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
  if (cudaGetLastError() != cudaSuccess) return VCS_ECUDA;
  const double total = (double)grid * block * (double)iters * OPS_PER_TRIP;
  *thread_instr_per_s = total / (best * 1e-3);
  if (seconds) *seconds = best * 1e-3;
  return VCS_OK;
}
