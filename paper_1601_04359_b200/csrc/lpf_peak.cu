// lpf_peak.cu -- integer-pipe throughput probe behind lpf_alu_peak (include/lpf.h): the measured counterpart
// of the derived ALU roofline denominator.
// Eight independent dependency chains per thread of one instruction kind, inline PTX so that ptxas keeps them:
//   0 LOP3   1 SHF.R.W   2 the eval kernel's PAIR pattern (SHF, SHF, LOP3 M & W1 & W2)   3 POPC
#include <cuda_runtime.h>

#include "lpf.h"

namespace lpf {

constexpr int PEAK_ITERS = 4096;
constexpr int PEAK_CHAINS = 8;

template <int MODE>
__global__ void __launch_bounds__(256) peak_kernel(unsigned* out, unsigned seed, unsigned sh) {
  unsigned a[PEAK_CHAINS], b[PEAK_CHAINS], c[PEAK_CHAINS];
#pragma unroll
  for (int i = 0; i < PEAK_CHAINS; ++i) {
    a[i] = seed + threadIdx.x * 7u + i;
    b[i] = seed * 3u + i;
    c[i] = 0xffffffffu - i;
  }
  for (int it = 0; it < PEAK_ITERS; ++it) {
#pragma unroll
    for (int i = 0; i < PEAK_CHAINS; ++i) {
      if (MODE == 0) {
        asm volatile("lop3.b32 %0, %0, %1, %2, 0x80;" : "+r"(c[i]) : "r"(a[i]), "r"(b[i]));
      } else if (MODE == 1) {
        asm volatile("shf.r.wrap.b32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(b[i]), "r"(sh));
      } else if (MODE == 2) {
        // both shifts update their own chain register, so nothing is loop invariant
        asm volatile("shf.r.wrap.b32 %0, %0, %1, %2;" : "+r"(a[i]) : "r"(b[i]), "r"(sh));
        asm volatile("shf.r.wrap.b32 %0, %0, %1, %2;" : "+r"(b[i]) : "r"(a[i]), "r"(sh + 1));
        asm volatile("lop3.b32 %0, %0, %1, %2, 0x80;" : "+r"(c[i]) : "r"(a[i]), "r"(b[i]));
      } else {
        asm volatile("popc.b32 %0, %0;" : "+r"(a[i]));
      }
    }
  }
  unsigned r = 0;
#pragma unroll
  for (int i = 0; i < PEAK_CHAINS; ++i) r ^= a[i] ^ b[i] ^ c[i];
  if (r == 0x12345678u) out[threadIdx.x] = r;      // never true in practice: keeps the chains alive
}

template <int MODE>
static cudaError_t time_mode(unsigned* d, int blocks, int instr_per_chain, double* lane_ops_per_s) {
  cudaEvent_t e0, e1;
  cudaError_t e = cudaEventCreate(&e0);
  if (e != cudaSuccess) return e;
  e = cudaEventCreate(&e1);
  if (e != cudaSuccess) { cudaEventDestroy(e0); return e; }
  float best = 1e30f;
  peak_kernel<MODE><<<blocks, 256>>>(d, 1u, 5u);   // warm-up
  for (int rep = 0; rep < 3; ++rep) {
    cudaEventRecord(e0);
    peak_kernel<MODE><<<blocks, 256>>>(d, 1u, 5u);
    cudaEventRecord(e1);
    e = cudaEventSynchronize(e1);
    if (e != cudaSuccess) break;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (ms < best) best = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  if (e != cudaSuccess) return e;
  e = cudaGetLastError();
  const double ops = (double)blocks * 256.0 * PEAK_ITERS * PEAK_CHAINS * instr_per_chain;
  *lane_ops_per_s = ops / ((double)best * 1e-3);
  return e;
}

}  // namespace lpf

extern "C" int lpf_alu_peak(int device, double* out4) {
  if (!out4 || device < 0) return LPF_E_INVAL;
  int prev = -1;
  if (cudaGetDevice(&prev) != cudaSuccess) return LPF_E_CUDA;
  if (prev != device && cudaSetDevice(device) != cudaSuccess) return LPF_E_CUDA;
  int n_sm = 0;
  unsigned* d = nullptr;
  cudaError_t e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, device);
  if (e == cudaSuccess) e = cudaMalloc(&d, 4096);
  if (e == cudaSuccess) e = lpf::time_mode<0>(d, n_sm * 8, 1, out4 + 0);
  if (e == cudaSuccess) e = lpf::time_mode<1>(d, n_sm * 8, 1, out4 + 1);
  if (e == cudaSuccess) e = lpf::time_mode<2>(d, n_sm * 8, 3, out4 + 2);
  if (e == cudaSuccess) e = lpf::time_mode<3>(d, n_sm * 8, 1, out4 + 3);
  if (d) cudaFree(d);
  if (prev != device) cudaSetDevice(prev);
  return e == cudaSuccess ? LPF_OK : LPF_E_CUDA;
}
