// lpf_static.cu -- lpf_swap_delta_static: the swap-delta evaluation for callers that
// cannot allocate device memory (CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).
//
// lpf_swap_delta keeps its scratch -- the compact bit images of stage 1, the bit planes padded with their halo of m
// pixels, the density mask -- in a workspace of the lpf_paths object that grows with cudaMalloc.  Here the same
// kernels get that scratch from ONE file-scope array in device memory, g_scratch, of LPF_STATIC_SCRATCH_BYTES: every
// GPU that loads the library holds it until the process exits, nothing is ever allocated or freed for it.
//
// g_scratch in HOST code is the host-side stand-in of the symbol, not a device address: a kernel given it would fault
// (or, where the GPU can reach host memory, silently use the wrong memory).  The device address is looked up once per
// device, with that device current, by cudaGetSymbolAddress (scratch_of below) and that pointer is what the kernels get.
#include <cuda_runtime.h>

#include <algorithm>
#include <mutex>

#include "lpf.h"
#include "lpf_internal.h"

// The scratch of every lpf_swap_delta_static call on this GPU: [0] work counter of the pack kernel, [1] dense planes,
// from word 64 on the bit images.  It keeps the last call's contents; calls that overlap on the GPU race on it.
static __device__ __align__(256) uint32_t g_scratch[LPF_STATIC_SCRATCH_BYTES / 4];

namespace lpf {

int cuda_fail(cudaError_t e);   // lpf_api.cu: records the code for lpf_last_cuda_error
// lpf_kernels.cu: memset of delta, pack (stage 1, padded planes, density mask), swap_delta_kernel_v3, mirror
cudaError_t launch_swap_delta(const uint8_t* image, uint32_t* bits, int H, int W, int m, int phase, const int* pairs,
                              long long n, const int32_t* rec, int n_nodes, const int32_t* rrec, int* delta,
                              long long plane_stride, unsigned int* counter, int n_sm, cudaStream_t st);

namespace {

constexpr size_t SCRATCH_WORDS = LPF_STATIC_SCRATCH_BYTES / 4;
constexpr size_t HEAD_WORDS = 64;          // 256 bytes: the bit images stay aligned

constexpr int MAX_DEVICES = 64;
std::mutex g_mu;
uint32_t* g_scratch_dev[MAX_DEVICES];      // device address of g_scratch on device d (nullptr: not looked up yet)

// device address of g_scratch on the CURRENT device `dev`; one lookup per device
cudaError_t scratch_of(int dev, uint32_t** out) {
  std::lock_guard<std::mutex> lk(g_mu);
  if (!g_scratch_dev[dev]) {
    void* ptr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&ptr, g_scratch);
    if (e != cudaSuccess) return e;
    g_scratch_dev[dev] = (uint32_t*)ptr;
  }
  *out = g_scratch_dev[dev];
  return cudaSuccess;
}

struct CurrentDevice {   // binds the calling thread to `dev` for the call, then restores
  int prev = -1;
  bool ok = true;
  explicit CurrentDevice(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; return; }
    if (prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
  }
  ~CurrentDevice() {
    int cur = -1;
    if (prev >= 0 && cudaGetDevice(&cur) == cudaSuccess && cur != prev) cudaSetDevice(prev);
  }
};

}  // namespace
}  // namespace lpf

extern "C" int lpf_swap_delta_static(const lpf_paths* p, const uint8_t* image, int H, int W, int phase,
                                     const int32_t* pairs, int64_t n, int32_t* delta, void* stream) {
  using namespace lpf;
  if (!p || !image || !pairs || !delta) return LPF_E_INVAL;
  if (p->device < 0 || p->device >= MAX_DEVICES || H < 1 || W < 1 || n < 0) return LPF_E_INVAL;
  if (phase != 0 && phase != 1) return LPF_E_INVAL;
  if (p->m > std::min(H, W) - 1) return LPF_E_INVAL;
  // the node records of the trie are tables of the lpf_paths object, uploaded by lpf_reserve: never here
  if (!p->d_swap_rec) return LPF_E_INVAL;
  // what lpf_swap_delta refuses: the padded bit plane and the warp stacks must fit the shared memory of one block
  const size_t padded_plane = (size_t)(H + 2 * p->m) * ((W + 2 * p->m + 31) / 32);
  if (padded_plane * 4 + 8 + 8 * 512 * 8 + 2048 > (size_t)p->max_smem) return LPF_E_UNSUPPORTED;
  // the scratch of this call: one phase plane of compact bit images (row-major and column-major) and its padded plane
  const size_t words = (size_t)H * ((W + 31) / 32) + (size_t)W * ((H + 31) / 32) + padded_plane;
  if (HEAD_WORDS + words > SCRATCH_WORDS) return LPF_E_TOO_LARGE;
  if (n == 0) return LPF_OK;
  CurrentDevice cd(p->device);
  if (!cd.ok) return LPF_E_CUDA;
  uint32_t* scratch = nullptr;
  cudaError_t e = scratch_of(p->device, &scratch);
  if (e != cudaSuccess) return cuda_fail(e);
  cudaStream_t st = (cudaStream_t)stream;
  // the array keeps the last call's contents: everything this call reads starts at zero
  e = cudaMemsetAsync(scratch, 0, (HEAD_WORDS + words) * 4, st);
  if (e != cudaSuccess) return cuda_fail(e);
  e = launch_swap_delta(image, scratch + HEAD_WORDS, H, W, p->m, phase, pairs, (long long)n, p->d_swap_rec,
                        (int)p->n_trie_nodes, p->d_swap_rrec, delta, 0, scratch, p->n_sm, st);
  if (e != cudaSuccess) return cuda_fail(e);
  return LPF_OK;
}
