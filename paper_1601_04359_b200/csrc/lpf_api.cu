// lpf_api.cu -- C ABI entry points of liblpf.so that touch the device (include/lpf.h).
// Host logic only: argument checks, geometry, workspace, program upload, launches.  Every step
// of the hot path runs in the kernels of lpf_kernels.cu.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstring>
#include <new>

#include "lpf_internal.h"
#include "lpf_kernels.cuh"

namespace lpf {

int build_host_table(lpf_paths* p);   // lpf_paths.cpp

static thread_local int g_last_cuda = 0;

static int cuda_fail(cudaError_t e) {
  g_last_cuda = (int)e;
  (void)cudaGetLastError();
  return e == cudaErrorMemoryAllocation ? LPF_E_NOMEM : LPF_E_CUDA;
}
#define LPF_CUDA(call)                                  \
  do {                                                  \
    cudaError_t e__ = (call);                           \
    if (e__ != cudaSuccess) return lpf::cuda_fail(e__); \
  } while (0)

struct DeviceGuard {   // binds the calling thread to the table's device for the call, then restores
  int prev = -1;
  bool ok = true;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; return; }
    if (prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
  }
  ~DeviceGuard() {
    int cur = -1;
    if (prev >= 0 && cudaGetDevice(&cur) == cudaSuccess && cur != prev) cudaSetDevice(prev);
  }
};

static void free_program(Program& pr) {
  if (pr.d_entries) cudaFree(pr.d_entries);
  if (pr.d_skip) cudaFree(pr.d_skip);
  if (pr.d_work) cudaFree(pr.d_work);
  pr.d_entries = nullptr; pr.d_skip = nullptr; pr.d_work = nullptr;
}

// uploads the program (once) and the work list expanded over (row band, strip band) of each octant
static int upload_program(Program& pr, const Geom& g) {
  if (!pr.d_entries) {
    // +64: the walker fetches 32 entries per warp, one chunk ahead
    LPF_CUDA(cudaMalloc(&pr.d_entries, sizeof(uint64_t) * (pr.entries.size() + 64)));
    LPF_CUDA(cudaMalloc(&pr.d_skip, sizeof(uint32_t) * std::max<size_t>(pr.skip.size(), 1)));
    LPF_CUDA(cudaMemset(pr.d_entries, 0, sizeof(uint64_t) * (pr.entries.size() + 64)));
    LPF_CUDA(cudaMemcpy(pr.d_entries, pr.entries.data(), sizeof(uint64_t) * pr.entries.size(), cudaMemcpyHostToDevice));
    LPF_CUDA(cudaMemcpy(pr.d_skip, pr.skip.data(), sizeof(uint32_t) * pr.skip.size(), cudaMemcpyHostToDevice));
  }
  int bands[4];
  bool same = pr.d_work != nullptr;
  for (int o = 0; o < 4; ++o) {
    const int sb = (g.v[o].n_strips + g.SB - 1) / g.SB;
    bands[o] = g.v[o].n_bands * 65536 + sb;
    same = same && bands[o] == pr.work_bands[o];
  }
  if (same) return LPF_OK;
  if (pr.d_work) { cudaFree(pr.d_work); pr.d_work = nullptr; }
  std::vector<int32_t> work;
  const size_t n_items = pr.items.size() / 4;
  for (size_t i = 0; i < n_items; ++i) {           // items are sorted big first; keep that order
    const int o = (int)pr.items[4 * i + 2];
    const int sb = (g.v[o].n_strips + g.SB - 1) / g.SB;
    for (int band = 0; band < g.v[o].n_bands; ++band)
      for (int s = 0; s < sb; ++s) {
        work.push_back((int32_t)pr.items[4 * i]);
        work.push_back((int32_t)pr.items[4 * i + 1]);
        work.push_back(o | (s << 4));
        work.push_back(band);
      }
  }
  pr.n_work = (int64_t)work.size() / 4;
  LPF_CUDA(cudaMalloc(&pr.d_work, sizeof(int32_t) * std::max<size_t>(work.size(), 4)));
  LPF_CUDA(cudaMemcpy(pr.d_work, work.data(), sizeof(int32_t) * work.size(), cudaMemcpyHostToDevice));
  for (int o = 0; o < 4; ++o) pr.work_bands[o] = bands[o];
  return LPF_OK;
}

}  // namespace lpf

using namespace lpf;

extern "C" int lpf_last_cuda_error(void) { return lpf::g_last_cuda; }

extern "C" int lpf_build_paths(int m, int device, lpf_paths** out) {
  if (!out) return LPF_E_INVAL;
  *out = nullptr;
  if (m < 0) return LPF_E_INVAL;
  if (m > MAX_M) return LPF_E_UNSUPPORTED;
  lpf_paths* p = new (std::nothrow) lpf_paths();
  if (!p) return LPF_E_NOMEM;
  p->m = m;
  p->device = device;
  int rc = build_host_table(p);
  if (rc != LPF_OK) { delete p; return rc; }
  if (device >= 0) {
    DeviceGuard g(device);
    cudaDeviceProp prop;
    cudaError_t e = g.ok ? cudaGetDeviceProperties(&prop, device) : cudaErrorInvalidDevice;
    if (e == cudaSuccess) e = cudaMalloc(&p->d_counter, sizeof(unsigned int) * 4);
    if (e != cudaSuccess) { rc = cuda_fail(e); delete p; return rc; }
    p->n_sm = prop.multiProcessorCount;
    p->max_smem = (int)prop.sharedMemPerBlockOptin;
  }
  *out = p;
  return LPF_OK;
}

extern "C" void lpf_free_paths(lpf_paths* p) {
  if (!p) return;
  if (p->device >= 0) {
    DeviceGuard g(p->device);
    for (auto& kv : p->programs) free_program(kv.second);
    if (p->d_packed) cudaFree(p->d_packed);
    if (p->d_counter) cudaFree(p->d_counter);
    if (p->d_swap_rec) cudaFree(p->d_swap_rec);
    if (p->d_swap_bits) cudaFree(p->d_swap_bits);
    if (p->d_io_in) cudaFree(p->d_io_in);
    if (p->d_io_out) cudaFree(p->d_io_out);
    if (p->io_stream) cudaStreamDestroy((cudaStream_t)p->io_stream);
    if (p->ev_start) cudaEventDestroy((cudaEvent_t)p->ev_start);
    if (p->ev_stop) cudaEventDestroy((cudaEvent_t)p->ev_stop);
  }
  delete p;
}

// ---- geometry ------------------------------------------------------------------------------------

namespace lpf {

cudaError_t launch_pack(const uint8_t* images, uint32_t* base, uint32_t* packed, const Geom& g, int B, int n_phase,
                        int phase0, unsigned int* counter, int n_sm, cudaStream_t st);
cudaError_t eval_occupancy(int TX, int TY, bool prune, int threads, size_t smem, int* blocks_per_sm);
cudaError_t launch_eval(const EvalParams& p, int grid, int threads, size_t smem, cudaStream_t st);
cudaError_t launch_mirror(unsigned long long* counts, int S, long long n_arrays, int n_sm, cudaStream_t st);
cudaError_t launch_objective(const long long* counts, const long long* target, int B, long long K,
                             unsigned long long* sse, int n_sm, cudaStream_t st);
cudaError_t launch_swap_delta(const uint8_t* image, uint32_t* bits, int H, int W, int m, int phase, const int* pairs,
                              long long n, const int32_t* rec, int n_nodes, int* delta, long long plane_stride,
                              unsigned int* counter, int n_sm, cudaStream_t st);

static int eval_impl(lpf_paths* p, const uint8_t* images, int B, int H, int W, int n_phase, int phase0,
                     int64_t* counts, unsigned flags, void* stream, const uint8_t* start_mask = nullptr) {
  if (!p || !images || !counts) return LPF_E_INVAL;
  if (p->device < 0) return LPF_E_INVAL;
  if (B < 1 || H < 1 || W < 1) return LPF_E_INVAL;
  if (n_phase == 1 && phase0 != 0 && phase0 != 1) return LPF_E_INVAL;
  if (p->m > std::min(H, W) - 1) return LPF_E_INVAL;
  if (flags & ~(LPF_PRUNE | LPF_NO_TRIE | LPF_S2 | LPF_NO_E2)) return LPF_E_INVAL;
  DeviceGuard dg(p->device);
  if (!dg.ok) return LPF_E_CUDA;
  cudaStream_t st = (cudaStream_t)stream;
  Geom g;
  // the eroded planes serve the trie program; m = 0 has nothing but the root, which only the plain program counts
  const bool use_e2 = !(flags & (LPF_NO_E2 | LPF_NO_TRIE | LPF_S2)) && p->m >= 1;
  if (!choose_geom(p->m, H, W, B, p->max_smem, p->tile_tx, p->tile_ty, p->cta_warps, use_e2, &g)) return LPF_E_UNSUPPORTED;
  const int Bpad = (B + g.G - 1) / g.G * g.G;
  long long off = 0;
  int work_per_item = 0;                           // (row band x strip band) pairs summed over the octants / 4
  for (int o = 0; o < 4; ++o) {
    g.v[o].packed_off = off;
    off += (long long)Bpad * g.v[o].view_words;
    work_per_item += g.v[o].n_bands * ((g.v[o].n_strips + g.SB - 1) / g.SB);
  }
  g.plane_words = off;
  work_per_item = std::max(1, work_per_item / 4);
  const int n_gp = (Bpad / g.G) * n_phase;

  // work items: about 20 per resident CTA (measured optimum on configs 2-4), pieces of 256 .. 16384 trie nodes; fewer mask slots than the
  // kernel provides (a smaller piece needs fewer)
  const int resident_guess = p->n_sm * 2;
  long long n_nodes = 0;
  for (int o = 0; o < 4; ++o) n_nodes += (long long)p->oct[o].size();
  const long long want_items = std::max<long long>(1, 32ll * resident_guess / ((long long)n_gp * work_per_item));
  long long piece = n_nodes / want_items;
  piece = std::max<long long>(256, std::min<long long>(piece, 16384));
  int q = 256;
  if (flags & LPF_S2) {                            // S2 items are lists of vectors, not trie pieces
    piece = std::max<long long>(32, std::min<long long>(p->n_half / want_items, 4096));
    q = 32;
  }
  while (q * 2 <= piece) q *= 2;                   // quantised so that nearby shapes share one cached program
  Program* pr = nullptr;
  for (;; q /= 2) {
    try {
      pr = &get_program(p, q, flags, g.v[0].stride, g.v[1].stride, g.v[0].e2_band_off, g.v[1].e2_band_off);
    } catch (const std::bad_alloc&) {
      return LPF_E_NOMEM;
    }
    if (pr->n_slots <= STACK_SLOTS_BUDGET) break;
    if (q <= 64) return LPF_E_UNSUPPORTED;
  }
  if (pr->entries.size() >= (size_t)1 << 30) return LPF_E_UNSUPPORTED;
  int rc = upload_program(*pr, g);
  if (rc != LPF_OK) return rc;

  const bool prune = (flags & LPF_PRUNE) != 0;
  const size_t smem_total = (size_t)g.smem_bytes;
  int occ = 0;
  LPF_CUDA(eval_occupancy(g.TX, g.TY, prune, g.threads, smem_total, &occ));
  if (occ < 1) return LPF_E_UNSUPPORTED;
  const int resident = p->n_sm * occ;

  // workspace: the packed octant views, then the compact row-major / column-major bit images of stage 1
  const size_t views_bytes = (size_t)n_phase * (size_t)g.plane_words * 4;
  const size_t base_words = (size_t)n_phase * B * ((size_t)H * ((W + 31) / 32) + (size_t)W * ((H + 31) / 32));
  // ... and, for lpf_eval_masked, the views and the base bit images of the start mask (one image, one plane)
  Geom gm = g;
  size_t mask_views_bytes = 0, mask_base_bytes = 0;
  if (start_mask) {
    long long moff = 0;
    for (int o = 0; o < 4; ++o) { gm.v[o].packed_off = moff; moff += gm.v[o].view_words; }
    gm.plane_words = moff;
    mask_views_bytes = (size_t)moff * 4;
    mask_base_bytes = ((size_t)H * ((W + 31) / 32) + (size_t)W * ((H + 31) / 32)) * 4;
  }
  const size_t need = views_bytes + base_words * 4 + mask_views_bytes + mask_base_bytes;
  if (need > p->packed_bytes) {
    if (p->d_packed) { LPF_CUDA(cudaStreamSynchronize(st)); cudaFree(p->d_packed); p->d_packed = nullptr; p->packed_bytes = 0; }
    LPF_CUDA(cudaMalloc(&p->d_packed, need));
    p->packed_bytes = need;
  }

  const int S = 2 * p->m + 1;
  LPF_CUDA(cudaMemsetAsync(counts, 0, sizeof(int64_t) * (size_t)B * n_phase * S * S, st));
  LPF_CUDA(launch_pack(images, p->d_packed + views_bytes / 4, p->d_packed, g, B, n_phase, phase0, p->d_counter,
                       p->n_sm, st));
  uint32_t* const d_mask = p->d_packed + views_bytes / 4 + base_words;
  if (start_mask)                                  // "phase" -1: a start pixel is selected iff its byte is non-zero
    LPF_CUDA(launch_pack(start_mask, d_mask + mask_views_bytes / 4, d_mask, gm, 1, 1, -1, p->d_counter, p->n_sm, st));

  EvalParams ep;
  ep.g = g;
  ep.entries = (const uint2*)pr->d_entries;
  ep.skip = pr->d_skip;
  ep.work = (const int4*)pr->d_work;
  ep.n_work = (int)pr->n_work;
  ep.n_gp = n_gp;
  ep.B = B;
  ep.n_phase = n_phase;
  ep.packed = p->d_packed;
  ep.Bpad = Bpad;
  ep.counts = (unsigned long long*)counts;
  ep.S = S;
  ep.counter = p->d_counter;
  ep.prune = prune ? 1 : 0;
  ep.n_slots = pr->n_slots;
  ep.mask = start_mask ? d_mask : nullptr;
  for (int o = 0; o < 4; ++o) ep.mask_off[o] = gm.v[o].packed_off;
  const long long total_work = (long long)ep.n_work * n_gp;
  if (total_work >= (1ll << 32)) return LPF_E_UNSUPPORTED;
  const int grid = (int)std::min<long long>(total_work, resident);
  if (p->timing) {
    if (!p->ev_start) {
      LPF_CUDA(cudaEventCreate((cudaEvent_t*)&p->ev_start));
      LPF_CUDA(cudaEventCreate((cudaEvent_t*)&p->ev_stop));
    }
    LPF_CUDA(cudaEventRecord((cudaEvent_t)p->ev_start, st));
  }
  LPF_CUDA(launch_eval(ep, grid, g.threads, smem_total, st));
  if (p->timing) LPF_CUDA(cudaEventRecord((cudaEvent_t)p->ev_stop, st));
  LPF_CUDA(launch_mirror((unsigned long long*)counts, S, (long long)B * n_phase, p->n_sm, st));

  p->last_info[0] = start_mask ? 6 : 4;                  // kernels launched (pack base, pack views, eval, mirror)
  p->last_info[1] = total_work;
  p->last_info[2] = (int64_t)pr->entries.size();         // program entries (all four octants)
  p->last_info[3] = grid;
  p->last_info[4] = g.threads;
  p->last_info[5] = (int64_t)smem_total;
  p->last_info[6] = g.TX * 1000 + g.TY * 100 + pr->n_slots;   // thread tile TX, TY and mask-stack slots
  p->last_info[7] = g.G;
  return LPF_OK;
}

}  // namespace lpf

extern "C" int lpf_eval(lpf_paths* p, const uint8_t* images, int B, int H, int W, int phase, int64_t* counts,
                        unsigned flags, void* stream) {
  return lpf::eval_impl(p, images, B, H, W, 1, phase, counts, flags, stream);
}

extern "C" int lpf_eval_both(lpf_paths* p, const uint8_t* images, int B, int H, int W, int64_t* counts,
                             unsigned flags, void* stream) {
  return lpf::eval_impl(p, images, B, H, W, 2, 0, counts, flags, stream);
}

extern "C" int lpf_eval_masked(lpf_paths* p, const uint8_t* images, int B, int H, int W, int phase,
                               const uint8_t* start_mask, int64_t* counts, unsigned flags, void* stream) {
  if (!start_mask || phase < -1 || phase > 1) return LPF_E_INVAL;
  return phase < 0 ? lpf::eval_impl(p, images, B, H, W, 2, 0, counts, flags, stream, start_mask)
                   : lpf::eval_impl(p, images, B, H, W, 1, phase, counts, flags, stream, start_mask);
}

extern "C" int lpf_set_timing(lpf_paths* p, int enable) {
  if (!p || p->device < 0) return LPF_E_INVAL;
  p->timing = enable ? 1 : 0;
  return LPF_OK;
}

extern "C" int lpf_set_tile(lpf_paths* p, int tx, int ty, int cta_warps) {
  if (!p) return LPF_E_INVAL;
  const bool known = (tx == 0 && ty == 0) || (tx == 4 && ty == 2) || (tx == 8 && ty == 1) || (tx == 4 && ty == 4) ||
                     (tx == 8 && ty == 2) || (tx == 16 && ty == 1);
  if (!known || cta_warps < 0 || cta_warps > 8) return LPF_E_INVAL;
  p->tile_tx = tx; p->tile_ty = ty; p->cta_warps = cta_warps;
  return LPF_OK;
}

extern "C" int lpf_last_eval_kernel_ms(lpf_paths* p, float* ms) {
  if (!p || !ms || p->device < 0 || !p->ev_start) return LPF_E_INVAL;
  DeviceGuard dg(p->device);
  if (!dg.ok) return LPF_E_CUDA;
  LPF_CUDA(cudaEventSynchronize((cudaEvent_t)p->ev_stop));
  LPF_CUDA(cudaEventElapsedTime(ms, (cudaEvent_t)p->ev_start, (cudaEvent_t)p->ev_stop));
  return LPF_OK;
}

extern "C" int lpf_last_launch_info(const lpf_paths* p, int64_t* out8) {
  if (!p || !out8) return LPF_E_INVAL;
  std::memcpy(out8, p->last_info, sizeof(p->last_info));
  return LPF_OK;
}

extern "C" int lpf_objective(const int64_t* counts, const int64_t* target, int B, int64_t K, uint64_t* sse,
                             void* stream) {
  if (!counts || !target || !sse || B < 1 || K < 1) return LPF_E_INVAL;
  int dev = 0, n_sm = 0;
  LPF_CUDA(cudaGetDevice(&dev));
  LPF_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
  LPF_CUDA(lpf::launch_objective((const long long*)counts, (const long long*)target, B, (long long)K,
                                 (unsigned long long*)sse, n_sm, (cudaStream_t)stream));
  return LPF_OK;
}

// ---- swap delta ----------------------------------------------------------------------------------

namespace lpf {

// node records of the image-coordinate trie for the swap-delta kernel, built and uploaded on first use
static int ensure_swap_table(lpf_paths* p) {
  if (p->d_swap_rec) return LPF_OK;
  try {
    std::vector<int32_t> rec;
    build_swap_records(p, rec);
    if ((int64_t)rec.size() != 4 * p->n_trie_nodes) return LPF_E_INVAL;
    LPF_CUDA(cudaMalloc(&p->d_swap_rec, sizeof(int32_t) * rec.size()));
    LPF_CUDA(cudaMemcpy(p->d_swap_rec, rec.data(), sizeof(int32_t) * rec.size(), cudaMemcpyHostToDevice));
  } catch (const std::bad_alloc&) {
    return LPF_E_NOMEM;
  }
  return LPF_OK;
}

}  // namespace lpf

namespace lpf {

// phase 0 | 1: delta [n][S][S] of that phase;  phase < 0: both phases in one pass over the trie, phase k written at
// delta + k * plane_stride (used by lpf_anneal)
int swap_delta_impl(lpf_paths* p, const uint8_t* image, int H, int W, int phase, const int32_t* pairs, int64_t n,
                    int32_t* delta, int64_t plane_stride, void* stream) {
  if (!p || !image || !pairs || !delta) return LPF_E_INVAL;
  if (p->device < 0 || H < 1 || W < 1 || n < 0) return LPF_E_INVAL;
  if (phase < -1 || phase > 1) return LPF_E_INVAL;
  if (p->m > std::min(H, W) - 1) return LPF_E_INVAL;
  if (n == 0) return LPF_OK;
  DeviceGuard dg(p->device);
  if (!dg.ok) return LPF_E_CUDA;
  const int n_planes = phase < 0 ? 2 : 1;
  // the padded base bit image(s) (halo of m pixels) and eight warp stacks of 4 KB live in shared memory; 24-bit node indices
  const size_t padded_words = (size_t)n_planes * (H + 2 * p->m) * ((W + 2 * p->m + 31) / 32);
  const size_t smem = padded_words * 4 + 8 + 8 * 512 * 8;
  if (smem + 2048 > (size_t)p->max_smem || p->n_trie_nodes >= (1 << 24)) return LPF_E_UNSUPPORTED;
  int rc = ensure_swap_table(p);
  if (rc != LPF_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  const size_t bits_bytes =
      (n_planes * ((size_t)H * ((W + 31) / 32) + (size_t)W * ((H + 31) / 32)) + padded_words) * 4;
  if (bits_bytes > p->swap_bits_bytes) {
    if (p->d_swap_bits) { LPF_CUDA(cudaStreamSynchronize(st)); cudaFree(p->d_swap_bits); p->d_swap_bits = nullptr; }
    p->swap_bits_bytes = 0;
    LPF_CUDA(cudaMalloc(&p->d_swap_bits, bits_bytes));
    p->swap_bits_bytes = bits_bytes;
  }
  LPF_CUDA(launch_swap_delta(image, p->d_swap_bits, H, W, p->m, phase, pairs, (long long)n, p->d_swap_rec,
                             (int)p->n_trie_nodes, delta, (long long)plane_stride, p->d_counter + 1, p->n_sm, st));
  return LPF_OK;
}

}  // namespace lpf

extern "C" int lpf_swap_delta(lpf_paths* p, const uint8_t* image, int H, int W, int phase, const int32_t* pairs,
                              int64_t n, int32_t* delta, void* stream) {
  if (phase != 0 && phase != 1) return LPF_E_INVAL;
  return lpf::swap_delta_impl(p, image, H, W, phase, pairs, n, delta, 0, stream);
}

// ---- host-buffer convenience (end-to-end measurement) ---------------------------------------------

extern "C" int lpf_eval_host(lpf_paths* p, const uint8_t* images_host, int B, int H, int W, int phase,
                             int64_t* counts_host, unsigned flags) {
  if (!p || !images_host || !counts_host) return LPF_E_INVAL;
  if (p->device < 0 || B < 1 || H < 1 || W < 1) return LPF_E_INVAL;
  DeviceGuard dg(p->device);
  if (!dg.ok) return LPF_E_CUDA;
  const int n_phase = phase < 0 ? 2 : 1;
  const int S = 2 * p->m + 1;
  const size_t in_bytes = (size_t)B * H * W;
  const size_t out_bytes = sizeof(int64_t) * (size_t)B * n_phase * S * S;
  if (in_bytes > p->io_in_bytes) {
    if (p->d_io_in) cudaFree(p->d_io_in);
    p->d_io_in = nullptr; p->io_in_bytes = 0;
    LPF_CUDA(cudaMalloc(&p->d_io_in, in_bytes));
    p->io_in_bytes = in_bytes;
  }
  if (out_bytes > p->io_out_bytes) {
    if (p->d_io_out) cudaFree(p->d_io_out);
    p->d_io_out = nullptr; p->io_out_bytes = 0;
    LPF_CUDA(cudaMalloc(&p->d_io_out, out_bytes));
    p->io_out_bytes = out_bytes;
  }
  if (!p->io_stream) LPF_CUDA(cudaStreamCreateWithFlags((cudaStream_t*)&p->io_stream, cudaStreamNonBlocking));
  cudaStream_t st = (cudaStream_t)p->io_stream;
  LPF_CUDA(cudaMemcpyAsync(p->d_io_in, images_host, in_bytes, cudaMemcpyHostToDevice, st));
  int rc = n_phase == 2 ? lpf_eval_both(p, (const uint8_t*)p->d_io_in, B, H, W, (int64_t*)p->d_io_out, flags, st)
                        : lpf_eval(p, (const uint8_t*)p->d_io_in, B, H, W, phase, (int64_t*)p->d_io_out, flags, st);
  if (rc != LPF_OK) return rc;
  LPF_CUDA(cudaMemcpyAsync(counts_host, p->d_io_out, out_bytes, cudaMemcpyDeviceToHost, st));
  LPF_CUDA(cudaStreamSynchronize(st));
  return LPF_OK;
}
