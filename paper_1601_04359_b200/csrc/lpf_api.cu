// lpf_api.cu -- C ABI entry points of liblpf.so that touch the device (include/lpf.h).
// Host logic only: argument checks, geometry, workspace, program upload, launches.  Every step
// of the hot path runs in the kernels of lpf_kernels.cu.
//
// Allocation discipline ("no hidden host sync except in lpf_build_paths"): everything that
// allocates, uploads or synchronises lives in lpf_reserve (reserve_* below).  The hot calls look their shape up in
// p->plans and only enqueue kernels and memsets on the caller's stream; a call for a shape that was never reserved
// reserves it first (documented in lpf.h) -- after that first call it is a pure enqueue as well.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstring>
#include <new>

#include "lpf_internal.h"
#include "lpf_kernels.cuh"

namespace lpf {

int build_host_table(lpf_paths* p);   // lpf_paths.cpp

static thread_local int g_last_cuda = 0;

int cuda_fail(cudaError_t e) {
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

// Consecutive calls on one lpf_paths share its workspace.  A call on a stream other than the previous call's first
// makes its stream wait (on the device) for the event recorded after that call; nothing blocks the host.  While a
// stream is being captured into a CUDA graph neither the wait nor the record is issued: the graph's own order holds.
struct StreamOrder {
  lpf_paths* p;
  cudaStream_t st;
  bool capturing = false;
  cudaError_t err = cudaSuccess;
  StreamOrder(lpf_paths* p_, cudaStream_t st_) : p(p_), st(st_) {
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    err = cudaStreamIsCapturing(st, &cs);
    capturing = cs != cudaStreamCaptureStatusNone;
    if (err == cudaSuccess && !capturing && p->last_stream_valid && p->last_stream != (void*)st)
      err = cudaStreamWaitEvent(st, (cudaEvent_t)p->ev_done, 0);
  }
  cudaError_t done() {
    if (capturing) return cudaSuccess;
    p->last_stream = (void*)st;
    p->last_stream_valid = 1;
    return cudaEventRecord((cudaEvent_t)p->ev_done, st);
  }
};

// growing a workspace buffer: work already enqueued may still read the old one
template <typename T>
static int grow(T** buf, size_t* have, size_t need) {
  if (need <= *have && *buf) return LPF_OK;
  if (*buf) {
    LPF_CUDA(cudaDeviceSynchronize());
    cudaFree(*buf);
    *buf = nullptr;
    *have = 0;
  }
  LPF_CUDA(cudaMalloc((void**)buf, std::max<size_t>(need, 16)));
  *have = need;
  return LPF_OK;
}

static void free_program(Program& pr) {
  if (pr.d_entries) cudaFree(pr.d_entries);
  if (pr.d_skip) cudaFree(pr.d_skip);
  if (pr.d_class_slots) cudaFree(pr.d_class_slots);
  if (pr.d_class_geom) cudaFree(pr.d_class_geom);
  pr.d_entries = nullptr;
  pr.d_skip = nullptr;
  pr.d_class_slots = nullptr;
  pr.d_class_geom = nullptr;
}

// uploads the program once; the device pointers are published only when every step has succeeded
static int upload_program(Program& pr) {
  if (pr.d_entries) return LPF_OK;
  uint64_t* d_e = nullptr;
  uint32_t* d_s = nullptr;
  signed char* d_c = nullptr;
  int* d_g = nullptr;
  const size_t ne = pr.entries.size() + 64;      // +64: the walker fetches 32 entries per warp, one chunk ahead
  std::vector<signed char> slots(std::max<size_t>(pr.classes.size(), 1) * MAX_PATTERNS, (signed char)-1);
  for (size_t c = 0; c < pr.classes.size(); ++c)
    std::memcpy(slots.data() + c * MAX_PATTERNS, pr.classes[c].slot_of, MAX_PATTERNS);
  std::vector<int> geom(std::max<size_t>(pr.classes.size(), 1) * 4, 0);
  for (size_t c = 0; c < pr.classes.size(); ++c) {
    geom[4 * c] = pr.classes[c].band_words;
    geom[4 * c + 1] = pr.classes[c].rows;
    geom[4 * c + 2] = pr.classes[c].n;
    geom[4 * c + 3] = pr.classes[c].level;
  }
  cudaError_t e = cudaMalloc(&d_e, sizeof(uint64_t) * ne);
  if (e == cudaSuccess) e = cudaMalloc(&d_s, sizeof(uint32_t) * std::max<size_t>(pr.skip.size(), 1));
  if (e == cudaSuccess) e = cudaMalloc(&d_c, slots.size());
  if (e == cudaSuccess) e = cudaMalloc(&d_g, sizeof(int) * geom.size());
  if (e == cudaSuccess) e = cudaMemset(d_e, 0, sizeof(uint64_t) * ne);
  if (e == cudaSuccess)
    e = cudaMemcpy(d_e, pr.entries.data(), sizeof(uint64_t) * pr.entries.size(), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(d_s, pr.skip.data(), sizeof(uint32_t) * pr.skip.size(), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(d_c, slots.data(), slots.size(), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(d_g, geom.data(), sizeof(int) * geom.size(), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) {
    if (d_e) cudaFree(d_e);
    if (d_s) cudaFree(d_s);
    if (d_c) cudaFree(d_c);
    if (d_g) cudaFree(d_g);
    return cuda_fail(e);
  }
  pr.d_entries = d_e;
  pr.d_skip = d_s;
  pr.d_class_slots = d_c;
  pr.d_class_geom = d_g;
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
    if (e == cudaSuccess) e = cudaEventCreateWithFlags((cudaEvent_t*)&p->ev_done, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreate((cudaEvent_t*)&p->ev_start);
    if (e == cudaSuccess) e = cudaEventCreate((cudaEvent_t*)&p->ev_stop);
    if (e != cudaSuccess) { rc = cuda_fail(e); lpf_free_paths(p); return rc; }
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
    cudaDeviceSynchronize();
    for (auto& kv : p->programs) free_program(kv.second);
    for (auto& kv : p->plans)
      if (kv.second.d_work) cudaFree(kv.second.d_work);
    if (p->d_packed) cudaFree(p->d_packed);
    if (p->d_counter) cudaFree(p->d_counter);
    if (p->d_swap_rec) cudaFree(p->d_swap_rec);
    if (p->d_swap_rrec) cudaFree(p->d_swap_rrec);
    if (p->d_swap_bits) cudaFree(p->d_swap_bits);
    if (p->d_an_state) cudaFree(p->d_an_state);
    if (p->d_an_delta) cudaFree(p->d_an_delta);
    if (p->d_an_dE) cudaFree(p->d_an_dE);
    if (p->d_io_in) cudaFree(p->d_io_in);
    if (p->d_io_out) cudaFree(p->d_io_out);
    if (p->io_stream) cudaStreamDestroy((cudaStream_t)p->io_stream);
    if (p->ev_done) cudaEventDestroy((cudaEvent_t)p->ev_done);
    if (p->ev_start) cudaEventDestroy((cudaEvent_t)p->ev_start);
    if (p->ev_stop) cudaEventDestroy((cudaEvent_t)p->ev_stop);
  }
  delete p;
}

// ---- plans: everything that allocates, uploads or synchronises ----------------------------------------

namespace lpf {

cudaError_t launch_pack(const uint8_t* images, uint32_t* base, uint32_t* packed, const Geom& g, int B, int Bpad,
                        int n_phase, int phase0, unsigned int* counter, int n_sm, cudaStream_t st);
cudaError_t eval_occupancy(int TX, int TY, bool prune, bool tm, int threads, size_t smem, int max_smem,
                           int* blocks_per_sm);
cudaError_t launch_eval(const EvalParams& p, int grid, int threads, size_t smem, cudaStream_t st);
cudaError_t launch_shallow(const EvalParams& p, const ShallowList& sl, int n_sm, cudaStream_t st);
cudaError_t launch_mirror(unsigned long long* counts, int S, long long n_arrays, int n_sm, cudaStream_t st);
cudaError_t launch_objective(const long long* counts, const long long* target, int B, long long K,
                             unsigned long long* sse, int n_sm, cudaStream_t st);
cudaError_t swap_delta_prepare(size_t smem);
cudaError_t launch_swap_delta(const uint8_t* image, uint32_t* bits, int H, int W, int m, int phase, const int* pairs,
                              long long n, const int32_t* rec, int n_nodes, const int32_t* rrec, int* delta,
                              long long plane_stride, unsigned int* counter, int n_sm, cudaStream_t st);

static std::array<int64_t, 8> plan_key(const lpf_paths* p, int B, int H, int W, int n_phase, unsigned flags,
                                       bool masked) {
  return {B, H, W, n_phase, (int64_t)flags, masked ? 1 : 0, 100 * p->tile_tx + p->tile_ty,
          p->cta_warps + 100 * p->n_teams + 10000 * (p->max_level + 1) + 100000 * (int64_t)p->smem_limit +
              (p->no_tmem ? (int64_t)1 << 50 : 0)};
}

static int check_eval_args(const lpf_paths* p, int B, int H, int W, unsigned flags) {
  if (!p || p->device < 0) return LPF_E_INVAL;
  if (B < 1 || H < 1 || W < 1) return LPF_E_INVAL;
  if (p->m > std::min(H, W) - 1) return LPF_E_INVAL;
  if (flags & ~(LPF_PRUNE | LPF_NO_TRIE | LPF_S2 | LPF_NO_E2)) return LPF_E_INVAL;
  return LPF_OK;
}

// builds the plan of one eval shape: geometry, program (built and uploaded), work list, launch configuration, and
// grows the packed-image workspace.  The only place of the eval path that allocates, copies or synchronises.
static int reserve_eval(lpf_paths* p, int B, int H, int W, int n_phase, unsigned flags, bool masked) {
  const auto key = plan_key(p, B, H, W, n_phase, flags, masked);
  if (p->plans.count(key)) return LPF_OK;
  EvalPlan pl;
  Geom& g = pl.g;
  // the eroded planes serve the trie program (choose_geom caps the level at m: m = 0 has nothing but the root)
  const int max_level = (flags & (LPF_NO_E2 | LPF_NO_TRIE | LPF_S2))
                            ? 0
                            : std::min(p->level_ok, p->max_level >= 0 ? p->max_level : MAX_LEVEL);
  const int max_teams = max_teams_of(p);
  if (!choose_geom(p->m, H, W, B, p->max_smem, p->smem_limit, p->tile_tx, p->tile_ty, p->cta_warps, max_level,
                   max_teams, p->path_patterns, &g))
    return LPF_E_UNSUPPORTED;
  pl.Bpad = (B + g.G - 1) / g.G * g.G;
  long long off = 0;
  int work_per_item = 0;                           // (row band x strip band) pairs summed over the octants / 4
  for (int o = 0; o < 4; ++o) {
    g.v[o].packed_off = off;
    off += (long long)pl.Bpad * g.v[o].view_words;
    work_per_item += g.v[o].n_bands * ((g.v[o].n_strips + g.SB - 1) / g.SB);
  }
  g.plane_words = off;
  work_per_item = std::max(1, work_per_item / 4);
  pl.n_gp = (pl.Bpad / g.G) * n_phase;

  DeviceGuard dg(p->device);
  if (!dg.ok) return LPF_E_CUDA;
  // teams per CTA: a CTA of NT teams shares its bands in shared memory, every team walks its own work unit.  Shared
  // memory per CTA does not grow with NT, so NT is the one that keeps the most warps resident (fewest teams on a tie).
  pl.prune = (flags & LPF_PRUNE) ? 1 : 0;
  pl.smem = (size_t)g.smem_bytes;
  int occ = 0;
  {
    int best_warps = 0;
    g.NT = 1;
    // teams of several warps meet at a named barrier of their own: ids 1 .. 15
    const int nt_max = g.threads > 32 ? 15 : 32;
    for (int nt = 1; nt * g.threads <= EVAL_CTA_MAX_THREADS && nt <= nt_max; ++nt) {
      if (p->n_teams > 0 ? nt != p->n_teams : nt > max_teams) continue;
      int o_nt = 0;
      LPF_CUDA(eval_occupancy(g.TX, g.TY, pl.prune != 0, false, nt * g.threads, pl.smem, p->max_smem, &o_nt));
      const int warps = o_nt * nt * (g.threads / 32);
      if (warps > best_warps) { best_warps = warps; g.NT = nt; occ = o_nt; }
    }
    if (best_warps < 1) return LPF_E_UNSUPPORTED;
  }

  // work units: about 20 per resident team (measured on configs 2-4: the optimum is flat between 10 and 30), pieces
  // of 256 .. 16384 trie nodes, and at least 4 pieces per team, octant and pattern class so that the teams of a CTA
  // stay busy until a key is exhausted (measured on config 3, level 6: 2 pieces 2.56 ms, 4 pieces 2.49 ms)
  const int resident_guess = p->n_sm * std::max(occ, 1);
  long long n_nodes = 0;
  for (int o = 0; o < 4; ++o) n_nodes += (long long)p->oct[o].size();
  const int planes_all = g.K > 0 ? balanced_count(g.K) : 0;
  const int classes_guess = (g.K > 0 && g.v[0].n_planes < planes_all) ? std::max(1, 2 * planes_all / g.v[0].n_planes) : 1;
  // wider classes for the shallow slopes (their bands are lower: more planes fit) mean more units per key but fewer
  // keys; only while about four keys per resident CTA remain (measured: config 3 2.49 -> 2.26 ms, but config 2, with 96
  // keys for 148 CTAs already, 0.125 -> 0.135 ms)
  const bool widen = (long long)pl.n_gp * work_per_item * 4 * classes_guess >= 4ll * resident_guess;
  const long long want_items = std::max<long long>(
      {1, 20ll * g.NT * resident_guess / ((long long)pl.n_gp * work_per_item), 16ll * g.NT * classes_guess});
  long long piece = n_nodes / want_items;
  piece = std::max<long long>(256, std::min<long long>(piece, 16384));
  int q = 256;
  if (flags & LPF_S2) {                            // S2 items are lists of vectors, not trie pieces
    piece = std::max<long long>(32, std::min<long long>(p->n_half / want_items, 4096));
    q = 32;
  }
  while ((long long)q * q * 2 <= piece * piece) q *= 2;   // nearest power of two: nearby shapes share one cached program
  Program* pr = nullptr;
  for (;; q /= 2) {
    try {
      pr = &get_program(p, q, flags, g.v[0].stride, g.v[1].stride, g.K, g.v[0].n_planes, g.v[0].band_words,
                        g.v[1].band_words, g.band_rows, widen);
    } catch (const std::bad_alloc&) {
      return LPF_E_NOMEM;
    }
    if (pr->n_slots <= STACK_SLOTS_BUDGET) break;
    drop_program(p, pr);                           // needs more mask slots than the kernel has: not kept
    if (q <= 64) return LPF_E_UNSUPPORTED;
  }
  if (pr->entries.size() >= (size_t)1 << 30) return LPF_E_UNSUPPORTED;
  int rc = upload_program(*pr);
  if (rc != LPF_OK) return rc;
  pl.pr = pr;

  // the work list: the items of one pattern class of an octant (one class at level 0) expanded over the strip bands
  // are the units of one (octant, row band, class), big first; a key of the kernel is such a triple on one (image group,
  // phase plane)
  std::vector<int32_t> units, obtab;
  const size_t n_items = pr->items.size() / 4;
  const int n_classes = std::max<int>(1, (int)pr->classes.size());
  for (int cls = 0; cls < n_classes; ++cls) {
    const int o = pr->classes.empty() ? -1 : pr->classes[cls].octant;
    for (int oo = 0; oo < 4; ++oo) {
      if (o >= 0 && oo != o) continue;
      const int sb = (g.v[oo].n_strips + g.SB - 1) / g.SB;
      for (int band = 0; band < g.v[oo].n_bands; ++band) {
        const int32_t first = (int32_t)(units.size() / 4);
        for (size_t i = 0; i < n_items; ++i) {             // items are sorted by size, descending
          if ((int)pr->items[4 * i + 2] != oo || (int)pr->items[4 * i + 3] != cls) continue;
          for (int s = 0; s < sb; ++s) {
            units.push_back((int32_t)pr->items[4 * i]);
            units.push_back((int32_t)pr->items[4 * i + 1]);
            units.push_back(s);
            units.push_back(0);
          }
        }
        const int32_t cnt = (int32_t)(units.size() / 4) - first;
        if (cnt == 0) continue;                            // an octant without vectors (tiny m)
        obtab.push_back(first);
        obtab.push_back(cnt);
        obtab.push_back(oo | (cls << 2));
        obtab.push_back(band);
      }
    }
  }
  pl.n_ob = (int)(obtab.size() / 4);
  pl.n_units = (int64_t)units.size() / 4;
  // the walker's loop replayed on the host (eval_kernel_v3: chunks of 32 entries, a PAIR entry that is not the last of
  // its chunk is folded with its successor): the data operations the design executes per start word
  pl.piece_nodes = q;
  for (size_t i = 0; i < n_items; ++i) {
    const int64_t first = pr->items[4 * i], cnt = pr->items[4 * i + 1];
    for (int64_t c0 = 0; c0 < cnt; c0 += 32) {
      const int n = (int)std::min<int64_t>(32, cnt - c0);
      for (int k = 0; k < n; ++k) {
        uint32_t x = (uint32_t)pr->entries[first + c0 + k];
        if (x & E_RELOAD) ++pl.reloads;
        if ((x & E_PAIR) && k + 1 < n) {
          ++pl.fused_pairs;
          ++k;
          x = (uint32_t)pr->entries[first + c0 + k];
          if (x & E_RELOAD) ++pl.reloads;
        } else {
          ++pl.singles;
        }
        if (x & E_TERMINAL) ++pl.terminals;
      }
    }
  }
  const long long n_keys = (long long)pl.n_ob * pl.n_gp;
  pl.grid = (int)std::max<long long>(0, std::min<long long>(pl.n_units * pl.n_gp, (long long)p->n_sm * occ));
  // passes of the share cursor over the keys: enough to attach every CTA of the grid, and two more for helping out
  const long long passes = n_keys > 0 ? (pl.grid + n_keys - 1) / n_keys + 2 : 0;
  if (n_keys * passes >= (1ll << 31)) return LPF_E_UNSUPPORTED;
  pl.n_keys = n_keys;
  pl.n_shares = n_keys * passes;
  pl.occ = occ;
  // The mask stack in tensor memory: a CTA allocates all 512 columns, so it must be alone on its SM, and the slots of the
  // ceil(warps / 4) warps of a lane quarter must fit them (config 3: 8 warps x 4 slots x 16 words).
  {
    const int warps = g.NT * g.threads / 32, T = g.TX * g.TY;
    pl.tmem_stack = occ == 1 && pr->n_slots > 0 && ((warps + 3) / 4) * pr->n_slots * T <= 512 && !p->no_tmem;
    if (pl.tmem_stack) {
      int o_tm = 0;
      LPF_CUDA(eval_occupancy(g.TX, g.TY, pl.prune != 0, true, g.NT * g.threads, pl.smem, p->max_smem, &o_tm));
      if (o_tm != 1) pl.tmem_stack = 0;
    }
  }
  shallow_terminals(p, pr->K, &pl.shallow);

  // workspace: the packed octant views, then the compact row-major / column-major bit images of stage 1, then (for
  // lpf_eval_masked) the views and the base bit images of the start mask (one image, one plane)
  pl.views_bytes = (size_t)n_phase * (size_t)g.plane_words * 4;
  pl.base_words = (size_t)n_phase * B * ((size_t)H * ((W + 31) / 32) + (size_t)W * ((H + 31) / 32));
  pl.gm = g;
  if (masked) {
    long long moff = 0;
    for (int o = 0; o < 4; ++o) { pl.gm.v[o].packed_off = moff; moff += pl.gm.v[o].view_words; }
    pl.gm.plane_words = moff;
    pl.mask_views_bytes = (size_t)moff * 4;
    pl.mask_base_bytes = ((size_t)H * ((W + 31) / 32) + (size_t)W * ((H + 31) / 32)) * 4;
  }
  pl.need = pl.views_bytes + pl.base_words * 4 + pl.mask_views_bytes + pl.mask_base_bytes;
  rc = grow(&p->d_packed, &p->packed_bytes, pl.need);
  if (rc != LPF_OK) return rc;
  // units, (octant, row band) table and the counters (share cursor + one per key) in one allocation
  int32_t* d_work = nullptr;
  const size_t work_ints = units.size() + obtab.size();
  cudaError_t e = cudaMalloc(&d_work, sizeof(int32_t) * (std::max<size_t>(work_ints, 4) + (size_t)n_keys + 4));
  if (e == cudaSuccess && !units.empty())
    e = cudaMemcpy(d_work, units.data(), sizeof(int32_t) * units.size(), cudaMemcpyHostToDevice);
  if (e == cudaSuccess && !obtab.empty())
    e = cudaMemcpy(d_work + units.size(), obtab.data(), sizeof(int32_t) * obtab.size(), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) {
    if (d_work) cudaFree(d_work);
    return cuda_fail(e);
  }
  pl.d_work = d_work;
  pl.d_obtab = d_work + units.size();
  pl.d_counters = (unsigned int*)(d_work + work_ints);
  try {
    p->plans[key] = pl;
  } catch (const std::bad_alloc&) {
    cudaFree(d_work);
    return LPF_E_NOMEM;
  }
  return LPF_OK;
}

// node records of the image-coordinate trie and the bit-image workspace of lpf_swap_delta on H x W images
static int reserve_swap(lpf_paths* p, int H, int W) {
  if (!p || p->device < 0 || H < 1 || W < 1 || p->m > std::min(H, W) - 1) return LPF_E_INVAL;
  // the padded base bit image(s) (halo of m pixels) and eight warp stacks of 4 KB live in shared memory; 24-bit node indices
  const size_t padded_words = (size_t)2 * (H + 2 * p->m) * ((W + 2 * p->m + 31) / 32);
  const size_t smem1 = padded_words / 2 * 4 + 8 + 8 * 512 * 8;
  if (smem1 + 2048 > (size_t)p->max_smem || p->n_trie_nodes >= (1 << 24)) return LPF_E_UNSUPPORTED;
  DeviceGuard dg(p->device);
  if (!dg.ok) return LPF_E_CUDA;
  if (!p->d_swap_rec) {
    try {
      std::vector<int32_t> rec, rrec;
      build_swap_records(p, rec, rrec, SWAP_REV_MAX_NODES);
      if ((int64_t)rec.size() != 4 * p->n_trie_nodes) return LPF_E_INVAL;
      int32_t* d = nullptr;
      int32_t* dr = nullptr;
      cudaError_t e = cudaMalloc(&d, sizeof(int32_t) * rec.size());
      if (e == cudaSuccess) e = cudaMemcpy(d, rec.data(), sizeof(int32_t) * rec.size(), cudaMemcpyHostToDevice);
      if (e == cudaSuccess && !rrec.empty()) {
        e = cudaMalloc(&dr, sizeof(int32_t) * rrec.size());
        if (e == cudaSuccess) e = cudaMemcpy(dr, rrec.data(), sizeof(int32_t) * rrec.size(), cudaMemcpyHostToDevice);
      }
      if (e != cudaSuccess) {
        if (d) cudaFree(d);
        if (dr) cudaFree(dr);
        return cuda_fail(e);
      }
      p->d_swap_rec = d;
      p->d_swap_rrec = dr;
      p->n_swap_rev = (int64_t)rrec.size() / 4;
      p->n_swap_rev1 = 0;                            // children of the reversed root: preorder, sibling chain from 1
      for (int64_t i = 1; i < p->n_swap_rev; i += rrec[4 * i + 2]) ++p->n_swap_rev1;
    } catch (const std::bad_alloc&) {
      return LPF_E_NOMEM;
    }
    LPF_CUDA(swap_delta_prepare((size_t)p->max_smem));
  }
  // both phase planes: compact bit images of stage 1, then the padded planes
  const size_t bits_bytes = (2 * ((size_t)H * ((W + 31) / 32) + (size_t)W * ((H + 31) / 32)) + padded_words) * 4;
  return grow(&p->d_swap_bits, &p->swap_bits_bytes, bits_bytes);
}

int anneal_kmax(int m, int n_ph) {       // batch size: at most 256 proposals and about 256 MB of delta arrays per buffer
  const long long K2 = (long long)(2 * m + 1) * (2 * m + 1);
  int K_max = 256;
  while (K_max > 8 && (long long)K_max * K2 * 4 * n_ph > (256ll << 20)) K_max /= 2;
  return K_max;
}

int reserve_anneal(lpf_paths* p, int H, int W) {
  int rc = reserve_eval(p, 1, H, W, 1, 0, false);
  if (rc == LPF_OK) rc = reserve_eval(p, 1, H, W, 2, 0, false);
  if (rc == LPF_OK) rc = reserve_swap(p, H, W);
  if (rc != LPF_OK) return rc;
  DeviceGuard dg(p->device);
  if (!dg.ok) return LPF_E_CUDA;
  const long long K2 = (long long)(2 * p->m + 1) * (2 * p->m + 1);
  const int K_max = std::max(anneal_kmax(p->m, 1), 2 * anneal_kmax(p->m, 2));   // arrays of either phase count
  if (!p->d_an_state) {
    LPF_CUDA(cudaMalloc(&p->d_an_state, 256));
    LPF_CUDA(cudaMalloc(&p->d_an_dE, sizeof(int64_t) * 256));
  }
  p->an_kmax = K_max;
  return grow(&p->d_an_delta, &p->an_delta_bytes, sizeof(int32_t) * 2 * (size_t)K_max * K2);   // two buffers (lpf_anneal.cu)
}

static int reserve_host(lpf_paths* p, int B, int H, int W) {
  DeviceGuard dg(p->device);
  if (!dg.ok) return LPF_E_CUDA;
  const int S = 2 * p->m + 1;
  int rc = grow((uint8_t**)&p->d_io_in, &p->io_in_bytes, (size_t)B * H * W);
  if (rc == LPF_OK) rc = grow((uint8_t**)&p->d_io_out, &p->io_out_bytes, sizeof(int64_t) * (size_t)B * 2 * S * S);
  if (rc != LPF_OK) return rc;
  if (!p->io_stream) LPF_CUDA(cudaStreamCreateWithFlags((cudaStream_t*)&p->io_stream, cudaStreamNonBlocking));
  return LPF_OK;
}

// ---- the eval calls: look the plan up, enqueue -------------------------------------------------------

// sum_over_batch: every image adds into ONE [n_phase][S][S] array (ensemble sum) instead of its own
static int eval_impl(lpf_paths* p, const uint8_t* images, int B, int H, int W, int n_phase, int phase0,
                     int64_t* counts, unsigned flags, void* stream, const uint8_t* start_mask = nullptr,
                     bool sum_over_batch = false) {
  if (!images || !counts) return LPF_E_INVAL;
  int rc = check_eval_args(p, B, H, W, flags);
  if (rc != LPF_OK) return rc;
  if (n_phase == 1 && phase0 != 0 && phase0 != 1) return LPF_E_INVAL;
  auto it = p->plans.find(plan_key(p, B, H, W, n_phase, flags, start_mask != nullptr));
  if (it == p->plans.end()) {                      // a shape that was not reserved: reserve it now (allocates, syncs)
    rc = reserve_eval(p, B, H, W, n_phase, flags, start_mask != nullptr);
    if (rc != LPF_OK) return rc;
    it = p->plans.find(plan_key(p, B, H, W, n_phase, flags, start_mask != nullptr));
  }
  const EvalPlan& pl = it->second;
  if (pl.need > p->packed_bytes) return LPF_E_INVAL;   // cannot happen: the workspace only grows
  DeviceGuard dg(p->device);
  if (!dg.ok) return LPF_E_CUDA;
  cudaStream_t st = (cudaStream_t)stream;
  StreamOrder order(p, st);
  LPF_CUDA(order.err);

  const int S = 2 * p->m + 1;
  const long long n_arrays = sum_over_batch ? n_phase : (long long)B * n_phase;
  LPF_CUDA(cudaMemsetAsync(counts, 0, sizeof(int64_t) * (size_t)n_arrays * S * S, st));
  LPF_CUDA(launch_pack(images, p->d_packed + pl.views_bytes / 4, p->d_packed, pl.g, B, pl.Bpad, n_phase, phase0,
                       p->d_counter, p->n_sm, st));
  uint32_t* const d_mask = p->d_packed + pl.views_bytes / 4 + pl.base_words;
  if (start_mask)                                  // "phase" -1: a start pixel is selected iff its byte is non-zero
    LPF_CUDA(launch_pack(start_mask, d_mask + pl.mask_views_bytes / 4, d_mask, pl.gm, 1, 1, 1, -1, p->d_counter,
                         p->n_sm, st));

  EvalParams ep;
  ep.g = pl.g;
  ep.entries = (const uint2*)pl.pr->d_entries;
  ep.skip = pl.pr->d_skip;
  ep.units = (const int4*)pl.d_work;
  ep.obtab = (const int4*)pl.d_obtab;
  ep.class_slots = pl.pr->d_class_slots;
  ep.class_geom = (const int4*)pl.pr->d_class_geom;
  ep.n_ob = pl.n_ob;
  ep.n_keys = (unsigned int)pl.n_keys;
  ep.n_shares = (unsigned int)pl.n_shares;
  ep.counters = pl.d_counters;
  ep.n_gp = pl.n_gp;
  ep.B = B;
  ep.n_phase = n_phase;
  ep.packed = p->d_packed;
  ep.Bpad = pl.Bpad;
  ep.counts = (unsigned long long*)counts;
  ep.S = S;
  ep.image_stride = sum_over_batch ? 0 : (long long)n_phase * S * S;
  ep.prune = pl.prune;
  ep.n_slots = pl.pr->n_slots;
  ep.tmem_stack = pl.tmem_stack;
  ep.mask = start_mask ? d_mask : nullptr;
  for (int o = 0; o < 4; ++o) ep.mask_off[o] = pl.gm.v[o].packed_off;
  const bool timed = p->timing && !order.capturing;
  if (pl.grid > 0)
    LPF_CUDA(cudaMemsetAsync(pl.d_counters, 0, sizeof(unsigned int) * ((size_t)pl.n_keys + 1), st));
  if (timed) LPF_CUDA(cudaEventRecord((cudaEvent_t)p->ev_start, st));
  if (pl.grid > 0) LPF_CUDA(launch_eval(ep, pl.grid, pl.g.NT * pl.g.threads, pl.smem, st));
  if (timed) {
    LPF_CUDA(cudaEventRecord((cudaEvent_t)p->ev_stop, st));
    p->timed_once = 1;
  }
  const int n_shallow = pl.shallow.n[0] + pl.shallow.n[1] + pl.shallow.n[2] + pl.shallow.n[3];
  if (n_shallow > 0) LPF_CUDA(launch_shallow(ep, pl.shallow, p->n_sm, st));   // level K: the vectors shorter than K
  LPF_CUDA(launch_mirror((unsigned long long*)counts, S, n_arrays, p->n_sm, st));
  LPF_CUDA(order.done());

  // kernels launched (pack base, pack views, eval, mirror; shallow kernel at level K; two more packs for a start mask)
  p->last_info[0] = (start_mask ? 6 : 4) + (n_shallow > 0 ? 1 : 0);
  p->last_info[1] = pl.n_units * pl.n_gp;                // work units x (image group, phase plane)
  p->last_info[2] = (int64_t)pl.pr->entries.size();      // program entries (all four octants)
  p->last_info[3] = pl.grid;
  p->last_info[4] = pl.g.NT * pl.g.threads;              // CTA = NT teams
  p->last_info[5] = (int64_t)pl.smem;
  p->last_info[6] = pl.g.TX * 1000 + pl.g.TY * 100 + pl.tmem_stack * 10 + pl.pr->n_slots;   // thread tile, mask stack
  p->last_info[7] = pl.g.G;
  p->last_info[8] = pl.g.K;                              // erosion level of the program (0: plain; classes may run lower)
  p->last_info[9] = pl.fused_pairs;                      // per image-phase and start word: 2 SHF + 1 LOP3 each
  p->last_info[10] = pl.singles;                         //   1 SHF + 1 LOP3 each
  p->last_info[11] = pl.terminals;                       //   1 POPC + 1 add each
  p->last_info[12] = pl.piece_nodes;
  p->last_info[13] = pl.g.NT;
  p->last_info[14] = pl.occ;
  p->last_info[15] = n_shallow;
  p->last_info[16] = pl.reloads;                         // entries that reload their row strip: TY * (TX + 1) LDS.32 each
  p->last_info[17] = (int64_t)pl.pr->classes.size();     // pattern classes (all octants)
  return LPF_OK;
}

}  // namespace lpf

extern "C" int lpf_reserve(lpf_paths* p, int B, int H, int W, unsigned flags, unsigned what) {
  if (!p || p->device < 0 || H < 1 || W < 1 || what == 0) return LPF_E_INVAL;
  if (what & ~(LPF_FOR_EVAL | LPF_FOR_EVAL_BOTH | LPF_FOR_MASKED | LPF_FOR_SWAP_DELTA | LPF_FOR_ANNEAL | LPF_FOR_HOST))
    return LPF_E_INVAL;
  int rc = LPF_OK;
  if (what & (LPF_FOR_EVAL | LPF_FOR_EVAL_BOTH | LPF_FOR_HOST)) {
    rc = check_eval_args(p, B, H, W, flags);
    if (rc != LPF_OK) return rc;
  }
  const bool masked = (what & LPF_FOR_MASKED) != 0;
  if (masked && !(what & (LPF_FOR_EVAL | LPF_FOR_EVAL_BOTH))) return LPF_E_INVAL;
  if (rc == LPF_OK && (what & LPF_FOR_EVAL)) rc = reserve_eval(p, B, H, W, 1, flags, masked);
  if (rc == LPF_OK && (what & LPF_FOR_EVAL_BOTH)) rc = reserve_eval(p, B, H, W, 2, flags, masked);
  if (rc == LPF_OK && (what & LPF_FOR_SWAP_DELTA)) rc = reserve_swap(p, H, W);
  if (rc == LPF_OK && (what & LPF_FOR_ANNEAL)) rc = reserve_anneal(p, H, W);
  if (rc == LPF_OK && (what & LPF_FOR_HOST)) {
    rc = reserve_host(p, B, H, W);
    if (rc == LPF_OK && !(what & (LPF_FOR_EVAL | LPF_FOR_EVAL_BOTH))) {
      rc = reserve_eval(p, B, H, W, 1, flags, false);
      if (rc == LPF_OK) rc = reserve_eval(p, B, H, W, 2, flags, false);
    }
  }
  if (rc == LPF_OK) {                              // uploads above used synchronous copies; leave nothing in flight
    DeviceGuard dg(p->device);
    if (!dg.ok) return LPF_E_CUDA;
    LPF_CUDA(cudaDeviceSynchronize());
  }
  return rc;
}

extern "C" int lpf_eval(const lpf_paths* p, const uint8_t* images, int B, int H, int W, int phase, int64_t* counts,
                        unsigned flags, void* stream) {
  return lpf::eval_impl(const_cast<lpf_paths*>(p), images, B, H, W, 1, phase, counts, flags, stream);
}

extern "C" int lpf_eval_both(const lpf_paths* p, const uint8_t* images, int B, int H, int W, int64_t* counts,
                             unsigned flags, void* stream) {
  return lpf::eval_impl(const_cast<lpf_paths*>(p), images, B, H, W, 2, 0, counts, flags, stream);
}

extern "C" int lpf_eval_masked(const lpf_paths* p, const uint8_t* images, int B, int H, int W, int phase,
                               const uint8_t* start_mask, int64_t* counts, unsigned flags, void* stream) {
  if (!start_mask || phase < -1 || phase > 1) return LPF_E_INVAL;
  lpf_paths* q = const_cast<lpf_paths*>(p);
  return phase < 0 ? lpf::eval_impl(q, images, B, H, W, 2, 0, counts, flags, stream, start_mask)
                   : lpf::eval_impl(q, images, B, H, W, 1, phase, counts, flags, stream, start_mask);
}

extern "C" int lpf_eval_sum(const lpf_paths* p, const uint8_t* images, int B, int H, int W, int phase,
                            int64_t* counts_sum, unsigned flags, void* stream) {
  if (phase < -1 || phase > 1) return LPF_E_INVAL;
  lpf_paths* q = const_cast<lpf_paths*>(p);
  return phase < 0 ? lpf::eval_impl(q, images, B, H, W, 2, 0, counts_sum, flags, stream, nullptr, true)
                   : lpf::eval_impl(q, images, B, H, W, 1, phase, counts_sum, flags, stream, nullptr, true);
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

extern "C" int lpf_set_level(lpf_paths* p, int max_level) {
  if (!p || max_level < -1 || max_level > MAX_LEVEL) return LPF_E_INVAL;
  p->max_level = max_level;
  return LPF_OK;
}

extern "C" int lpf_set_shared_memory(lpf_paths* p, int bytes) {
  if (!p || bytes < 0 || (bytes > 0 && bytes < 16384)) return LPF_E_INVAL;
  p->smem_limit = bytes;
  return LPF_OK;
}

extern "C" int lpf_set_tmem_stack(lpf_paths* p, int enable) {
  if (!p || (enable != 0 && enable != 1)) return LPF_E_INVAL;
  p->no_tmem = !enable;
  return LPF_OK;
}

extern "C" int lpf_set_teams(lpf_paths* p, int n_teams) {
  if (!p || n_teams < 0 || n_teams > EVAL_CTA_MAX_THREADS / 32) return LPF_E_INVAL;
  p->n_teams = n_teams;
  return LPF_OK;
}

extern "C" int lpf_last_eval_kernel_ms(const lpf_paths* p, float* ms) {
  if (!p || !ms || p->device < 0 || !p->timed_once) return LPF_E_INVAL;
  DeviceGuard dg(p->device);
  if (!dg.ok) return LPF_E_CUDA;
  LPF_CUDA(cudaEventSynchronize((cudaEvent_t)p->ev_stop));
  LPF_CUDA(cudaEventElapsedTime(ms, (cudaEvent_t)p->ev_start, (cudaEvent_t)p->ev_stop));
  return LPF_OK;
}

extern "C" int lpf_last_launch_info(const lpf_paths* p, int64_t* out18) {
  if (!p || !out18) return LPF_E_INVAL;
  std::memcpy(out18, p->last_info, sizeof(p->last_info));
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

// phase 0 | 1: delta [n][S][S] of that phase;  phase < 0: both phases in one pass over the trie, phase k written at
// delta + k * plane_stride (used by lpf_anneal)
int swap_delta_impl(lpf_paths* p, const uint8_t* image, int H, int W, int phase, const int32_t* pairs, int64_t n,
                    int32_t* delta, int64_t plane_stride, void* stream) {
  if (!p || !image || !pairs || !delta) return LPF_E_INVAL;
  if (p->device < 0 || H < 1 || W < 1 || n < 0) return LPF_E_INVAL;
  if (phase < -1 || phase > 1) return LPF_E_INVAL;
  if (p->m > std::min(H, W) - 1) return LPF_E_INVAL;
  if (n == 0) return LPF_OK;
  const size_t padded_words = (size_t)2 * (H + 2 * p->m) * ((W + 2 * p->m + 31) / 32);
  const size_t bits_bytes = (2 * ((size_t)H * ((W + 31) / 32) + (size_t)W * ((H + 31) / 32)) + padded_words) * 4;
  if (!p->d_swap_rec || bits_bytes > p->swap_bits_bytes) {   // not reserved: reserve now (allocates, syncs)
    const int rc = reserve_swap(p, H, W);
    if (rc != LPF_OK) return rc;
  }
  if (phase < 0 && padded_words * 4 + 8 + 8 * 512 * 8 + 2048 > (size_t)p->max_smem) return LPF_E_UNSUPPORTED;
  DeviceGuard dg(p->device);
  if (!dg.ok) return LPF_E_CUDA;
  cudaStream_t st = (cudaStream_t)stream;
  StreamOrder order(p, st);
  LPF_CUDA(order.err);
  LPF_CUDA(launch_swap_delta(image, p->d_swap_bits, H, W, p->m, phase, pairs, (long long)n, p->d_swap_rec,
                             (int)p->n_trie_nodes, p->d_swap_rrec, delta, (long long)plane_stride, p->d_counter + 1,
                             p->n_sm, st));
  LPF_CUDA(order.done());
  return LPF_OK;
}

}  // namespace lpf

extern "C" int lpf_swap_delta(const lpf_paths* p, const uint8_t* image, int H, int W, int phase, const int32_t* pairs,
                              int64_t n, int32_t* delta, void* stream) {
  if (phase != 0 && phase != 1) return LPF_E_INVAL;
  return lpf::swap_delta_impl(const_cast<lpf_paths*>(p), image, H, W, phase, pairs, n, delta, 0, stream);
}

// ---- host-buffer convenience (end-to-end measurement) ---------------------------------------------

extern "C" int lpf_eval_host(lpf_paths* p, const uint8_t* images_host, int B, int H, int W, int phase,
                             int64_t* counts_host, unsigned flags) {
  if (!p || !images_host || !counts_host) return LPF_E_INVAL;
  if (p->device < 0 || B < 1 || H < 1 || W < 1) return LPF_E_INVAL;
  const int n_phase = phase < 0 ? 2 : 1;
  const int S = 2 * p->m + 1;
  const size_t in_bytes = (size_t)B * H * W;
  const size_t out_bytes = sizeof(int64_t) * (size_t)B * n_phase * S * S;
  if (in_bytes > p->io_in_bytes || sizeof(int64_t) * (size_t)B * 2 * S * S > p->io_out_bytes || !p->io_stream) {
    int rc = check_eval_args(p, B, H, W, flags);
    if (rc == LPF_OK) rc = reserve_host(p, B, H, W);
    if (rc != LPF_OK) return rc;
  }
  DeviceGuard dg(p->device);
  if (!dg.ok) return LPF_E_CUDA;
  // the private stream: lpf_eval below orders it after earlier work on this table (StreamOrder)
  cudaStream_t st = (cudaStream_t)p->io_stream;
  {
    StreamOrder order(p, st);                      // the H2D copy overwrites d_io_in: wait for the previous call first
    LPF_CUDA(order.err);
    LPF_CUDA(cudaMemcpyAsync(p->d_io_in, images_host, in_bytes, cudaMemcpyHostToDevice, st));
    LPF_CUDA(order.done());
  }
  int rc = n_phase == 2 ? lpf_eval_both(p, (const uint8_t*)p->d_io_in, B, H, W, (int64_t*)p->d_io_out, flags, st)
                        : lpf_eval(p, (const uint8_t*)p->d_io_in, B, H, W, phase, (int64_t*)p->d_io_out, flags, st);
  if (rc != LPF_OK) return rc;
  LPF_CUDA(cudaMemcpyAsync(counts_host, p->d_io_out, out_bytes, cudaMemcpyDeviceToHost, st));
  LPF_CUDA(cudaStreamSynchronize(st));
  return LPF_OK;
}
