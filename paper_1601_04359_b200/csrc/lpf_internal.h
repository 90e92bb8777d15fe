// lpf_internal.h -- shared between the host table builder (lpf_paths.cpp) and the CUDA side
// (lpf_kernels.cu / lpf_api.cu) of liblpf.so.  Not part of the C ABI (include/lpf.h).
// Nothing here is used by, or shared with, oracle/.
#pragma once
#include <cstdint>
#include <map>
#include <utility>
#include <vector>

#include "lpf.h"

namespace lpf {

// ---- node program entry (uint64), DESIGN.md "Node program" -------------------------------
// low word x:
//   [ 0.. 4] sh    = a & 31          bit offset of the window inside its word
//   [ 5..10] col   = (a >> 5) + 16   word-column offset of the window, arithmetic shift
//   [11..20] b                        row offset (0..m; canonical half has b >= 0)
//   [21] TERMINAL  this prefix is a whole path P_v: count it
//   [22] SAVE      copy the running mask to stack slot sslot (node has >= 2 children in its piece)
//   [23] RESTORE   parent mask comes from stack slot rslot (not from the previous entry)
//   [24] INIT      parent mask is "every valid start pixel" (first entry of a work item / chain)
//   [25] ADV       (direct descents only) b == previous b + 1
//   [26] RELOAD    (direct descents only) col differs from the previous entry's col
// high word y:
//   [ 0..19] cidx  = (b + m) * (2m + 1) + (a + m), index into counts[2m+1][2m+1]
//   [20..25] rslot
//   [26..31] sslot
constexpr uint32_t E_SH_MASK = 31u;
constexpr int E_COL_SHIFT = 5;
constexpr uint32_t E_COL_MASK = 63u;
constexpr int E_COL_BIAS = 16;
constexpr int E_B_SHIFT = 11;
constexpr uint32_t E_B_MASK = 1023u;
constexpr uint32_t E_TERMINAL = 1u << 21;
constexpr uint32_t E_SAVE = 1u << 22;
constexpr uint32_t E_RESTORE = 1u << 23;
constexpr uint32_t E_INIT = 1u << 24;
constexpr uint32_t E_ADV = 1u << 25;
constexpr uint32_t E_RELOAD = 1u << 26;
constexpr uint32_t E_CIDX_MASK = (1u << 20) - 1u;
constexpr int E_RSLOT_SHIFT = 20;
constexpr int E_SSLOT_SHIFT = 26;
constexpr uint32_t E_SLOT_MASK = 63u;

constexpr int MAX_M = 511;
constexpr int MAX_SLOTS = 28;   // mask-stack slots the kernels reserve per thread

struct Node {
  int16_t a, b;          // pixel offset of this node (last pixel of the prefix)
  int32_t parent;
  int32_t first_child;
  int32_t next_sibling;
  int32_t size;          // nodes in the subtree (self included)
  int32_t depth;         // root = 0
  uint8_t terminal;      // this prefix equals P_(a,b)
};

struct Program {         // one linearisation of the trie (host copy + optional device copy)
  std::vector<uint64_t> entries;
  std::vector<uint32_t> skip;          // entries in the subtree below each entry (LPF_PRUNE jump)
  std::vector<int64_t> items;          // [n_items][2] = first entry, count; sorted by count, descending
  int n_slots = 0;
  uint64_t* d_entries = nullptr;
  uint32_t* d_skip = nullptr;
  int64_t* d_items = nullptr;
};

}  // namespace lpf

struct lpf_paths {
  int m = 0;
  int device = -1;
  int n_sm = 0;                      // multiprocessors of `device`
  int max_smem = 0;                  // opt-in dynamic shared memory per block, bytes
  int64_t n_half = 0;
  int64_t sum_len = 0;
  std::vector<lpf::Node> nodes;                          // nodes[0] = root (0,0)
  std::map<std::pair<int, unsigned>, lpf::Program> programs;   // key: (piece_nodes, flags & LPF_NO_TRIE)
  // device workspace (grown on demand)
  uint32_t* d_packed = nullptr;
  size_t packed_bytes = 0;
  unsigned int* d_counter = nullptr;
  // swap-delta path table: canonical paths, flattened (built lazily)
  int16_t* d_path_xy = nullptr;      // [sum_len][2]
  int32_t* d_path_off = nullptr;     // [n_half + 1]
  int16_t* d_vecs = nullptr;         // [n_half][2] = dx, dy of each canonical vector
  // device staging buffers of lpf_eval_host (grown on demand) and its private stream
  void* d_io_in = nullptr;
  size_t io_in_bytes = 0;
  void* d_io_out = nullptr;
  size_t io_out_bytes = 0;
  void* io_stream = nullptr;
  // lpf_set_timing: CUDA events recorded around the eval kernel alone
  int timing = 0;
  void* ev_start = nullptr;
  void* ev_stop = nullptr;
  int64_t last_info[8] = {0, 0, 0, 0, 0, 0, 0, 0};
};

namespace lpf {

// closed-form rasteriser: P_v for v in the canonical half (lpf_paths.cpp)
int canonical_path(int dx, int dy, int16_t* xy);
inline bool in_half(int dx, int dy) { return dy > 0 || (dy == 0 && dx >= 0); }

// builds (or returns the cached) program for (piece_nodes, flags); host side only
Program& get_program(lpf_paths* p, int piece_nodes, unsigned flags);

}  // namespace lpf
