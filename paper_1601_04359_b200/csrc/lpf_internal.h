// lpf_internal.h -- shared between the host table builder (lpf_paths.cpp) and the CUDA side
// (lpf_kernels.cu / lpf_api.cu) of liblpf.so.  Not part of the C ABI (include/lpf.h).
// Nothing here is used by, or shared with, oracle/.
#pragma once
#include <cstdint>
#include <array>
#include <map>
#include <tuple>
#include <utility>
#include <vector>

#include "lpf.h"
#include "lpf_kernels.cuh"

namespace lpf {

// ---- octant views ----------------------------------------------
// Every canonical vector v = (dx,dy) in D belongs to one octant; its path is walked on a
// transposed / flipped VIEW of the image in which it is an x-major first-octant path
// (a' >= 0, 0 <= b' <= a'), so that the walker only ever moves right along a row or steps down.
//   o = 0: dx >= 0, dy <= dx      view (x',y') = I[y'][x']        (a',b') = ( a,  b)
//   o = 1: dx >= 0, dy >  dx      view (x',y') = I[x'][y']        (a',b') = ( b,  a)
//   o = 2: dx <  0, dy > -dx      view (x',y') = I[x'][-y' mod W] (a',b') = ( b, -a)
//   o = 3: dx <  0, dy <= -dx     view (x',y') = I[y'][-x' mod W] (a',b') = (-a,  b)
// The start pixels of a view are a bijection of the start pixels of the image, so the count of
// a path is the same in its view.
inline int octant_of(int dx, int dy) {
  if (dx >= 0) return dy <= dx ? 0 : 1;
  return dy > -dx ? 2 : 3;
}
inline void to_view(int o, int a, int b, int* av, int* bv) {
  switch (o) {
    case 0: *av = a; *bv = b; break;
    case 1: *av = b; *bv = a; break;
    case 2: *av = b; *bv = -a; break;
    default: *av = -a; *bv = b; break;
  }
}
inline void from_view(int o, int av, int bv, int* a, int* b) {
  switch (o) {
    case 0: *a = av; *b = bv; break;
    case 1: *a = bv; *b = av; break;
    case 2: *a = -bv; *b = av; break;
    default: *a = -av; *b = bv; break;
  }
}

// ---- node program entry (uint64), DESIGN.md "Node program" -------------------------------
// low word x:
//   [ 0.. 4] sh      = a' & 31        bit offset of the window inside its word
//   [ 5] RELOAD      row, word column or plane differs from the previous entry: reload the row strip
//   [ 6] TERMINAL    the last node of the entry is a whole path P_v: count it
//   [ 7] SAVE        copy the running mask to stack slot sslot (the last node has >= 2 children in its piece)
//   [ 8] RESTORE     parent mask comes from stack slot rslot (not from the previous entry)
//   [ 9] INIT        parent mask is "every valid start pixel" (first entry of a work item, and only there)
//   [10] PAIR        this entry's own mask is never needed (not TERMINAL, not SAVE) and the next entry continues from
//                    it: the walker fuses both windows into one 3-input AND (M & W1 & W2)
//   [11] ERODED      level K >= 1: the window is read from eroded plane q (high word) and covers the K + 1 pixels
//                    (a' + j, b' + s_1 + .. + s_j), j = 0..K, s_j = bit j-1 of q; the first `back` of them are nodes
//                    already in the mask (AND is idempotent), the rest are the nodes of this entry, the last of which
//                    owns TERMINAL, SAVE and cidx.  The word offset of the plane (its slot in the item's pattern class
//                    times band_words) is already added to `off`.
//   [12..31] off     = b' * stride + (a' >> 5) (+ slot * band_words), word offset of the window in shared memory
// high word y:
//   [ 0..19] cidx    = (dy + m) * (2m + 1) + (dx + m), index into counts[2m+1][2m+1] (image coordinates)
//   [20..22] rslot   [23..25] sslot
//   [26..31] q       step pattern of the window (for the host test; the kernel needs only `off`)
constexpr uint32_t E_SH_MASK = 31u;
constexpr uint32_t E_RELOAD = 1u << 5;
constexpr uint32_t E_TERMINAL = 1u << 6;
constexpr uint32_t E_SAVE = 1u << 7;
constexpr uint32_t E_RESTORE = 1u << 8;
constexpr uint32_t E_INIT = 1u << 9;
constexpr uint32_t E_PAIR = 1u << 10;
constexpr uint32_t E_ERODED = 1u << 11;
constexpr int E_OFF_SHIFT = 12;
constexpr uint32_t E_CIDX_MASK = (1u << 20) - 1u;
constexpr int E_RSLOT_SHIFT = 20;
constexpr int E_SSLOT_SHIFT = 23;
constexpr uint32_t E_SLOT_MASK = 7u;
constexpr int E_Q_SHIFT = 26;
static_assert(STACK_SLOTS_BUDGET <= 8, "three bits per mask-stack slot");

constexpr int MAX_M = 511;
constexpr int64_t SWAP_REV_MAX_NODES = 4 << 20;   // reversed trie of lpf_swap_delta: 64 MB of records at most (m <= ~100)

struct Node {
  int16_t a, b;          // pixel offset of this node (last pixel of the prefix), view coordinates
  int32_t parent;
  int32_t first_child;
  int32_t next_sibling;
  int32_t size;          // nodes in the subtree (self included)
  int32_t depth;         // root = 0
  uint8_t terminal;      // this prefix is a whole path
};

struct Program {         // one linearisation of the four octant tries for one set of view strides
  std::vector<uint64_t> entries;
  std::vector<uint32_t> skip;          // entries in the subtree below each entry (LPF_PRUNE jump)
  std::vector<int64_t> items;          // [n_items][4] = first entry, count, octant, 0; sorted by count, descending
  int n_slots = 0;
  int stride[4] = {0, 0, 0, 0};
  int K = 0;                           // erosion level (0: plain program)
  int n_planes = 0;                    // full-height planes the geometry reserved per image (beside the plain band)
  int band_rows = 0;                   // start rows of a band
  bool widen = false;                  // classes of shallow slopes take the planes their lower bands leave room for
  int band_words[4] = {0, 0, 0, 0};    // level K: the plane in slot s of view o sits at s * band_words[o] in shared memory
  // level K: pattern classes (slope sectors of one octant whose paths use at most n_planes patterns); items[4 i + 3] is
  // the class of item i
  struct Class {
    int octant = 0;
    int rows = 0;                      // rows of the class's band: band_rows + the largest b' of its paths + 1
    int band_words = 0;                // words of one of its planes in shared memory (rows * stride, padded)
    int level = 0;                     // its own level K_c <= the program's (steep classes of large templates: lower)
    int n = 0;                         // patterns used
    int pattern[MAX_PATTERNS];         // slot -> pattern q
    signed char slot_of[MAX_PATTERNS]; // rank of a balanced pattern -> slot, or -1
  };
  std::vector<Class> classes;
  signed char* d_class_slots = nullptr;  // device: [classes][MAX_PATTERNS]
  int* d_class_geom = nullptr;           // device: [classes][4] = band words, rows, planes, level
  uint64_t* d_entries = nullptr;       // device copy, uploaded by lpf_reserve (lpf_api.cu)
  uint32_t* d_skip = nullptr;
};

// Everything one eval call needs for one (B, H, W, phases, flags, masked, tile) shape; built by lpf_reserve (or by the
// first call for the shape), after which an eval only enqueues work (lpf_api.cu).
struct EvalPlan {
  Geom g;                              // views with their offsets inside one phase plane of the packed workspace
  Geom gm;                             // the same views for the start mask of lpf_eval_masked (one image, one plane)
  ShallowList shallow;                 // level K: terminals above depth K
  Program* pr = nullptr;
  int32_t* d_work = nullptr;           // work units [n_units][4] = first entry, entries, strip band, 0 (one allocation
  int32_t* d_obtab = nullptr;          //   with) the (octant, row band) table [n_ob][4] = first unit, units, octant, band
  unsigned int* d_counters = nullptr;  //   and the share cursor + one unit counter per key
  int64_t n_units = 0, n_keys = 0, n_shares = 0;
  int n_ob = 0;
  int Bpad = 0, n_gp = 0, grid = 0, prune = 0, occ = 0, tmem_stack = 0;
  size_t smem = 0;
  size_t views_bytes = 0, base_words = 0, mask_views_bytes = 0, mask_base_bytes = 0, need = 0;
  // what the walker executes per image-phase and start word (lpf_last_launch_info): pairs of entries folded into one
  // 3-input AND, entries executed on their own, terminal entries (POPC + add), trie nodes per piece
  int64_t fused_pairs = 0, singles = 0, terminals = 0, piece_nodes = 0, reloads = 0;
};

}  // namespace lpf

struct lpf_paths {
  int m = 0;
  int device = -1;
  int n_sm = 0;                      // multiprocessors of `device`
  int max_smem = 0;                  // opt-in dynamic shared memory per block, bytes
  int64_t n_half = 0;
  int64_t sum_len = 0;
  int64_t n_trie_nodes = 0;          // distinct prefixes of all P_v, v in D (one trie, image coordinates)
  std::vector<lpf::Node> oct[4];     // per-octant prefix tries in view coordinates; [0] = root (0,0)
  // key: (piece_nodes, program kind, stride0, stride1, 100 K + planes per class, band words 0, band words 1)
  std::map<std::tuple<int, unsigned, int, int, int, int, int>, lpf::Program> programs;
  int level_ok = 0;                  // highest level whose path windows are all balanced words (build_host_table)
  int path_patterns[lpf::MAX_LEVEL + 1] = {0, 0, 0, 0, 0, 0, 0};   // most patterns of length K on one path
  // key: B, H, W, phases, flags, masked, 100 tile_tx + tile_ty, cta_warps
  std::map<std::array<int64_t, 8>, lpf::EvalPlan> plans;
  // device workspace (sized by lpf_reserve; a call for a shape that was not reserved reserves it first)
  uint32_t* d_packed = nullptr;
  size_t packed_bytes = 0;
  unsigned int* d_counter = nullptr;
  // swap-delta node records: the image-coordinate trie in preorder, 16 bytes per node (built by lpf_reserve)
  int32_t* d_swap_rec = nullptr;     // [n_trie_nodes][4]
  int32_t* d_swap_rrec = nullptr;    // reversed trie [n_swap_rev][4], or null (table too large: per-node walks instead)
  int64_t n_swap_rev = 0;
  int n_swap_rev1 = 0;               // children of the reversed trie's root (the unit of slicing)
  uint32_t* d_swap_bits = nullptr;   // packed base image of the last lpf_swap_delta call
  size_t swap_bits_bytes = 0;
  // lpf_anneal: chain state, speculative deltas and their error changes
  void* d_an_state = nullptr;
  int32_t* d_an_delta = nullptr;
  int64_t* d_an_dE = nullptr;
  size_t an_delta_bytes = 0;
  int an_kmax = 0;
  // stream order: work of consecutive calls shares the workspace, so a call on another stream first waits for the
  // event recorded after the previous call (no host synchronisation)
  void* ev_done = nullptr;
  void* last_stream = nullptr;
  int last_stream_valid = 0;
  // device staging buffers of lpf_eval_host and its private stream
  void* d_io_in = nullptr;
  size_t io_in_bytes = 0;
  void* d_io_out = nullptr;
  size_t io_out_bytes = 0;
  void* io_stream = nullptr;
  // lpf_set_timing: CUDA events recorded around the eval kernel alone
  int tile_tx = 0, tile_ty = 0, cta_warps = 0;   // lpf_set_tile overrides (0 = automatic)
  int n_teams = 0;                   // teams per CTA override (0 = automatic)
  int max_level = -1;                // erosion level cap (lpf_set_level; -1 = automatic)
  int smem_limit = 0;                // shared memory one eval CTA may use, bytes (lpf_set_shared_memory; 0 = all)
  int no_tmem = 0;                   // keep the mask stack in local memory (lpf_set_tmem_stack(p, 0))
  int timing = 0;
  int timed_once = 0;                // a timed eval has been issued: ev_start / ev_stop hold a measurement
  void* ev_start = nullptr;
  void* ev_stop = nullptr;
  int64_t last_info[18] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
};

namespace lpf {

// closed-form rasteriser: P_v for v in the canonical half (lpf_paths.cpp)
int canonical_path(int dx, int dy, int16_t* xy);
inline bool in_half(int dx, int dy) { return dy > 0 || (dy == 0 && dx >= 0); }

// lpf_swap_delta for one phase (0 | 1) or for both in one pass (phase < 0: phase k at delta + k * plane_stride); lpf_api.cu
int swap_delta_impl(lpf_paths* p, const uint8_t* image, int H, int W, int phase, const int32_t* pairs, int64_t n,
                    int32_t* delta, int64_t plane_stride, void* stream);

// the image-coordinate trie in preorder for lpf_swap_delta (lpf_paths.cpp)
// also the reversed trie (rrec, left empty if it would exceed max_rev nodes)
void build_swap_records(const lpf_paths* p, std::vector<int32_t>& rec, std::vector<int32_t>& rrec, int64_t max_rev);

// builds (or returns the cached) program for (piece_nodes, flags, view strides); host side only
Program& get_program(lpf_paths* p, int piece_nodes, unsigned flags, int stride03, int stride12, int K, int n_planes,
                     int bw03, int bw12, int band_rows, bool widen);
int max_teams_of(const lpf_paths* p);
// the terminals above depth K of every octant trie (counted by shallow_kernel, not by the program)
void shallow_terminals(const lpf_paths* p, int K, ShallowList* out);
// forgets a cached program that was never uploaded (one the kernel cannot take)
void drop_program(lpf_paths* p, const Program* pr);

// largest proposal batch of lpf_anneal for n_ph phase planes; plans + swap tables + batch buffers of lpf_anneal on
// H x W images (lpf_api.cu; allocates and synchronises)
int anneal_kmax(int m, int n_ph);
int reserve_anneal(lpf_paths* p, int H, int W);

}  // namespace lpf
