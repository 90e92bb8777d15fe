// lpf_kernels.cuh -- geometry and launch parameter blocks shared by lpf_paths.cpp (host geometry),
// lpf_kernels.cu and lpf_api.cu.  Plain structs, no CUDA types.
#pragma once
#include <cstdint>
#include <vector_types.h>

#ifdef __CUDACC__
#define LPF_HD __host__ __device__
#else
#define LPF_HD
#endif

namespace lpf {

// ---- step patterns ------------------------------------------------
// Every step of a first-octant path is (+1, 0) or (+1, +1); a K-step pattern q has bit j-1 set iff step j goes one row
// down.  The patterns of K consecutive steps of a digital straight segment are the BALANCED words of length K: any two
// factors of equal length differ by at most one in their number of down steps (2, 4, 8, 14, 24, 36 of them for
// K = 1 .. 6, not 2^K).  The host checks that every window of every path of the table is balanced before it uses a
// level; the eval kernel derives the planes of all balanced patterns of its level with compile-time recursion.
LPF_HD constexpr bool balanced_word(unsigned q, int K) {
  for (int L = 1; L <= K; ++L) {
    int lo = 99, hi = -1;
    for (int s = 0; s + L <= K; ++s) {
      int c = 0;
      for (int t = 0; t < L; ++t) c += (int)((q >> (s + t)) & 1u);
      lo = c < lo ? c : lo;
      hi = c > hi ? c : hi;
    }
    if (hi - lo > 1) return false;
  }
  return true;
}
// position of q among the balanced words of length K in ascending order
LPF_HD constexpr int balanced_rank(unsigned q, int K) {
  int r = 0;
  for (unsigned t = 0; t < q; ++t) r += balanced_word(t, K) ? 1 : 0;
  return r;
}
LPF_HD constexpr int balanced_count(int K) { return balanced_rank(1u << K, K); }
constexpr int MAX_LEVEL = 6;
constexpr int MAX_PATTERNS = 36;          // balanced_count(MAX_LEVEL)
static_assert(balanced_count(MAX_LEVEL) == MAX_PATTERNS, "pattern table size");

// One octant view of one image in HBM / shared memory.
//   word (r, i), r in [0, rows), i in [0, stride): bit k holds [ view(x' = (32 i + k) mod Wv, y' = r mod Hv) == phase ]
//   rows = n_bands * band_rows + m (periodic halo below), stride = n_strips * TX + m / 32 + 1, made odd
constexpr int STACK_SLOTS_BUDGET = 8;   // mask-stack slots per thread (local memory, T words each)

struct ViewGeom {
  int Hv, Wv;        // view height (rows) and width (pixels): octants 0,3: H,W; octants 1,2: W,H
  int Wc;            // ceil(Wv / 32) words that hold start pixels
  int n_strips;      // ceil(Wc / TX) strips of TX words per row
  int stride;        // words per packed row
  int n_bands;       // ceil(Hv / band_rows) bands of start rows
  int band_words;    // (band_rows + m) * stride rounded up to a multiple of 4: one band of one plane in shared memory
  int n_planes;      // full-height eroded planes that fit in shared memory beside the plain band: 0 = plain mode (the
                     // plain band alone).  A pattern class keeps only the rows its paths reach and may hold more.
  int band_pitch;    // words per image in shared memory: band_words (plain mode), else (n_planes + 1) * band_words:
                     // the planes, then the plain band they are derived from
  int plane_words;   // words of the plain view of one image in HBM (rows * stride, padded)
  int view_words;    // whole packed block of one image (= plane_words: only the plain view is kept in HBM)
  long long packed_off;   // word offset of this octant's [Bpad][view_words] block inside one phase plane
};

struct Geom {
  int H, W, m;
  int K;             // erosion level: 0 = plain plane; K >= 1: one plane per K-step pattern of a class
  int TX, TY;        // thread tile: TX adjacent words x TY start rows (32 rows apart)
  int band_rows;     // start rows per work item, multiple of 32 * TY
  int SB;            // strips per work item (<= 8)
  int wpi;           // warps per image band = SB * band_rows / (32 TY)
  int G;             // images per CTA
  int NT;            // teams per CTA: every team (G * wpi warps) walks its own work unit on the CTA's shared bands
  int threads;       // threads of one team: G * wpi * 32 (the CTA has NT times as many)
  int smem_bytes;    // G * max band_words * 4
  ViewGeom v[4];
  long long plane_words;  // words of one phase plane: Bpad * sum_o view_words
};

// host: pick the geometry for (m, H, W, B); false if one band does not fit in shared memory
//   tx, ty > 0 override the thread tile; cta_warps (1..8) the warps per CTA
constexpr int EVAL_CTA_MAX_THREADS = 1024;  // a CTA of NT teams (the eval kernel is compiled for 64 registers per thread)
//   max_level: highest erosion level allowed (0: plain plane only); at level K a window covers K + 1 path pixels: plane
//   q at (a, b) = AND of the pixels (a + j, b + s_1 + .. + s_j), j = 0..K, s_j = bit j-1 of q.  The vectors of an octant
//   are split by slope into CLASSES whose paths use at most n_planes patterns; the planes of one class are derived in
//   shared memory from the plain band when a CTA takes a key of that class
//   max_teams: teams of one CTA that can find work on one key (lpf_internal.h: max_teams_of)
//   path_patterns[K]: most patterns of length K on one path of the table (a class needs as many planes; where the
//   bands cannot be made low enough for that, the classes of steep slopes run at lower levels: Program::Class::level)
//   max_smem: opt-in shared memory of an SM's CTA; cta_smem: what one CTA may use of it (0 = all; lpf_set_shared_memory)
bool choose_geom(int m, int H, int W, int B, int max_smem, int cta_smem, int tx, int ty, int cta_warps, int max_level,
                 int max_teams, const int* path_patterns, Geom* out);

// terminals above depth K have no program entry at level K (a window covers K + 1 pixels): shallow_kernel counts them
constexpr int MAX_SHALLOW = 21;   // 1 + 2 + .. + MAX_LEVEL vectors of fewer than MAX_LEVEL steps per octant
// prefix tree of the balanced step patterns of fewer than MAX_LEVEL steps: node (J steps, pattern PRE) has the index
// shallow_base(J) + balanced_rank(PRE, J)
LPF_HD constexpr int shallow_base(int J) { int b = 0; for (int j = 0; j < J; ++j) b += balanced_count(j); return b; }
constexpr int SHALLOW_NODES = shallow_base(MAX_LEVEL);   // 1 + 2 + 4 + 8 + 14 + 24
struct ShallowList {
  int n[4];                          // vectors per octant
  int cidx[4][MAX_SHALLOW];          // their index into counts[S][S]
  signed char node[4][SHALLOW_NODES];// prefix-tree node -> position in the octant's list, or -1
};

struct EvalParams {
  Geom g;
  const uint2* entries;
  const uint32_t* skip;
  const int4* units;          // work units = first entry, entries, strip band, 0; the units of one (octant, row band)
                              // are consecutive, big first
  const int4* obtab;          // [n_ob] (octant, row band, class) triples = first unit, units, octant | class << 2, row band
  const signed char* class_slots;  // level K: [n_classes][MAX_PATTERNS] plane slot of each balanced pattern (by rank), or -1
  const int4* class_geom;          // level K: [n_classes] = words of one band of the class, its rows, its planes, its level
  int n_ob;
  unsigned int n_keys;        // n_gp * n_ob keys = (image group, phase plane, octant, row band, class); key = gp * n_ob + ob
  unsigned int n_shares;      // n_keys * passes: how often the cursor hands out every key
  unsigned int* counters;     // [0] the share cursor, [1 + key] units of the key handed out; zeroed before the launch
  int n_gp;                   // ceil(B / G) * n_phase (image group x phase plane)
  int B;
  int n_phase;                // 1 or 2 phase planes in `packed`
  const uint32_t* packed;     // [n_phase][4 octants][Bpad][view_words]
  int Bpad;
  unsigned long long* counts; // [B][n_phase][S][S]  (lpf_eval_sum: [n_phase][S][S], image_stride 0)
  long long image_stride;     // elements between the count arrays of consecutive images: n_phase * S * S, or 0
  int S;                      // 2m + 1
  int prune;
  int n_slots;                // mask-stack slots of the program (<= STACK_SLOTS_BUDGET)
  int tmem_stack;             // the mask stack lives in tensor memory (one CTA per SM, the slots of all warps fit 512 columns)
  const uint32_t* mask;       // lpf_eval_masked: packed views of the start mask (one image), or nullptr
  long long mask_off[4];      // word offset of each octant view inside `mask`
};

}  // namespace lpf
