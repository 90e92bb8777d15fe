// lpf_kernels.cuh -- launch parameter blocks shared by lpf_kernels.cu and lpf_api.cu.
#pragma once
#include <cstdint>

namespace lpf {

// Geometry of one packed image in HBM / shared memory.
//   word (r, i), r in [0, rows), i in [0, stride): bit k holds [ I[r mod H][(32 (i - CL) + k) mod W] == phase ]
//   rows   = Hpad + m            Hpad = ceil(H / T) * T   (start rows padded to whole threads)
//   stride = Wc + CL + CR (+pad) Wc = ceil(W / 32), CL = ceil(m / 32), CR = floor(m / 32) + 1
struct Geom {
  int H, W, m;
  int T;            // start rows per thread
  int Wc;           // start word columns
  int CL;           // halo words on the left
  int stride;       // words per packed row
  int rows;         // packed rows
  int img_words;    // rows * stride rounded up to a multiple of 4 (16-byte TMA granule)
  int tpi;          // threads per image = Wc * ceil(H / T)
  int wpi;          // warps per image
  int G;            // images per CTA
};

struct EvalParams {
  Geom g;
  const uint64_t* entries;
  const uint32_t* skip;
  const int64_t* items;       // [n_items][2]
  int n_items;
  int n_groups;               // ceil(B / G) * n_phase
  int B;
  int n_phase;                // 1 or 2 phase planes in `packed`
  const uint32_t* packed;     // [n_phase][Bpad][img_words], Bpad = ceil(B / G) * G
  int Bpad;
  unsigned long long* counts; // [B][n_phase][S][S]
  int S;                      // 2m + 1
  unsigned int* counter;      // dynamic work-item counter, zeroed by the pack kernel
  int prune;
};

}  // namespace lpf
