// lpf_kernels.cu -- CUDA kernels of liblpf.so (sm_100a).
//   pack_base_kernel  uint8 image -> row-major and column-major bit images, 32 px / word, one coalesced pass
//   pack_views_kernel the four octant views per image, each with its periodic halo laid out exactly as the eval kernel
//                     wants a row band in shared memory (a2)
//   eval_kernel_v3<.> the hot loop: TMA-stage a row band, derive the eroded planes of a pattern class from it, walk
//                     the node program with a running AND mask (a3), POPC + warp reduce at terminals (a4), optional
//                     zero-mask pruning (a5)
//   shallow_kernel    the vectors of fewer steps than a window of the eroded program covers
//   mirror_kernel     counts[-v] = counts[v] (a6)
//   objective_kernel  sum (c - t)^2 per image (a8, Eq. 14/19)
//   swap_delta_kernel_v3 + swap_mirror_kernel  per-proposal count deltas (a9)
#include <cuda_runtime.h>

#include <algorithm>

#include "lpf_internal.h"
#include "lpf_kernels.cuh"
#include "lpf_swap.cuh"

namespace lpf {


// ---------------------------------------------------------------------------------------------
// bit-pack, stage 1: uint8 image -> two compact bit images per phase plane, from ONE coalesced pass.
//   One warp per 32 x 32 pixel tile: lane k reads byte (y0 + j, x0 + k) for j = 0..31 (32 coalesced row
//   segments).  Row words come from __ballot_sync (bit k of Brow[y][x0/32] = [I[y][x0+k] == phase]); every
//   lane also assembles its own COLUMN word (bit j of Bcol[x][y0/32] = [I[y0+j][x] == phase]), so the
//   transposed octant views never read the image with a stride.
//   base layout per plane and image: Brow [H][Wc] then Bcol [W][Hc]   (Wc = ceil(W/32), Hc = ceil(H/32))
// Also zeroes the work counter of the eval kernel that follows on the same stream.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) pack_base_kernel(const uint8_t* __restrict__ images,
                                                        uint32_t* __restrict__ base, int B, int H, int W,
                                                        int n_phase, int phase0, unsigned int* counter) {
  if (blockIdx.x == 0 && threadIdx.x == 0) *counter = 0u;
  const int lane = threadIdx.x & 31;
  const int Wc = (W + 31) >> 5, Hc = (H + 31) >> 5;
  const long long img_words = (long long)H * Wc + (long long)W * Hc;
  const long long tiles = (long long)B * Hc * Wc;
  const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
  for (long long t = warp; t < tiles; t += nwarps) {
    const int b = (int)(t / (Hc * Wc));
    const int rem = (int)(t - (long long)b * Hc * Wc);
    const int ty = rem / Wc, tx = rem - ty * Wc;
    const int x = tx * 32 + lane;
    const uint8_t* src = images + ((size_t)b * H + (size_t)ty * 32) * W + x;
    unsigned col0 = 0, col1 = 0, row0 = 0, row1 = 0;
    int vv[32];                          // all 32 byte loads of the tile in flight before the first ballot (config 4:
                                         // 42 -> 25 us, config 3: 18 -> 6 us; with 8 in flight the kernel waited four times)
#pragma unroll
    for (int j = 0; j < 32; ++j) {
      vv[j] = 255;
      if (x < W && ty * 32 + j < H) vv[j] = src[(size_t)j * W];
    }
#pragma unroll
    for (int j = 0; j < 32; ++j) {
      const int y = ty * 32 + j;
      const int v = vv[j];
      const bool b0 = n_phase == 2 ? (v == 0) : (phase0 < 0 ? (v != 0 && x < W && y < H) : (v == phase0));
      const bool b1 = n_phase == 2 && (v == 1);
      const unsigned r0 = __ballot_sync(0xffffffffu, b0);
      const unsigned r1 = __ballot_sync(0xffffffffu, b1);
      if (lane == j) { row0 = r0; row1 = r1; }
      col0 |= (unsigned)b0 << j;
      col1 |= (unsigned)b1 << j;
    }
    uint32_t* o0 = base + (size_t)b * img_words;
    const int y = ty * 32 + lane;
    if (y < H) o0[(size_t)y * Wc + tx] = row0;
    if (x < W) o0[(size_t)H * Wc + (size_t)x * Hc + ty] = col0;
    if (n_phase == 2) {
      uint32_t* o1 = o0 + (size_t)B * img_words;
      if (y < H) o1[(size_t)y * Wc + tx] = row1;
      if (x < W) o1[(size_t)H * Wc + (size_t)x * Hc + ty] = col1;
    }
  }
}

// 32 consecutive view pixels x' = xs .. xs+31 (no wrap inside) of one source row of `words` words
__device__ __forceinline__ uint32_t window32(const uint32_t* __restrict__ row, int words, int xs) {
  const int w = xs >> 5;
  const uint32_t lo = row[w];
  const uint32_t hi = (w + 1 < words) ? row[w + 1] : 0u;
  return __funnelshift_r(lo, hi, xs & 31);
}

// 32 pixels x .. x+31 of the MIRRORED row msrc[x] = src[(Wv - x) mod Wv], x in [0, Wv), zero beyond Wv (view 3).
// For x + k >= 1 the sources are src[Wv - x - k], descending: the bit-reversed window of src at s = Wv - x - 31.
// Source index 0 inside that window would be pixel x + k = Wv (beyond the row) and is cleared, indices < 0 shift in
// as zeros; pixel 0 of the mirrored row is src[0].
__device__ __forceinline__ uint32_t mirrored_window32(const uint32_t* __restrict__ src, int words, int Wv, int x) {
  const int s = Wv - x - 31;
  uint32_t w;
  if (s > 0) w = window32(src, words, s);
  else if (s > -32) w = (window32(src, words, 0) & ~1u) << (-s);
  else w = 0u;
  return __brev(w) | (x == 0 ? (src[0] & 1u) : 0u);
}

// word of the periodic extension of a view row: 32 view pixels x' = (x0 + k) mod Wv, x0 in [0, Wv).  One window of
// the source row, and one more per wrap (a word wraps at most once unless Wv < 32).  No per-bit work, no division.
template <bool MIRROR>
__device__ __forceinline__ uint32_t periodic_word(const uint32_t* __restrict__ src, int words, int Wv, int x0) {
  uint32_t word = MIRROR ? mirrored_window32(src, words, Wv, x0) : window32(src, words, x0);
  int filled = Wv - x0;                                  // valid bits so far; the bits above them are zero
  if (filled < 32) {
    const uint32_t head = MIRROR ? mirrored_window32(src, words, Wv, 0) : window32(src, words, 0);
    do {
      word |= head << filled;
      filled += Wv;
    } while (filled < 32);
  }
  return word;
}

// ---------------------------------------------------------------------------------------------
// bit-pack, stage 2: the four octant views with their periodic halo.
//   view o of image I (lpf_internal.h): 0: I[y'][x']  1: I[x'][y']  2: I[x'][-y' mod W]  3: I[y'][-x' mod W]
//   word (r, i) of a view holds x' = (32 i + k) mod Wv, y' = r mod Hv.  Views 0 and 3 read Brow, views 1 and 2 Bcol.
//   One thread per word: a funnel shift of two base words, a word that wraps around the row end two of them; fully
//   coalesced stores (the eroded planes are derived from these words in the eval kernel's shared memory).
// ---------------------------------------------------------------------------------------------
constexpr int PACK_TILE = 4096;

__global__ void __launch_bounds__(256) pack_views_kernel(const uint32_t* __restrict__ base,
                                                         uint32_t* __restrict__ packed, Geom g, int B, int Bpad,
                                                         int4 tiles, long long ctas_per_plane) {
  const int Wc = (g.W + 31) >> 5, Hc = (g.H + 31) >> 5;
  const long long img_words = (long long)g.H * Wc + (long long)g.W * Hc;
  // CTA -> (phase plane, view, image, tile)
  const long long cta = blockIdx.x;
  const int plane = (int)(cta / ctas_per_plane);
  long long rem = cta - (long long)plane * ctas_per_plane;
  int o = 0, tl = tiles.x;
  if (rem >= (long long)Bpad * tl) { rem -= (long long)Bpad * tl; o = 1; tl = tiles.y; }
  if (o == 1 && rem >= (long long)Bpad * tl) { rem -= (long long)Bpad * tl; o = 2; tl = tiles.z; }
  if (o == 2 && rem >= (long long)Bpad * tl) { rem -= (long long)Bpad * tl; o = 3; tl = tiles.w; }
  const ViewGeom& v = g.v[o];
  const int b = (int)(rem / tl);
  const int tile = (int)(rem - (long long)b * tl);
  const int pv = v.plane_words;                            // words of the view of one image (rows * stride + padding)
  const int stride = v.stride, rows = v.n_bands * g.band_rows + g.m;
  const int w0 = tile * PACK_TILE, w1 = min(pv, w0 + PACK_TILE);
  uint32_t* dst = packed + (size_t)plane * g.plane_words + v.packed_off + (size_t)b * v.view_words;
  if (b >= B) {                                            // padding images of the last CTA group: all-zero views
    for (int L = w0 + threadIdx.x; L < w1; L += blockDim.x) dst[L] = 0u;
    return;
  }
  const uint32_t* bimg = base + ((size_t)plane * B + b) * img_words;
  const bool rowmajor = (o == 0 || o == 3);
  const int words = rowmajor ? Wc : Hc;
  for (int L = w0 + threadIdx.x; L < w1; L += blockDim.x) {
    uint32_t w = 0u;
    if (L < rows * stride) {
      const int r = L / stride, i = L - r * stride;
      int yv = r;                                          // r < rows <= 2 Hv + band_rows: a few subtractions at most
      while (yv >= v.Hv) yv -= v.Hv;
      // source row of a view row: views 0, 3: image row yv (Brow); view 1: image column yv; view 2: column -yv
      const uint32_t* src = rowmajor ? bimg + (size_t)yv * Wc
                                     : bimg + (size_t)g.H * Wc + (size_t)((o == 1) ? yv : (yv ? g.W - yv : 0)) * Hc;
      const int x0 = (int)((32u * (unsigned)i) % (unsigned)v.Wv);
      w = (o == 3) ? periodic_word<true>(src, words, v.Wv, x0) : periodic_word<false>(src, words, v.Wv, x0);
    }
    dst[L] = w;
  }
}

// ---------------------------------------------------------------------------------------------
// mbarrier / TMA bulk-copy helpers (cp.async.bulk -> SASS UBLKCP)
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, unsigned parity) {
  uint32_t ok;
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
      "selp.u32 %0, 1, 0, p;\n"
      "}\n"
      : "=r"(ok)
      : "r"(smem_u32(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity) {
  while (!mbar_try_wait(bar, parity)) {
  }
}
__device__ __forceinline__ void tma_bulk_g2s(void* dst, const void* src, unsigned bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

// ---------------------------------------------------------------------------------------------
// eval kernel, version 3: register strips on octant views, lean interpreter.
//   CTA = NT teams of G images x wpi warps.  The CTA holds the bands of one KEY -- (image group, phase plane, octant,
//   row band, pattern class) -- in shared memory; every team walks its own work UNIT = (program item, strip band) of
//   that key.  Lane = start row inside a block of 32 rows, warp = (strip, row block): a thread
//   owns the TX x-adjacent start words [strip*TX, strip*TX+TX) of TY start rows (32 apart).
//   It keeps the TX+1 words of the CURRENT path row in registers (R), so an entry that stays in the same row, word
//   column and plane costs TX x (SHF + LOP3) and no load at all; any other reloads TX+1 words (odd row stride: the 32
//   lanes hit 32 different banks).
//   Program fetch: each warp loads 32 entries at a time, one per lane (one coalesced 256 B request, issued a
//   whole chunk ahead), and broadcasts them entry by entry with SHFL; the high word (count index, slots) is
//   fetched only by the rare entries that need it.
//   Saved masks of the depth-first walk live in LOCAL memory (saves/restores are a few % of the entries each; the
//   lines stay in L1), so the hot loop carries no stack registers.
//   The walker does not know about planes: at level K >= 1 shared memory holds the eroded
//   planes of the key's pattern class (derived from the plain band when the key is taken), an entry's offset field
//   already points into the right plane, and one window covers K + 1 path pixels.  PAIR entries fold their window
//   into the next entry's 3-input AND.
//   The mask of an item is initialised once, before the loop (INIT is only ever an item's first entry).
// ---------------------------------------------------------------------------------------------
// ---------------------------------------------------------------------------------------------
// Level K: the eroded planes of one pattern class, derived in shared memory from the plain band (DESIGN.md "Eroded
// planes").  The window of pattern q at a word is the AND of the plain windows j pixels to the right and rho_j =
// s_1 + .. + s_j rows below, j = 0..K.  Compile-time recursion over the balanced words of length K: the patterns are
// the leaves of a prefix tree, every tree edge is one funnel shift + AND, and a leaf is stored only if the class holds
// the pattern (slot[rank] >= 0, a uniform test).
// ---------------------------------------------------------------------------------------------
__host__ __device__ constexpr int popcount_c(unsigned x) { int c = 0; for (; x; x >>= 1) c += (int)(x & 1u); return c; }

template <int K, int J, unsigned PRE>
__device__ __forceinline__ void derive_rec(uint32_t acc, const uint32_t (&lo)[K + 1], const uint32_t (&hi)[K + 1],
                                           uint32_t* out, const signed char* slot, int band_words) {
  if constexpr (J == K) {
    const int s = slot[balanced_rank(PRE, K)];
    if (s >= 0) out[(size_t)s * band_words] = acc;
  } else {
    constexpr int rho = popcount_c(PRE);
    if constexpr (balanced_word(PRE, J + 1))
      derive_rec<K, J + 1, PRE>(acc & __funnelshift_r(lo[rho], hi[rho], J + 1), lo, hi, out, slot, band_words);
    if constexpr (balanced_word(PRE | (1u << J), J + 1))
      derive_rec<K, J + 1, (PRE | (1u << J))>(acc & __funnelshift_r(lo[rho + 1], hi[rho + 1], J + 1), lo, hi, out, slot,
                                              band_words);
  }
}

// planes: [n_planes][band_words] of one image; plain: its plain band [rows][stride] (rows = band_rows + m)
template <int K>
__device__ __forceinline__ void derive_planes(uint32_t* planes, const uint32_t* plain, int rows, int stride,
                                              int band_words, const signed char* slot) {
  const int n = rows * stride;
  const int dr = (int)blockDim.x / stride, di = (int)blockDim.x - dr * stride;
  int r = (int)threadIdx.x / stride, i = (int)threadIdx.x - r * stride;
  for (int idx = threadIdx.x; idx < n; idx += blockDim.x) {
    uint32_t lo[K + 1], hi[K + 1];
    const bool more = i + 1 < stride;                      // the word right of the last one of a row reads as zero
#pragma unroll
    for (int rr = 0; rr <= K; ++rr) {
      const bool ok = r + rr < rows;                       // below the band everything reads as zero
      lo[rr] = ok ? plain[idx + rr * stride] : 0u;
      hi[rr] = (ok && more) ? plain[idx + rr * stride + 1] : 0u;
    }
    derive_rec<K, 0, 0u>(lo[0], lo, hi, planes + idx, slot, band_words);
    i += di;
    r += dr;
    if (i >= stride) { i -= stride; ++r; }
  }
}

// ---------------------------------------------------------------------------------------------
// Tensor memory as the mask stack (TM variant of the eval kernel).  A saved mask is T words that only the thread that
// saved them ever reads back: exactly the access of tcgen05.st / tcgen05.ld with the 32x32b shape (thread i of a warp
// <-> TMEM lane 32 (warp % 4) + i, T consecutive columns).  In local memory a save or a restore moves as many bytes
// through L1 as a row-strip reload (a tenth of that pipe's traffic on config 3); TMEM has its own datapath.  One CTA
// per SM owns all 512 columns: ceil(warps / 4) warps share a lane quarter, n_slots x T columns each.
// ---------------------------------------------------------------------------------------------
template <int T>
__device__ __forceinline__ void tmem_save(uint32_t taddr, const uint32_t (&v)[T]) {
  static_assert(T == 8 || T == 16, "thread tile of 8 or 16 words");
  if constexpr (T == 16)
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
                 ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]),
                 "r"(v[8]), "r"(v[9]), "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15])
                 : "memory");
  else
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"r"(taddr), "r"(v[0]),
                 "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7])
                 : "memory");
  asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}
template <int T>
__device__ __forceinline__ void tmem_restore(uint32_t taddr, uint32_t (&v)[T]) {
  if constexpr (T == 16)
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                   "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
                 : "r"(taddr)
                 : "memory");
  else
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
                 : "r"(taddr)
                 : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// 64 registers per thread: CTAs of up to 1024 threads, 32 warps resident per SM (measured against 72 registers and 24
// warps: config 3 5.33 vs 5.38 ms, config 4 3.67 vs 3.76 ms; the few spilled words sit next to the mask stack in L1)
#ifndef LPF_EVAL_ATTR
#define LPF_EVAL_ATTR __maxnreg__(64)
#endif
template <int TX, int TY, bool PRUNE, bool TM>
__global__ void LPF_EVAL_ATTR eval_kernel_v3(const EvalParams p) {
  constexpr int T = TX * TY;
  constexpr unsigned FULL = 0xffffffffu;
  extern __shared__ __align__(128) uint32_t smem[];
  __shared__ __align__(8) uint64_t bar;
  __shared__ unsigned int s_key;
  __shared__ unsigned int s_unit[2][32];
  __shared__ signed char s_slot[MAX_PATTERNS];

  const Geom& g = p.g;
  const int tid = threadIdx.x, lane = tid & 31;
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);   // provably warp-uniform: the team's unit stays in uniform registers
  const int team_warps = g.G * g.wpi;
  const int team = warp / team_warps;                   // teams walk different units on the same bands
  const int wteam = warp - team * team_warps;
  const int img_local = wteam / g.wpi;
  const int ww = wteam - img_local * g.wpi;
  const int strip_l = ww % g.SB, rblk = ww / g.SB;
  const int row0 = rblk * 32 * TY + lane;               // band-local start row of ty = 0
  uint32_t stk[TM ? 1 : STACK_SLOTS_BUDGET * T];   // the mask stack in local memory (TM: in tensor memory)
  __shared__ uint32_t s_tmem;
  uint32_t tm_mine = 0;                            // TMEM address of this warp's slot 0
  if constexpr (TM) {
    if (tid < 32) {                                // one warp allocates all 512 columns: one CTA per SM (lpf_api.cu)
      asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(&s_tmem)) : "memory");
      asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    tm_mine = s_tmem + ((32u * ((unsigned)warp & 3u)) << 16) + ((unsigned)warp >> 2) * (unsigned)(p.n_slots * T);
  }

  uint32_t M[T];
  uint32_t R[TY][TX + 1];

  if (tid == 0) {
    mbar_init(&bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  unsigned parity = 0;
  const int groups_per_plane = p.Bpad / g.G;
  unsigned flip = 0;

  // A key = (image group, phase plane, octant, row band): the bands one CTA holds in shared memory.  Shares of the keys
  // are handed out by one cursor, pass after pass over all keys in alternating direction: the first passes attach every
  // CTA of the grid to a key, the later ones let a CTA that has run out of work help on a key that is still open (the
  // most recently started ones come first).  The units of a key (program item x strip band, big first) are handed out
  // to the TEAMS by the key's own counter, so a team never waits for another one before the key is exhausted.
  for (;;) {
    __syncthreads();                 // everybody is done reading the previous bands (and the mbarrier is initialised)
    if (tid == 0) {
      unsigned key = 0xffffffffu;
      for (;;) {
        const unsigned s = atomicAdd(p.counters, 1u);
        if (s >= p.n_shares) break;
        const unsigned pass = s / p.n_keys, idx = s - pass * p.n_keys;
        const unsigned k = (pass & 1u) ? p.n_keys - 1u - idx : idx;
        const int4 ob = __ldg(p.obtab + k % (unsigned)p.n_ob);
        if (*(volatile unsigned int*)(p.counters + 1 + k) < (unsigned)ob.y) { key = k; break; }
      }
      s_key = key;
      if (key != 0xffffffffu) {
        const int4 ob = __ldg(p.obtab + key % (unsigned)p.n_ob);
        const int gp = (int)(key / (unsigned)p.n_ob);
        const int plane = gp / groups_per_plane;
        const int b0 = (gp - plane * groups_per_plane) * g.G;
        const ViewGeom& v = g.v[ob.z & 3];
        // the plain band of every image of the group: level 0 walks it; level K derives its planes from it (it sits
        // behind them).  A pattern class keeps only the rows its paths reach: its own band words, rows and planes.
        int bw = v.band_words, np_c = 0;
        if (g.K > 0) {
          const int4 cg = __ldg(p.class_geom + (ob.z >> 2));
          bw = cg.x;
          np_c = cg.z;
        }
        const unsigned bytes = (unsigned)bw * 4u;
        mbar_expect_tx(&bar, bytes * (unsigned)g.G);
        const uint32_t* src = p.packed + (size_t)plane * g.plane_words + v.packed_off + (size_t)b0 * v.view_words +
                              (size_t)ob.w * g.band_rows * v.stride;
        for (int gi = 0; gi < g.G; ++gi)
          tma_bulk_g2s(smem + (size_t)gi * v.band_pitch + (size_t)np_c * bw, src + (size_t)gi * v.view_words, bytes,
                       &bar);
      }
    }
    __syncthreads();
    const unsigned key = __shfl_sync(FULL, s_key, 0);
    if (key == 0xffffffffu) break;
    const int4 ob = __ldg(p.obtab + key % (unsigned)p.n_ob);     // first unit, units, octant, row band
    const int gp = (int)(key / (unsigned)p.n_ob);
    const int plane = gp / groups_per_plane;
    const int b0 = (gp - plane * groups_per_plane) * g.G;
    const int o = ob.z & 3, band = ob.w;
    const ViewGeom& v = g.v[o];
    const int stride = v.stride;
    const int rowstep = 32 * stride * 4;                     // bytes between the TY start rows of a thread
    const int b_img = b0 + img_local;
    unsigned long long* cnt = p.counts + (size_t)b_img * p.image_stride + (size_t)plane * p.S * p.S;
    const bool store = (lane == 0) && (b_img < p.B);
    mbar_wait(&bar, parity);
    parity ^= 1u;
    if (g.K > 0) {                   // the planes of the key's pattern class
      const signed char* slot = p.class_slots + (size_t)(ob.z >> 2) * MAX_PATTERNS;
      const int4 cg = __ldg(p.class_geom + (ob.z >> 2));     // band words, rows, planes, level of the class
      for (int i = tid; i < MAX_PATTERNS; i += (int)blockDim.x) s_slot[i] = slot[i];   // a CTA may be one warp
      __syncthreads();
      for (int gi = 0; gi < g.G; ++gi) {
        uint32_t* planes = smem + (size_t)gi * v.band_pitch;
        const uint32_t* plain = planes + (size_t)cg.z * cg.x;
        switch (cg.w) {
          case 1: derive_planes<1>(planes, plain, cg.y, stride, cg.x, s_slot); break;
          case 2: derive_planes<2>(planes, plain, cg.y, stride, cg.x, s_slot); break;
          case 3: derive_planes<3>(planes, plain, cg.y, stride, cg.x, s_slot); break;
          case 4: derive_planes<4>(planes, plain, cg.y, stride, cg.x, s_slot); break;
          case 5: derive_planes<5>(planes, plain, cg.y, stride, cg.x, s_slot); break;
          default: derive_planes<6>(planes, plain, cg.y, stride, cg.x, s_slot); break;
        }
      }
      __syncthreads();
    }

   for (;;) {                        // the team's units of this key
    unsigned u;
    if (team_warps == 1) {
      u = 0;
      if (lane == 0) u = atomicAdd(p.counters + 1 + key, 1u);
    } else {
      if (wteam == 0 && lane == 0) s_unit[flip][team] = atomicAdd(p.counters + 1 + key, 1u);
      asm volatile("bar.sync %0, %1;" ::"r"(1 + team), "r"(team_warps * 32) : "memory");
      u = s_unit[flip][team];
      flip ^= 1u;                    // the other slot next time: nobody can still be reading it
    }
    u = __shfl_sync(FULL, u, 0);     // provably warp-uniform: the walker's control flow stays on the uniform datapath
    if (__all_sync(FULL, u >= (unsigned)ob.y)) break;     // a vote: ptxas keeps the loop on the uniform datapath
    const int4 wk = __ldg(p.units + ob.x + u);               // first entry, entries, strip band
    const int sband = wk.z;
    // per-unit thread geometry (the octant decides the view size)
    const int strip = sband * g.SB + strip_l;
    const bool active = strip < v.n_strips;
    const char* base =
        (const char*)(smem + (size_t)img_local * v.band_pitch + row0 * stride + (active ? strip : 0) * TX);
    int e = wk.x;
    const int e1 = e + wk.y;
    uint2 cur = __ldg(p.entries + e + lane);                 // the entry array is padded by 64
    // Every item begins with its only INIT entry: the parent mask is "every valid start pixel" (of the selected ones
    // for L2~).
#pragma unroll
    for (int ty = 0; ty < TY; ++ty) {
      const bool rowok = active && (band * g.band_rows + row0 + ty * 32 < v.Hv);
#pragma unroll
      for (int t = 0; t < TX; ++t) {
        const int nb = v.Wv - 32 * (strip * TX + t);         // start pixels x' < Wv only
        const uint32_t cm = nb >= 32 ? 0xffffffffu : (nb <= 0 ? 0u : ((1u << nb) - 1u));
        M[ty * TX + t] = rowok ? cm : 0u;
      }
      if (p.mask != nullptr && rowok) {                      // L2~: only the selected start pixels
        const uint32_t* mw =
            p.mask + p.mask_off[o] + (size_t)(band * g.band_rows + row0 + ty * 32) * stride + strip * TX;
#pragma unroll
        for (int t = 0; t < TX; ++t) M[ty * TX + t] &= __ldg(mw + t);
      }
    }
    while (e < e1) {
      const uint2 nxt = __ldg(p.entries + e + 32 + lane);
      const int n = min(32, e1 - e);
      int jump = -1;
      uint32_t x = __shfl_sync(FULL, cur.x, 0);
#pragma unroll 1
      for (int i = 0; i < n; ++i) {
        // the next program word, broadcast by a warp reduction: REDUX writes a uniform register directly and leaves the
        // shared-memory pipe, which the strip reloads keep busy, one instruction per entry (a shuffle goes through it)
        uint32_t xn = __reduce_or_sync(FULL, lane == i + 1 ? cur.x : 0u);
        if (x & E_RESTORE) {
          const uint32_t y = __shfl_sync(FULL, cur.y, i);
          if constexpr (TM) {
            tmem_restore<T>(tm_mine + ((y >> E_RSLOT_SHIFT) & E_SLOT_MASK) * T, M);
          } else {
            const uint32_t* s = stk + ((y >> E_RSLOT_SHIFT) & E_SLOT_MASK) * T;
#pragma unroll
            for (int t = 0; t < T; ++t) M[t] = s[t];
          }
        }
        if (x & E_RELOAD) {
          const char* rp = base + ((x >> (E_OFF_SHIFT - 2)) & ~3u);
#pragma unroll
          for (int ty = 0; ty < TY; ++ty)
#pragma unroll
            for (int k = 0; k <= TX; ++k) R[ty][k] = *(const uint32_t*)(rp + ty * rowstep + 4 * k);
        }
        if ((x & E_PAIR) && i + 1 < n) {
          // this node's mask is never needed on its own: fold its window and its child's into one 3-input AND
          uint32_t Wp[T];
#pragma unroll
          for (int ty = 0; ty < TY; ++ty)
#pragma unroll
            for (int t = 0; t < TX; ++t) Wp[ty * TX + t] = __funnelshift_r(R[ty][t], R[ty][t + 1], x);
          x = xn;
          ++i;
          xn = __reduce_or_sync(FULL, lane == i + 1 ? cur.x : 0u);
          if (x & E_RELOAD) {
            const char* rp = base + ((x >> (E_OFF_SHIFT - 2)) & ~3u);
#pragma unroll
            for (int ty = 0; ty < TY; ++ty)
#pragma unroll
              for (int k = 0; k <= TX; ++k) R[ty][k] = *(const uint32_t*)(rp + ty * rowstep + 4 * k);
          }
#pragma unroll
          for (int ty = 0; ty < TY; ++ty)
#pragma unroll
            for (int t = 0; t < TX; ++t)
              M[ty * TX + t] &= Wp[ty * TX + t] & __funnelshift_r(R[ty][t], R[ty][t + 1], x);
        } else {
#pragma unroll
          for (int ty = 0; ty < TY; ++ty)
#pragma unroll
            for (int t = 0; t < TX; ++t) M[ty * TX + t] &= __funnelshift_r(R[ty][t], R[ty][t + 1], x);
        }
        if (x & (E_TERMINAL | E_SAVE)) {
          const uint32_t y = __shfl_sync(FULL, cur.y, i);
          if (x & E_SAVE) {
            if constexpr (TM) {
              tmem_save<T>(tm_mine + ((y >> E_SSLOT_SHIFT) & E_SLOT_MASK) * T, M);
            } else {
              uint32_t* s = stk + ((y >> E_SSLOT_SHIFT) & E_SLOT_MASK) * T;
#pragma unroll
              for (int t = 0; t < T; ++t) s[t] = M[t];
            }
          }
          if (x & E_TERMINAL) {
            int c = 0;
#pragma unroll
            for (int t = 0; t < T; ++t) c += __popc(M[t]);
            c = __reduce_add_sync(FULL, c);
            if (c != 0) {

              if (store) atomicAdd(cnt + (y & E_CIDX_MASK), (unsigned long long)c);
            } else if (PRUNE) {          // paper's "enhanced" rule: nothing below can count
              const int sk = (int)__ldg(p.skip + e + i);
              if (sk) {
                jump = e + i + 1 + sk;
                break;
              }
            }
          }
        }
        x = xn;
      }
      if (PRUNE && jump >= 0) {
        e = jump;
        if (e < e1) cur = __ldg(p.entries + e + lane);
      } else {
        e += 32;
        cur = nxt;
      }
    }
   }
  }
  if constexpr (TM) {                              // every warp is done with its columns
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (tid < 32) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(s_tmem) : "memory");
  }
}

typedef void (*eval_fn)(const EvalParams);
static eval_fn eval_fn_for(int TX, int TY, bool prune, bool tm) {
#define LPF_PICK(tx, ty)                                                                              \
  if (TX == tx && TY == ty)                                                                           \
    return tm ? (prune ? eval_kernel_v3<tx, ty, true, true> : eval_kernel_v3<tx, ty, false, true>)    \
              : (prune ? eval_kernel_v3<tx, ty, true, false> : eval_kernel_v3<tx, ty, false, false>);
  LPF_PICK(4, 2)
  LPF_PICK(8, 1)
  LPF_PICK(4, 4)
  LPF_PICK(8, 2)
  LPF_PICK(16, 1)
#undef LPF_PICK
  return nullptr;
}
// ---------------------------------------------------------------------------------------------
// mirror: counts[-v] = counts[v] for v in D.  n_arrays = B * n_phase arrays of S*S.
// ---------------------------------------------------------------------------------------------
__global__ void mirror_kernel(unsigned long long* counts, int S) {
  // grid = (chunks, arrays).  In the row-major [S][S] array the vectors outside D (dy < 0, or dy = 0 and dx < 0) are
  // exactly the indices below the centre, and -v sits at K - 1 - k: no division, coalesced both ways.
  const long long K = (long long)S * S;
  const long long half = K / 2;
  unsigned long long* c = counts + (size_t)blockIdx.y * K;
  for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < half; k += (long long)gridDim.x * blockDim.x)
    c[k] = c[K - 1 - k];
}

// ---------------------------------------------------------------------------------------------
// shallow vectors (level K >= 1): a window of the eroded program covers K + 1 path pixels, so the vectors whose paths
// are shorter (depth < K in their octant trie: at most 1 + 2 + .. + K of them per octant) have no entry.  They are
// counted here from the plain view in HBM: grid = (n_phase * B, 4 octants, row chunks).  A thread loads the plain
// words of 32 start pixels and of the K - 1 rows below and walks the prefix tree of the balanced step patterns with
// compile-time recursion (one funnel shift + AND per edge, as derive_planes does); where a prefix is one of the
// octant's short vectors (sl.node, a uniform test) it counts: POPC, warp reduce, one shared-memory atomic per warp.
// ---------------------------------------------------------------------------------------------
template <int J, unsigned PRE>
__device__ __forceinline__ void shallow_rec(uint32_t acc, const uint32_t (&lo)[MAX_LEVEL], const uint32_t (&hi)[MAX_LEVEL],
                                            int K, const signed char* node, int* s_cnt, bool lane0) {
  const int t = node[shallow_base(J) + balanced_rank(PRE, J)];
  if (t >= 0) {
    const int c = __reduce_add_sync(0xffffffffu, __popc(acc));
    if (lane0 && c) atomicAdd(&s_cnt[t], c);
  }
  if constexpr (J + 1 < MAX_LEVEL) {
    if (J + 1 < K) {
      constexpr int rho = popcount_c(PRE);
      if constexpr (balanced_word(PRE, J + 1))
        shallow_rec<J + 1, PRE>(acc & __funnelshift_r(lo[rho], hi[rho], J + 1), lo, hi, K, node, s_cnt, lane0);
      if constexpr (balanced_word(PRE | (1u << J), J + 1))
        shallow_rec<J + 1, (PRE | (1u << J))>(acc & __funnelshift_r(lo[rho + 1], hi[rho + 1], J + 1), lo, hi, K, node,
                                              s_cnt, lane0);
    }
  }
}

__global__ void __launch_bounds__(256) shallow_kernel(const EvalParams p, const ShallowList sl, int rows_per_chunk) {
  const Geom& g = p.g;
  const int o = blockIdx.y;
  const int n = sl.n[o];
  if (n == 0) return;
  const ViewGeom& v = g.v[o];
  const int b = blockIdx.x % p.B, plane = blockIdx.x / p.B;
  const uint32_t* plain = p.packed + (size_t)plane * g.plane_words + v.packed_off + (size_t)b * v.view_words;
  const uint32_t* mask = p.mask ? p.mask + p.mask_off[o] : nullptr;
  const int stride = v.stride;
  __shared__ int s_cnt[MAX_SHALLOW];
  if (threadIdx.x < MAX_SHALLOW) s_cnt[threadIdx.x] = 0;
  __syncthreads();
  const int r0 = blockIdx.z * rows_per_chunk, r1 = min(v.Hv, r0 + rows_per_chunk);
  const int n_words = max(0, r1 - r0) * v.Wc;
  const bool lane0 = (threadIdx.x & 31) == 0;
  for (int base = 0; base < n_words; base += blockDim.x) {   // uniform trip count: the warp reduces together
    const int idx = base + threadIdx.x;
    uint32_t lo[MAX_LEVEL], hi[MAX_LEVEL];
#pragma unroll
    for (int rr = 0; rr < MAX_LEVEL; ++rr) lo[rr] = hi[rr] = 0u;
    uint32_t w0 = 0u;
    if (idx < n_words) {
      const int r = r0 + idx / v.Wc, i = idx % v.Wc;
      const int nb = v.Wv - 32 * i;
      const uint32_t* q = plain + (size_t)r * stride + i;    // the view has m >= K - 1 halo rows below and one word right
#pragma unroll
      for (int rr = 0; rr < MAX_LEVEL; ++rr)
        if (rr < g.K) { lo[rr] = q[(size_t)rr * stride]; hi[rr] = q[(size_t)rr * stride + 1]; }
      w0 = lo[0] & (nb >= 32 ? 0xffffffffu : ((1u << nb) - 1u));   // start pixels x' < Wv only
      if (mask) w0 &= mask[(size_t)r * stride + i];
    }
    shallow_rec<0, 0u>(w0, lo, hi, g.K, sl.node[o], s_cnt, lane0);
  }
  __syncthreads();
  if (threadIdx.x < n && s_cnt[threadIdx.x])
    atomicAdd(p.counts + (size_t)b * p.image_stride + (size_t)plane * p.S * p.S + sl.cidx[o][threadIdx.x],
              (unsigned long long)s_cnt[threadIdx.x]);
}

// ---------------------------------------------------------------------------------------------
// objective: sse[b] = sum_k (c[b][k] - t[k])^2, exact in uint64 (Eq. 14 / Eq. 19).
// grid = (chunks, B); partial sums are combined with one 64-bit atomic per block.
// ---------------------------------------------------------------------------------------------
__global__ void objective_kernel(const long long* __restrict__ counts, const long long* __restrict__ target,
                                 long long K, unsigned long long* sse) {
  const int b = blockIdx.y;
  const long long* c = counts + (size_t)b * K;
  unsigned long long s = 0;
  for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < K; k += (long long)gridDim.x * blockDim.x) {
    const long long d = c[k] - target[k];
    s += (unsigned long long)(d * d);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
  __shared__ unsigned long long ws[32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0) ws[warp] = s;
  __syncthreads();
  if (warp == 0) {
    s = (lane < (int)(blockDim.x >> 5)) ? ws[lane] : 0ull;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    if (lane == 0) atomicAdd(sse + b, s);
  }
}

// ---------------------------------------------------------------------------------------------
// swap delta, version 3: the device code is in lpf_swap.cuh.
// ---------------------------------------------------------------------------------------------
// the base bit image with a periodic halo of m pixels on every side: bit (X, Y) of the padded image, X in
// [0, W + 2m), Y in [0, H + 2m), is pixel ((X - m) mod W, (Y - m) mod H).  One thread per output word.  With it a
// segment that starts inside the image never needs a modulo.
__global__ void pack_padded_kernel(const uint32_t* __restrict__ brow, uint32_t* __restrict__ padded, int H, int W,
                                   int m, long long brow_plane_stride) {
  const int Wc = (W + 31) >> 5, PWc = (W + 2 * m + 31) >> 5, PH = H + 2 * m;
  brow += blockIdx.y * brow_plane_stride;                  // one phase plane per blockIdx.y
  padded += (size_t)blockIdx.y * PH * PWc;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < PH * PWc; i += gridDim.x * blockDim.x) {
    const int Y = i / PWc, wi = i - Y * PWc;
    int y = (Y - m) % H;
    y += y < 0 ? H : 0;
    const uint32_t* srow = brow + (size_t)y * Wc;
    int x0 = (32 * wi - m) % W;
    x0 += x0 < 0 ? W : 0;
    uint32_t word = 0;
    if (x0 + 32 <= W) word = window32(srow, Wc, x0);
    else
      for (int k = 0; k < 32; ++k) {
        const int xs = (x0 + k) % W;
        word |= ((srow[xs >> 5] >> (xs & 31)) & 1u) << k;
      }
    padded[i] = word;
  }
}

// which phase planes are DENSE (more than half of the pixels in phase): bit k of *mask for plane k.  In a dense phase
// the backward walks of the reversed trie rarely die, and the per-node walks of swap_delta_unit are cheaper (measured on
// config 5: phase 1, fraction 0.30, 1.9e6 swaps/s with the reversed trie against 7.7e5 without; phase 0, fraction 0.70,
// 5.2e4 against 6.8e4).  One CTA; brow = the compact row-major bit images of stage 1, one per plane.
__global__ void __launch_bounds__(256) phase_density_kernel(const uint32_t* __restrict__ brow, int H, int W, int n_planes,
                                                            long long plane_stride, unsigned int* mask) {
  __shared__ unsigned long long s_sum;
  const int Wc = (W + 31) >> 5;
  unsigned int dense = 0;
  for (int pl = 0; pl < n_planes; ++pl) {
    if (threadIdx.x == 0) s_sum = 0ull;
    __syncthreads();
    unsigned long long c = 0;
    for (int i = threadIdx.x; i < H * Wc; i += blockDim.x) c += __popc(brow[pl * plane_stride + i]);
    atomicAdd(&s_sum, c);
    __syncthreads();
    if (2ull * s_sum > (unsigned long long)H * W) dense |= 1u << pl;
    __syncthreads();
  }
  if (threadIdx.x == 0) *mask = dense;
}

// CTA = sw proposals (1 .. SWAP_SW: 8 when there are many proposals -- the node records are fetched once for all of
// them -- fewer for a small batch, so that its passes run in parallel CTAs instead of one after the other) x one node
// slice (gridDim.y slices, so that a small batch still fills the chip); image bits in shared memory.
// delta must be zero on entry; only the canonical half is written (swap_mirror_kernel fills the rest).
__global__ void __launch_bounds__(256) swap_delta_kernel_v3(const uint32_t* __restrict__ bits, int H, int W, int m,
                                                             const int* __restrict__ pairs, long long n,
                                                             const int4* __restrict__ rec, int n_nodes,
                                                             const int4* __restrict__ rrec,
                                                             const unsigned int* __restrict__ dense,
                                                             int* __restrict__ delta, int n_planes,
                                                             long long plane_stride, int sw) {
  extern __shared__ __align__(16) uint32_t sm[];
  __shared__ SwapShared sh;
  const int plane_words = (H + 2 * m) * ((W + 2 * m + 31) >> 5);
  uint2* stk = (uint2*)(sm + ((n_planes * plane_words + 1) & ~1));
  for (int i = threadIdx.x; i < n_planes * plane_words; i += blockDim.x) sm[i] = bits[i];
  const long long S2 = (long long)(2 * m + 1) * (2 * m + 1);
  swap_delta_unit<3, true>(sm, stk, sh, H, W, m, pairs, n, (long long)blockIdx.x * sw, rec, n_nodes, rrec, __ldg(dense),
                  delta + (long long)blockIdx.x * sw * S2, n_planes, plane_stride, sw, blockIdx.y, gridDim.y);
}

// delta(-v) = delta(v) (Eq. 12): fills the half outside D of every [S][S] array
__global__ void swap_mirror_kernel(int* __restrict__ delta, int S, long long n_arrays) {
  const long long K = (long long)S * S;
  const long long half = K / 2;                            // indices below the centre are outside D
  const long long total = n_arrays * half;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total;
       i += (long long)gridDim.x * blockDim.x) {
    const long long arr = i / half;
    const long long k = i - arr * half;
    delta[arr * K + k] = delta[arr * K + (K - 1 - k)];
  }
}

// ---------------------------------------------------------------------------------------------
// host launch wrappers (called from lpf_api.cu)
// ---------------------------------------------------------------------------------------------
// Bpad: images per octant block of the packed layout (B rounded up to the CTA group; 1 for a start mask)
cudaError_t launch_pack(const uint8_t* images, uint32_t* base, uint32_t* packed, const Geom& g, int B, int Bpad,
                        int n_phase, int phase0, unsigned int* counter, int n_sm, cudaStream_t st) {
  const long long tiles = (long long)B * ((g.H + 31) / 32) * ((g.W + 31) / 32);
  long long blocks = (tiles + 7) / 8;
  blocks = std::max(1ll, std::min(blocks, (long long)n_sm * 16));
  pack_base_kernel<<<(unsigned)blocks, 256, 0, st>>>(images, base, B, g.H, g.W, n_phase, phase0, counter);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  int tl[4], stride_max = 0;
  long long per_plane = 0;
  for (int o = 0; o < 4; ++o) {
    tl[o] = (g.v[o].plane_words + PACK_TILE - 1) / PACK_TILE;
    per_plane += (long long)Bpad * tl[o];
    stride_max = std::max(stride_max, g.v[o].stride);
  }
  if (per_plane * n_phase >= (1ll << 31)) return cudaErrorInvalidValue;
  pack_views_kernel<<<(unsigned)(per_plane * n_phase), 256, 0, st>>>(base, packed, g, B, Bpad,
                                                                     make_int4(tl[0], tl[1], tl[2], tl[3]), per_plane);
  return cudaGetLastError();
}

// also raises the kernel's dynamic shared memory limit to the device maximum (once is enough, repeating is harmless),
// so that launches of any plan fit whatever order the plans were made in
cudaError_t eval_occupancy(int TX, int TY, bool prune, bool tm, int threads, size_t smem, int max_smem,
                           int* blocks_per_sm) {
  eval_fn f = eval_fn_for(TX, TY, prune, tm);
  if (!f) return cudaErrorInvalidValue;
  cudaFuncAttributes fa;
  cudaError_t e = cudaFuncGetAttributes(&fa, f);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem - (int)fa.sharedSizeBytes);
  if (e != cudaSuccess) return e;
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_per_sm, f, threads, smem);
}

cudaError_t launch_eval(const EvalParams& p, int grid, int threads, size_t smem, cudaStream_t st) {
  eval_fn f = eval_fn_for(p.g.TX, p.g.TY, p.prune != 0, p.tmem_stack != 0);
  if (!f) return cudaErrorInvalidValue;
  f<<<grid, threads, smem, st>>>(p);
  return cudaGetLastError();
}

cudaError_t launch_shallow(const EvalParams& p, const ShallowList& sl, int n_sm, cudaStream_t st) {
  // row chunks: about two CTAs per SM in all
  int hv_max = 0;
  for (int o = 0; o < 4; ++o) hv_max = std::max(hv_max, p.g.v[o].Hv);
  const long long blocks = (long long)p.B * p.n_phase * 4;
  int nz = (int)std::max<long long>(1, std::min<long long>((2ll * n_sm + blocks - 1) / blocks, (hv_max + 7) / 8));
  const int rows_per_chunk = (hv_max + nz - 1) / nz;
  nz = (hv_max + rows_per_chunk - 1) / rows_per_chunk;
  shallow_kernel<<<dim3((unsigned)(p.B * p.n_phase), 4u, (unsigned)nz), 256, 0, st>>>(p, sl, rows_per_chunk);
  return cudaGetLastError();
}

cudaError_t launch_mirror(unsigned long long* counts, int S, long long n_arrays, int n_sm, cudaStream_t st) {
  const long long half = (long long)S * S / 2;
  long long chunks = std::max<long long>(1, (half + 1023) / 1024);
  chunks = std::min(chunks, std::max<long long>(1, (8ll * n_sm + n_arrays - 1) / n_arrays));
  for (long long a0 = 0; a0 < n_arrays; a0 += 65535) {      // gridDim.y <= 65535: fold larger batches
    const long long na = std::min<long long>(n_arrays - a0, 65535);
    mirror_kernel<<<dim3((unsigned)chunks, (unsigned)na), 256, 0, st>>>(counts + (size_t)a0 * S * S, S);
  }
  return cudaGetLastError();
}

cudaError_t launch_objective(const long long* counts, const long long* target, int B, long long K,
                             unsigned long long* sse, int n_sm, cudaStream_t st) {
  cudaError_t e = cudaMemsetAsync(sse, 0, sizeof(unsigned long long) * (size_t)B, st);
  if (e != cudaSuccess) return e;
  long long chunks = (K + 256 * 8 - 1) / (256 * 8);
  const long long want = ((long long)n_sm * 32 + B - 1) / B;    // enough blocks to fill the chip and keep loads in flight
  if (chunks > want) chunks = want;
  if (chunks < 1) chunks = 1;
  // gridDim.y <= 65535: fold larger batches
  for (int b0 = 0; b0 < B; b0 += 65535) {
    const int nb = (B - b0 < 65535) ? (B - b0) : 65535;
    objective_kernel<<<dim3((unsigned)chunks, (unsigned)nb), 256, 0, st>>>(counts + (size_t)b0 * K, target, K,
                                                                             sse + b0);
  }
  return cudaGetLastError();
}

cudaError_t swap_delta_prepare(size_t max_smem) {
  cudaFuncAttributes fa;
  cudaError_t e = cudaFuncGetAttributes(&fa, swap_delta_kernel_v3);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(swap_delta_kernel_v3, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              (int)max_smem - (int)fa.sharedSizeBytes);
}

// the padded bit planes of the base image for the swap-delta kernel: stage 1 of the bit-pack gives the row-major bit
// image(s) (the column-major half is unused), pack_padded_kernel adds the periodic halo of m pixels.
// bits: [n_planes compact images][n_planes padded planes]; returns the padded planes through *padded.
cudaError_t launch_swap_bits(const uint8_t* image, uint32_t* bits, int H, int W, int m, int phase,
                             unsigned int* counter, int n_sm, cudaStream_t st, uint32_t** padded_out) {
  const int n_planes = phase < 0 ? 2 : 1;
  const int Wc = (W + 31) / 32, Hc = (H + 31) / 32;
  const int PWc = (W + 2 * m + 31) / 32, PH = H + 2 * m;
  const long long img_words = (long long)H * Wc + (long long)W * Hc;
  uint32_t* const padded = bits + (size_t)n_planes * img_words;
  pack_base_kernel<<<(unsigned)std::max(1, (Hc * Wc + 7) / 8), 256, 0, st>>>(image, bits, 1, H, W, n_planes,
                                                                             phase < 0 ? 0 : phase, counter);
  pack_padded_kernel<<<dim3((unsigned)std::max(1, std::min((PH * PWc + 255) / 256, n_sm * 8)), (unsigned)n_planes), 256,
                       0, st>>>(bits, padded, H, W, m, img_words);
  phase_density_kernel<<<1, 256, 0, st>>>(bits, H, W, n_planes, img_words, counter + 1);   // counter[1]: dense planes
  *padded_out = padded;
  return cudaGetLastError();
}

// the swap-delta kernel alone on the n_launch proposals of `pairs`: delta must be zero, only the canonical half is written
static cudaError_t launch_swap_core(const uint32_t* padded, int H, int W, int m, int n_planes, const int* pairs,
                                    long long n_launch, const int32_t* rec, int n_nodes, const int32_t* rrec,
                                    const unsigned int* dense, int* delta, long long plane_stride, int n_sm,
                                    cudaStream_t st) {
  const int PWc = (W + 2 * m + 31) / 32, PH = H + 2 * m;
  const size_t smem = (size_t)((n_planes * PH * PWc + 1) & ~1) * 4 + (size_t)8 * SWAP_STACK * 8;
  const long long S2 = (long long)(2 * m + 1) * (2 * m + 1);
  // proposals per CTA: 8 for big batches; a small batch is spread over about four CTAs per SM instead
  int sw = SWAP_SW;
  while (sw > 1 && (n_launch + sw - 1) / sw < 4ll * n_sm) sw /= 2;
  const long long ctas = (n_launch + sw - 1) / sw;
  for (long long c0 = 0; c0 < ctas; c0 += (1ll << 30)) {
    const long long cnt = std::min(ctas - c0, 1ll << 30);
    const long long s0 = c0 * sw;
    // node slices: about four CTAs per SM in total, at least 256 nodes per slice
    const int slices =
        (int)std::max(1ll, std::min<long long>({(4ll * n_sm + cnt - 1) / cnt, (n_nodes + 255) / 256, 65535ll}));
    swap_delta_kernel_v3<<<dim3((unsigned)cnt, (unsigned)slices), 256, smem, st>>>(
        padded, H, W, m, pairs + 4 * s0, n_launch - s0, (const int4*)rec, n_nodes, (const int4*)rrec, dense,
        delta + s0 * S2, n_planes, plane_stride, sw);
  }
  return cudaGetLastError();
}

// phase 0 | 1: one plane, delta [n][S][S];  phase < 0: both planes, phase k at delta + k * plane_stride
cudaError_t launch_swap_delta(const uint8_t* image, uint32_t* bits, int H, int W, int m, int phase, const int* pairs,
                              long long n, const int32_t* rec, int n_nodes, const int32_t* rrec, int* delta,
                              long long plane_stride, unsigned int* counter, int n_sm, cudaStream_t st) {
  const int n_planes = phase < 0 ? 2 : 1;
  const long long S2 = (long long)(2 * m + 1) * (2 * m + 1);
  cudaError_t e = cudaSuccess;
  for (int pl = 0; pl < n_planes; ++pl) {
    e = cudaMemsetAsync(delta + pl * plane_stride, 0, sizeof(int) * (size_t)n * S2, st);
    if (e != cudaSuccess) return e;
  }
  uint32_t* padded = nullptr;
  e = launch_swap_bits(image, bits, H, W, m, phase, counter, n_sm, st, &padded);
  if (e != cudaSuccess) return e;
  e = launch_swap_core(padded, H, W, m, n_planes, pairs, n, rec, n_nodes, rrec, counter + 1, delta, plane_stride, n_sm, st);
  if (e != cudaSuccess) return e;
  const long long blocks = std::max(1ll, std::min<long long>((n * (S2 / 2) + 255) / 256, (long long)n_sm * 16));
  for (int pl = 0; pl < n_planes; ++pl)
    swap_mirror_kernel<<<(unsigned)blocks, 256, 0, st>>>(delta + pl * plane_stride, 2 * m + 1, n);
  return cudaGetLastError();
}

}  // namespace lpf
