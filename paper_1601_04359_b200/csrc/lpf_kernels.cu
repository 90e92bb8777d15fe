// lpf_kernels.cu -- CUDA kernels of liblpf.so (sm_100a).
//   pack_base_kernel  uint8 image -> row-major and column-major bit images, 32 px / word, one coalesced pass
//   pack_views_kernel the four octant views per image (plain, and the eroded planes E2 / D2), each with its periodic
//                     halo laid out exactly as the eval kernel wants it in shared memory (a2)
//   eval_kernel_v3<.> the hot loop: walk the node program with a running AND mask (a3), POPC +
//                     warp reduce at terminals (a4), optional zero-mask pruning (a5)
//   mirror_kernel     counts[-v] = counts[v] (a6)
//   objective_kernel  sum (c - t)^2 per image (a8, Eq. 14/19)
//   swap_delta_kernel_v3 + swap_mirror_kernel  per-proposal count deltas (a9)
#include <cuda_runtime.h>

#include <algorithm>

#include "lpf_internal.h"
#include "lpf_kernels.cuh"

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
#pragma unroll 8
    for (int j = 0; j < 32; ++j) {
      const int y = ty * 32 + j;
      int v = 255;
      if (x < W && y < H) v = src[(size_t)j * W];
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
//   One CTA per tile of PACK_TILE consecutive words of one (phase plane, view, image): it stages the plain words of
//   the tile and of the row below it in shared memory (each a funnel shift of two base words, wrap words two of them),
//   derives E2 = pixel & right neighbour and D2 = pixel & lower-right neighbour there (across word and row boundaries)
//   and writes the planes with fully coalesced stores (a tile is one contiguous block of every plane).
// ---------------------------------------------------------------------------------------------
constexpr int PACK_TILE = 4096;

__global__ void __launch_bounds__(256) pack_views_kernel(const uint32_t* __restrict__ base,
                                                         uint32_t* __restrict__ packed, Geom g, int B, int Bpad,
                                                         int4 tiles, long long ctas_per_plane) {
  extern __shared__ uint32_t s_plain[];                    // [PACK_TILE + stride + 2]
  const int Wc = (g.W + 31) >> 5, Hc = (g.H + 31) >> 5;
  const long long img_words = (long long)g.H * Wc + (long long)g.W * Hc;
  const int np = g.v[0].e2_view_off > 0 ? 3 : 1;
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
  const int pv = v.view_words / np;                        // words of one plane of one image (rows * stride + padding)
  const int stride = v.stride, rows = v.n_bands * g.band_rows + g.m;
  const int w0 = tile * PACK_TILE, w1 = min(pv, w0 + PACK_TILE);
  const int n_stage = min(w1 + stride + 2, rows * stride) - w0;      // staged words; beyond them everything is zero
  uint32_t* dst = packed + (size_t)plane * g.plane_words + v.packed_off + (size_t)b * v.view_words;
  if (b >= B) {                                            // padding images of the last CTA group: all-zero planes
    for (int L = w0 + threadIdx.x; L < w1; L += blockDim.x) {
      dst[L] = 0u;
      if (np == 3) { dst[L + v.e2_view_off] = 0u; dst[L + 2 * (size_t)v.e2_view_off] = 0u; }
    }
    return;
  }
  const uint32_t* bimg = base + ((size_t)plane * B + b) * img_words;
  const bool rowmajor = (o == 0 || o == 3);
  const int words = rowmajor ? Wc : Hc;
  for (int j = threadIdx.x; j < n_stage; j += blockDim.x) {
    const int L = w0 + j;
    const int r = L / stride, i = L - r * stride;
    int yv = r;                                            // r < rows <= 2 Hv + band_rows: a few subtractions at most
    while (yv >= v.Hv) yv -= v.Hv;
    // source row of a view row: views 0, 3: image row yv (Brow); view 1: image column yv; view 2: column -yv
    const uint32_t* src = rowmajor ? bimg + (size_t)yv * Wc
                                   : bimg + (size_t)g.H * Wc + (size_t)((o == 1) ? yv : (yv ? g.W - yv : 0)) * Hc;
    const int x0 = (int)((32u * (unsigned)i) % (unsigned)v.Wv);
    s_plain[j] = (o == 3) ? periodic_word<true>(src, words, v.Wv, x0) : periodic_word<false>(src, words, v.Wv, x0);
  }
  __syncthreads();
  for (int L = w0 + threadIdx.x; L < w1; L += blockDim.x) {
    const int j = L - w0;
    const uint32_t w00 = j < n_stage ? s_plain[j] : 0u;
    dst[L] = w00;
    if (np == 3) {
      const int r = L / stride, i = L - r * stride;
      const bool more = i + 1 < stride;                    // the word right of the last one of a row reads as zero
      const uint32_t w01 = (more && j + 1 < n_stage) ? s_plain[j + 1] : 0u;
      const uint32_t w10 = (j + stride < n_stage) ? s_plain[j + stride] : 0u;
      const uint32_t w11 = (more && j + stride + 1 < n_stage) ? s_plain[j + stride + 1] : 0u;
      dst[L + v.e2_view_off] = w00 & __funnelshift_r(w00, w01, 1);
      dst[L + 2 * (size_t)v.e2_view_off] = w00 & __funnelshift_r(w10, w11, 1);
    }
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
//   CTA = G images x wpi warps; every warp of the CTA walks the same work item = (program item, row band,
//   strip band) on the same phase plane.  Lane = start row inside a block of 32 rows, warp = (strip, row
//   block): a thread owns the TX x-adjacent start words [strip*TX, strip*TX+TX) of TY start rows (32 apart).
//   It keeps the TX+1 words of the CURRENT path row in registers (R), so a node that stays in the same row
//   and word column costs TX x (SHF + LOP3) and no load at all; a node that changes row reloads TX+1 words
//   (odd row stride: the 32 lanes hit 32 different banks).
//   Program fetch: each warp loads 32 entries at a time, one per lane (one coalesced 256 B request, issued a
//   whole chunk ahead), and broadcasts them node by node with SHFL; the high word (count index, slots) is
//   fetched only by the rare entries that need it.
//   Saved masks of the depth-first walk live in LOCAL memory (saves/restores are ~2.6 % of the nodes each;
//   the lines stay in L1), so the hot loop carries no stack registers and shared memory holds only the
//   bands: 4-5 CTAs per SM instead of 2 (measured: config 3 15.4 -> 11.6 ms against a shared-memory stack).
//   The kernel does not know about planes: in eroded mode shared memory holds the E2 and
//   the D2 band instead of the plain one, an entry's offset field already points into the right plane, and one
//   window then covers two path pixels.  PAIR entries fold their window into the next entry's 3-input AND.
//   The mask of an item is initialised once, before the loop (INIT is only ever an item's first entry).
// ---------------------------------------------------------------------------------------------
template <int TX, int TY, bool PRUNE>
__global__ void __launch_bounds__(256) eval_kernel_v3(const EvalParams p) {
  constexpr int T = TX * TY;
  constexpr unsigned FULL = 0xffffffffu;
  extern __shared__ __align__(128) uint32_t smem[];
  __shared__ __align__(8) uint64_t bar;
  __shared__ unsigned int s_work;

  const Geom& g = p.g;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int img_local = warp / g.wpi;
  const int ww = warp - img_local * g.wpi;
  const int strip_l = ww % g.SB, rblk = ww / g.SB;
  const int row0 = rblk * 32 * TY + lane;               // band-local start row of ty = 0
  uint32_t stk[STACK_SLOTS_BUDGET * T];

  uint32_t M[T];
  uint32_t R[TY][TX + 1];

  if (tid == 0) {
    mbar_init(&bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  unsigned parity = 0;
  const unsigned total_work = (unsigned)p.n_work * (unsigned)p.n_gp;
  const int groups_per_plane = p.Bpad / g.G;

  for (;;) {
    if (tid == 0) s_work = atomicAdd(p.counter, 1u);
    __syncthreads();                 // everybody is also done reading the previous band
    const unsigned work = s_work;
    if (work >= total_work) break;
    const int wi = (int)(work / (unsigned)p.n_gp);          // big items first, over all groups
    const int gp = (int)(work - (unsigned)wi * (unsigned)p.n_gp);
    const int plane = gp / groups_per_plane;
    const int b0 = (gp - plane * groups_per_plane) * g.G;
    const int4 wk = __ldg(p.work + wi);
    const int o = wk.z & 15, sband = wk.z >> 4, band = wk.w;
    const ViewGeom& v = g.v[o];
    const int stride = v.stride;
    if (tid == 0) {
      const unsigned bytes = (unsigned)v.band_words * 4u;
      mbar_expect_tx(&bar, bytes * (unsigned)g.G * (v.e2_band_off ? 2u : 1u));
      const uint32_t* src = p.packed + (size_t)plane * g.plane_words + v.packed_off + (size_t)b0 * v.view_words +
                            (size_t)band * g.band_rows * stride;
      for (int gi = 0; gi < g.G; ++gi) {
        if (v.e2_band_off) {        // eroded mode: shared memory holds the E2 and the D2 band, the plain view stays in HBM
          tma_bulk_g2s(smem + (size_t)gi * v.band_pitch, src + (size_t)gi * v.view_words + v.e2_view_off, bytes, &bar);
          tma_bulk_g2s(smem + (size_t)gi * v.band_pitch + v.e2_band_off,
                       src + (size_t)gi * v.view_words + 2 * (size_t)v.e2_view_off, bytes, &bar);
        } else {
          tma_bulk_g2s(smem + (size_t)gi * v.band_pitch, src + (size_t)gi * v.view_words, bytes, &bar);
        }
      }
    }
    // per-item thread geometry (the octant decides the view size)
    const int strip = sband * g.SB + strip_l;
    const bool active = strip < v.n_strips;
    const char* base =
        (const char*)(smem + (size_t)img_local * v.band_pitch + row0 * stride + (active ? strip : 0) * TX);
    const int rowstep = 32 * stride * 4;                     // bytes between the TY start rows of a thread
    const int b_img = b0 + img_local;
    unsigned long long* cnt = p.counts + (size_t)b_img * p.image_stride + (size_t)plane * p.S * p.S;
    const bool store = (lane == 0) && (b_img < p.B);
    mbar_wait(&bar, parity);
    parity ^= 1u;
    __syncthreads();                 // s_work may be rewritten only after everyone has read it

    int e = wk.x;
    const int e1 = e + wk.y;
    uint2 cur = __ldg(p.entries + e + lane);                 // the entry array is padded by 64
    // Every item begins with its only INIT entry: the parent mask is "every valid start pixel" (of the selected ones
    // for L2~; in eroded mode AND the plain word of the start pixels themselves, i.e. the root pixel, from HBM).
#pragma unroll
    for (int ty = 0; ty < TY; ++ty) {
      const bool rowok = active && (band * g.band_rows + row0 + ty * 32 < v.Hv);
#pragma unroll
      for (int t = 0; t < TX; ++t) {
        const int nb = v.Wv - 32 * (strip * TX + t);         // start pixels x' < Wv only
        const uint32_t cm = nb >= 32 ? 0xffffffffu : (nb <= 0 ? 0u : ((1u << nb) - 1u));
        M[ty * TX + t] = rowok ? cm : 0u;
      }
      if (v.e2_band_off && rowok) {
        const uint32_t* pw = p.packed + (size_t)plane * g.plane_words + v.packed_off + (size_t)b_img * v.view_words +
                             (size_t)(band * g.band_rows + row0 + ty * 32) * stride + strip * TX;
#pragma unroll
        for (int t = 0; t < TX; ++t) M[ty * TX + t] &= __ldg(pw + t);
      }
      if (p.mask != nullptr && rowok) {                      // L2~: only the selected start pixels
        const uint32_t* mw =
            p.mask + p.mask_off[o] + (size_t)(band * g.band_rows + row0 + ty * 32) * stride + strip * TX;
#pragma unroll
        for (int t = 0; t < TX; ++t) M[ty * TX + t] &= __ldg(mw + t);
      }
    }
    if (__shfl_sync(FULL, cur.y, 0) & E_ROOTCOUNT_HI) {      // eroded mode has no entry for the root: v = 0 is counted here
      int c = 0;
#pragma unroll
      for (int t = 0; t < T; ++t) c += __popc(M[t]);
      c = __reduce_add_sync(FULL, c);
      if (c != 0 && store) atomicAdd(cnt + (size_t)(p.S / 2) * p.S + p.S / 2, (unsigned long long)c);
    }
    while (e < e1) {
      const uint2 nxt = __ldg(p.entries + e + 32 + lane);
      const int n = min(32, e1 - e);
      int jump = -1;
      uint32_t x = __shfl_sync(FULL, cur.x, 0);
#pragma unroll 1
      for (int i = 0; i < n; ++i) {
        uint32_t xn = __shfl_sync(FULL, cur.x, i + 1);
        if (x & E_RESTORE) {
          const uint32_t y = __shfl_sync(FULL, cur.y, i);
          const uint32_t* s = stk + ((y >> E_RSLOT_SHIFT) & E_SLOT_MASK) * T;
#pragma unroll
          for (int t = 0; t < T; ++t) M[t] = s[t];
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
          xn = __shfl_sync(FULL, cur.x, i + 1);
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
            uint32_t* s = stk + ((y >> E_SSLOT_SHIFT) & E_SLOT_MASK) * T;
#pragma unroll
            for (int t = 0; t < T; ++t) s[t] = M[t];
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

typedef void (*eval_fn)(const EvalParams);
static eval_fn eval_fn_for(int TX, int TY, bool prune) {
#define LPF_PICK(tx, ty) \
  if (TX == tx && TY == ty) return prune ? eval_kernel_v3<tx, ty, true> : eval_kernel_v3<tx, ty, false>;
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
__global__ void mirror_kernel(unsigned long long* counts, int S, long long n_arrays) {
  const int m = S / 2;
  const long long K = (long long)S * S;
  const long long total = n_arrays * K;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total;
       i += (long long)gridDim.x * blockDim.x) {
    const long long arr = i / K;
    const int k = (int)(i - arr * K);
    const int dy = k / S - m, dx = k % S - m;
    if (!(dy > 0 || (dy == 0 && dx >= 0))) counts[i] = counts[arr * K + (K - 1 - k)];
  }
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
// swap delta, version 3.
//   For one proposal let u be the pixel whose bit becomes 1 and w the one whose bit becomes 0:
//     delta(v) = #{segments of vector v that contain u and lie in phase in I'}
//              - #{segments of vector v that contain w and lie in phase in I }
//   A segment of v that has pixel px at path position k starts at s = px - P_v[k]; P_v[0..k] is a trie node N, so
//   the candidates are exactly the pairs (trie node N, terminal D in the subtree of N) with start s_N = px - o_N.
//   (A) lane per node N: the prefix root -> N must be in phase from s_N.  The parent's pixel is one of the 8
//       neighbours of px (register mask lookup: most nodes stop there); the other ancestors' pixels are stepped
//       backwards with Bresenham error arithmetic on a vector that runs through N -- no loads but the image bits.
//   (B) the subtree of every surviving (N, start) is explored by the whole warp from a per-warp stack in shared
//       memory: a lane pops one node, tests its pixel, counts it if it is a terminal, and pushes its next sibling
//       (always) and its first child (if the pixel is in phase).  A dead prefix kills every vector below it at once.
//   CTA = SW proposals (node records are fetched once for all of them); image bits in shared memory.
//   delta must be zero on entry; only the canonical half is written (swap_mirror_kernel fills the rest).
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

constexpr int SWAP_SW = 8;          // proposals per CTA
constexpr int SWAP_STACK = 512;     // items per warp stack (8 bytes each)

__device__ __forceinline__ int wrap_coord(int x, int n) {
  x += (x < 0) ? n : 0;
  x -= (x >= n) ? n : 0;
  return x;
}

struct SwapPass {                   // one (proposal, pixel) pass, in shared memory
  int px, py;                       // the swapped pixel the segments must contain
  int ox, oy;                       // pixel that reads as out of phase in this pass (w in I'), or -1
  unsigned nb;                      // in-phase bits of the 8 neighbours px - step, by step code
  int sign;                         // +1: u on I', -1: w on I
  int pbase;                        // word offset of this pass's phase plane in the shared-memory bit images
  long long out_off;                // offset of this pass's [S][S] delta array from the CTA's first one
};

__global__ void __launch_bounds__(256) swap_delta_kernel_v3(const uint32_t* __restrict__ bits, int H, int W, int m,
                                                             const int* __restrict__ pairs, long long n,
                                                             const int4* __restrict__ rec, int n_nodes,
                                                             int* __restrict__ delta, int n_planes,
                                                             long long plane_stride) {
  extern __shared__ __align__(16) uint32_t sm[];
  __shared__ SwapPass s_pass[4 * SWAP_SW];                            // (proposal, phase plane, pixel)
  __shared__ int s_n;
  const int PWc = (W + 2 * m + 31) >> 5, PH = H + 2 * m;                // padded bit image: halo of m pixels all round
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  uint32_t* P = sm;                                                   // [n_planes][PH][PWc] bits of the base image I
  const int plane_words = PH * PWc;
  uint2* stk = (uint2*)(sm + ((n_planes * plane_words + 1) & ~1)) + (size_t)warp * SWAP_STACK;
  // pixel (x, y) of the plane at Pq, x in [-m, W + m), y in [-m, H + m)
  auto pbit = [&](const uint32_t* Pq, int x, int y) -> unsigned {
    const int X = x + m;
    return (Pq[(y + m) * PWc + (X >> 5)] >> (X & 31)) & 1u;
  };
  const int S = 2 * m + 1;
  const long long K = (long long)S * S;
  for (int i = tid; i < n_planes * plane_words; i += blockDim.x) P[i] = bits[i];
  __syncthreads();
  if (tid == 0) {
    int cnt = 0;
    for (int j = 0; j < SWAP_SW; ++j) {
      const long long sw = (long long)blockIdx.x * SWAP_SW + j;
      if (sw >= n) break;
      const int xp = pairs[4 * sw], yp = pairs[4 * sw + 1], xq = pairs[4 * sw + 2], yq = pairs[4 * sw + 3];
      const bool ok = xp >= 0 && xp < W && xq >= 0 && xq < W && yp >= 0 && yp < H && yq >= 0 && yq < H;
      if (!ok) continue;
      for (int pl = 0; pl < n_planes; ++pl) {
        const uint32_t* Pq = P + pl * plane_words;
        const int bp = (int)pbit(Pq, xp, yp), bq = (int)pbit(Pq, xq, yq);
        if (bp == bq) continue;                            // nothing changes for this phase
        const int ux = bp ? xq : xp, uy = bp ? yq : yp;    // bit 0 -> 1
        const int wx = bp ? xp : xq, wy = bp ? yp : yq;    // bit 1 -> 0
        for (int pass = 0; pass < 2; ++pass) {
          SwapPass sp;
          sp.px = pass ? wx : ux; sp.py = pass ? wy : uy;
          sp.ox = pass ? -1 : wx; sp.oy = pass ? -1 : wy;
          sp.nb = 0;
          for (int code = 0; code < 9; ++code) {
            const int x = wrap_coord(sp.px - (code / 3 - 1), W), y = wrap_coord(sp.py - (code % 3 - 1), H);
            unsigned bit = pbit(Pq, x, y);
            if (x == sp.ox && y == sp.oy) bit = 0;
            sp.nb |= bit << code;
          }
          sp.sign = pass ? -1 : 1;
          sp.pbase = pl * plane_words;
          sp.out_off = (long long)pl * plane_stride + (long long)j * K;
          s_pass[cnt++] = sp;
        }
      }
    }
    s_n = cnt;
  }
  __syncthreads();
  const int np = s_n;
  if (np == 0) return;
  int* const out0 = delta + (long long)blockIdx.x * SWAP_SW * K;
  const unsigned lt = (1u << lane) - 1u;
  int top = 0;                                             // warp-uniform: items on this warp's stack

  // blockIdx.y slices the node range, so that a small batch of proposals still fills the chip
  const int slice = (n_nodes + gridDim.y - 1) / gridDim.y;
  const int n_begin = blockIdx.y * slice, n_end = min(n_nodes, n_begin + slice);
  for (int N0 = n_begin + warp * 32; N0 < n_end; N0 += blockDim.x) {
    const int N = N0 + lane;
    int4 rN = make_int4(0, 0, 0, 0);
    if (N < n_end) rN = __ldg(rec + N);
    const int oNx = (short)(rN.x & 0xffff), oNy = rN.x >> 16;
    const int codeN = (rN.w >> 20) & 15;
    const int d = max(abs(oNx), abs(oNy));                 // depth of N
    // Bresenham state of the representative vector at position d (reading D2, closed form)
    const int vx = (short)(rN.y & 0xffff), vy = rN.y >> 16;
    const int ax = abs(vx), ay = abs(vy);
    const bool xmaj = ax >= ay;
    const int nn = xmaj ? ax : ay, mn = xmaj ? ay : ax;
    const int sxs = (vx > 0) - (vx < 0), sys = (vy > 0) - (vy < 0);
    const int q0 = xmaj ? abs(oNy) : abs(oNx);
    const int e0 = 2 * d * mn + nn - 2 * nn * q0;
    for (int q = 0; q < np; ++q) {
      const unsigned nb = s_pass[q].nb;
      const uint32_t* Pq = P + s_pass[q].pbase;
      bool alive = (N < n_end) && (d == 0 || ((nb >> codeN) & 1u));
      if (__any_sync(0xffffffffu, alive)) {                // (not so: typical for u, an isolated pixel kills all 32 at once)
      const int ox = s_pass[q].ox, oy = s_pass[q].oy;
      const int sx = wrap_coord(s_pass[q].px - oNx, W), sy = wrap_coord(s_pass[q].py - oNy, H);
      if (alive && d >= 2)                                 // the far end first: a long prefix usually dies at its start
        alive = pbit(Pq, sx, sy) && !(sx == ox && sy == oy);
      if (alive) {
        // (A) ancestors at positions d-2 .. 1 (d-1 was the neighbour test, 0 the start), stepping the error term backwards
        int e = e0, qq = q0;
        if (ox < 0) {
          // fast walk (the w pass on I: nothing to mask): one linear bit index into the padded image, no modulo
          const int PW = PWc * 32;
          const int dmaj = xmaj ? sxs : sys * PW, dmin = xmaj ? sys * PW : sxs;
          int L = (sy + m + oNy) * PW + (sx + m + oNx);      // pixel px itself (position d)
          for (int k = d - 1; k >= 1; --k) {
            e -= 2 * mn;
            L -= dmaj;
            if (e < 0) { e += 2 * nn; L -= dmin; }
            if (k == d - 1) continue;
            if (!((Pq[L >> 5] >> (L & 31)) & 1u)) { alive = false; break; }
          }
        } else {
          for (int k = d - 1; k >= 1; --k) {
            e -= 2 * mn;
            if (e < 0) { e += 2 * nn; --qq; }
            if (k == d - 1) continue;
            const int ax_ = xmaj ? sxs * k : sxs * qq, ay_ = xmaj ? sys * qq : sys * k;
            const int x = wrap_coord(sx + ax_, W), y = wrap_coord(sy + ay_, H);
            if (!pbit(Pq, x, y) || (x == ox && y == oy)) { alive = false; break; }
          }
        }
      }
      int* const out = out0 + s_pass[q].out_off;
      const int sign = s_pass[q].sign;
      if (alive && (rN.w & 0xFFFFF) != 0xFFFFF) atomicAdd(out + (rN.w & 0xFFFFF), sign);
      // (B) push the first child of every survivor, then drain the warp stack
      const bool push = alive && rN.z > 1;
      const unsigned pm = __ballot_sync(0xffffffffu, push);
      if (push)
        stk[top + __popc(pm & lt)] =
            make_uint2((unsigned)(N + 1) | ((unsigned)q << 24), (unsigned)sx | ((unsigned)sy << 16));
      top += __popc(pm);
      __syncwarp();
      }
      // the survivors of all passes are explored together (the depth of the live region is paid once, not once
      // per pass); the stack is drained early only when the next 32 pushes might not fit
      if (top <= SWAP_STACK - 32 && q + 1 < np) continue;
      while (top > 0) {
        const int take = min(top, 32);
        uint2 it = make_uint2(0, 0);
        if (lane < take) it = stk[top - 1 - lane];
        top -= take;
        __syncwarp();
        bool p_sib = false, p_child = false;
        int i = 0;
        if (lane < take) {
          i = (int)(it.x & 0xFFFFFF);
          const int qi = (int)(it.x >> 24);
          const int4 r = __ldg(rec + i);
          const int isx = (int)(it.y & 0xffff), isy = (int)(it.y >> 16);
          const int x = wrap_coord(isx + (short)(r.x & 0xffff), W), y = wrap_coord(isy + (r.x >> 16), H);
          const bool in = pbit(P + s_pass[qi].pbase, x, y) && !(x == s_pass[qi].ox && y == s_pass[qi].oy);
          if (in && (r.w & 0xFFFFF) != 0xFFFFF)
            atomicAdd(out0 + s_pass[qi].out_off + (r.w & 0xFFFFF), s_pass[qi].sign);
          p_sib = (r.w >> 24) & 1;
          p_child = in && r.z > 1;
          if (p_sib) it.x += (unsigned)r.z;                // next sibling = i + subtree size
        }
        const unsigned ms = __ballot_sync(0xffffffffu, p_sib);
        const unsigned mc = __ballot_sync(0xffffffffu, p_child);
        const int ns = __popc(ms), nc = __popc(mc);
        if (top + ns + nc > SWAP_STACK) {
          // the stack cannot take this batch: every lane walks its own item's remainder serially (rare)
          if (lane < take) {
            const int qi = (int)(it.x >> 24);                // it.x may already point at the sibling: undo
            const int isx = (int)(it.y & 0xffff), isy = (int)(it.y >> 16);
            const int4 r0 = __ldg(rec + i);
            // serial preorder scan of: the subtree of i below i (if in phase), then all later siblings' subtrees
            int j = p_child ? i + 1 : i + r0.z;
            // end of the scan: the parent's subtree end is unknown here, so follow sibling flags
            bool more = true;
            int cur_top = i;                                  // the sibling-level node whose subtree is scanned
            int4 rt = r0;
            while (more) {
              const int end = cur_top + rt.z;
              while (j < end) {
                const int4 r = __ldg(rec + j);
                const int x = wrap_coord(isx + (short)(r.x & 0xffff), W), y = wrap_coord(isy + (r.x >> 16), H);
                const bool in = pbit(P + s_pass[qi].pbase, x, y) &&
                                !(x == s_pass[qi].ox && y == s_pass[qi].oy);
                if (in) {
                  if ((r.w & 0xFFFFF) != 0xFFFFF)
                    atomicAdd(out0 + s_pass[qi].out_off + (r.w & 0xFFFFF), s_pass[qi].sign);
                  ++j;
                } else {
                  j += r.z;
                }
              }
              more = (rt.w >> 24) & 1;
              if (more) {                                     // move to the next sibling: test it like any node
                cur_top = end;
                rt = __ldg(rec + cur_top);
                const int x = wrap_coord(isx + (short)(rt.x & 0xffff), W), y = wrap_coord(isy + (rt.x >> 16), H);
                const bool in = pbit(P + s_pass[qi].pbase, x, y) &&
                                !(x == s_pass[qi].ox && y == s_pass[qi].oy);
                if (in && (rt.w & 0xFFFFF) != 0xFFFFF)
                  atomicAdd(out0 + s_pass[qi].out_off + (rt.w & 0xFFFFF), s_pass[qi].sign);
                j = in ? cur_top + 1 : cur_top + rt.z;
              }
            }
          }
        } else {
          if (p_sib) stk[top + __popc(ms & lt)] = it;
          if (p_child) stk[top + ns + __popc(mc & lt)] = make_uint2((unsigned)(i + 1) | (it.x & 0xFF000000u), it.y);
          top += ns + nc;
        }
        __syncwarp();
      }
    }
  }
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
  const int np = g.v[0].e2_view_off > 0 ? 3 : 1;
  int tl[4], stride_max = 0;
  long long per_plane = 0;
  for (int o = 0; o < 4; ++o) {
    tl[o] = (g.v[o].view_words / np + PACK_TILE - 1) / PACK_TILE;
    per_plane += (long long)Bpad * tl[o];
    stride_max = std::max(stride_max, g.v[o].stride);
  }
  if (per_plane * n_phase >= (1ll << 31)) return cudaErrorInvalidValue;
  pack_views_kernel<<<(unsigned)(per_plane * n_phase), 256, (size_t)(PACK_TILE + stride_max + 2) * 4, st>>>(
      base, packed, g, B, Bpad, make_int4(tl[0], tl[1], tl[2], tl[3]), per_plane);
  return cudaGetLastError();
}

// also raises the kernel's dynamic shared memory limit to the device maximum (once is enough, repeating is harmless),
// so that launches of any plan fit whatever order the plans were made in
cudaError_t eval_occupancy(int TX, int TY, bool prune, int threads, size_t smem, int max_smem, int* blocks_per_sm) {
  eval_fn f = eval_fn_for(TX, TY, prune);
  if (!f) return cudaErrorInvalidValue;
  cudaFuncAttributes fa;
  cudaError_t e = cudaFuncGetAttributes(&fa, f);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem - (int)fa.sharedSizeBytes);
  if (e != cudaSuccess) return e;
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_per_sm, f, threads, smem);
}

cudaError_t launch_eval(const EvalParams& p, int grid, int threads, size_t smem, cudaStream_t st) {
  eval_fn f = eval_fn_for(p.g.TX, p.g.TY, p.prune != 0);
  if (!f) return cudaErrorInvalidValue;
  f<<<grid, threads, smem, st>>>(p);
  return cudaGetLastError();
}

cudaError_t launch_mirror(unsigned long long* counts, int S, long long n_arrays, int n_sm, cudaStream_t st) {
  const long long total = n_arrays * S * S;
  long long blocks = (total + 255) / 256;
  if (blocks > (long long)n_sm * 8) blocks = (long long)n_sm * 8;
  mirror_kernel<<<(unsigned)blocks, 256, 0, st>>>(counts, S, n_arrays);
  return cudaGetLastError();
}

cudaError_t launch_objective(const long long* counts, const long long* target, int B, long long K,
                             unsigned long long* sse, int n_sm, cudaStream_t st) {
  cudaError_t e = cudaMemsetAsync(sse, 0, sizeof(unsigned long long) * (size_t)B, st);
  if (e != cudaSuccess) return e;
  long long chunks = (K + 256 * 8 - 1) / (256 * 8);
  const long long want = ((long long)n_sm * 8 + B - 1) / B;     // enough blocks to fill the chip
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

// phase 0 | 1: one plane, delta [n][S][S];  phase < 0: both planes, phase k at delta + k * plane_stride
cudaError_t launch_swap_delta(const uint8_t* image, uint32_t* bits, int H, int W, int m, int phase, const int* pairs,
                              long long n, const int32_t* rec, int n_nodes, int* delta, long long plane_stride,
                              unsigned int* counter, int n_sm, cudaStream_t st) {
  const int n_planes = phase < 0 ? 2 : 1;
  const int Wc = (W + 31) / 32, Hc = (H + 31) / 32;
  const int PWc = (W + 2 * m + 31) / 32, PH = H + 2 * m;
  const size_t smem = (size_t)((n_planes * PH * PWc + 1) & ~1) * 4 + (size_t)8 * SWAP_STACK * 8;
  const long long img_words = (long long)H * Wc + (long long)W * Hc;
  uint32_t* const padded = bits + (size_t)n_planes * img_words;
  cudaError_t e = cudaSuccess;
  const long long S2 = (long long)(2 * m + 1) * (2 * m + 1);
  for (int pl = 0; pl < n_planes; ++pl) {
    e = cudaMemsetAsync(delta + pl * plane_stride, 0, sizeof(int) * (size_t)n * S2, st);
    if (e != cudaSuccess) return e;
  }
  // stage 1 of the bit-pack gives the row-major bit image(s) of the base image (the column-major half is unused)
  pack_base_kernel<<<(unsigned)std::max(1, (Hc * Wc + 7) / 8), 256, 0, st>>>(image, bits, 1, H, W, n_planes,
                                                                             phase < 0 ? 0 : phase, counter);
  pack_padded_kernel<<<dim3((unsigned)std::max(1, std::min((PH * PWc + 255) / 256, n_sm * 8)), (unsigned)n_planes), 256,
                       0, st>>>(bits, padded, H, W, m, img_words);
  const long long ctas = (n + SWAP_SW - 1) / SWAP_SW;
  for (long long c0 = 0; c0 < ctas; c0 += (1ll << 30)) {
    const long long cnt = std::min(ctas - c0, 1ll << 30);
    const long long s0 = c0 * SWAP_SW;
    // node slices: about two CTAs per SM in total, at least 256 nodes per slice
    const int slices =
        (int)std::max(1ll, std::min<long long>({(2ll * n_sm + cnt - 1) / cnt, (n_nodes + 255) / 256, 65535ll}));
    swap_delta_kernel_v3<<<dim3((unsigned)cnt, (unsigned)slices), 256, smem, st>>>(
        padded, H, W, m, pairs + 4 * s0, n - s0, (const int4*)rec, n_nodes, delta + s0 * S2, n_planes, plane_stride);
  }
  const long long blocks = std::max(1ll, std::min<long long>((n * (S2 / 2) + 255) / 256, (long long)n_sm * 16));
  for (int pl = 0; pl < n_planes; ++pl)
    swap_mirror_kernel<<<(unsigned)blocks, 256, 0, st>>>(delta + pl * plane_stride, 2 * m + 1, n);
  return cudaGetLastError();
}

}  // namespace lpf
