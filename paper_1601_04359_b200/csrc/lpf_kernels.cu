// lpf_kernels.cu -- CUDA kernels of liblpf.so (sm_100a).
//   pack_base_kernel  uint8 image -> row-major and column-major bit images, 32 px / word, one coalesced pass
//   pack_views_kernel the four octant views per image, each with its periodic halo laid out exactly as the
//                     eval kernel wants it in shared memory (a2)
//   eval_kernel_v3<.> the hot loop: walk the node program with a running AND mask (a3), POPC +
//                     warp reduce at terminals (a4), optional zero-mask pruning (a5)
//   mirror_kernel     counts[-v] = counts[v] (a6)
//   objective_kernel  sum (c - t)^2 per image (a8, Eq. 14/19)
//   swap_delta_kernel per-proposal count deltas (a9)
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
      const bool b0 = n_phase == 2 ? (v == 0) : (v == phase0);
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

// ---------------------------------------------------------------------------------------------
// bit-pack, stage 2: the four octant views with their periodic halo, one thread per output word.
//   view o of image I (lpf_internal.h): 0: I[y'][x']  1: I[x'][y']  2: I[x'][-y' mod W]  3: I[y'][-x' mod W]
//   word (r, i) of a view holds x' = (32 i + k) mod Wv, y' = r mod Hv.  Views 0 and 3 read Brow, views 1 and 2
//   read Bcol; a word whose 32 pixels do not wrap is one funnel shift of two base words (view 3: of the
//   bit-reversed pair), the others are gathered bit by bit.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) pack_views_kernel(const uint32_t* __restrict__ base,
                                                         uint32_t* __restrict__ packed, Geom g, int B, int n_phase) {
  const int Wc = (g.W + 31) >> 5, Hc = (g.H + 31) >> 5;
  const long long img_words = (long long)g.H * Wc + (long long)g.W * Hc;
  const long long total = (long long)n_phase * g.plane_words;
  for (long long w = (long long)blockIdx.x * blockDim.x + threadIdx.x; w < total;
       w += (long long)gridDim.x * blockDim.x) {
    const int plane = (int)(w / g.plane_words);
    const long long wp = w - (long long)plane * g.plane_words;
    int o = 0;
#pragma unroll
    for (int k = 1; k < 4; ++k)
      if (wp >= g.v[k].packed_off) o = k;
    const ViewGeom& v = g.v[o];
    const long long rem = wp - v.packed_off;
    const int b = (int)(rem / v.view_words);
    const int idx = (int)(rem - (long long)b * v.view_words);
    const int r = idx / v.stride, i = idx - r * v.stride;
    const int rows = v.n_bands * g.band_rows + g.m;
    uint32_t word = 0;
    if (b < B && r < rows) {
      const int yv = r % v.Hv;
      const int x0 = (32 * i) % v.Wv;
      const uint32_t* bimg = base + ((size_t)plane * B + b) * img_words;
      // source row of this view row: views 0, 3: image row yv (Brow); view 1: image column yv; view 2: column -yv
      const uint32_t* srow;
      int words;
      if (o == 0 || o == 3) { srow = bimg + (size_t)yv * Wc; words = Wc; }
      else {
        const int c = (o == 1) ? yv : (yv ? g.W - yv : 0);
        srow = bimg + (size_t)g.H * Wc + (size_t)c * Hc;
        words = Hc;
      }
      if (o != 3) {
        if (x0 + 32 <= v.Wv) word = window32(srow, words, x0);
        else
          for (int k = 0; k < 32; ++k) {
            const int xs = (x0 + k) % v.Wv;
            word |= ((srow[xs >> 5] >> (xs & 31)) & 1u) << k;
          }
      } else {
        // bit k = source bit (Wv - x0 - k) mod Wv: for 1 <= x0 and x0 + 31 <= Wv the sources are the 32
        // consecutive pixels Wv - x0 - 31 .. Wv - x0 in descending order
        if (x0 >= 1 && x0 + 31 <= v.Wv) word = __brev(window32(srow, words, v.Wv - x0 - 31));
        else
          for (int k = 0; k < 32; ++k) {
            const int xv = (x0 + k) % v.Wv;
            const int xs = xv ? v.Wv - xv : 0;
            word |= ((srow[xs >> 5] >> (xs & 31)) & 1u) << k;
          }
      }
    }
    packed[w] = word;
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
      mbar_expect_tx(&bar, bytes * (unsigned)g.G);
      const uint32_t* src = p.packed + (size_t)plane * g.plane_words + v.packed_off + (size_t)b0 * v.view_words +
                            (size_t)band * g.band_rows * stride;
      for (int gi = 0; gi < g.G; ++gi)
        tma_bulk_g2s(smem + (size_t)gi * v.band_words, src + (size_t)gi * v.view_words, bytes, &bar);
    }
    // per-item thread geometry (the octant decides the view size)
    const int strip = sband * g.SB + strip_l;
    const bool active = strip < v.n_strips;
    const char* base =
        (const char*)(smem + (size_t)img_local * v.band_words + row0 * stride + (active ? strip : 0) * TX);
    const int rowstep = 32 * stride * 4;                     // bytes between the TY start rows of a thread
    const int b_img = b0 + img_local;
    unsigned long long* cnt = p.counts + ((size_t)b_img * p.n_phase + plane) * (size_t)p.S * p.S;
    const bool store = (lane == 0) && (b_img < p.B);
    mbar_wait(&bar, parity);
    parity ^= 1u;
    __syncthreads();                 // s_work may be rewritten only after everyone has read it

    int e = wk.x;
    const int e1 = e + wk.y;
    uint2 cur = __ldg(p.entries + e + lane);                 // the entry array is padded by 64
    while (e < e1) {
      const uint2 nxt = __ldg(p.entries + e + 32 + lane);
      const int n = min(32, e1 - e);
      int jump = -1;
      uint32_t x = __shfl_sync(FULL, cur.x, 0);
#pragma unroll 1
      for (int i = 0; i < n; ++i) {
        uint32_t xn = __shfl_sync(FULL, cur.x, i + 1);
        if (x & (E_INIT | E_RESTORE)) {
          if (x & E_INIT) {
#pragma unroll
            for (int ty = 0; ty < TY; ++ty) {
              const bool rowok = active && (band * g.band_rows + row0 + ty * 32 < v.Hv);
#pragma unroll
              for (int t = 0; t < TX; ++t) {
                const int nb = v.Wv - 32 * (strip * TX + t);   // start pixels x' < Wv only
                const uint32_t cm = nb >= 32 ? 0xffffffffu : (nb <= 0 ? 0u : ((1u << nb) - 1u));
                M[ty * TX + t] = rowok ? cm : 0u;
              }
            }
          } else {
            const uint32_t y = __shfl_sync(FULL, cur.y, i);
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
// swap delta, version 1.  One CTA per proposal.
//   Bit plane Bp of the base image in shared memory (no halo, modular addressing), and a second
//   copy Bq with the two bits exchanged.  If the two bits are equal nothing changes.  Otherwise let
//   u be the pixel whose bit becomes 1 and w the one whose bit becomes 0:
//     delta(v) = #{k : segment started at u - P_v[k] lies in phase in I'}   (it contains u)
//              - #{k : segment started at w - P_v[k] lies in phase in I }   (it contains w)
//   Warp per vector of D, lane per candidate k; the other half is the mirror delta(-v) = delta(v).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ bool seg_in_phase(const uint32_t* plane, int Wc, int H, int W, const short2* path,
                                             int len, int sx, int sy) {
  for (int jx = 0; jx < len; ++jx) {
    const short2 o = path[jx];
    int x = sx + o.x, y = sy + o.y;
    x += (x < 0) ? W : 0;
    x -= (x >= W) ? W : 0;
    y += (y < 0) ? H : 0;
    y -= (y >= H) ? H : 0;
    if (!((plane[y * Wc + (x >> 5)] >> (x & 31)) & 1u)) return false;
  }
  return true;
}

__global__ void __launch_bounds__(256) swap_delta_kernel_v1(const uint8_t* __restrict__ image, int H, int W, int m,
                                                             int phase, const int* __restrict__ pairs,
                                                             const short2* __restrict__ path_xy,
                                                             const int* __restrict__ path_off,
                                                             const short2* __restrict__ vecs, int n_half,
                                                             int* __restrict__ delta) {
  extern __shared__ __align__(16) uint32_t sm[];
  const int Wc = (W + 31) >> 5;
  uint32_t* P0 = sm;                  // base image plane
  uint32_t* P1 = sm + H * Wc;         // plane after the swap
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nw = blockDim.x >> 5;
  const long long sw = blockIdx.x;
  const int S = 2 * m + 1;
  int* out = delta + sw * (long long)S * S;
  const int xp = pairs[4 * sw], yp = pairs[4 * sw + 1], xq = pairs[4 * sw + 2], yq = pairs[4 * sw + 3];
  const bool ok = xp >= 0 && xp < W && xq >= 0 && xq < W && yp >= 0 && yp < H && yq >= 0 && yq < H;
  for (int w = warp; w < H * Wc; w += nw) {
    const int y = w / Wc, x = (w - y * Wc) * 32 + lane;
    const bool bit = (x < W) && image[(size_t)y * W + x] == (uint8_t)phase;
    const unsigned v = __ballot_sync(0xffffffffu, bit);
    if (lane == 0) { P0[w] = v; P1[w] = v; }
  }
  __syncthreads();
  int bp = 0, bq = 0;
  if (ok) {
    bp = (P0[yp * Wc + (xp >> 5)] >> (xp & 31)) & 1;
    bq = (P0[yq * Wc + (xq >> 5)] >> (xq & 31)) & 1;
  }
  if (!ok || bp == bq) {              // nothing changes for this phase
    for (int k = tid; k < S * S; k += blockDim.x) out[k] = 0;
    return;
  }
  __syncthreads();
  if (tid == 0) {                     // exchange the two bits in P1
    P1[yp * Wc + (xp >> 5)] ^= 1u << (xp & 31);
    P1[yq * Wc + (xq >> 5)] ^= 1u << (xq & 31);
  }
  __syncthreads();
  const int ux = bp ? xq : xp, uy = bp ? yq : yp;   // bit 0 -> 1
  const int wx = bp ? xp : xq, wy = bp ? yp : yq;   // bit 1 -> 0
  for (int v = warp; v < n_half; v += nw) {
    const int off = path_off[v], len = path_off[v + 1] - off;
    const short2* path = path_xy + off;
    int d = 0;
    for (int c = lane; c < 2 * len; c += 32) {
      const int k = (c < len) ? c : c - len;
      const short2 o = path[k];
      if (c < len) d += seg_in_phase(P1, Wc, H, W, path, len, ux - o.x, uy - o.y) ? 1 : 0;
      else d -= seg_in_phase(P0, Wc, H, W, path, len, wx - o.x, wy - o.y) ? 1 : 0;
    }
    d = __reduce_add_sync(0xffffffffu, d);
    if (lane == 0) {
      const short2 vv = vecs[v];
      out[(vv.y + m) * S + (vv.x + m)] = d;
      out[(-vv.y + m) * S + (-vv.x + m)] = d;
    }
  }
}

// ---------------------------------------------------------------------------------------------
// host launch wrappers (called from lpf_api.cu)
// ---------------------------------------------------------------------------------------------
cudaError_t launch_pack(const uint8_t* images, uint32_t* base, uint32_t* packed, const Geom& g, int B, int n_phase,
                        int phase0, unsigned int* counter, int n_sm, cudaStream_t st) {
  const long long tiles = (long long)B * ((g.H + 31) / 32) * ((g.W + 31) / 32);
  long long blocks = (tiles + 7) / 8;
  blocks = std::max(1ll, std::min(blocks, (long long)n_sm * 16));
  pack_base_kernel<<<(unsigned)blocks, 256, 0, st>>>(images, base, B, g.H, g.W, n_phase, phase0, counter);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  const long long total = (long long)n_phase * g.plane_words;
  blocks = (total + 255) / 256;
  blocks = std::max(1ll, std::min(blocks, (long long)n_sm * 32));
  pack_views_kernel<<<(unsigned)blocks, 256, 0, st>>>(base, packed, g, B, n_phase);
  return cudaGetLastError();
}

cudaError_t eval_occupancy(int TX, int TY, bool prune, int threads, size_t smem, int* blocks_per_sm) {
  eval_fn f = eval_fn_for(TX, TY, prune);
  if (!f) return cudaErrorInvalidValue;
  cudaError_t e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
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

cudaError_t launch_swap_delta(const uint8_t* image, int H, int W, int m, int phase, const int* pairs, long long n,
                              const int16_t* path_xy, const int* path_off, const int16_t* vecs, int n_half,
                              int* delta, cudaStream_t st) {
  const size_t smem = (size_t)2 * H * ((W + 31) / 32) * 4;
  cudaError_t e = cudaFuncSetAttribute(swap_delta_kernel_v1, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  const long long S2 = (long long)(2 * m + 1) * (2 * m + 1);
  for (long long s0 = 0; s0 < n; s0 += (1ll << 30)) {
    const long long cnt = (n - s0 < (1ll << 30)) ? (n - s0) : (1ll << 30);
    swap_delta_kernel_v1<<<(unsigned)cnt, 256, smem, st>>>(image, H, W, m, phase, pairs + 4 * s0,
                                                          (const short2*)path_xy, path_off, (const short2*)vecs,
                                                          n_half, delta + s0 * S2);
  }
  return cudaGetLastError();
}

}  // namespace lpf
