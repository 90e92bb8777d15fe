// lpf_swap.cuh -- device code of the swap-delta evaluation,
// shared by swap_delta_kernel_v3 (lpf_kernels.cu) and the persistent annealing kernel (lpf_anneal.cu).
//   For one proposal let u be the pixel whose bit becomes 1 and w the one whose bit becomes 0:
//     delta(v) = #{segments of vector v that contain u and lie in phase in I'}
//              - #{segments of vector v that contain w and lie in phase in I }
//   A segment of v that has pixel px at path position k starts at s = px - P_v[k]; P_v[0..k] is a trie node N, so
//   the candidates are exactly the pairs (trie node N, terminal D in the subtree of N) with start s_N = px - o_N.
//   (A) the prefix root -> N must be in phase from s_N.  With the REVERSED trie (lpf_paths.cpp; tables of m up to
//       about 100): the walks N -> root of all nodes, read as offsets from px, share their beginnings, so they are
//       explored depth-first from px like the subtrees of (B) -- one pixel test per distinct backward walk that is still
//       in phase; a walk that is complete for a node N makes (N, its end pixel) a survivor.  Without it (large tables):
//       lane per node N; the parent's pixel is one of the 8 neighbours of px (register mask lookup: most nodes stop
//       there), then the far end, then the other ancestors' pixels are stepped backwards with Bresenham error
//       arithmetic on a vector that runs through N -- no loads but the image bits.
//   (B) the subtrees of all surviving (N, start) are explored by the whole CTA from one stack in shared memory: a
//       thread pops one node, tests its pixel, counts it if it is a terminal, and pushes its next sibling (always)
//       and its first child (if the pixel is in phase).  A dead prefix kills every vector below it at once.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

namespace lpf {

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
  int rev;                          // (A) by the reversed trie (else by the per-node walks)
  int pbase;                        // word offset of this pass's phase plane in the shared-memory bit images
  long long out_off;                // offset of this pass's [S][S] delta array from the CTA's first one
};

struct SwapShared {                 // per-CTA scratch of swap_delta_unit
  SwapPass pass[4 * SWAP_SW];       // (proposal, phase plane, pixel)
  int n;                            // passes
  int top;                          // items on the CTA's stack (may run past its capacity: see swap_delta_unit)
};

// One unit of swap-delta work of a CTA of 256 threads: the proposals pairs[first_prop .. first_prop + sw) (those below
// n; sw <= SWAP_SW) against node slice `slice` of `n_slices` equal slices of the trie (passes on a dense phase plane,
// bit k of dense_mask, or rrec == nullptr) and against the children c of the reversed trie's root with c % n_slices ==
// slice (passes on a sparse plane).  Adds into out0 [sw][S][S]
// (canonical half only; plane k at + k * plane_stride), which must have been zeroed.
//   P    shared memory: [n_planes][H + 2m][ceil((W + 2m) / 32)] bits of the base image with its halo of m pixels
//   stk  shared memory: the CTA's stack of 8 * SWAP_STACK items (8 bytes each)
//   CHAIN: trie nodes of an only-child chain visited per pop of (B); FAST_WALK: the branch-free form of the backward walk
//   of (A).  Measured on config 5 / the annealing benchmark: the batched kernel is fastest with 3 and the branch-free
//   walk (phase 1 1.90e6 -> 2.25e6 swaps/s, phase 0 6.5e4 -> 9.9e4), the annealing chain (small units) with 2 and the
//   plain walk (1.96e4 -> 2.14e4 proposals/s; 3 nodes per pop: 2.04e4, the branch-free walk: 1.79e4).
template <int CHAIN, bool FAST_WALK>
__device__ __forceinline__ void swap_delta_unit(const uint32_t* P, uint2* stk, SwapShared& sh, int H, int W, int m,
                                                const int* __restrict__ pairs, long long n, long long first_prop,
                                                const int4* __restrict__ rec, int n_nodes,
                                                const int4* __restrict__ rrec, unsigned dense_mask,
                                                int* __restrict__ out0, int n_planes, long long plane_stride, int sw,
                                                int slice, int n_slices) {
  const int PWc = (W + 2 * m + 31) >> 5, PH = H + 2 * m;                // padded bit image: halo of m pixels all round
  const int tid = threadIdx.x, lane = tid & 31;
  const int plane_words = PH * PWc;
  // pixel (x, y) of the plane at Pq, x in [-m, W + m), y in [-m, H + m)
  auto pbit = [&](const uint32_t* Pq, int x, int y) -> unsigned {
    const int X = x + m;
    return (Pq[(y + m) * PWc + (X >> 5)] >> (X & 31)) & 1u;
  };
  const int S = 2 * m + 1;
  const long long K = (long long)S * S;
  __syncthreads();                                        // the previous unit of this CTA is finished with sh
  if (tid == 0) { sh.n = 0; sh.top = 0; }
  __syncthreads();
  // one thread per (proposal of this CTA, phase plane): its two passes (u on I', w on I) go to the next free slots
  if (tid < sw * n_planes) {
    const int j = tid / n_planes, pl = tid - j * n_planes;
    const long long swi = first_prop + j;
    if (swi < n) {
      const int xp = pairs[4 * swi], yp = pairs[4 * swi + 1], xq = pairs[4 * swi + 2], yq = pairs[4 * swi + 3];
      const bool ok = xp >= 0 && xp < W && xq >= 0 && xq < W && yp >= 0 && yp < H && yq >= 0 && yq < H;
      const uint32_t* Pq = P + pl * plane_words;
      const int bp = ok ? (int)pbit(Pq, xp, yp) : 0, bq = ok ? (int)pbit(Pq, xq, yq) : 0;
      if (bp != bq) {                                        // otherwise nothing changes for this phase
        const int ux = bp ? xq : xp, uy = bp ? yq : yp;      // bit 0 -> 1
        const int wx = bp ? xp : xq, wy = bp ? yp : yq;      // bit 1 -> 0
        const int slot = atomicAdd(&sh.n, 2);
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
          sp.rev = (rrec != nullptr) && !((dense_mask >> pl) & 1u);
          sp.pbase = pl * plane_words;
          sp.out_off = (long long)pl * plane_stride + (long long)j * K;
          sh.pass[slot + pass] = sp;
        }
      }
    }
  }
  __syncthreads();
  const int np = sh.n;
  if (np == 0) return;
  const unsigned lt = (1u << lane) - 1u;
  constexpr int CAP = 8 * SWAP_STACK;                      // the CTA's stack: the eight warp stacks as one
  constexpr unsigned DUMMY = 0xFFFFFFFFu;                  // a reserved slot that was not filled
  // test node i of pass qi from start (isx, isy): in phase?  counts it if it is a whole path
  auto visit = [&](int i, int qi, int isx, int isy, const int4& r) -> bool {
    const int x = wrap_coord(isx + (short)(r.x & 0xffff), W), y = wrap_coord(isy + (r.x >> 16), H);
    const bool in = pbit(P + sh.pass[qi].pbase, x, y) && !(x == sh.pass[qi].ox && y == sh.pass[qi].oy);
    if (in && (r.w & 0xFFFFF) != 0xFFFFF) atomicAdd(out0 + sh.pass[qi].out_off + (r.w & 0xFFFFF), sh.pass[qi].sign);
    return in;
  };
  // serial fall-backs for a full stack (rare): the preorder range [j, end) with dead subtrees skipped; node `cur`, its
  // later siblings and everything below them
  auto scan_range = [&](int j, int end, int qi, int isx, int isy) {
    while (j < end) {
      const int4 r = __ldg(rec + j);
      j += visit(j, qi, isx, isy, r) ? 1 : r.z;
    }
  };
  auto scan_siblings = [&](int cur, int qi, int isx, int isy) {
    for (;;) {
      const int4 r = __ldg(rec + cur);
      if (visit(cur, qi, isx, isy, r)) scan_range(cur + 1, cur + r.z, qi, isx, isy);
      if (!((r.w >> 24) & 1)) break;
      cur += r.z;
    }
  };
  // the same for the reversed trie: node j of rrec is the end of a backward walk from the pass's pixel; if it is in
  // phase and complete for trie node N, then (N, that pixel) is a survivor: N is counted and its subtree scanned
  auto rvisit_serial = [&](int j, int qi, const int4& r) -> bool {
    const int x = wrap_coord(sh.pass[qi].px + (short)(r.x & 0xffff), W), y = wrap_coord(sh.pass[qi].py + (r.x >> 16), H);
    const bool in = pbit(P + sh.pass[qi].pbase, x, y) && !(x == sh.pass[qi].ox && y == sh.pass[qi].oy);
    if (in && r.y >= 0) {
      const int4 rN = __ldg(rec + r.y);
      if ((rN.w & 0xFFFFF) != 0xFFFFF) atomicAdd(out0 + sh.pass[qi].out_off + (rN.w & 0xFFFFF), sh.pass[qi].sign);
      scan_range(r.y + 1, r.y + rN.z, qi, x, y);
    }
    return in;
  };
  auto rscan_range = [&](int j, int end, int qi) {
    while (j < end) {
      const int4 r = __ldg(rrec + j);
      j += rvisit_serial(j, qi, r) ? 1 : r.z;
    }
  };
  auto rscan_siblings = [&](int cur, int qi) {
    for (;;) {
      const int4 r = __ldg(rrec + cur);
      if (rvisit_serial(cur, qi, r)) rscan_range(cur + 1, cur + r.z, qi);
      if (!(r.w & 1)) break;
      cur += r.z;
    }
  };
  // reserves cnt slots of the CTA's stack for this warp and returns the first; slots at or beyond CAP do not exist:
  // their owners walk their items serially instead, and the stack top is clamped before the next pop
  auto reserve = [&](int cnt) -> int {
    int base = 0;
    if (lane == 0) base = atomicAdd(&sh.top, cnt);
    return __shfl_sync(0xffffffffu, base, 0);
  };

  constexpr unsigned REV = 0x80000000u;                    // stack item: a node of the reversed trie
  // the node range is sliced, so that a small batch of proposals still fills the chip
  const int slice_nodes = (n_nodes + n_slices - 1) / n_slices;
  bool any_scan = false;
  for (int q = 0; q < np; ++q) any_scan |= !sh.pass[q].rev;
  const int n_begin = slice * slice_nodes, n_end = any_scan ? min(n_nodes, n_begin + slice_nodes) : n_begin;
  const int n_iter = max(1, (n_end - n_begin + (int)blockDim.x - 1) / (int)blockDim.x);
  if (tid < np && sh.pass[tid].rev) {
    // (A) with the reversed trie: v = 0 (the pixel itself is in phase by construction) and the segments that START at
    // the pixel, then this slice's children of the reversed root go on the stack; each is pushed on its own, so the
    // sibling chain is not followed for them
    const int q = tid;
    if (slice == 0) {                                      // the root is a survivor at the pixel itself: (B) from there
      atomicAdd(out0 + sh.pass[q].out_off + (__ldg(rec).w & 0xFFFFF), sh.pass[q].sign);
      if (n_nodes > 1) {
        const int pos = atomicAdd(&sh.top, 1);
        const int px = sh.pass[q].px, py = sh.pass[q].py;
        if (pos < CAP) stk[pos] = make_uint2(1u | ((unsigned)q << 24), (unsigned)px | ((unsigned)py << 16));
        else scan_siblings(1, q, px, py);
      }
    }
    int c = 1, k = 0;
    for (;;) {
      const int4 r = __ldg(rrec + c);
      if (k % n_slices == slice) {
        const int pos = atomicAdd(&sh.top, 1);
        if (pos < CAP) stk[pos] = make_uint2((unsigned)c | ((unsigned)q << 24) | REV, 1u);   // y = 1: no sibling push
        else if (rvisit_serial(c, q, r)) rscan_range(c + 1, c + r.z, q);
      }
      if (!(r.w & 1)) break;
      c += r.z;
      ++k;
    }
  }
  for (int itn = 0; itn < n_iter; ++itn) {
    const int N = n_begin + itn * blockDim.x + tid;
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
      const unsigned nb = sh.pass[q].nb;
      const uint32_t* Pq = P + sh.pass[q].pbase;
      bool alive = (N < n_end) && !sh.pass[q].rev && (d == 0 || ((nb >> codeN) & 1u));
      if (!__any_sync(0xffffffffu, alive)) continue;       // typical for u: an isolated pixel kills all 32 at once
      const int ox = sh.pass[q].ox, oy = sh.pass[q].oy;
      const int sx = wrap_coord(sh.pass[q].px - oNx, W), sy = wrap_coord(sh.pass[q].py - oNy, H);
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
          if constexpr (FAST_WALK) {
            // branch-free steps and a 32-bit shared-memory address: 11 instructions per pixel instead of 29
            const int two_mn = 2 * mn, two_nn = 2 * nn;
            const unsigned pq_s = (unsigned)__cvta_generic_to_shared(Pq);
            {                                                // position d - 1 was the neighbour test
              e -= two_mn;
              const int neg = e >> 31;
              e += neg & two_nn;
              L -= dmaj + (neg & dmin);
            }
            for (int k = d - 2; k >= 1; --k) {
              e -= two_mn;
              const int neg = e >> 31;
              e += neg & two_nn;
              L -= dmaj + (neg & dmin);
              unsigned wv;
              asm volatile("ld.shared.u32 %0, [%1];" : "=r"(wv) : "r"(pq_s + 4u * (unsigned)(L >> 5)));
              if (!((wv >> (L & 31)) & 1u)) { alive = false; break; }
            }
          } else {
            for (int k = d - 1; k >= 1; --k) {
              e -= 2 * mn;
              L -= dmaj;
              if (e < 0) { e += 2 * nn; L -= dmin; }
              if (k == d - 1) continue;
              if (!((Pq[L >> 5] >> (L & 31)) & 1u)) { alive = false; break; }
            }
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
      if (alive && (rN.w & 0xFFFFF) != 0xFFFFF) atomicAdd(out0 + sh.pass[q].out_off + (rN.w & 0xFFFFF), sh.pass[q].sign);
      // (B) the first child of every survivor goes on the CTA's stack
      const bool push = alive && rN.z > 1;
      const unsigned pm = __ballot_sync(0xffffffffu, push);
      if (pm) {
        const int pos = reserve(__popc(pm)) + __popc(pm & lt);
        if (push) {
          if (pos < CAP) stk[pos] = make_uint2((unsigned)(N + 1) | ((unsigned)q << 24), (unsigned)sx | ((unsigned)sy << 16));
          else scan_siblings(N + 1, q, sx, sy);
        }
      }
    }
    // The survivors of all passes and of all warps are explored together, by the whole CTA (a deep live region is
    // paid once, and a big one is shared by eight warps): now, if the stack is half full or the slice is finished.
    if (!__syncthreads_or(itn + 1 == n_iter || sh.top > CAP / 2)) continue;   // one decision for the whole CTA
    for (;;) {
      const int n = min(sh.top, CAP);                      // slots beyond CAP were never written: their owners scanned
      if (n == 0) break;
      const int take = min(n, (int)blockDim.x);
      uint2 it = make_uint2(DUMMY, 0);
      if (tid < take) it = stk[n - 1 - tid];
      __syncthreads();                                     // every thread has read top and its item
      if (tid == 0) sh.top = n - take;
      __syncthreads();
      bool p_sib = false, p_child = false, p_fwd = false, rev = false;
      int i = 0, qi = 0, isx = 0, isy = 0, size_i = 0, fN = 0, fsize = 0, fx = 0, fy = 0;
      if (it.x != DUMMY) {
        i = (int)(it.x & 0xFFFFFF);
        qi = (int)((it.x >> 24) & 0x7Fu);
        rev = (it.x & REV) != 0;
        if (!rev) {
          isx = (int)(it.y & 0xffff);
          isy = (int)(it.y >> 16);
          // An only child follows its parent in the preorder array, and most of the trie is unary chains (about 36
          // nodes per vector at m = 64): the next CHAIN - 1 records are loaded with the node's own (independent loads
          // of one or two cache lines), and a chain of only children is visited in this pop instead of going through
          // the stack node by node.
          int4 r[CHAIN];
#pragma unroll
          for (int c = 0; c < CHAIN; ++c) r[c] = __ldg(rec + min(i + c, n_nodes - 1));
          p_sib = (r[0].w >> 24) & 1;
          if (p_sib) it.x += (unsigned)r[0].z;             // next sibling = i + subtree size
          bool in = visit(i, qi, isx, isy, r[0]);
          size_i = r[0].z;
#pragma unroll
          for (int c = 1; c < CHAIN; ++c) {
            if (in && size_i > 1 && !((r[c].w >> 24) & 1)) {   // alive, has a child, and that child has no sibling
              ++i;
              size_i = r[c].z;
              in = visit(i, qi, isx, isy, r[c]);
            } else {
              break;
            }
          }
          p_child = in && size_i > 1;
        } else {
          // the end of a backward walk from the pass's pixel: in phase -> its extensions; complete for trie node fN ->
          // (fN, this pixel) is a survivor of (A): count it, and its first child is the start of (B)
          const int4 r = __ldg(rrec + i);
          size_i = r.z;
          fx = wrap_coord(sh.pass[qi].px + (short)(r.x & 0xffff), W);
          fy = wrap_coord(sh.pass[qi].py + (r.x >> 16), H);
          const bool in = pbit(P + sh.pass[qi].pbase, fx, fy) && !(fx == sh.pass[qi].ox && fy == sh.pass[qi].oy);
          p_child = in && r.z > 1;
          p_sib = (r.w & 1) && it.y == 0u;                 // the root's children were pushed one by one (y = 1)
          if (p_sib) it.x += (unsigned)r.z;
          if (in && r.y >= 0) {
            fN = r.y;
            const int4 rN = __ldg(rec + fN);
            fsize = rN.z;
            if ((rN.w & 0xFFFFF) != 0xFFFFF) atomicAdd(out0 + sh.pass[qi].out_off + (rN.w & 0xFFFFF), sh.pass[qi].sign);
            p_fwd = rN.z > 1;
          }
        }
      }
      const unsigned ms = __ballot_sync(0xffffffffu, p_sib);
      const unsigned mc = __ballot_sync(0xffffffffu, p_child);
      const unsigned mf = __ballot_sync(0xffffffffu, p_fwd);
      const int ns = __popc(ms), nc = __popc(mc), nf = __popc(mf);
      if (ns + nc + nf) {
        const int base = reserve(ns + nc + nf);
        if (base + ns + nc + nf <= CAP) {
          if (p_sib) stk[base + __popc(ms & lt)] = make_uint2(it.x, rev ? 0u : it.y);
          if (p_child)
            stk[base + ns + __popc(mc & lt)] = make_uint2((unsigned)(i + 1) | (it.x & 0xFF000000u), rev ? 0u : it.y);
          if (p_fwd)
            stk[base + ns + nc + __popc(mf & lt)] =
                make_uint2((unsigned)(fN + 1) | ((unsigned)qi << 24), (unsigned)fx | ((unsigned)fy << 16));
        } else {
          // the stack cannot take this warp's pushes: every lane walks the remainder of its own item serially, and
          // the part of the reservation that lies inside the stack is marked unused
          for (int k = base + lane; k < min(base + ns + nc + nf, CAP); k += 32) stk[k] = make_uint2(DUMMY, 0);
          if (!rev) {
            if (p_child) scan_range(i + 1, i + size_i, qi, isx, isy);
            if (p_sib) scan_siblings((int)(it.x & 0xFFFFFFu), qi, isx, isy);   // it.x was advanced to the sibling
          } else {
            if (p_fwd) scan_range(fN + 1, fN + fsize, qi, fx, fy);
            if (p_child) rscan_range(i + 1, i + size_i, qi);
            if (p_sib) rscan_siblings(i + size_i, qi);
          }
        }
      }
      __syncthreads();                                     // all pushes of this round are in
    }
  }
}

}  // namespace lpf
