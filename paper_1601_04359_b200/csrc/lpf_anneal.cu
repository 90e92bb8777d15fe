// lpf_anneal.cu -- simulated annealing of Alg. 3 on the device.
// The chain itself is sequential (one proposal, one Metropolis decision at a time); what is parallel is the
// EVALUATION: a batch of K consecutive proposals is evaluated speculatively against the current image by the swap-delta
// kernel (which reads them straight from the caller's proposal list at the device-resident progress counter), the
// decisions are then taken in order by one thread, the first accepted proposal is applied and the proposals after it
// are thrown away and re-evaluated in the next batch -- so the result is exactly the sequential chain, whatever K is.
// The whole chain runs in ONE cooperative launch (anneal_chain_kernel): the host never sees a decision, it reads the
// final state when the chain is finished.
// Readings A1-A5 of the garbled listing are those of DESIGN.md "Annealing readings" (the oracle states them too).
#include <cooperative_groups.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>

#include "lpf_internal.h"
#include "lpf_swap.cuh"

namespace cg = cooperative_groups;

namespace lpf {

cudaError_t launch_swap_bits(const uint8_t* image, uint32_t* bits, int H, int W, int m, int phase,
                             unsigned int* counter, int n_sm, cudaStream_t st, uint32_t** padded_out);

struct AnnealState {
  long long next;        // proposals consumed so far (reading A1: the one counter that runs to N)
  long long c, s;        // per-temperature counters of Alg. 3 lines 6-8 (s: accepted, reading A1)
  long long accepted, levels;
  long long E;           // Eq. 19 over D and the requested phases on integer counts (reading A4), exact
  double T;
  int acc_idx;           // index inside the current batch of the accepted proposal, or -1
  int ticket;            // blocks of anneal_decide_kernel that have delivered their dE
  int acc_pair[4];       // the accepted proposal's pixels (x_p, y_p, x_q, y_q) if it exchanged two bytes, else -1
  int acc_bytes[2];      // ... and the bytes that are at p and at q after the exchange
};

// E of the start image: sum over the canonical half of (t - c)^2, all phases.  One block.
__global__ void anneal_e0_kernel(const long long* __restrict__ counts, const long long* __restrict__ target, int S,
                                 int n_ph, AnnealState* st) {
  const long long K = (long long)S * S, c0 = K / 2;
  long long s = 0;
  for (long long i = threadIdx.x; i < (long long)n_ph * (K - c0); i += blockDim.x) {
    const long long ph = i / (K - c0), k = c0 + (i - ph * (K - c0));
    const long long d = target[ph * K + k] - counts[ph * K + k];
    s += d * d;
  }
  __shared__ long long red[256];
  red[threadIdx.x] = s;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) st->E = red[0];
}

struct AnnealArgs {
  AnnealState* state;
  const uint32_t* padded;      // [n_ph] padded bit planes of the START image (lpf_swap.cuh layout)
  int H, W, m, phase, n_ph;
  const int* pairs;            // [N][4] the proposals (policy 0: the caller's list; else = pairs_out)
  int* pairs_out;              // policy 1 | 2: [N][4], every proposal is written here when it is generated
  int policy;                  // 0: list; 1: opposite bytes; 2: opposite bytes, both interfacial (reading A7)
  unsigned long long seed;
  const double* log_u;         // [N]
  long long N;
  const int4* rec;             // swap-delta node records
  int n_nodes;
  const int4* rrec;            // reversed trie of the swap delta, or null
  const unsigned int* dense;   // bit k: phase plane k is dense (per-node walks instead of the reversed trie)
  int* delta;                  // two buffers of [n_ph][K_max][S][S], zero on entry and again on exit
  long long ph_stride, buf_stride;
  int K_max;
  long long* dE;               // [K_max], zero on entry
  long long* counts;           // [n_ph][S][S]: descriptor of P
  const long long* target;
  uint8_t* image;
  uint8_t* accept_log;
  double wh2, T_mult;
  long long c_max, s_max;
};

__device__ __forceinline__ long long ld_cg(const long long* p) { return __ldcg(p); }

// n-th output of SplitMix64 for `seed` (Steele, Lea, Flood 2014): the counter-based generator of reading A7
__device__ __forceinline__ unsigned long long splitmix64(unsigned long long seed, unsigned long long n) {
  unsigned long long z = seed + n * 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

// The modification operator drawing its own pixels from the CURRENT image (reading A7),
// by one warp: lane t tries attempts t and t + 32 of a side, the first qualifying attempt wins (ballot).  The image
// bytes are read with ld.global.cg: the deciding thread of an earlier batch may have exchanged two of them.
//   policy 1: p = attempt 0 (any pixel), q = first attempt with another byte
//   policy 2: p = first interfacial attempt, q = first interfacial attempt with another byte
//   nothing qualifies in 64 attempts: q = p (identity move).  Every lane returns the same pair.
__device__ __forceinline__ int4 propose_pair(const uint8_t* image, int H, int W, int policy, unsigned long long seed,
                                             long long k, int lane) {
  auto byte_at = [&](int x, int y) -> int { return __ldcg(image + (size_t)y * W + x); };
  auto wrap = [](int v, int n) { return v < 0 ? v + n : (v >= n ? v - n : v); };
  int px = -1, py = -1, qx = -1, qy = -1, bp = -1;
  for (int side = 0; side < 2; ++side) {
    for (int round = 0; round < 2; ++round) {
      const int t = lane + 32 * round;
      const unsigned long long u = splitmix64(seed, 1ull + 2ull * (64ull * (unsigned long long)k + t) + side);
      const int x = (int)(((u >> 32) * (unsigned long long)W) >> 32);
      const int y = (int)(((u & 0xffffffffull) * (unsigned long long)H) >> 32);
      const int b = byte_at(x, y);
      bool ok = side == 0 || b != bp;
      if (policy == 2 && ok)
        ok = byte_at(wrap(x + 1, W), y) != b || byte_at(wrap(x - 1, W), y) != b || byte_at(x, wrap(y + 1, H)) != b ||
             byte_at(x, wrap(y - 1, H)) != b;
      if (policy == 1 && side == 0) ok = (t == 0);
      const unsigned hit = __ballot_sync(0xffffffffu, ok);
      if (hit) {
        const int src = __ffs(hit) - 1;
        const int wx = __shfl_sync(0xffffffffu, x, src), wy = __shfl_sync(0xffffffffu, y, src);
        if (side == 0) { px = wx; py = wy; bp = __shfl_sync(0xffffffffu, b, src); }
        else { qx = wx; qy = wy; }
        break;
      }
    }
    if (side == 0 && px < 0) {                               // no interfacial pixel met: attempt 0, identity move
      const unsigned long long u = splitmix64(seed, 1ull + 2ull * (64ull * (unsigned long long)k));
      px = (int)(((u >> 32) * (unsigned long long)W) >> 32);
      py = (int)(((u & 0xffffffffull) * (unsigned long long)H) >> 32);
      return make_int4(px, py, px, py);
    }
  }
  if (qx < 0) { qx = px; qy = py; }
  return make_int4(px, py, qx, qy);
}

// The whole chain in ONE cooperative launch (one CTA set resident on every SM, grid-wide barriers between the phases of
// a batch): the padded bit planes of the current image stay in every CTA's shared memory and are patched after an
// acceptance; nothing goes back to the host until the chain is finished.  Per batch of K proposals:
//   (A) Q = modify(P), SDQ = evaluate(Q) for proposals next .. next + K - 1, speculatively against P: swap_delta_unit
//       on (proposal, node slice) units spread over the grid  (Alg. 3 lines 9-10)
//   (B) dE[j] = E(Q_j) - E(P) = sum_phases sum_{v in D} [ (t - c - delta)^2 - (t - c)^2 ], exact, by (proposal, chunk)
//       units; the CTA that finishes LAST takes the decisions in order -- lines 7-17 -- up to and including the first
//       accepted proposal, whose two bytes it exchanges (P = Q)
//   (C) SDP = SDQ: the accepted proposal's delta is added to the descriptor (both halves), every delta is zeroed
//       again, every CTA patches its bit planes.
// Two grid barriers per batch: (C) of a batch and (A) of the next one run in the same phase -- a CTA patches its planes,
// does its share of (C), then evaluates its units of the next batch into the OTHER of two delta buffers; (B) of that
// batch reads the descriptor (C) has updated only after the barrier that follows.
// The proposals after an accepted one saw a stale image: they are not consumed and come back in the next batch, so
// the chain is exactly the sequential one for any K; K follows the acceptance rate (about 1 / rate + 1).  Memory that
// other CTAs write during the launch (state, delta, dE, counts) is read with ld.global.cg.
__global__ void __launch_bounds__(256) anneal_chain_kernel(const AnnealArgs a) {
  cg::grid_group grid = cg::this_grid();
  extern __shared__ __align__(16) uint32_t sm[];
  __shared__ SwapShared sh;
  __shared__ long long s_red[8];
  __shared__ long long s_dE[256];
  __shared__ double s_lu[256];
  __shared__ int s_last;
  __shared__ int s_pair[4];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int H = a.H, W = a.W, m = a.m, n_ph = a.n_ph;
  const int PWc = (W + 2 * m + 31) >> 5, PH = H + 2 * m;
  const int plane_words = PH * PWc;
  uint2* stk = (uint2*)(sm + ((n_ph * plane_words + 1) & ~1));
  for (int i = tid; i < n_ph * plane_words; i += blockDim.x) sm[i] = a.padded[i];
  const int S = 2 * m + 1;
  const long long K2 = (long long)S * S, c0 = K2 / 2, half = K2 - c0;
  const long long per_prop = n_ph * half;                       // elements of D over the phases
  const int n_chunks = (int)((per_prop + 1023) / 1024);
  int K = min(4, a.K_max);                                // proposals of the batch being decided
  long long win_next = 0, win_acc = 0;
  const unsigned int dense_mask = __ldg(a.dense);         // swaps keep the volume fractions: fixed for the chain
  // The reversed trie only if no plane of the chain is dense: a unit walks all planes of its proposal, and with one dense
  // plane the few slices that also explore the reversed trie of the sparse one would finish last (measured on the 100 x
  // 100 two-phase benchmark: 1.85e4 proposals/s with it, 1.94e4 without).
  const int4* const rrec = dense_mask == 0u ? a.rrec : nullptr;
  // (A): the deltas of proposals first .. first + Kb - 1 against the image in this CTA's shared memory, into dbuf
  auto evaluate = [&](long long first, int Kb, int* dbuf) {
    const int n_slices = max(1, min((int)gridDim.x / Kb, (a.n_nodes + 255) / 256));
    for (int unit = blockIdx.x; unit < Kb * n_slices; unit += gridDim.x) {
      const int j = unit / n_slices, slice = unit - j * n_slices;
      if (first + j >= a.N) continue;
      if (a.policy == 0) {
        swap_delta_unit<2, false>(sm, stk, sh, H, W, m, a.pairs, a.N, first + j, a.rec, a.n_nodes, rrec, dense_mask,
                                  dbuf + (long long)j * K2, n_ph, a.ph_stride, 1, slice, n_slices);
      } else {                                               // Q = modify(P): the operator draws its pixels from P
        __syncthreads();                                     // the previous unit is finished with s_pair
        if (warp == 0) {
          const int4 pr = propose_pair(a.image, H, W, a.policy, a.seed, first + j, lane);
          if (lane == 0) {
            s_pair[0] = pr.x; s_pair[1] = pr.y; s_pair[2] = pr.z; s_pair[3] = pr.w;
            if (slice == 0) {                                // for the decisions and for the caller
              int* po = a.pairs_out + 4 * (first + j);
              po[0] = pr.x; po[1] = pr.y; po[2] = pr.z; po[3] = pr.w;
            }
          }
        }
        __syncthreads();
        swap_delta_unit<2, false>(sm, stk, sh, H, W, m, s_pair, 1, 0, a.rec, a.n_nodes, rrec, dense_mask,
                                  dbuf + (long long)j * K2, n_ph, a.ph_stride, 1, slice, n_slices);
      }
    }
  };
  long long next = ld_cg(&a.state->next);
  if (next < a.N) evaluate(next, K, a.delta);
  grid.sync();
  for (int batch = 0; next < a.N; ++batch) {
    int* const dcur = a.delta + (long long)(batch & 1) * a.buf_stride;   // the deltas of this batch
    // ---- (B)
    for (int unit = blockIdx.x; unit < K * n_chunks; unit += gridDim.x) {
      const int j = unit / n_chunks, chunk = unit - j * n_chunks;
      long long s = 0;
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        const long long i = (long long)chunk * 1024 + r * 256 + tid;
        if (i < per_prop) {
          const long long ph = i / half, k = c0 + (i - ph * half);
          const long long dv = __ldcg(dcur + ph * a.ph_stride + (long long)j * K2 + k);
          if (dv != 0) {
            const long long d = a.target[ph * K2 + k] - ld_cg(a.counts + ph * K2 + k);
            s += dv * dv - 2 * d * dv;
          }
        }
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
      __syncthreads();
      if (lane == 0) s_red[warp] = s;
      __syncthreads();
      if (tid == 0) {
        long long t = 0;
        for (int w8 = 0; w8 < 8; ++w8) t += s_red[w8];
        if (t != 0) atomicAdd((unsigned long long*)(a.dE + j), (unsigned long long)t);
      }
    }
    if (tid == 0) {
      __threadfence();
      s_last = (atomicAdd(&a.state->ticket, 1) == (int)gridDim.x - 1);
    }
    __syncthreads();
    if (s_last) {                                                // every dE[j] of this batch is complete
      __threadfence();
      if (tid < K) {
        s_dE[tid] = ld_cg(a.dE + tid);
        a.dE[tid] = 0;
        s_lu[tid] = (next + tid < a.N) ? a.log_u[next + tid] : 0.0;
      }
      __syncthreads();
      if (tid == 0) {
        AnnealState st;
        st.next = next;
        st.c = ld_cg(&a.state->c); st.s = ld_cg(&a.state->s);
        st.accepted = ld_cg(&a.state->accepted); st.levels = ld_cg(&a.state->levels);
        st.E = ld_cg(&a.state->E);
        st.T = __longlong_as_double(ld_cg((const long long*)&a.state->T));
        int acc_idx = -1;
        long long consumed = 0;
        for (int jj = 0; jj < K; ++jj) {
          const long long idx = next + jj;
          if (idx >= a.N) break;
          ++consumed;
          st.c += 1;                                            // line 8
          const long long de = s_dE[jj];
          const double num = (double)(-de);                     // E_P - E_Q, exact
          const double den = a.wh2 * st.T;
          const bool acc = s_lu[jj] < num / den;                // line 11, reading A3
          if (a.accept_log) a.accept_log[idx] = acc ? 1 : 0;
          if (acc) {                                            // lines 12-13
            st.s += 1;
            st.accepted += 1;
            st.E += de;
            acc_idx = jj;
          }
          if (st.c >= a.c_max || st.s >= a.s_max) {             // the temperature level is complete: line 17
            st.T = st.T * a.T_mult;
            st.levels += 1;
            st.c = 0;
            st.s = 0;
          }
          if (acc) break;                                       // the later proposals saw a stale image
        }
        st.acc_idx = acc_idx;
        st.acc_pair[0] = st.acc_pair[1] = st.acc_pair[2] = st.acc_pair[3] = -1;
        st.acc_bytes[0] = st.acc_bytes[1] = 0;
        if (acc_idx >= 0) {                                     // P = Q: exchange the two bytes (reading A5)
          const long long idx = next + acc_idx;
          const int xp = __ldcg(a.pairs + 4 * idx), yp = __ldcg(a.pairs + 4 * idx + 1),
                    xq = __ldcg(a.pairs + 4 * idx + 2), yq = __ldcg(a.pairs + 4 * idx + 3);
          if (xp >= 0 && xp < W && xq >= 0 && xq < W && yp >= 0 && yp < H && yq >= 0 && yq < H) {
            volatile uint8_t* img = a.image;
            const uint8_t bp = img[(size_t)yp * W + xp], bq = img[(size_t)yq * W + xq];
            img[(size_t)yp * W + xp] = bq;
            img[(size_t)yq * W + xq] = bp;
            st.acc_pair[0] = xp; st.acc_pair[1] = yp; st.acc_pair[2] = xq; st.acc_pair[3] = yq;
            st.acc_bytes[0] = bq; st.acc_bytes[1] = bp;         // the bytes now at p and at q
          }
        }
        st.next = next + consumed;
        st.ticket = 0;
        *a.state = st;
      }
    }
    grid.sync();
    // ---- (C) of this batch, then (A) of the next one into the other delta buffer
    const int acc_idx = __ldcg(&a.state->acc_idx);
    if (acc_idx >= 0 && tid < 18 * n_ph) {                       // the two exchanged pixels, every periodic replica
      const int ph = tid / 18, r = tid % 18, which = r / 9, rep = r % 9;
      const int x = __ldcg(&a.state->acc_pair[2 * which]), y = __ldcg(&a.state->acc_pair[2 * which + 1]);
      if (x >= 0) {
        const int X = x + m + (rep / 3 - 1) * W, Y = y + m + (rep % 3 - 1) * H;
        if (X >= 0 && X < W + 2 * m && Y >= 0 && Y < PH) {
          const int want = (a.phase < 0) ? ph : a.phase;
          uint32_t* wp = sm + (size_t)ph * plane_words + (size_t)Y * PWc + (X >> 5);
          const uint32_t bit = 1u << (X & 31);
          if (__ldcg(&a.state->acc_bytes[which]) == want) atomicOr(wp, bit); else atomicAnd(wp, ~bit);
        }
      }
    }
    for (int unit = blockIdx.x; unit < K * n_chunks; unit += gridDim.x) {
      const int j = unit / n_chunks, chunk = unit - j * n_chunks;
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        const long long i = (long long)chunk * 1024 + r * 256 + tid;
        if (i < per_prop) {
          const long long ph = i / half, k = c0 + (i - ph * half);
          int* dp = dcur + ph * a.ph_stride + (long long)j * K2 + k;
          const int dv = __ldcg(dp);
          if (dv != 0) {
            if (j == acc_idx) {
              const long long nv = ld_cg(a.counts + ph * K2 + k) + dv;
              a.counts[ph * K2 + k] = nv;
              a.counts[ph * K2 + (K2 - 1 - k)] = nv;                     // count(-v) = count(v); v = 0 never changes
            }
            *dp = 0;
          }
        }
      }
    }
    next = ld_cg(&a.state->next);
    // Batch size for the next rounds, revised every 16 batches: one more than the expected run up to the first acceptance.
    // A batch costs about a + b K (a: the two grid barriers and the deepest exploration, b: the work of one proposal,
    // a / b ~ 10 on the 100 x 100 benchmark) and consumes (1 - (1 - r)^K) / r proposals at acceptance rate r; the ratio
    // peaks near K = 1 / r + 1 (measured against three expected acceptances per batch in powers of two, the rule before:
    // r = 0.85: 2.1e4 -> 3.4e4 proposals/s, 0.45: 1.5e4 -> 2.2e4, 0.11: 3.1e4 -> 5.0e4, 0.03: 3.8e4 -> 7.3e4).
    if ((batch & 15) == 15) {
      const long long ac = ld_cg(&a.state->accepted);
      const long long dn = next - win_next, da = ac - win_acc;
      win_next = next;
      win_acc = ac;
      if (dn > 0) {
        const double rate = (double)max(1ll, da) / (double)dn;
        K = min(a.K_max, (int)fmin(256.0, fmax(2.0, 1.0 / rate + 1.5)));
      }
    }
    __syncthreads();                                             // the patched bit planes, for every thread of this CTA
    if (next < a.N) evaluate(next, K, a.delta + (long long)((batch + 1) & 1) * a.buf_stride);
    grid.sync();
  }
}

}  // namespace lpf

using namespace lpf;

static int anneal_impl(lpf_paths* p, uint8_t* image, int H, int W, int phase, const int64_t* target,
                       const int32_t* pairs, int policy, uint64_t seed, int32_t* pairs_out, const double* log_u,
                       int64_t N, double T_max, double T_min, int64_t c_max, int64_t s_max, int64_t* counts,
                       uint8_t* accept_log, double* stats5, void* stream) {
  if (!p || !image || !target || !counts || !stats5 || (N > 0 && (!pairs || !log_u))) return LPF_E_INVAL;
  if (p->device < 0 || N < 0 || phase < -1 || phase > 1 || c_max < 1 || s_max < 1) return LPF_E_INVAL;
  if (!(T_max > 0.0) || !(T_min > 0.0)) return LPF_E_INVAL;
  cudaStream_t st = (cudaStream_t)stream;
  const int n_ph = phase < 0 ? 2 : 1;
  const int S = 2 * p->m + 1;
  const long long K2 = (long long)S * S;
  // SDP = evaluate(P) (line 2)
  int rc = phase < 0 ? lpf_eval_both(p, image, 1, H, W, counts, 0, stream)
                     : lpf_eval(p, image, 1, H, W, phase, counts, 0, stream);
  if (rc != LPF_OK) return rc;
  int prev = -1;
  if (cudaGetDevice(&prev) != cudaSuccess) return LPF_E_CUDA;
  if (prev != p->device && cudaSetDevice(p->device) != cudaSuccess) return LPF_E_CUDA;

  // chain state, proposal batch, deltas and error changes live in the table (lpf_reserve with LPF_FOR_ANNEAL)
  const int K_max = anneal_kmax(p->m, n_ph);
  if (!p->d_an_state || p->an_delta_bytes < sizeof(int) * 2 * (size_t)n_ph * K_max * K2) {
    rc = reserve_anneal(p, H, W);
    if (rc != LPF_OK) { if (prev != p->device) cudaSetDevice(prev); return rc; }
  }
  AnnealState* d_state = (AnnealState*)p->d_an_state;
  int* d_delta = p->d_an_delta;
  long long* d_dE = (long long*)p->d_an_dE;
  cudaError_t e = cudaSuccess;
  AnnealState h{};
  h.T = T_max;                                                   // line 3
  h.acc_idx = -1;
  const double T_mult = N > 0 ? std::pow(T_min / T_max, (double)s_max / (double)N) : 1.0;   // line 4, reading A2
  const double wh2 = (double)W * (double)H * (double)W * (double)H;
  const long long ph_stride = (long long)K_max * K2;
  // the chain's workspace: state, zeroed delta arrays, the padded bit planes of the start image (kept up to date by
  // anneal_apply_kernel from then on), E of the start image
  uint32_t* padded = nullptr;
  if (e == cudaSuccess) e = cudaMemcpyAsync(d_state, &h, sizeof(h), cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) e = cudaMemsetAsync(d_delta, 0, sizeof(int) * 2 * (size_t)n_ph * K_max * K2, st);
  if (e == cudaSuccess) e = cudaMemsetAsync(d_dE, 0, sizeof(long long) * 256, st);
  if (e == cudaSuccess)
    e = launch_swap_bits(image, p->d_swap_bits, H, W, p->m, phase, p->d_counter + 1, p->n_sm, st, &padded);
  if (e == cudaSuccess) {
    anneal_e0_kernel<<<1, 256, 0, st>>>((const long long*)counts, (const long long*)target, S, n_ph, d_state);
    e = cudaGetLastError();
  }
  rc = LPF_OK;
  if (e == cudaSuccess && N > 0) {
    // the whole chain: one cooperative launch, as many CTAs as are resident at once
    const size_t smem = (size_t)((n_ph * (H + 2 * p->m) * ((W + 2 * p->m + 31) / 32) + 1) & ~1) * 4 +
                        (size_t)8 * SWAP_STACK * 8;
    cudaFuncAttributes fa;
    e = cudaFuncGetAttributes(&fa, anneal_chain_kernel);
    if (e == cudaSuccess)
      e = cudaFuncSetAttribute(anneal_chain_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                               p->max_smem - (int)fa.sharedSizeBytes);
    int occ = 0;
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, anneal_chain_kernel, 256, smem);
    if (e == cudaSuccess && occ < 1) rc = LPF_E_UNSUPPORTED;
    if (e == cudaSuccess && rc == LPF_OK) {
      AnnealArgs a;
      a.state = d_state; a.padded = padded; a.H = H; a.W = W; a.m = p->m; a.phase = phase; a.n_ph = n_ph;
      a.pairs = pairs; a.pairs_out = pairs_out; a.policy = policy; a.seed = seed; a.log_u = log_u; a.N = N; a.rec = (const int4*)p->d_swap_rec; a.n_nodes = (int)p->n_trie_nodes;
      a.rrec = (const int4*)p->d_swap_rrec; a.dense = p->d_counter + 2;
      a.delta = d_delta; a.ph_stride = ph_stride; a.buf_stride = (long long)n_ph * ph_stride; a.K_max = K_max; a.dE = d_dE; a.counts = (long long*)counts;
      a.target = (const long long*)target; a.image = image; a.accept_log = accept_log; a.wh2 = wh2; a.T_mult = T_mult;
      a.c_max = c_max; a.s_max = s_max;
      void* args[] = {&a};
      e = cudaLaunchCooperativeKernel((const void*)anneal_chain_kernel, dim3((unsigned)(occ * p->n_sm)), dim3(256),
                                      args, smem, st);
    }
  }
  if (e == cudaSuccess && rc == LPF_OK) {
    e = cudaMemcpyAsync(&h, d_state, sizeof(h), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  }
  stats5[0] = (double)h.next;
  stats5[1] = (double)h.accepted;
  stats5[2] = (double)h.levels;
  stats5[3] = h.T;
  stats5[4] = (double)h.E;
  if (prev != p->device) cudaSetDevice(prev);
  if (rc != LPF_OK) return rc;
  if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? LPF_E_NOMEM : LPF_E_CUDA;
  return LPF_OK;
}

extern "C" int lpf_anneal(lpf_paths* p, uint8_t* image, int H, int W, int phase, const int64_t* target,
                          const int32_t* pairs, const double* log_u, int64_t N, double T_max, double T_min,
                          int64_t c_max, int64_t s_max, int64_t* counts, uint8_t* accept_log, double* stats5,
                          void* stream) {
  return anneal_impl(p, image, H, W, phase, target, pairs, 0, 0, nullptr, log_u, N, T_max, T_min, c_max, s_max, counts,
                     accept_log, stats5, stream);
}

extern "C" int lpf_anneal_generate(lpf_paths* p, uint8_t* image, int H, int W, int phase, const int64_t* target,
                                   int policy, uint64_t seed, int32_t* pairs_out, const double* log_u, int64_t N,
                                   double T_max, double T_min, int64_t c_max, int64_t s_max, int64_t* counts,
                                   uint8_t* accept_log, double* stats5, void* stream) {
  if (policy != LPF_PROPOSE_OPPOSITE && policy != LPF_PROPOSE_INTERFACIAL) return LPF_E_INVAL;
  if (N > 0 && !pairs_out) return LPF_E_INVAL;
  return anneal_impl(p, image, H, W, phase, target, pairs_out, policy, seed, pairs_out, log_u, N, T_max, T_min, c_max,
                     s_max, counts, accept_log, stats5, stream);
}
