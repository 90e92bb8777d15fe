// lpf_anneal.cu -- simulated annealing of Alg. 3 on the device.
// The chain itself is sequential (one proposal, one Metropolis decision at a time); what is parallel is the
// EVALUATION: a batch of K consecutive proposals is evaluated speculatively against the current image with
// lpf_swap_delta, the decisions are then taken in order by one thread, the first accepted proposal is applied and the
// proposals after it are thrown away and re-evaluated in the next batch -- so the result is exactly the sequential
// chain, whatever K is.  The host never sees a decision: it only reads the progress counter every few batches.
// Readings A1-A5 of the garbled listing are those of DESIGN.md "Annealing readings" (the oracle states them too).
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>

#include "lpf_internal.h"

namespace lpf {

struct AnnealState {
  long long next;        // proposals consumed so far (reading A1: the one counter that runs to N)
  long long c, s;        // per-temperature counters of Alg. 3 lines 6-8 (s: accepted, reading A1)
  long long accepted, levels;
  long long E;           // Eq. 19 over D and the requested phases on integer counts (reading A4), exact
  double T;
  int acc_idx;           // index inside the current batch of the accepted proposal, or -1
  int pad;
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

// the next K proposals, or (-1,-1,-1,-1) past the end (lpf_swap_delta gives those an all-zero delta)
__global__ void anneal_gather_kernel(const int* __restrict__ pairs, long long N, const AnnealState* st,
                                     int* __restrict__ batch, int K) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= K) return;
  const long long idx = st->next + j;
#pragma unroll
  for (int t = 0; t < 4; ++t) batch[4 * j + t] = idx < N ? pairs[4 * idx + t] : -1;
}

// dE[j] = E(Q_j) - E(P) = sum_phases sum_{v in D} [ (t - c - delta)^2 - (t - c)^2 ], exact.  One block per proposal.
__global__ void anneal_de_kernel(const int* __restrict__ delta, long long ph_stride,
                                 const long long* __restrict__ counts, const long long* __restrict__ target, int S,
                                 int n_ph, long long* __restrict__ dE) {
  const long long K = (long long)S * S, c0 = K / 2;
  const int j = blockIdx.x;
  long long s = 0;
  for (int ph = 0; ph < n_ph; ++ph) {
    const int* dl = delta + ph * ph_stride + (long long)j * K;
    for (long long k = c0 + threadIdx.x; k < K; k += blockDim.x) {
      const long long dv = dl[k];
      if (dv != 0) {
        const long long d = target[ph * K + k] - counts[ph * K + k];
        s += dv * dv - 2 * d * dv;
      }
    }
  }
  __shared__ long long red[256];
  red[threadIdx.x] = s;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) dE[j] = red[0];
}

// Alg. 3 lines 7-17 for the proposals of this batch, in order, up to and including the first accepted one.
__global__ void anneal_decide_kernel(AnnealState* state, const long long* __restrict__ dE,
                                     const double* __restrict__ log_u, long long N, int K, double wh2, double T_mult,
                                     long long c_max, long long s_max, const int* __restrict__ batch,
                                     uint8_t* image, int H, int W, uint8_t* accept_log) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  AnnealState st = *state;
  int acc_idx = -1;
  long long consumed = 0;
  for (int j = 0; j < K; ++j) {
    const long long idx = st.next + j;
    if (idx >= N) break;
    ++consumed;
    st.c += 1;                                                  // line 8
    const double num = (double)(-dE[j]);                        // E_P - E_Q, exact
    const double den = wh2 * st.T;
    const bool acc = log_u[idx] < num / den;                    // line 11, reading A3
    if (accept_log) accept_log[idx] = acc ? 1 : 0;
    if (acc) {                                                  // lines 12-13
      st.s += 1;
      st.accepted += 1;
      st.E += dE[j];
      acc_idx = j;
    }
    if (st.c >= c_max || st.s >= s_max) {                       // the temperature level is complete: line 17
      st.T = st.T * T_mult;
      st.levels += 1;
      st.c = 0;
      st.s = 0;
    }
    if (acc) break;                                             // the later proposals saw a stale image
  }
  st.next += consumed;
  st.acc_idx = acc_idx;
  *state = st;
  if (acc_idx >= 0) {                                           // P = Q: exchange the two bytes (reading A5)
    const int xp = batch[4 * acc_idx], yp = batch[4 * acc_idx + 1], xq = batch[4 * acc_idx + 2],
              yq = batch[4 * acc_idx + 3];
    if (xp >= 0 && xp < W && xq >= 0 && xq < W && yp >= 0 && yp < H && yq >= 0 && yq < H) {
      const uint8_t bp = image[(size_t)yp * W + xp], bq = image[(size_t)yq * W + xq];
      image[(size_t)yp * W + xp] = bq;
      image[(size_t)yq * W + xq] = bp;
    }
  }
}

// SDP = SDQ: counts += delta of the accepted proposal (the delta arrays are full templates, mirrored)
__global__ void anneal_apply_kernel(const AnnealState* state, const int* __restrict__ delta, long long ph_stride,
                                    long long* __restrict__ counts, int S, int n_ph) {
  const int j = state->acc_idx;
  if (j < 0) return;
  const long long K = (long long)S * S;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < (long long)n_ph * K;
       i += (long long)gridDim.x * blockDim.x) {
    const long long ph = i / K, k = i - ph * K;
    counts[i] += delta[ph * ph_stride + (long long)j * K + k];
  }
}

}  // namespace lpf

using namespace lpf;

extern "C" int lpf_anneal(lpf_paths* p, uint8_t* image, int H, int W, int phase, const int64_t* target,
                          const int32_t* pairs, const double* log_u, int64_t N, double T_max, double T_min,
                          int64_t c_max, int64_t s_max, int64_t* counts, uint8_t* accept_log, double* stats5,
                          void* stream) {
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
  if (!p->d_an_state || p->an_delta_bytes < sizeof(int) * (size_t)n_ph * K_max * K2) {
    rc = reserve_anneal(p, H, W);
    if (rc != LPF_OK) { if (prev != p->device) cudaSetDevice(prev); return rc; }
  }
  AnnealState* d_state = (AnnealState*)p->d_an_state;
  int* d_batch = p->d_an_batch;
  int* d_delta = p->d_an_delta;
  long long* d_dE = (long long*)p->d_an_dE;
  cudaError_t e = cudaSuccess;
  AnnealState h{};
  h.T = T_max;                                                   // line 3
  h.acc_idx = -1;
  const double T_mult = N > 0 ? std::pow(T_min / T_max, (double)s_max / (double)N) : 1.0;   // line 4, reading A2
  const double wh2 = (double)W * (double)H * (double)W * (double)H;
  if (e == cudaSuccess) e = cudaMemcpyAsync(d_state, &h, sizeof(h), cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) {
    anneal_e0_kernel<<<1, 256, 0, st>>>((const long long*)counts, (const long long*)target, S, n_ph, d_state);
    e = cudaGetLastError();
  }
  const long long ph_stride = (long long)K_max * K2;
  int K = 16;
  long long last_next = 0, last_acc = 0;
  rc = LPF_OK;
  while (e == cudaSuccess && rc == LPF_OK && h.next < N) {
    K = std::min(K, K_max);
    for (int rep = 0; rep < 8 && rc == LPF_OK && e == cudaSuccess; ++rep) {
      anneal_gather_kernel<<<(K + 63) / 64, 64, 0, st>>>(pairs, N, d_state, d_batch, K);
      // Q = modify(P), SDQ = evaluate(Q): lines 9-10 (both phases in one pass over the trie if asked)
      rc = swap_delta_impl(p, image, H, W, phase, d_batch, K, d_delta, ph_stride, stream);
      if (rc != LPF_OK) break;
      anneal_de_kernel<<<K, 256, 0, st>>>(d_delta, ph_stride, (const long long*)counts, (const long long*)target, S,
                                          n_ph, d_dE);
      anneal_decide_kernel<<<1, 32, 0, st>>>(d_state, d_dE, log_u, N, K, wh2, T_mult, c_max, s_max, d_batch, image,
                                             H, W, accept_log);
      anneal_apply_kernel<<<std::max(1, std::min(p->n_sm * 4, (int)((n_ph * K2 + 255) / 256))), 256, 0, st>>>(
          d_state, d_delta, ph_stride, (long long*)counts, S, n_ph);
      e = cudaGetLastError();
    }
    if (e != cudaSuccess || rc != LPF_OK) break;
    e = cudaMemcpyAsync(&h, d_state, sizeof(h), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    // batch size for the next rounds: about three expected acceptances per batch
    const long long dn = h.next - last_next, da = h.accepted - last_acc;
    last_next = h.next;
    last_acc = h.accepted;
    if (dn > 0) {
      const double rate = std::max(1.0, (double)da) / (double)dn;
      int want = (int)std::min(256.0, std::max(8.0, 3.0 / rate));
      K = 8;
      while (K < want) K *= 2;
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
