// The schedule stage of ONE layer, as a device function: straggler
// mask, peer choice, push-sum weight halving / adding, mixing coefficients, AdamW bias corrections,
// written to the global schedule tables; the layer's round counter is read and advanced.
// Called by layup_schedule_kernel (schedule.cu: one CTA per layer in front of the update kernel).
// Thread i < K works for replica i; every thread of the CTA must call it (it contains CTA
// barriers); blockDim.x >= K.  (It is a device function because a "leader" form of the update
// kernel -- the first CTA of every layer runs this stage and the others poll a flag, one launch for
// any size -- was built on it and measured: bit-exact, 9-10 % slower on HBM-sized rounds.)
//
// PAPER.md:101  "Randomly select a peer: j ~ Random(M-1);  w_i <- w_i/2;  ...
//                Peer Update: x^{j,l} <- w_j/(w_i+w_j) x^{j,l} + w_i/(w_i+w_j) x^{i,l};
//                w_j <- w_j + w_i"
// Colliding pushes are folded in ascending sender index (R3): for receiver j,
// alpha_k = wh_i / (W + wh_i), W <- W + wh_i, starting from W = wh_j.
#pragma once
#include "layup_internal.cuh"
#include "philox.cuh"

namespace layup {

__host__ __device__ inline size_t schedule_scratch_bytes(int K) { return sizeof(double) * K + sizeof(int) * 2 * (size_t)K; }

// scratch: schedule_scratch_bytes(K) of shared memory, 8-byte aligned
__device__ __forceinline__ void schedule_layer(const SchedParams &p, int layer, unsigned char *scratch) {
  const int K = p.K;
  double *s_wh = reinterpret_cast<double *>(scratch);            // [K]
  int *s_peer = reinterpret_cast<int *>(s_wh + K);               // [K]
  int *s_cnt = s_peer + K;                                       // [K]
  const int i = threadIdx.x;
  const size_t row = (size_t)layer * K;
  // the round number is device state (layup.h "CUDA-graph capture"): every thread reads it here,
  // thread 0 advances it after the barrier below
  const uint32_t step = p.step_dev[layer];

  bool act = false;
  if (i < K) {
    act = draw_active(p.seed, step, i, p.skip_thr, p.delay_replica, p.delay_rounds);
    int peer = -1;
    double wh = p.w[row + i];
    if (act && K >= 2) {
      peer = draw_peer(p.seed, step, p.peer_mode == 0 ? (uint32_t)layer : kNoLayer, i, K);
      if (p.mix_mode != kMixSymmetric) wh = wh * 0.5;            // w_i <- w_i / 2 (exact)
    }
    if (p.adamw && act) {                                        // this worker takes its t-th step
      const double p1 = __dmul_rn(p.bpow[2 * (row + i)], p.beta1);   // no contraction into 1 - p1
      const double p2 = __dmul_rn(p.bpow[2 * (row + i) + 1], p.beta2);
      p.bpow[2 * (row + i)] = p1;
      p.bpow[2 * (row + i) + 1] = p2;
      p.t.c1[row + i] = (float)(p.lr / (1.0 - p1));
      p.t.c2[row + i] = (float)(1.0 / sqrt(1.0 - p2));
    }
    s_peer[i] = peer;
    s_wh[i] = wh;
    p.t.peer[row + i] = peer;
  }
  __syncthreads();
  if (i == 0) p.step_dev[layer] = step + 1u;

  // CSR by receiver without a serial prefix sum: the senders of receivers below i are exactly the
  // pushes whose peer index is below i; one pass over the K peers gives count, offset and last writer
  int cnt = 0, off = 0, last = -1;
  if (i < K) {
    for (int s = 0; s < K; ++s) {
      const int pr = s_peer[s];
      cnt += (pr == i);
      off += (pr >= 0 && pr < i);
      if (pr == i) last = s;
    }
  }
  // entries of the sender list: all pushes, the last writer only, or none (symmetric)
  const int n_list = p.mix_mode == kMixPushSum ? cnt : p.mix_mode == kMixLossy ? (cnt > 0 ? 1 : 0) : 0;
  if (p.mix_mode != kMixPushSum) {
    // shortened lists: offset = entries of the receivers below i
    if (i < K) s_cnt[i] = n_list;
    __syncthreads();
    off = 0;
    if (i < K)
      for (int r = 0; r < i; ++r) off += s_cnt[r];
  }

  if (i < K) {
    double W = s_wh[i];
    int k = off;
    for (int s = 0; s < K && p.mix_mode != kMixSymmetric; ++s) {
      if (s_peer[s] != i) continue;
      if (p.mix_mode == kMixLossy && s != last) continue;        // overwritten: skipped
      const double ws = s_wh[s];
      p.t.senders[row + k] = s;
      p.t.alpha[row + k] = (float)(ws / (W + ws));               // one rounding to fp32
      W = W + ws;                                                // w_j <- w_j + w_i
      ++k;
    }
    if (p.mix_mode != kMixSymmetric) p.w[row + i] = W;
    p.t.flags[row + i] = (unsigned char)((act ? kFlagActive : 0) | (cnt > 0 ? kFlagRecv : 0));
    p.t.recv_off[(size_t)layer * (K + 1) + i] = off;
    if (i == K - 1) p.t.recv_off[(size_t)layer * (K + 1) + K] = off + n_list;
  }
}

}  // namespace layup
