// Schedule stage: straggler mask, peer choice, push-sum
// weight halving / adding, and the mixing coefficients, for every layer of a launch.
// O(L*K) integer + fp64 scalar work; one CTA per layer, one thread per replica.
//
// PAPER.md:101  "Randomly select a peer: j ~ Random(M-1);  w_i <- w_i/2;  ...
//                Peer Update: x^{j,l} <- w_j/(w_i+w_j) x^{j,l} + w_i/(w_i+w_j) x^{i,l};
//                w_j <- w_j + w_i"
// Colliding pushes are folded in ascending sender index (R3): for receiver j,
// alpha_k = wh_i / (W + wh_i), W <- W + wh_i, starting from W = wh_j.
// Variant mixers: kMixLossy keeps only the last writer of every
// receiver (R22) -- the update kernel is unchanged, it just sees a shorter
// sender list; kMixSymmetric exchanges no weight (R23) and the update kernel
// walks the peer table instead of a sender list.
// AdamW (NEXT-3): the per-(layer, replica) bias corrections, from running products
// beta^t kept in fp64, narrowed once: c1 = eta/(1-b1^t), c2 = 1/sqrt(1-b2^t).
#include "layup_internal.cuh"
#include "philox.cuh"

namespace layup {

__global__ void __launch_bounds__(1024) layup_schedule_kernel(const SchedParams p) {
  extern __shared__ __align__(8) unsigned char sm[];
  const int K = p.K;
  double *s_wh = reinterpret_cast<double *>(sm);                 // [K]
  int *s_peer = reinterpret_cast<int *>(s_wh + K);               // [K]
  int *s_cnt = s_peer + K;                                       // [K]

  // the update kernel behind this one on the stream may start now (it waits for this grid's
  // completion with griddepcontrol.wait before it reads the tables)
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const int layer = p.layer_begin + blockIdx.x;
  const int i = threadIdx.x;
  const size_t row = (size_t)layer * K;
  if (blockIdx.x == 0)                                           // tile tickets of the persistent update launches
    for (int t = i; t < p.n_ps_ticket; t += blockDim.x) p.ps_ticket[t] = 0;
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

// Introspection: peers and mask of an arbitrary round, no state touched.
__global__ void layup_peers_only_kernel(uint64_t seed, uint32_t step, uint32_t skip_thr, int K, int L,
                                        int peer_mode, int delay_replica, int delay_rounds, int32_t *peer,
                                        unsigned char *active) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= L * K) return;
  const int layer = idx / K, i = idx - layer * K;
  const bool act = draw_active(seed, step, i, skip_thr, delay_replica, delay_rounds);
  peer[idx] = (act && K >= 2) ? draw_peer(seed, step, peer_mode == 0 ? (uint32_t)layer : kNoLayer, i, K) : -1;
  if (layer == 0) active[i] = act ? 1 : 0;
}

cudaError_t launch_schedule(const SchedParams &p, int n_layers, cudaStream_t s) {
  const int threads = ((p.K + 31) / 32) * 32;
  const size_t smem = sizeof(double) * p.K + sizeof(int) * 2 * (size_t)p.K;
  layup_schedule_kernel<<<n_layers, threads, smem, s>>>(p);
  return cudaGetLastError();
}

cudaError_t launch_peers_only(uint64_t seed, uint32_t step, uint32_t skip_thr, int K, int L, int peer_mode,
                              int delay_replica, int delay_rounds, int32_t *peer_dev, unsigned char *active_dev,
                              cudaStream_t s) {
  const int n = K * L;
  layup_peers_only_kernel<<<(n + 255) / 256, 256, 0, s>>>(seed, step, skip_thr, K, L, peer_mode, delay_replica,
                                                          delay_rounds, peer_dev, active_dev);
  return cudaGetLastError();
}

}  // namespace layup
