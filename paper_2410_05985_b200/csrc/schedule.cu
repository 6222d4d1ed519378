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
#include "schedule_body.cuh"

namespace layup {

__global__ void __launch_bounds__(1024) layup_schedule_kernel(const SchedParams p) {
  extern __shared__ __align__(8) unsigned char sm[];
  // the update kernel behind this one on the stream may start now (it waits for this grid's
  // completion with griddepcontrol.wait before it reads the tables)
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  // tile tickets of the persistent update launches behind this kernel: one slot per work-list position
  // (position q = layer L-1-q; a launch draws from the slot of its FIRST position).  Only the slots of
  // this call's own layers are re-armed, so per-layer events on other streams keep theirs.
  if (p.n_ps_ticket > 0 && threadIdx.x == 0) p.ps_ticket[p.L - 1 - (p.layer_begin + (int)blockIdx.x)] = 0;
  schedule_layer(p, p.layer_begin + blockIdx.x, sm);
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
  const size_t smem = schedule_scratch_bytes(p.K);
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
