// Counter-based peer selector and straggler mask of the library (host + device).
// Philox4x32 with 10 rounds (Salmon et al., SC'11), keyed on (seed, step, layer, replica)
// as BASELINE.json:north_star item 2 asks; written from the published algorithm, shares
// nothing with oracle/ and does not include cuRAND.
#pragma once
#include <stdint.h>

#if defined(__CUDACC__)
#define LAYUP_HD __host__ __device__ __forceinline__
#else
#define LAYUP_HD inline
#endif

namespace layup {

constexpr uint32_t kTagPeer = 0u;        // counter word 3 of a peer draw
constexpr uint32_t kTagSkip = 1u;        // counter word 3 of a straggler draw
constexpr uint32_t kNoLayer = 0xFFFFFFFFu;

LAYUP_HD uint32_t mulhi32(uint32_t a, uint32_t b) {
#if defined(__CUDA_ARCH__)
  return __umulhi(a, b);
#else
  return (uint32_t)(((uint64_t)a * (uint64_t)b) >> 32);
#endif
}

// first output word of Philox4x32-10(counter = (c0,c1,c2,c3), key = (k0,k1))
LAYUP_HD uint32_t philox_first_word(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                    uint32_t k0, uint32_t k1) {
  constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
  constexpr uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = mulhi32(M0, c0), lo0 = M0 * c0;
    const uint32_t hi1 = mulhi32(M1, c2), lo1 = M1 * c2;
    const uint32_t n0 = hi1 ^ c1 ^ k0;
    const uint32_t n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += W0; k1 += W1;
  }
  return c0;
}

// PAPER.md:101 "j ~ Random(M-1)": uniform over the K-1 other workers, never self.
// layer_field = layer (peer_mode 0) or kNoLayer (peer_mode 1, one peer per iteration).
LAYUP_HD int32_t draw_peer(uint64_t seed, uint32_t step, uint32_t layer_field, int32_t replica, int32_t K) {
  const uint32_t r = philox_first_word(step, layer_field, (uint32_t)replica, kTagPeer,
                                       (uint32_t)seed, (uint32_t)(seed >> 32));
  const uint32_t q = mulhi32(r, (uint32_t)(K - 1));
  return (int32_t)(q + (q >= (uint32_t)replica ? 1u : 0u));
}

// Straggler mask: one draw per (step, replica); skip iff r < thr.
// Delay mode: replica delay_replica completes one iteration every delay_rounds+1
// rounds, i.e. is active only when (step+1) % (delay_rounds+1) == 0; ANDed with the random mask.
LAYUP_HD bool draw_active(uint64_t seed, uint32_t step, int32_t replica, uint32_t skip_thr,
                          int32_t delay_replica = 0, int32_t delay_rounds = 0) {
  if (delay_rounds > 0 && replica == delay_replica &&
      (((uint64_t)step + 1u) % ((uint64_t)delay_rounds + 1u)) != 0u) return false;
  if (skip_thr == 0u) return true;
  const uint32_t r = philox_first_word(step, kNoLayer, (uint32_t)replica, kTagSkip,
                                       (uint32_t)seed, (uint32_t)(seed >> 32));
  return !(r < skip_thr);
}

}  // namespace layup
