/* The C-ABI of include/layup.h driven from plain C99, without Python's hand-mirrored structs
 * (SURVEY.md 8(b)).  Two programs from one source:
 *   -DLAYOUT_ONLY : prints sizeof / offsetof of layup_config and layup_tuning (no CUDA, no library);
 *                   tests/test_library_cpu.py compares them with the ctypes mirror in binding.py.
 *   default       : cudaMalloc an arena, layup_init, two replicas holding 1.0 and 3.0 everywhere,
 *                   zero gradients, one layup_round: with K = 2 each replica's only possible peer
 *                   is the other one, both weights are halved to 1/4, so every push mixes with
 *                   alpha = 1/2 and both replicas become exactly 2.0 ("Peer Update");
 *                   the push-sum weights still sum to 1.  Prints "C_ABI_OK".
 */
#include <stddef.h>
#include <stdio.h>
#include <stdlib.h>

#include "layup.h"

#ifdef LAYOUT_ONLY
#define OFF(T, f) printf(#T "." #f " %zu\n", offsetof(T, f))
int main(void) {
  printf("sizeof.layup_config %zu\n", sizeof(layup_config));
  printf("sizeof.layup_tuning %zu\n", sizeof(layup_tuning));
  OFF(layup_config, K); OFF(layup_config, L); OFF(layup_config, numel); OFF(layup_config, lr);
  OFF(layup_config, momentum); OFF(layup_config, seed); OFF(layup_config, peer_mode); OFF(layup_config, skip_prob);
  OFF(layup_config, device); OFF(layup_config, delay_replica); OFF(layup_config, delay_rounds);
  OFF(layup_config, optimizer); OFF(layup_config, mix_mode); OFF(layup_config, weight_decay);
  OFF(layup_config, beta1); OFF(layup_config, beta2); OFF(layup_config, eps); OFF(layup_config, tuning);
  OFF(layup_tuning, engine); OFF(layup_tuning, launch_shape); OFF(layup_tuning, fused); OFF(layup_tuning, fused_waves);
  OFF(layup_tuning, tile_items); OFF(layup_tuning, variant); OFF(layup_tuning, ctas_per_sm); OFF(layup_tuning, pdl);
  OFF(layup_tuning, tma2d); OFF(layup_tuning, stages); OFF(layup_tuning, group_threads);
  return 0;
}
#else
#include <cuda_runtime_api.h>

#define CHECK(call)                                                                              \
  do {                                                                                           \
    int rc__ = (call);                                                                           \
    if (rc__ != LAYUP_OK) {                                                                      \
      fprintf(stderr, "%s -> %d: %s\n", #call, rc__, layup_last_error(ctx));                     \
      return 1;                                                                                  \
    }                                                                                            \
  } while (0)

int main(void) {
  layup_ctx *ctx = NULL;
  const int64_t numel[3] = {5000, 33, 70001};          /* several tiles, ragged tails */
  layup_config cfg = {0};
  cfg.K = 2; cfg.L = 3; cfg.numel = numel; cfg.lr = 0.125f; cfg.seed = 7; cfg.device = 0;
  size_t bytes = 0;
  CHECK(layup_arena_bytes(&cfg, &bytes));
  void *arena = NULL;
  if (cudaMalloc(&arena, bytes) != cudaSuccess) { fprintf(stderr, "cudaMalloc failed\n"); return 1; }
  CHECK(layup_init(&cfg, arena, bytes, &ctx));
  float *host = (float *)malloc(sizeof(float) * 70001);
  for (int l = 0; l < 3; ++l)
    for (int i = 0; i < 2; ++i) {
      float *d = NULL; int64_t n = 0;
      CHECK(layup_ptr(ctx, LAYUP_WHAT_X, i, l, &d, &n));
      if (n != numel[l]) { fprintf(stderr, "layup_ptr numel\n"); return 1; }
      for (int64_t e = 0; e < n; ++e) host[e] = i == 0 ? 1.0f : 3.0f;
      if (cudaMemcpy(d, host, sizeof(float) * (size_t)n, cudaMemcpyHostToDevice) != cudaSuccess) return 1;
    }
  CHECK(layup_round(ctx, 0, NULL));                     /* gradients are zero: the arena was zeroed by layup_init */
  CHECK(layup_sync(ctx));
  double w[6];
  CHECK(layup_weights(ctx, w));
  for (int l = 0; l < 3; ++l) {
    if (w[2 * l] + w[2 * l + 1] != 1.0 || w[2 * l] != 0.5) { fprintf(stderr, "weights of layer %d: %g %g\n", l, w[2 * l], w[2 * l + 1]); return 1; }
    for (int i = 0; i < 2; ++i) {
      float *d = NULL; int64_t n = 0;
      CHECK(layup_ptr(ctx, LAYUP_WHAT_X, i, l, &d, &n));
      if (cudaMemcpy(host, d, sizeof(float) * (size_t)n, cudaMemcpyDeviceToHost) != cudaSuccess) return 1;
      for (int64_t e = 0; e < n; ++e)
        if (host[e] != 2.0f) { fprintf(stderr, "layer %d replica %d element %lld = %g, want 2\n", l, i, (long long)e, host[e]); return 1; }
    }
  }
  int32_t order[3], n_order = 0;
  CHECK(layup_last_order(ctx, order, &n_order));
  if (n_order != 3 || order[0] != 2 || order[2] != 0) { fprintf(stderr, "issue order\n"); return 1; }   /* output layer first */
  if (layup_round(ctx, 0, NULL) != LAYUP_ESTATE) { fprintf(stderr, "round 0 twice was accepted\n"); return 1; }
  CHECK(layup_destroy(ctx));
  cudaFree(arena);
  free(host);
  printf("C_ABI_OK\n");
  return 0;
}
#endif
