// Internal declarations shared by the library's translation units (not part of the C-ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace layup {

constexpr int kFlagActive = 1;         // replica takes its local step and pushes this round
constexpr int kFlagRecv = 2;           // replica receives at least one push this round

// One (replica-major) layer of the arena; offsets in floats inside a section.
struct LayerDesc {
  long long base;      // offset of replica 0's slice
  long long pad;       // slice stride (numel rounded up to 32 floats = 128 B)
  long long numel;     // unpadded elements
};

// Per-(layer) schedule tables, written by the schedule kernel, read by the update kernel.
struct SchedTables {
  int32_t *peer;            // [L*K]   chosen peer or -1
  int32_t *recv_off;        // [L*(K+1)] CSR by receiver
  int32_t *senders;         // [L*K]   senders of each receiver, ascending
  float *alpha;             // [L*K]   mixing coefficient of each push, same order
  unsigned char *flags;     // [L*K]   kFlagActive | kFlagRecv
  float *c1, *c2;           // [L*K]   AdamW step scalars eta/(1-b1^t), 1/sqrt(1-b2^t) (else nullptr)
};

constexpr int kMixPushSum = 0;         // lossless push-sum fold (R3)
constexpr int kMixLossy = 1;           // contention: only the last writer's push lands (R22)
constexpr int kMixSymmetric = 2;       // AD-PSGD pairwise averaging (R23)

// fp32 scalars of the local step (narrowed once on the host)
struct StepScalars {
  float neg_lr, mu, wd;                 // SGD: -eta, momentum, coupled weight decay
  float b1, b2, omb1, omb2, eps, decay; // AdamW: betas, 1-betas, eps, 1 - eta*wd
};

struct SchedParams {
  SchedTables t;
  double *w;                // [L*K] push-sum weights, updated in place
  uint64_t seed;
  uint32_t *step_dev;       // [L] the round each layer runs next: read, then advanced, by the schedule stage
  uint32_t skip_thr;        // skip iff draw < skip_thr; 0 = straggler mode off
  int32_t K, L;
  int32_t layer_begin;      // blockIdx.x + layer_begin = layer
  int32_t peer_mode;
  int32_t delay_replica, delay_rounds;   // deterministic straggler (0 rounds = off)
  int32_t mix_mode;         // kMix*
  int32_t adamw;            // 1: maintain bpow and emit c1, c2
  double *bpow;             // [L*K*2] (beta1^t, beta2^t) per (layer, replica), AdamW only
  double lr, beta1, beta2;  // fp32 values widened
  int32_t *ticket;          // [L] zero between launches; fused single-launch path only (update_tma.cu)
  int32_t *ps_ticket;       // [L] tile tickets of persistent update launches (update_persist.cu), by work-list
  int32_t n_ps_ticket;      //   position; the schedule kernel zeroes the slots of its own layers; 0 = none
};
constexpr int kFusedMaxK = 64;         // the in-kernel schedule stage is O(K) per thread

struct UpdateParams {
  float *x, *g, *m, *v;             // section bases (m / v == nullptr when the optimiser has none)
  const LayerDesc *layers;          // [L]
  const long long *tile_prefix;     // [L+1] by position; position p holds layer L-1-p
  SchedTables t;
  long long tile_begin, tile_end;   // work-list range of this launch
  int32_t K, L;
  int32_t C, log2C;                 // float4 columns per tile (power of two)
  int32_t pos_begin, pos_end;       // positions covered by [tile_begin, tile_end)
  StepScalars s;
  int32_t opt;                      // OPT_* of rule.cuh
  int32_t symmetric;                // mix_mode == kMixSymmetric
  int32_t all_active;               // skip_prob == 0: every replica is active in every round
  SchedParams sched;                // fused single-launch path: the schedule stage's inputs
  const void *tmaps;                // [n_sections][L] CUtensorMap (128 B each) of the layer sections, or nullptr
  const void *tmaps_g4;             // same views with a one-row box, for tile::gather4 (straggler mode), or nullptr
  unsigned long long *trace;        // [L] first CTA start per layer (%globaltimer, atomicMin), or nullptr (layup_trace)
  int32_t *ps_ticket;               // persistent shape: this launch's tile ticket (zero at launch)
};

// layup_trace: the first CTA of a (step, layer) event to start leaves the GPU nanosecond timer
__device__ __forceinline__ void trace_start(unsigned long long *trace, int layer) {
  if (trace != nullptr && threadIdx.x == 0) {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    atomicMin(trace + layer, t);
  }
}

// Work-list table of one launch, passed by value in the kernel parameters (constant bank):
// the launch covers positions [0, n) of this table; position q holds layer `layer[q]`
// (reverse layer order) and the tiles [prefix[q], prefix[q+1]) of the launch.
constexpr int kMaxPos = 160;
struct PosTable {
  long long prefix[kMaxPos + 1];
  LayerDesc lay[kMaxPos];
  int32_t layer[kMaxPos];
  int32_t n;
};

// The dynamic shared memory a kernel may be launched with is an attribute of the FUNCTION on the device,
// shared by every ctx of the process: a ctx that set it to its own (smaller) need would break the launches
// of an older ctx that needs more (two LayUp objects alive at once: "invalid argument" at launch).  So the
// library always opens a kernel up to the device's opt-in maximum; a launch still gets what it asks for.
inline cudaError_t allow_max_dynamic_smem(const void *fn, int need_bytes) {
  int dev = 0, optin = 0;
  cudaFuncAttributes fa;
  cudaError_t e;
  if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
  if ((e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev)) != cudaSuccess) return e;
  if ((e = cudaFuncGetAttributes(&fa, fn)) != cudaSuccess) return e;
  const int most = optin - (int)fa.sharedSizeBytes;
  if (need_bytes > most) return cudaErrorInvalidValue;
  return cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, most);
}

// api.cu
void note_error(const char *text);     // becomes the text of layup_last_error(NULL) on this host thread
// schedule.cu
cudaError_t launch_schedule(const SchedParams &p, int n_layers, cudaStream_t s);
cudaError_t launch_peers_only(uint64_t seed, uint32_t step, uint32_t skip_thr, int K, int L, int peer_mode,
                              int delay_replica, int delay_rounds, int32_t *peer_dev, unsigned char *active_dev,
                              cudaStream_t s);
// diagnose.cu
cudaError_t diag_plan(int K, size_t smem_optin, int *C, int *stages, int *smem_bytes, int *ctas_per_sm);
cudaError_t launch_disagreement(const float *x, const double *w, double *dist, int K, int C, int log2C, int stages,
                                const PosTable &tab, int grid, int smem_bytes, cudaStream_t s);
// update.cu
int update_num_variants();
cudaError_t update_kernel_setup(int variant, int opt, bool symmetric, int smem_bytes, int *threads, int *ctas_per_sm);
cudaError_t launch_update(const UpdateParams &p, int variant, bool persistent, int grid, int smem_bytes,
                          cudaStream_t s);
size_t update_smem_bytes(int K, int C);
// update_tma.cu -- TMA-bulk staged variants
int tma_num_variants();
int tma_default_variant(int n_items, int n_sections);
int tma_bulk_variant(int n_items, int n_sections, bool straggler_mode);
size_t tma_smem_bytes(int K, int C, int opt, bool fused, int rega, bool gather4);
int tma_variant_rega(int variant, int opt);        // arrays this thread shape stages through registers
int tma_variant_max_items(int variant);            // ... and the largest tile it takes (0 = any)
bool tma_has_fused(int variant);
cudaError_t tma_kernel_setup(int variant, int opt, bool symmetric, bool strag, int smem_bytes, int *threads, int *ctas_per_sm);
cudaError_t launch_update_tma(const UpdateParams &p, const PosTable &tab, int variant, bool fused, bool pdl, int grid,
                              int smem_bytes, cudaStream_t s);

// update_persist.cu -- persistent warp-specialised ring form (layup_tuning.launch_shape = 2)
int persist_max_k();
int persist_stages(int K, int C, int opt, size_t smem_optin, int ctas, int want);
size_t persist_smem_bytes(int K, int C, int opt, int stages);
cudaError_t persist_kernel_setup(int opt, bool symmetric, int smem_bytes, int *ctas_per_sm);
void persist_shape(int *stages, int n_items, int want_groups, int want_gs, int *groups, int *gs);
cudaError_t launch_update_persist(const UpdateParams &p, const PosTable &tab, int grid, int smem_bytes, int stages,
                                  int groups, int group_threads, bool pdl, cudaStream_t s);

}  // namespace layup
