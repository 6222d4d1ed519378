/*
 * layup.h -- C-ABI boundary of the B200-native LayUp hot path.
 *
 * What the library computes: the "Updater Thread i" of Algorithm 1 of LayUp
 * (arXiv 2410.05985) for K workers held as K fp32
 * replicas of every layer in ONE device arena:  per layer, as soon as its gradient
 * exists, the local SGD step on each worker's copy
 * ("Local Update"), then the push-sum gossip mix of that copy into a
 * randomly chosen peer's copy of the same layer ("Peer Update",
 * PAPER.md:104-106 weights), with no buffer or queue.  The
 * deterministic reading of the paper's racy system is DESIGN.md "Readings" R1-R25.
 *
 * Conventions
 *  - All functions return int: LAYUP_OK (0) or a negative LAYUP_E* code; no exceptions,
 *    no abort, nothing printed.  layup_last_error() gives the text of the last failure.
 *  - Pointers are HOST pointers unless the comment says DEVICE.
 *  - Launching calls (layup_layer_update, layup_round) are ASYNCHRONOUS on the given
 *    CUDA stream; device-side failures surface at layup_sync().  If a launching call fails
 *    after one of its kernels was already enqueued (the schedule stage advances the device's
 *    round counter), the ctx is POISONED: every later launching call returns LAYUP_ECUDA.
 *  - Ownership: the caller allocates the arena (device memory) and the streams and keeps
 *    them alive until layup_destroy(); the library borrows them.  It owns only its small
 *    tables (layer table, schedule tables, weights w[L][K]); it never allocates
 *    parameter-sized memory ("without buffering").
 *  - A ctx is used from one host thread at a time.  Every call leaves the calling thread's
 *    current CUDA device as it found it.
 *  - There is no CPU fallback: without a CUDA device every launching call fails with
 *    LAYUP_ECUDA.
 *
 * Arena layout (DEVICE, fp32): sections X | G | M | V (M only if momentum != 0 or AdamW, V
 * only for AdamW), each
 * `section_floats` long.  Inside a section layers are stored in order 0..L-1; layer l
 * holds its K replicas back to back, each slice padded to a multiple of 32 floats
 * (128 B):   addr(what, i, l, e) = arena + what*section + base[l] + i*pad[l] + e.
 * The arena base must be 128-byte aligned.  layup_init() zeroes the whole arena, so the
 * pads are zero and stay zero; fill x (and g before every step) through layup_ptr().
 */
#ifndef LAYUP_H_
#define LAYUP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LAYUP_OK      0
#define LAYUP_EINVAL -1   /* bad argument, misaligned or too-small arena              */
#define LAYUP_ESTATE -2   /* (step, layer) applied out of order or twice              */
#define LAYUP_ECUDA  -3   /* CUDA failure (no device, launch or runtime error)        */

#define LAYUP_WHAT_X 0    /* parameters x^{i,l}                 */
#define LAYUP_WHAT_G 1    /* gradient of this step   ("Backward pass")    */
#define LAYUP_WHAT_M 2    /* momentum buffer / AdamW first moment, local to the worker (R8, R21) */
#define LAYUP_WHAT_V 3    /* AdamW second moment, local to the worker (R21)           */

#define LAYUP_OPT_SGD   0 /* x <- x - eta*(g + wd*x), optional heavy-ball momentum */
#define LAYUP_OPT_ADAMW 1 /* AdamW, PyTorch's convention (Tables A7/A8 469-491)        */

#define LAYUP_MIX_PUSHSUM   0 /* push-sum fold, every colliding push applied (R3)      */
#define LAYUP_MIX_LOSSY     1 /* contention: only the last writer's push and weight land
                                 ("one of the peers will be skipped", 106; R22)         */
#define LAYUP_MIX_SYMMETRIC 2 /* AD-PSGD-style pairwise averaging x_i,x_j <- (x_i+x_j)/2, ascending
                                 worker index, no push-sum weights (R23)               */

#define LAYUP_MAX_K 1024  /* replicas (workers) per ctx.  Accepted up to here; the kernels are tuned for
                             the paper's worker counts and run at HBM speed for K <= 128 (>= 6.0 TB/s);
                             K = 256 reaches 3.8-5.9 TB/s, K = 512 2.8-4.1 TB/s          */

typedef struct layup_ctx layup_ctx;       /* opaque */
typedef struct layup_graph layup_graph;   /* opaque: a captured sequence of launching calls */

/* Launch tuning, all optional: 0 in a field = the library's default, and a NULL pointer in
 * layup_config.tuning = all defaults.  None of them changes a single result bit (every launch
 * shape is parity-tested against the oracle); they select WHICH of the library's kernels runs.
 * This block is the only switch: the library reads no environment variable. */
typedef struct {
  int32_t engine;       /* 0 auto: TMA-staged kernel while the tile of all K replicas fits in shared
                           memory, else the LDG kernel; 1 TMA-staged; 2 LDG                         */
  int32_t launch_shape; /* 0 auto = 1; 1 grouped: one CTA per (layer, tile) work item, the list in
                           reverse layer order; 2 persistent: resident CTAs drain the same list
                           through a multi-stage TMA ring                             */
  int32_t fused;        /* 0 auto = 1; 1: launches of at most fused_waves waves of work items run the
                           schedule stage inside the update kernel (ONE launch); 2: never            */
  int32_t fused_waves;  /* default 4 (K <= 16), 2 (K <= 32), 1 (larger K)                            */
  int32_t tile_items;   /* float4 items (replicas x columns) per work item; default 1024            */
  int32_t variant;      /* grouped shape: thread shape of the update kernel, an index into update_tma.cu's
                           table (0 = the library's choice; 1 128 threads x 8 CTAs/SM, 2 512 x 2,
                           3 256 x 2, 4 512 x 3, 5 256 x 5 with the last array of x, g, m, v staged
                           through registers instead of shared memory -- what straggler-mode launches
                           take by default when the optimiser has state, 6 256 x 6 -- the default for
                           SGD without momentum and tiles of <= 1024 items, 7 512 x 3 with the same
                           split staging for tiles of 2048 items);
                           persistent shape: consumer groups per CTA (0 = as many as the ring feeds) */
  int32_t ctas_per_sm;  /* cap on resident CTAs per SM of persistent grids; default: all that fit   */
  int32_t pdl;          /* 0 auto = 1; 1: the update kernel is a programmatic dependent launch behind
                           the schedule kernel; 2: plain stream order                               */
  int32_t tma2d;        /* 0 auto (by K and optimiser); 1: tensor-map loads -- one 2-D tiled
                           TMA load per array and tile, and in straggler mode (skip_prob > 0 or a delay
                           straggler) tile::gather4 requests of four replica rows each; 2: 1-D bulk
                           copies, one per (replica, array) row the round needs (what auto takes in
                           straggler mode unless a tile row is only 128 B long, i.e. 8 float4 columns:
                           K > 64 at the default tile_items, smaller K with tile_items < 1024)      */
  int32_t stages;       /* persistent shape: depth of the TMA ring; default: as deep as fits        */
  int32_t group_threads;/* persistent shape: threads per consumer group (multiple of 32); default
                           512 with one group (768 for tiles of 2048+ items), 256 with more         */
} layup_tuning;

typedef struct {
  int32_t  K;          /* workers M of the paper, 1 <= K <= LAYUP_MAX_K    */
  int32_t  L;          /* layers                                                          */
  const int64_t *numel;/* [L] HOST: elements per layer (unpadded), each >= 1              */
  float    lr;         /* eta                                               */
  float    momentum;   /* mu; 0 => no M section in the arena                              */
  uint64_t seed;       /* Philox key of the peer selector and of the straggler mask       */
  int32_t  peer_mode;  /* 0: peer per (step, layer, replica)  [BASELINE.json north_star]
                          1: peer per (step, replica), all layers [Alg. 1, PAPER.md:101,453] */
  float    skip_prob;  /* straggler mode: P(replica idles this round); 0 = off            */
  int32_t  device;     /* CUDA ordinal                                                    */
  int32_t  delay_replica; /* delay-mode straggler: this replica ...           */
  int32_t  delay_rounds;  /* ... completes one iteration every delay_rounds+1 rounds (active
                          only when (step+1) % (delay_rounds+1) == 0) and keeps receiving in
                          between; 0 = off.  ANDed with the skip_prob mask    */
  int32_t  optimizer;  /* LAYUP_OPT_*: the local step of every worker                      */
  int32_t  mix_mode;   /* LAYUP_MIX_*: how a push meets the peer's copy                    */
  float    weight_decay; /* SGD: coupled, d = g + wd*x; AdamW: decoupled, x <- x(1-eta*wd)
                          (the weight_decay rows of PAPER.md:416-443, 469-491)             */
  float    beta1;      /* AdamW only: 0 <= beta1 < 1                                       */
  float    beta2;      /* AdamW only: 0 <= beta2 < 1                                       */
  float    eps;        /* AdamW only: >= 0                                                 */
  const layup_tuning *tuning; /* HOST, may be NULL (defaults); read during layup_init only         */
} layup_config;

/* Bytes of device memory the arena needs for this config (X + G (+ M (+ V)), padded). Pure. */
int layup_arena_bytes(const layup_config *cfg, size_t *bytes);

/* Create a ctx over a caller-owned DEVICE arena (128-B aligned, >= layup_arena_bytes).
 * Zeroes the arena, sets w[l][i] = 1/K and the step counters to 0.
 * Synchronous. */
int layup_init(const layup_config *cfg, void *arena_dev, size_t arena_bytes, layup_ctx **out);

/* Waits for the ctx's pending work, frees the library's tables.  The arena is untouched. */
int layup_destroy(layup_ctx *ctx);

/* Borrowed DEVICE pointer to slice (what, replica, layer) and its unpadded length. */
int layup_ptr(layup_ctx *ctx, int32_t what, int32_t replica, int32_t layer,
              float **dptr, int64_t *numel);

/* Learning-rate schedules live outside the path: lr is a scalar that
 * the next launching call picks up. */
int layup_set_lr(layup_ctx *ctx, float lr);

/* The paper's per-layer event ("Notify" / "Wait for notification"):
 * for ALL K replicas of `layer`, round `step`: straggler mask, peer choice, weight
 * halving, local step, push, peer update, weight add.  The layer's gradients must
 * already be in the arena in `cuda_stream` order.  Each layer must see step = 0,1,2,...
 * exactly once each (LAYUP_ESTATE otherwise); layers may be issued in any order and on
 * any streams -- they are independent -- but the paper's order is L-1 first
 * (PAPER.md:23,25).  cuda_stream: a cudaStream_t (NULL = legacy default stream). */
int layup_layer_update(layup_ctx *ctx, int64_t step, int32_t layer, void *cuda_stream);

/* All layers L-1 .. 0 of round `step` as ONE work list in reverse layer order:
 * by default a grouped launch, one CTA per (layer, tile) work item, which the hardware CTA
 * scheduler drains in list order (two kernels: schedule stage + update; one kernel when the
 * launch is small, see layup_tuning.fused; lists of more than 160 layers are split into
 * consecutive launches); with layup_tuning.launch_shape = 2 a persistent kernel whose resident
 * CTAs walk the same list.  Bit-identical to L calls of layup_layer_update. */
int layup_round(layup_ctx *ctx, int64_t step, void *cuda_stream);

/* layup_round with HOST buffers, layer-pipelined: for l = L-1..0 copy layer l's
 * gradients host->device, update it, copy its new parameters device->host, the three
 * stages of consecutive layers overlapping on the library's own streams.
 * g_host, x_host: [sum_l K*numel[l]] fp32, layer-major then replica (no padding), should
 * be pinned for the copies to be asynchronous; x_host may be NULL (no read-back).
 * Returns after the last copy has completed (synchronous).  The step bookkeeping is committed
 * only when the whole round succeeded; on a mid-round CUDA failure the library first waits for
 * its copy streams (the host buffers are no longer in use when the call returns), and the ctx
 * is POISONED: every later launching call returns LAYUP_ECUDA (the arena holds a partial round). */
int layup_round_host(layup_ctx *ctx, int64_t step, const float *g_host, float *x_host);

/* Wait for every stream the ctx has launched on; report the first sticky CUDA error. */
int layup_sync(layup_ctx *ctx);

/* ---- introspection for parity (read-only) ---------------------------------------- */

/* Host-side pure function: the peer replica `replica` pushes to in (step, layer), as
 * the kernels draw it: Philox4x32-10, key = seed, counter = (step, layer, replica, 0);
 * pass layer = -1 for peer_mode 1.  K >= 2. */
int layup_peer(uint64_t seed, int64_t step, int32_t layer, int32_t replica, int32_t K,
               int32_t *peer);

/* The peer choice and straggler mask of an ARBITRARY round `step`, drawn on the device by a
 * read-only kernel (the same draw_peer / draw_active device functions the schedule stage calls;
 * no state touched): peer[l*K+i] (-1 if replica i is inactive) and active[i].  What the update
 * kernel actually consumed in the last issued round is layup_schedule_tables().  Synchronous. */
int layup_schedule(layup_ctx *ctx, int64_t step, int32_t *peer /*[L*K]*/, uint8_t *active /*[K]*/);

/* The schedule tables the update kernel CONSUMED for the most recent (step, layer) event of
 * `layer`, as the schedule stage left them on the device (two-launch path: written by the
 * schedule kernel and read by the update kernel; single-launch path: the copy the update kernel
 * computed in shared memory, written out by the CTA that retires the layer):
 *   peer[i]      chosen peer of replica i, -1 if inactive
 *   flags[i]     bit 0: active (local step + push), bit 1: receives >= 1 push
 *   recv_off[j]  CSR by receiver: entries [recv_off[j], recv_off[j+1]) of senders/alpha
 *   senders[k]   sender of entry k, ascending within a receiver (R3)
 *   alpha[k]     w_i/(w_i+w_j) of that push, fp64 divide rounded once to fp32
 * With the symmetric mixer only peer and flags are meaningful (no sender list).  Any pointer may
 * be NULL.  step_done receives the step that event applied.  Waits for the ctx's work.  HOST. */
int layup_schedule_tables(layup_ctx *ctx, int32_t layer, int64_t *step_done, int32_t *peer /*[K]*/,
                          uint8_t *flags /*[K]*/, int32_t *recv_off /*[K+1]*/, int32_t *senders /*[K]*/,
                          float *alpha /*[K]*/);

/* Issue order ("output layer first"): the layers of the most recent launching
 * call in the order the library put them on the device -- the work-list positions of layup_round
 * / a graph, the per-layer launches of layup_round_host, the single layer of layup_layer_update.
 * layers: HOST [L]; *n = entries written. */
int layup_last_order(layup_ctx *ctx, int32_t *layers /*[L]*/, int32_t *n);

/* Device-side evidence of the same order: while enabled, the first CTA of every (step, layer)
 * event to start records the GPU's nanosecond timer (%globaltimer, atomicMin per layer).
 * layup_trace(ctx, 1) arms and clears; layup_trace_read copies out first_ns[l] (UINT64_MAX = layer
 * not started since arming) after waiting for the ctx's work.  HOST array. */
int layup_trace(layup_ctx *ctx, int32_t enable);
int layup_trace_read(layup_ctx *ctx, uint64_t *first_ns /*[L]*/);

/* Current push-sum weights w[l*K+i], after all work issued so far. */
int layup_weights(layup_ctx *ctx, double *w /*[L*K]*/);

/* Checkpoint / resume.  Everything the library owns besides the caller's arena: the push-sum
 * weights w[L*K], AdamW's running beta powers bpow[L*K*2] = (beta1^t, beta2^t)
 * per (layer, replica) (NULL unless the optimizer is AdamW) and the step each layer expects
 * next, next_step[L].  HOST arrays.  A ctx created with the same config over a copy of the
 * arena and given these three continues bit-identically.  Synchronous. */
int layup_state_export(layup_ctx *ctx, double *w, double *bpow, int64_t *next_step);
int layup_state_import(layup_ctx *ctx, const double *w, const double *bpow, const int64_t *next_step);

/* Model disagreement (PAPER.md:389-395 Fig. A1; eq. (9)): for every layer l and
 * replica i, dist[l*K+i] = sum_e (x_i[e] - xbar[e])^2, where xbar = (1/K) sum_i x_i (weighted == 0,
 * the paper's plain average) or xbar = sum_i w_i x_i with the current push-sum weights
 * (weighted != 0).  Runs a read-only reduction kernel (fp64 accumulation, 4 B of HBM traffic per
 * parameter) on `cuda_stream` -- after everything the ctx has issued so far (the library waits
 * for its own streams) and in stream order after the caller's own writes to x on that stream --
 * then copies dist to the HOST array and returns.  Synchronous. */
int layup_disagreement(layup_ctx *ctx, int32_t weighted, double *dist /*[L*K]*/, void *cuda_stream);
/* Device time of the reduction kernel(s) of the last layup_disagreement call (CUDA events). */
int layup_disagreement_ms(layup_ctx *ctx, double *ms);

/* ---- the same diagnostic for callers that must not allocate device memory ------------ */
/* Who this is for.  LayUp's per-layer events are issued from backward hooks while the backward
 * pass and earlier layers' gossip are still running on other streams.  A
 * monitoring hook that wants the disagreement curve of Fig. A1 from inside
 * that window must not call cudaMalloc / cudaFree: both wait for the whole device, which would
 * serialise exactly the overlap the method exists for.  The same holds for a job that has
 * handed all of HBM to the arena and to a framework's caching allocator (nothing is left for a
 * raw cudaMalloc to succeed with), and for a process that only borrows a parameter buffer in the
 * arena layout and never created a ctx -- layup_init allocates the library's tables, so a
 * ctx-based call is no use to it.
 *
 * layup_disagreement_static computes what layup_disagreement computes, with the same kernels,
 * without a ctx and without allocating anything, on the calling thread's CURRENT device.  The
 * accumulators the reduction kernel adds into, and the device copy of the weights, live in
 * one array compiled into the library: 2 * LAYUP_STATIC_MAX_PAIRS doubles (256 KiB) of device
 * memory on every GPU the process uses with this library, held from the moment the library's
 * code is loaded on that GPU until the process exits.
 *   x_dev    DEVICE, 128-B aligned, on the current device: one X section in the arena layout
 *            above for (K, L, numel) -- layer l starts at sum_{l'<l} K*pad(numel[l']) floats, its
 *            K slices pad(numel[l]) floats apart, pad(n) = n rounded up to 32, pad floats ZERO.
 *            layup_ptr(ctx, LAYUP_WHAT_X, 0, 0) of a ctx with the same (K, numel) is such a pointer.
 *   numel    HOST [L], each >= 1.        K in [1, LAYUP_MAX_K],  L >= 1.
 *   w        HOST [L*K] consensus coefficients (the push-sum weights of layup_weights for the
 *            weighted consensus), or NULL for the plain mean 1/K.
 *   dist     HOST [L*K] output, dist[l*K+i] as in layup_disagreement.
 * Limits and errors: L*K > LAYUP_STATIC_MAX_PAIRS, bad sizes, a misaligned x_dev or one that is
 * not device memory of the current device give LAYUP_EINVAL before anything is enqueued (text:
 * layup_last_error(NULL)); CUDA failures give LAYUP_ECUDA.  The call issues a memset of its
 * accumulators, the copy of w, the kernel(s) and the read-back on `cuda_stream`, in stream order
 * after the caller's writes to x on that stream, and returns when dist is complete (synchronous;
 * it does NOT wait for other streams -- order the writers of x before it yourself).  It calls no
 * cudaMalloc / cudaFree, creates no stream or event and uses no allocating library routine.
 * First call on each device: it looks up the device address of the array (cudaGetSymbolAddress)
 * and the SM count, once, and keeps them; make that first call outside any stream capture.
 * Sharing: every call on a device uses the one array, which still holds the previous call's
 * sums (each call clears the part it uses before its kernel).  Two calls that overlapped on the
 * GPU would race on it, so the library holds a process-wide lock from the first enqueue to the
 * final stream synchronise: calls from several host threads run one after the other. */
#define LAYUP_STATIC_MAX_PAIRS 16384   /* (layer, replica) pairs: L*K <= this                  */
int layup_disagreement_static(const float *x_dev, int32_t K, int32_t L, const int64_t *numel,
                              const double *w, double *dist, void *cuda_stream);

/* ---- CUDA-graph capture of launching calls ------------------------------------------ */
/* The round number is DEVICE state (one counter per layer, read and advanced by the schedule
 * stage), not a kernel argument, so a recorded sequence of launches can be replayed for later
 * rounds.  layup_graph_begin puts `cuda_stream` (not the legacy default stream) into capture;
 * the layup_layer_update / layup_round calls that follow ON THAT STREAM are recorded, not run
 * (their `step` arguments are checked as usual and count on from the ctx's state);
 * layup_graph_end closes the capture and instantiates it; layup_graph_launch replays the
 * recorded (layer) events for whatever rounds come next, advancing the ctx's step bookkeeping
 * by what was recorded.  Capture-time state is baked into the graph: the learning rate
 * (layup_set_lr needs a new capture) and whether layup_trace was armed (a graph captured while
 * tracing keeps stamping on every replay, one captured without never stamps; layup_trace calls
 * after the capture do not change either).  Typical use: one graph = one backward's worth of
 * per-layer events, or one or several whole rounds of an L2-resident model, where the launch
 * overhead, not HBM, is the cost.  layup_sync checks the device counters against
 * the host's bookkeeping (LAYUP_ESTATE on disagreement). */
int layup_graph_begin(layup_ctx *ctx, void *cuda_stream);
int layup_graph_end(layup_ctx *ctx, layup_graph **out);
int layup_graph_launch(layup_ctx *ctx, layup_graph *g, void *cuda_stream);
int layup_graph_destroy(layup_ctx *ctx, layup_graph *g);

/* Device time of the path's kernels, measured with CUDA events on the launch stream around
 * every launching call's kernels (the schedule kernel, a few microseconds, and the fused update
 * kernel): enable, run, layup_sync(), read (and reset).  launches = launching calls timed,
 * total_ms = sum of their durations. */
int layup_profile(layup_ctx *ctx, int32_t enable);
int layup_profile_read(layup_ctx *ctx, int64_t *launches, double *total_ms);

/* Kernels launched by this ctx so far (schedule + update kernels). */
int layup_launch_count(layup_ctx *ctx, int64_t *launches);

/* Text of the last error on this ctx (ctx may be NULL: last error of a ctx-less call). */
const char *layup_last_error(layup_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* LAYUP_H_ */
