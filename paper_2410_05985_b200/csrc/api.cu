// C-ABI of liblayup (include/layup.h): argument checking, arena layout, step bookkeeping,
// launches.  Every step of the path itself runs in the kernels of schedule.cu / update.cu.
#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "../../include/layup.h"
#include "layup_internal.cuh"
#include "philox.cuh"
#include "rule.cuh"

using namespace layup;

struct layup_ctx {
  int32_t K = 0, L = 0, device = 0, peer_mode = 0;
  float lr = 0.f, mu = 0.f, skip_prob = 0.f;
  int32_t optimizer = 0, mix_mode = 0, opt = 0, n_sections = 2;  // opt: OPT_* of rule.cuh
  float wd = 0.f, beta1 = 0.f, beta2 = 0.f, eps = 0.f;
  uint32_t skip_thr = 0;
  uint64_t seed = 0;
  std::vector<LayerDesc> layers;          // host copy
  std::vector<long long> tile_prefix;     // host copy, by position (pos p = layer L-1-p)
  std::vector<int64_t> next_step;         // per layer
  long long section = 0;                  // floats per section
  float *arena = nullptr;
  int C = 0, log2C = 0, smem = 0, ctas_per_sm = 1, n_sm = 1;
  layup_tuning tune{};                                 // layup_config.tuning (zeros = defaults)
  int variant = 0, threads = 256;
  int rega = 0;                                        // arrays the thread shape stages through registers
  bool straggler_mode = false;                         // skip_prob > 0 or a delay-mode straggler
  int split_variant = -1, split_smem = 0;              // thread shape of the launches that are not latency bound (-1: ctx->variant)
  bool persistent = false;                             // tuning.launch_shape == 2
  int engine = 1;                                      // 1: TMA-staged kernel, 0: LDG kernel
  int32_t delay_replica = 0, delay_rounds = 0;
  int diag_C = 0, diag_log2C = 0, diag_smem = 0, diag_ctas = 1;
  int diag_stages = 0;
  double *d_dist = nullptr;
  // device tables
  LayerDesc *d_layers = nullptr;
  long long *d_tile_prefix = nullptr;
  double *d_w = nullptr, *d_bpow = nullptr;
  SchedTables t{};
  int32_t *d_peer_scratch = nullptr, *d_ticket = nullptr;
  void *d_tmaps = nullptr;                // [n_sections][L] CUtensorMap: 2-D tiled view [K][pad] of every layer section
  void *d_tmaps_g4 = nullptr;             // ... with a one-row box, for tile::gather4 (straggler mode, grouped shape)
  bool ps_ok = false;                     // tuning.launch_shape == 2: persistent form of the TMA kernel
  int ps_smem = 0, ps_ctas = 0, ps_stages = 0, ps_groups = 1, ps_gs = 256;
  bool pdl = true;                        // programmatic dependent launch of the update kernel behind the schedule kernel
  bool fused_ok = false;                  // the single-launch path exists for this ctx (K, engine, variant)
  long long fused_max_tiles = 0;          // ... and is taken by launches of at most this many work items
  unsigned char *d_active_scratch = nullptr;
  uint32_t *d_step = nullptr;             // [L] round each layer runs next (device state, see layup.h graphs)
  int32_t *d_ps_ticket = nullptr;         // [L] tile tickets of persistent update launches, by work-list position
  int n_ps_ticket = 0;
  unsigned long long *d_trace = nullptr;  // [L] layup_trace
  bool tracing = false;
  // bookkeeping
  bool poisoned = false;                  // a launching call failed half way (layup_round_host)
  std::vector<int32_t> last_order;        // layup_last_order
  std::vector<int64_t> last_event_step;   // [L] step of the most recent event of each layer (-1: none)
  bool capturing = false;                 // between layup_graph_begin and layup_graph_end
  cudaStream_t cap_stream = nullptr;
  std::vector<int64_t> cap_next_step, cap_last_event;
  std::vector<int32_t> cap_order;
  int64_t cap_launches = 0;
  cudaEvent_t diag_ev0 = nullptr, diag_ev1 = nullptr;
  bool diag_timed = false;
  std::vector<cudaStream_t> streams;      // every stream launched on
  cudaStream_t own_stream = nullptr;      // introspection / init
  cudaStream_t s_h2d = nullptr, s_cmp = nullptr, s_d2h = nullptr;
  std::vector<cudaEvent_t> ev_h2d, ev_done;
  bool profiling = false;
  std::vector<std::pair<cudaEvent_t, cudaEvent_t>> prof_pending, prof_pool;
  int64_t launches = 0;
  std::string err;
};

struct layup_graph {
  cudaGraph_t graph = nullptr;
  cudaGraphExec_t exec = nullptr;
  layup_ctx *owner = nullptr;
  std::vector<int64_t> advance;           // [L] rounds each layer moves per replay
  std::vector<int32_t> order;             // layers in recorded issue order
  int64_t launches = 0;                   // kernels per replay
};

static thread_local std::string g_err;

// every entry point leaves the caller's current device as it found it
struct DeviceGuard {
  int prev = -1;
  cudaError_t err;
  explicit DeviceGuard(int dev) {
    err = cudaGetDevice(&prev);
    if (err == cudaSuccess && prev != dev) err = cudaSetDevice(dev);
  }
  ~DeviceGuard() {
    int cur = -1;
    if (prev >= 0 && cudaGetDevice(&cur) == cudaSuccess && cur != prev) cudaSetDevice(prev);
  }
};
#define LAYUP_ON_DEVICE(ctx)       \
  DeviceGuard guard__((ctx)->device); \
  CU_TRY(ctx, guard__.err)

static int fail(layup_ctx *ctx, int code, const char *fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  if (ctx) ctx->err = buf;
  g_err = buf;
  return code;
}

// ctx-less entry points of other translation units (diagnose.cu) leave their text behind layup_last_error(NULL)
void layup::note_error(const char *text) { g_err = text; }

#define CU_TRY(ctx, expr)                                                                      \
  do {                                                                                         \
    cudaError_t e__ = (expr);                                                                  \
    if (e__ != cudaSuccess)                                                                    \
      return fail(ctx, LAYUP_ECUDA, "%s: %s (%s:%d)", #expr, cudaGetErrorString(e__), __FILE__, __LINE__); \
  } while (0)

static long long pad32(long long n) { return (n + 31) / 32 * 32; }

static int check_config(const layup_config *cfg) {
  if (!cfg) return fail(nullptr, LAYUP_EINVAL, "config is NULL");
  if (cfg->K < 1 || cfg->K > LAYUP_MAX_K) return fail(nullptr, LAYUP_EINVAL, "K=%d outside [1,%d]", cfg->K, LAYUP_MAX_K);
  if (cfg->L < 1 || !cfg->numel) return fail(nullptr, LAYUP_EINVAL, "L=%d / numel invalid", cfg->L);
  for (int l = 0; l < cfg->L; ++l)
    if (cfg->numel[l] < 1) return fail(nullptr, LAYUP_EINVAL, "numel[%d]=%lld < 1", l, (long long)cfg->numel[l]);
  if (!(cfg->skip_prob >= 0.f && cfg->skip_prob <= 1.f)) return fail(nullptr, LAYUP_EINVAL, "skip_prob outside [0,1]");
  if (cfg->peer_mode != 0 && cfg->peer_mode != 1) return fail(nullptr, LAYUP_EINVAL, "peer_mode must be 0 or 1");
  if (!(cfg->momentum >= 0.f) || !(cfg->lr == cfg->lr)) return fail(nullptr, LAYUP_EINVAL, "lr / momentum invalid");
  if (cfg->optimizer != LAYUP_OPT_SGD && cfg->optimizer != LAYUP_OPT_ADAMW) return fail(nullptr, LAYUP_EINVAL, "optimizer must be 0 (SGD) or 1 (AdamW)");
  if (cfg->mix_mode < LAYUP_MIX_PUSHSUM || cfg->mix_mode > LAYUP_MIX_SYMMETRIC) return fail(nullptr, LAYUP_EINVAL, "mix_mode must be 0, 1 or 2");
  if (!(cfg->weight_decay >= 0.f)) return fail(nullptr, LAYUP_EINVAL, "weight_decay invalid");
  if (cfg->optimizer == LAYUP_OPT_ADAMW &&
      !(cfg->beta1 >= 0.f && cfg->beta1 < 1.f && cfg->beta2 >= 0.f && cfg->beta2 < 1.f && cfg->eps >= 0.f))
    return fail(nullptr, LAYUP_EINVAL, "AdamW needs 0 <= beta1, beta2 < 1 and eps >= 0");
  if (cfg->delay_rounds < 0 || (cfg->delay_rounds > 0 && (cfg->delay_replica < 0 || cfg->delay_replica >= cfg->K)))
    return fail(nullptr, LAYUP_EINVAL, "delay_replica / delay_rounds invalid");
  if (cfg->tuning) {
    const layup_tuning &t = *cfg->tuning;
    if (t.engine < 0 || t.engine > 2 || t.launch_shape < 0 || t.launch_shape > 2 || t.fused < 0 || t.fused > 2 ||
        t.pdl < 0 || t.pdl > 2 || t.tma2d < 0 || t.tma2d > 2 || t.fused_waves < 0 || t.tile_items < 0 ||
        t.variant < 0 || t.ctas_per_sm < 0 || t.stages < 0 || t.group_threads < 0)
      return fail(nullptr, LAYUP_EINVAL, "layup_tuning field out of range");
  }
  return LAYUP_OK;
}

static int n_sections(const layup_config *cfg) {      // X, G (, M (, V))
  return cfg->optimizer == LAYUP_OPT_ADAMW ? 4 : cfg->momentum != 0.f ? 3 : 2;
}

static long long section_floats(const layup_config *cfg) {
  long long s = 0;
  for (int l = 0; l < cfg->L; ++l) s += (long long)cfg->K * pad32(cfg->numel[l]);
  return s;
}

extern "C" int layup_arena_bytes(const layup_config *cfg, size_t *bytes) {
  int rc = check_config(cfg);
  if (rc) return rc;
  if (!bytes) return fail(nullptr, LAYUP_EINVAL, "bytes is NULL");
  *bytes = (size_t)section_floats(cfg) * sizeof(float) * n_sections(cfg);
  return LAYUP_OK;
}

static void note_stream(layup_ctx *ctx, cudaStream_t s) {
  if (std::find(ctx->streams.begin(), ctx->streams.end(), s) == ctx->streams.end()) ctx->streams.push_back(s);
}

extern "C" int layup_init(const layup_config *cfg, void *arena_dev, size_t arena_bytes, layup_ctx **out) {
  int rc = check_config(cfg);
  if (rc) return rc;
  if (!out) return fail(nullptr, LAYUP_EINVAL, "out is NULL");
  *out = nullptr;
  size_t need = 0;
  layup_arena_bytes(cfg, &need);
  if (!arena_dev || ((uintptr_t)arena_dev & 127u)) return fail(nullptr, LAYUP_EINVAL, "arena NULL or not 128-byte aligned");
  if (arena_bytes < need) return fail(nullptr, LAYUP_EINVAL, "arena too small: %zu < %zu", arena_bytes, need);

  int ndev = 0;
  CU_TRY(nullptr, cudaGetDeviceCount(&ndev));
  if (cfg->device < 0 || cfg->device >= ndev) return fail(nullptr, LAYUP_EINVAL, "device %d of %d", cfg->device, ndev);
  DeviceGuard guard(cfg->device);
  CU_TRY(nullptr, guard.err);

  layup_ctx *ctx = new layup_ctx();
  if (cfg->tuning) ctx->tune = *cfg->tuning;
  const layup_tuning &tune = ctx->tune;
  ctx->K = cfg->K; ctx->L = cfg->L; ctx->device = cfg->device; ctx->peer_mode = cfg->peer_mode;
  ctx->lr = cfg->lr; ctx->mu = cfg->momentum; ctx->skip_prob = cfg->skip_prob; ctx->seed = cfg->seed;
  {
    double th = (double)cfg->skip_prob * 4294967296.0;     // DESIGN R10: threshold in double, clamped
    if (th > 4294967295.0) th = 4294967295.0;
    ctx->skip_thr = cfg->skip_prob > 0.f ? (uint32_t)th : 0u;
  }
  ctx->delay_replica = cfg->delay_replica; ctx->delay_rounds = cfg->delay_rounds;
  ctx->optimizer = cfg->optimizer; ctx->mix_mode = cfg->mix_mode; ctx->wd = cfg->weight_decay;
  ctx->beta1 = cfg->beta1; ctx->beta2 = cfg->beta2; ctx->eps = cfg->eps;
  ctx->n_sections = n_sections(cfg);
  ctx->opt = cfg->optimizer == LAYUP_OPT_ADAMW ? OPT_ADAMW : cfg->momentum != 0.f ? OPT_SGD_MOM : OPT_SGD;
  ctx->arena = (float *)arena_dev;
  ctx->section = section_floats(cfg);

  // tile shape: C float4 columns per replica (power of two, >= 8), K*C items per tile.
  // Measured on B200: ~1024 items per CTA (48 KB staged with momentum, 4 CTAs/SM) is
  // best while a replica's row of the tile is >= 1 KB; for K >= 32 rows of 1 KB (C = 64) beat more
  // CTAs per SM as long as two CTAs still fit (staged bytes <= 112 KB).
  const int items_env = tune.tile_items;
  const int items_target = std::max(256, items_env > 0 ? items_env : 1024);
  int C = 8;
  while ((long long)cfg->K * C * 2 <= items_target && C < 4096) C *= 2;
  if (items_env <= 0)
    while (C < 64 && (long long)cfg->K * (2 * C) * 16 * ctx->n_sections <= 112 * 1024) C *= 2;
  // (smaller tiles for rounds of only a few work items per SM were tried: more CTAs repeating the
  //  fused schedule stage made configs[0] slower, 6.2 -> 8.2 us per round.)
  ctx->C = C;
  ctx->log2C = 0;
  while ((1 << ctx->log2C) < C) ++ctx->log2C;
  ctx->smem = (int)update_smem_bytes(cfg->K, C);

  const int K = cfg->K, L = cfg->L;
  ctx->layers.resize(L);
  long long base = 0;
  for (int l = 0; l < L; ++l) {
    ctx->layers[l] = LayerDesc{base, pad32(cfg->numel[l]), cfg->numel[l]};
    base += (long long)K * ctx->layers[l].pad;
  }
  ctx->tile_prefix.assign(L + 1, 0);
  for (int p = 0; p < L; ++p) {
    const LayerDesc &d = ctx->layers[L - 1 - p];
    const long long cols = d.pad / 4;
    ctx->tile_prefix[p + 1] = ctx->tile_prefix[p] + (cols + C - 1) / C;
  }
  ctx->next_step.assign(L, 0);

  cudaDeviceProp prop;
  auto bail = [&](int code) { layup_destroy(ctx); return code; };
#define CU_TRY_INIT(expr)                                                                               \
  do {                                                                                                  \
    cudaError_t e__ = (expr);                                                                           \
    if (e__ != cudaSuccess) {                                                                           \
      fail(nullptr, LAYUP_ECUDA, "%s: %s (%s:%d)", #expr, cudaGetErrorString(e__), __FILE__, __LINE__); \
      return bail(LAYUP_ECUDA);                                                                         \
    }                                                                                                   \
  } while (0)
  CU_TRY_INIT(cudaGetDeviceProperties(&prop, cfg->device));
  ctx->n_sm = prop.multiProcessorCount;
  if ((size_t)ctx->smem > prop.sharedMemPerBlockOptin) {
    fail(nullptr, LAYUP_EINVAL, "K=%d needs %d B of shared memory per CTA", K, ctx->smem);
    return bail(LAYUP_EINVAL);
  }
  ctx->engine = tune.engine == 2 ? 0 : 1;
  ctx->straggler_mode = ctx->skip_thr != 0u || ctx->delay_rounds != 0;     // some replicas may idle in a round
  // Straggler mode fetches exactly the rows a round needs: row-by-row bulk copies, or tile::gather4
  // requests of four rows each.  Measured on B200 the two tie while a row is >= 256 B
  // and gather4 wins once rows shrink to 128 B (K >= 128: up to 18 %), so auto takes it there.
  const bool want_g4 = ctx->straggler_mode && tune.launch_shape != 2 && C * 4 <= 256 &&
                       (tune.tma2d == 1 || (tune.tma2d == 0 && C <= 8));
  ctx->persistent = tune.launch_shape == 2;
  ctx->variant = (ctx->persistent && tune.engine != 2) ? 0 : tune.variant;   // persistent TMA shape: variant = consumer groups
  ctx->pdl = tune.pdl != 2;
  if (ctx->engine == 1) {
    // TMA-staged kernel stages x, g (, m) of the whole tile: fall back to the LDG kernel if it does not fit
    if (ctx->variant < 0 || ctx->variant >= tma_num_variants()) ctx->variant = 0;
    if (tune.variant == 0) ctx->variant = tma_default_variant(K * C, ctx->n_sections);
    ctx->fused_ok = K <= kFusedMaxK && tma_has_fused(ctx->variant) && tune.fused != 2;
    ctx->rega = tma_variant_rega(ctx->variant, ctx->opt);
    const int max_items = tma_variant_max_items(ctx->variant);
    if (max_items > 0 && K * C > max_items) {
      fail(nullptr, LAYUP_EINVAL, "thread shape %d takes tiles of at most %d items (this ctx: %d)", ctx->variant, max_items, K * C);
      return bail(LAYUP_EINVAL);
    }
    const size_t need_smem = tma_smem_bytes(K, C, ctx->opt, ctx->fused_ok, ctx->rega, want_g4);
    if (need_smem > prop.sharedMemPerBlockOptin) { ctx->engine = 0; ctx->fused_ok = false; }
    else ctx->smem = (int)need_smem;
  }
  if (ctx->engine == 1) {
    CU_TRY_INIT(tma_kernel_setup(ctx->variant, ctx->opt, ctx->mix_mode == kMixSymmetric, ctx->straggler_mode, ctx->smem, &ctx->threads, &ctx->ctas_per_sm));
    // Launches that are not latency bound may take a thread shape of their own: split
    // staging (last array through registers, five CTAs per SM) in straggler mode with optimiser
    // state, six CTAs per SM for two-array tiles of <= 1024 items
    if (tune.variant == 0) {
      ctx->split_variant = tma_bulk_variant(K * C, ctx->n_sections, ctx->straggler_mode);
      if (ctx->split_variant >= 0) {
        int thr = 0, occ = 0;
        ctx->split_smem = (int)tma_smem_bytes(K, C, ctx->opt, false, tma_variant_rega(ctx->split_variant, ctx->opt), want_g4);
        CU_TRY_INIT(tma_kernel_setup(ctx->split_variant, ctx->opt, ctx->mix_mode == kMixSymmetric, ctx->straggler_mode, ctx->split_smem, &thr, &occ));
      }
    }
  } else {
    if (ctx->variant < 0 || ctx->variant >= update_num_variants()) ctx->variant = 0;
    CU_TRY_INIT(update_kernel_setup(ctx->variant, ctx->opt, ctx->mix_mode == kMixSymmetric, ctx->smem, &ctx->threads, &ctx->ctas_per_sm));
  }
  if (ctx->ctas_per_sm < 1) ctx->ctas_per_sm = 1;
  // launches of up to this many work items are launch-latency bound: one fused launch beats two
  // (measured on B200 with every launch fused: K = 8 ties, K = 16 loses 8 %, K = 64 loses 45 % on
  //  HBM-sized rounds -- the redundant schedule stage is only free while the launch is latency bound)
  //  (K = 8 always fused: per-layer events 3.03 -> 2.97 ms per round, but AdamW rounds -0.7 % and
  //  straggler rounds -12 %, where the schedule stage sits in front of the loads: not done.)
  //  (the redundant stage is O(K) per CTA: per-layer events of configs[4], K = 64, 1.005 ms per round with a
  //  4-wave bound, 0.957 with 1 wave; configs[1], K = 8: 2.99 ms with 4 waves, 3.03 with 1 or 2)
  const int waves = tune.fused_waves > 0 ? tune.fused_waves : (K <= 16 ? 4 : K <= 32 ? 2 : 1);
  ctx->fused_max_tiles = (long long)waves * ctx->n_sm * ctx->ctas_per_sm;
  const int cap = tune.ctas_per_sm;
  if (cap > 0 && cap < ctx->ctas_per_sm) ctx->ctas_per_sm = cap;

  CU_TRY_INIT(cudaStreamCreateWithFlags(&ctx->own_stream, cudaStreamNonBlocking));
  CU_TRY_INIT(cudaMalloc(&ctx->d_layers, sizeof(LayerDesc) * L));
  CU_TRY_INIT(cudaMalloc(&ctx->d_tile_prefix, sizeof(long long) * (L + 1)));
  CU_TRY_INIT(cudaMalloc(&ctx->d_w, sizeof(double) * L * K));
  CU_TRY_INIT(cudaMalloc(&ctx->t.peer, sizeof(int32_t) * L * K));
  CU_TRY_INIT(cudaMalloc(&ctx->t.recv_off, sizeof(int32_t) * L * (K + 1)));
  CU_TRY_INIT(cudaMalloc(&ctx->t.senders, sizeof(int32_t) * L * K));
  CU_TRY_INIT(cudaMalloc(&ctx->t.alpha, sizeof(float) * L * K));
  CU_TRY_INIT(cudaMalloc(&ctx->t.flags, (size_t)L * K));
  if (ctx->opt == OPT_ADAMW) {
    CU_TRY_INIT(cudaMalloc(&ctx->t.c1, sizeof(float) * L * K));
    CU_TRY_INIT(cudaMalloc(&ctx->t.c2, sizeof(float) * L * K));
    CU_TRY_INIT(cudaMalloc(&ctx->d_bpow, sizeof(double) * 2 * L * K));
    std::vector<double> ones((size_t)2 * L * K, 1.0);                    // beta^0
    CU_TRY_INIT(cudaMemcpy(ctx->d_bpow, ones.data(), sizeof(double) * 2 * L * K, cudaMemcpyHostToDevice));
    CU_TRY_INIT(cudaMemset(ctx->t.c1, 0, sizeof(float) * L * K));
    CU_TRY_INIT(cudaMemset(ctx->t.c2, 0, sizeof(float) * L * K));
  }
  CU_TRY_INIT(cudaMalloc(&ctx->d_peer_scratch, sizeof(int32_t) * L * K));
  CU_TRY_INIT(cudaMalloc(&ctx->d_ticket, sizeof(int32_t) * L));
  CU_TRY_INIT(cudaMemset(ctx->d_ticket, 0, sizeof(int32_t) * L));
  CU_TRY_INIT(cudaMalloc(&ctx->d_active_scratch, (size_t)K));
  CU_TRY_INIT(cudaMalloc(&ctx->d_dist, sizeof(double) * L * K));
  CU_TRY_INIT(cudaMalloc(&ctx->d_step, sizeof(uint32_t) * L));
  CU_TRY_INIT(cudaMemset(ctx->d_step, 0, sizeof(uint32_t) * L));
  ctx->n_ps_ticket = L;                   // one per work-list position: launches on different streams never share one
  CU_TRY_INIT(cudaMalloc(&ctx->d_ps_ticket, sizeof(int32_t) * ctx->n_ps_ticket));
  CU_TRY_INIT(cudaMemset(ctx->d_ps_ticket, 0, sizeof(int32_t) * ctx->n_ps_ticket));
  CU_TRY_INIT(cudaMalloc(&ctx->d_trace, sizeof(unsigned long long) * L));
  CU_TRY_INIT(cudaMemset(ctx->d_trace, 0xFF, sizeof(unsigned long long) * L));
  ctx->last_event_step.assign(L, -1);
  // 2-D tile loads replace K*arrays 1-D bulk copies per CTA by one per array.  Measured on B200: a
  // clear win without momentum (K = 16: 6.27 -> 6.94 TB/s) and from 64 copies per CTA up; at
  // K = 16 with momentum (48 copies) the 1-D form is 0.2 % ahead, so it is kept there.
  // (the persistent shape issues a tile's loads from one warp: always the 2-D form there)
  // Straggler mode with tma2d = 1 (grouped shape): the same views with a ONE-row box, read four
  // arbitrary rows at a time with tile::gather4.
  const int n_staged = ctx->n_sections - ctx->rega;
  const bool want_2d = tune.tma2d == 1 || (tune.tma2d == 0 && (n_staged <= 2 || K * n_staged >= 64 || ctx->persistent));
  if (ctx->engine == 1 && C * 4 <= 256 && (want_g4 || (!ctx->straggler_mode && want_2d && K <= 256))) {
    // One tensor map per (section, layer): rank 2, inner dim = the padded slice, outer dim = the K
    // replicas (stride = pad), box = [K][C*4 floats] ([1][C*4] for gather4), no swizzle, zero fill
    // past the slice end.
    typedef CUresult (*EncodeTiled)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                    const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    bool ok = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) == cudaSuccess &&
              qres == cudaDriverEntryPointSuccess && fn != nullptr;
    std::vector<CUtensorMap> maps((size_t)ctx->n_sections * L);
    for (int a = 0; ok && a < ctx->n_sections; ++a)
      for (int l = 0; ok && l < L; ++l) {
        const LayerDesc &d = ctx->layers[l];
        if (d.pad >= (1ll << 31)) { ok = false; break; }                  // box coordinates are int32
        const cuuint64_t gdim[2] = {(cuuint64_t)d.pad, (cuuint64_t)K};
        const cuuint64_t gstride[1] = {(cuuint64_t)d.pad * sizeof(float)};
        const cuuint32_t box[2] = {(cuuint32_t)(C * 4), want_g4 ? 1u : (cuuint32_t)K};
        const cuuint32_t estride[2] = {1, 1};
        void *base_ptr = ctx->arena + (long long)a * ctx->section + d.base;
        ok = ((EncodeTiled)fn)(&maps[(size_t)a * L + l], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, base_ptr, gdim, gstride, box,
                               estride, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                               CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
      }
    cudaGetLastError();
    if (ok) {
      void **slot = want_g4 ? &ctx->d_tmaps_g4 : &ctx->d_tmaps;
      CU_TRY_INIT(cudaMalloc(slot, sizeof(CUtensorMap) * maps.size()));
      CU_TRY_INIT(cudaMemcpy(*slot, maps.data(), sizeof(CUtensorMap) * maps.size(), cudaMemcpyHostToDevice));
    }
  }
  if (ctx->engine == 1 && ctx->persistent) {
    // no silent fallback: the persistent shape either exists for this ctx or init says why not
    if (K > persist_max_k()) {
      fail(nullptr, LAYUP_EINVAL, "launch_shape = persistent needs K <= %d with the TMA engine", persist_max_k());
      return bail(LAYUP_EINVAL);
    }
    const int want_ctas = tune.ctas_per_sm > 0 ? tune.ctas_per_sm : 1;
    ctx->ps_stages = persist_stages(K, C, ctx->opt, prop.sharedMemPerBlockOptin, want_ctas, tune.stages);
    if (ctx->ps_stages < 2) {
      fail(nullptr, LAYUP_EINVAL, "launch_shape = persistent: two stages of this tile do not fit in shared memory");
      return bail(LAYUP_EINVAL);
    }
    persist_shape(&ctx->ps_stages, K * C, tune.variant, tune.group_threads, &ctx->ps_groups, &ctx->ps_gs);
    ctx->ps_smem = (int)persist_smem_bytes(K, C, ctx->opt, ctx->ps_stages);
    CU_TRY_INIT(persist_kernel_setup(ctx->opt, ctx->mix_mode == kMixSymmetric, ctx->ps_smem, &ctx->ps_ctas));
    if (ctx->ps_ctas > want_ctas) ctx->ps_ctas = want_ctas;
    if (ctx->ps_ctas < 1) {
      fail(nullptr, LAYUP_EINVAL, "launch_shape = persistent: the kernel does not fit on an SM");
      return bail(LAYUP_EINVAL);
    }
    ctx->ps_ok = true;
  }
  CU_TRY_INIT(cudaMemcpy(ctx->d_layers, ctx->layers.data(), sizeof(LayerDesc) * L, cudaMemcpyHostToDevice));
  CU_TRY_INIT(cudaMemcpy(ctx->d_tile_prefix, ctx->tile_prefix.data(), sizeof(long long) * (L + 1), cudaMemcpyHostToDevice));
  std::vector<double> w0((size_t)L * K, 1.0 / (double)K);              // PAPER.md:106  w_i = 1/M
  CU_TRY_INIT(cudaMemcpy(ctx->d_w, w0.data(), sizeof(double) * L * K, cudaMemcpyHostToDevice));
  CU_TRY_INIT(cudaMemset(ctx->t.recv_off, 0, sizeof(int32_t) * L * (K + 1)));
  CU_TRY_INIT(cudaMemset(ctx->t.flags, 0, (size_t)L * K));
  CU_TRY_INIT(cudaMemset(ctx->t.peer, 0xFF, sizeof(int32_t) * L * K));
  CU_TRY_INIT(cudaMemset(ctx->t.senders, 0, sizeof(int32_t) * L * K));
  CU_TRY_INIT(cudaMemset(ctx->t.alpha, 0, sizeof(float) * L * K));
  CU_TRY_INIT(cudaMemset(arena_dev, 0, need));                          // pads are zero and stay zero
  CU_TRY_INIT(cudaDeviceSynchronize());
#undef CU_TRY_INIT
  *out = ctx;
  return LAYUP_OK;
}

extern "C" int layup_destroy(layup_ctx *ctx) {
  if (!ctx) return LAYUP_OK;
  DeviceGuard guard(ctx->device);
  if (ctx->capturing) {                                    // abandon an open capture
    cudaGraph_t g = nullptr;
    cudaStreamEndCapture(ctx->cap_stream, &g);
    if (g) cudaGraphDestroy(g);
    cudaGetLastError();
  }
  for (cudaStream_t s : ctx->streams) cudaStreamSynchronize(s);
  for (cudaStream_t s : {ctx->own_stream, ctx->s_h2d, ctx->s_cmp, ctx->s_d2h})
    if (s) { cudaStreamSynchronize(s); cudaStreamDestroy(s); }
  for (auto &v : {ctx->ev_h2d, ctx->ev_done})
    for (cudaEvent_t e : v) cudaEventDestroy(e);
  for (auto &pr : ctx->prof_pending) { cudaEventDestroy(pr.first); cudaEventDestroy(pr.second); }
  for (auto &pr : ctx->prof_pool) { cudaEventDestroy(pr.first); cudaEventDestroy(pr.second); }
  if (ctx->diag_ev0) cudaEventDestroy(ctx->diag_ev0);
  if (ctx->diag_ev1) cudaEventDestroy(ctx->diag_ev1);
  cudaFree(ctx->d_layers); cudaFree(ctx->d_tile_prefix); cudaFree(ctx->d_w);
  cudaFree(ctx->t.peer); cudaFree(ctx->t.recv_off); cudaFree(ctx->t.senders); cudaFree(ctx->t.alpha);
  cudaFree(ctx->t.c1); cudaFree(ctx->t.c2); cudaFree(ctx->d_bpow);
  cudaFree(ctx->t.flags); cudaFree(ctx->d_peer_scratch); cudaFree(ctx->d_ticket); cudaFree(ctx->d_tmaps); cudaFree(ctx->d_tmaps_g4);
  cudaFree(ctx->d_active_scratch); cudaFree(ctx->d_dist); cudaFree(ctx->d_step); cudaFree(ctx->d_trace); cudaFree(ctx->d_ps_ticket);
  delete ctx;
  return LAYUP_OK;
}

extern "C" int layup_ptr(layup_ctx *ctx, int32_t what, int32_t replica, int32_t layer, float **dptr, int64_t *numel) {
  if (!ctx || !dptr) return fail(ctx, LAYUP_EINVAL, "ctx or dptr is NULL");
  if (what < 0 || what >= ctx->n_sections) return fail(ctx, LAYUP_EINVAL, "what=%d not in this arena", what);
  if (replica < 0 || replica >= ctx->K || layer < 0 || layer >= ctx->L) return fail(ctx, LAYUP_EINVAL, "replica %d / layer %d out of range", replica, layer);
  const LayerDesc &d = ctx->layers[layer];
  *dptr = ctx->arena + (long long)what * ctx->section + d.base + (long long)replica * d.pad;
  if (numel) *numel = d.numel;
  return LAYUP_OK;
}

extern "C" int layup_set_lr(layup_ctx *ctx, float lr) {
  if (!ctx || !(lr == lr)) return fail(ctx, LAYUP_EINVAL, "ctx NULL or lr NaN");
  ctx->lr = lr;
  return LAYUP_OK;
}

// what every launching call checks first
static int check_launchable(layup_ctx *ctx, int64_t step, cudaStream_t s) {
  if (ctx->poisoned) return fail(ctx, LAYUP_ECUDA, "ctx is poisoned: an earlier launching call failed half way through a round");
  if (step < 0 || step > 0xFFFFFFFFll) return fail(ctx, LAYUP_EINVAL, "step %lld outside [0, 2^32)", (long long)step);
  if (ctx->capturing && s != ctx->cap_stream)
    return fail(ctx, LAYUP_EINVAL, "a graph capture is open on another stream (layup_graph_begin)");
  return LAYUP_OK;
}

// schedule kernel + update kernel for positions [pos_begin, pos_end) of the reverse-ordered list.
// The round number itself is device state (d_step); `step` only feeds the host's bookkeeping.
static int issue_kernels(layup_ctx *ctx, int pos_begin, int pos_end, cudaStream_t s, int *n_kernels) {
  const int L = ctx->L;
  SchedParams sp{};
  sp.t = ctx->t; sp.w = ctx->d_w; sp.seed = ctx->seed; sp.step_dev = ctx->d_step; sp.skip_thr = ctx->skip_thr;
  sp.K = ctx->K; sp.L = L; sp.peer_mode = ctx->peer_mode;
  sp.delay_replica = ctx->delay_replica; sp.delay_rounds = ctx->delay_rounds;
  sp.layer_begin = L - pos_end;                       // layers [L-pos_end, L-pos_begin)
  sp.mix_mode = ctx->mix_mode; sp.adamw = ctx->opt == OPT_ADAMW ? 1 : 0; sp.bpow = ctx->d_bpow;
  sp.lr = (double)ctx->lr; sp.beta1 = (double)ctx->beta1; sp.beta2 = (double)ctx->beta2;
  sp.ticket = ctx->d_ticket;
  sp.ps_ticket = ctx->d_ps_ticket; sp.n_ps_ticket = ctx->ps_ok ? ctx->n_ps_ticket : 0;
  const bool fused = ctx->fused_ok && ctx->tile_prefix[pos_end] - ctx->tile_prefix[pos_begin] <= ctx->fused_max_tiles;
  *n_kernels = 0;                                     // kernels enqueued so far (the caller poisons the ctx on a late failure)
  if (!fused) {
    CU_TRY(ctx, launch_schedule(sp, pos_end - pos_begin, s));
    *n_kernels += 1;
  }

  UpdateParams up{};
  up.x = ctx->arena;
  up.g = ctx->arena + ctx->section;
  up.m = ctx->n_sections >= 3 ? ctx->arena + 2 * ctx->section : nullptr;
  up.v = ctx->n_sections >= 4 ? ctx->arena + 3 * ctx->section : nullptr;
  up.layers = ctx->d_layers; up.tile_prefix = ctx->d_tile_prefix; up.t = ctx->t;
  up.tile_begin = ctx->tile_prefix[pos_begin]; up.tile_end = ctx->tile_prefix[pos_end];
  up.K = ctx->K; up.L = L; up.C = ctx->C; up.log2C = ctx->log2C; up.pos_begin = pos_begin; up.pos_end = pos_end;
  up.s.neg_lr = -ctx->lr; up.s.mu = ctx->mu; up.s.wd = ctx->opt == OPT_ADAMW ? 0.f : ctx->wd;
  up.s.b1 = ctx->beta1; up.s.b2 = ctx->beta2; up.s.eps = ctx->eps;
  up.s.omb1 = (float)(1.0 - (double)ctx->beta1); up.s.omb2 = (float)(1.0 - (double)ctx->beta2);
  up.s.decay = (float)(1.0 - (double)ctx->lr * (double)ctx->wd);          // AdamW: x <- x (1 - eta*wd)
  up.opt = ctx->opt; up.symmetric = ctx->mix_mode == kMixSymmetric ? 1 : 0;
  up.all_active = (ctx->skip_thr == 0u && ctx->delay_rounds == 0) ? 1 : 0;
  up.sched = sp;
  up.tmaps = ctx->d_tmaps;
  up.tmaps_g4 = ctx->d_tmaps_g4;
  up.trace = ctx->tracing ? ctx->d_trace : nullptr;
  const long long tiles = up.tile_end - up.tile_begin;
  const long long resident = (long long)ctx->n_sm * ctx->ctas_per_sm;

  int n_launch = 0;
  if (ctx->engine == 1) {
    // one launch per <= kMaxPos positions: the work-list table travels in the kernel parameters
    for (int q0 = pos_begin; q0 < pos_end;) {
      PosTable tab;
      int n = 0;
      const long long t0 = ctx->tile_prefix[q0];
      while (q0 + n < pos_end && n < kMaxPos && ctx->tile_prefix[q0 + n + 1] - t0 <= 0x7FFFFFFFll) {
        tab.prefix[n] = ctx->tile_prefix[q0 + n] - t0;
        tab.lay[n] = ctx->layers[L - 1 - (q0 + n)];
        tab.layer[n] = L - 1 - (q0 + n);
        ++n;
      }
      if (n == 0) return fail(ctx, LAYUP_EINVAL, "layer %d has more than 2^31 tiles", L - 1 - q0);
      tab.prefix[n] = ctx->tile_prefix[q0 + n] - t0;
      tab.n = n;
      // only the first update launch directly follows the schedule kernel on the stream
      if (ctx->ps_ok && !fused) {
        up.ps_ticket = ctx->d_ps_ticket + q0;          // the slot of this launch's first position (schedule.cu re-arms it)
        const int grid = (int)std::min<long long>(tab.prefix[n], (long long)ctx->n_sm * ctx->ps_ctas);
        CU_TRY(ctx, launch_update_persist(up, tab, grid, ctx->ps_smem, ctx->ps_stages, ctx->ps_groups, ctx->ps_gs, ctx->pdl && n_launch == 0, s));
      } else {
        const bool split = !fused && ctx->split_variant >= 0;
        CU_TRY(ctx, launch_update_tma(up, tab, split ? ctx->split_variant : ctx->variant, fused, ctx->pdl && n_launch == 0,
                                      (int)tab.prefix[n], split ? ctx->split_smem : ctx->smem, s));
      }
      q0 += n;
      ++n_launch;
      *n_kernels += 1;
    }
  } else {
    // LDG kernel: grouped (one CTA per work item) unless a persistent grid was asked for
    const bool persistent = ctx->persistent || tiles > 0x7FFFFFFFll;
    const int grid = (int)(persistent ? std::min<long long>(tiles, resident) : tiles);
    CU_TRY(ctx, launch_update(up, ctx->variant, persistent, grid, ctx->smem, s));
    *n_kernels += 1;
  }
  return LAYUP_OK;
}

static int issue(layup_ctx *ctx, int64_t step, int pos_begin, int pos_end, cudaStream_t s) {
  // profiling brackets the whole issue: the schedule kernel (a few us, overlapped with the update
  // kernel's prologue by the programmatic dependent launch) and the update kernel(s); not while
  // a graph is being captured (nothing runs then)
  std::pair<cudaEvent_t, cudaEvent_t> ev{nullptr, nullptr};
  const bool prof = ctx->profiling && !ctx->capturing;
  if (prof) {
    if (!ctx->prof_pool.empty()) { ev = ctx->prof_pool.back(); ctx->prof_pool.pop_back(); }
    else {
      CU_TRY(ctx, cudaEventCreate(&ev.first));
      cudaError_t e = cudaEventCreate(&ev.second);
      if (e != cudaSuccess) { cudaEventDestroy(ev.first); CU_TRY(ctx, e); }
    }
  }
  int n_kernels = 0;
  int rc = LAYUP_OK;
  if (prof && cudaEventRecord(ev.first, s) != cudaSuccess) rc = fail(ctx, LAYUP_ECUDA, "cudaEventRecord failed");
  if (rc == LAYUP_OK) rc = issue_kernels(ctx, pos_begin, pos_end, s, &n_kernels);
  if (rc == LAYUP_OK && prof && cudaEventRecord(ev.second, s) != cudaSuccess) rc = fail(ctx, LAYUP_ECUDA, "cudaEventRecord failed");
  if (prof) (rc == LAYUP_OK ? ctx->prof_pending : ctx->prof_pool).push_back(ev);   // never leaked
  if (rc != LAYUP_OK) {
    // a kernel of this call is already on the stream (the schedule stage advances the device's round
    // counter and halves the weights): the host's bookkeeping can no longer be trusted to match
    if (n_kernels > 0 && !ctx->capturing) ctx->poisoned = true;
    return rc;
  }
  ctx->launches += n_kernels;
  for (int p = pos_begin; p < pos_end; ++p) {
    ctx->last_order.push_back(ctx->L - 1 - p);
    ctx->last_event_step[ctx->L - 1 - p] = step;
  }
  note_stream(ctx, s);
  return LAYUP_OK;
}

extern "C" int layup_layer_update(layup_ctx *ctx, int64_t step, int32_t layer, void *cuda_stream) {
  if (!ctx) return fail(nullptr, LAYUP_EINVAL, "ctx is NULL");
  if (layer < 0 || layer >= ctx->L) return fail(ctx, LAYUP_EINVAL, "layer %d out of range", layer);
  int rc = check_launchable(ctx, step, (cudaStream_t)cuda_stream);
  if (rc) return rc;
  if (ctx->next_step[layer] != step)
    return fail(ctx, LAYUP_ESTATE, "layer %d expects step %lld, got %lld", layer, (long long)ctx->next_step[layer], (long long)step);
  LAYUP_ON_DEVICE(ctx);
  const int pos = ctx->L - 1 - layer;
  if (!ctx->capturing) ctx->last_order.clear();
  rc = issue(ctx, step, pos, pos + 1, (cudaStream_t)cuda_stream);
  if (rc == LAYUP_OK) ctx->next_step[layer] = step + 1;
  return rc;
}

extern "C" int layup_round(layup_ctx *ctx, int64_t step, void *cuda_stream) {
  if (!ctx) return fail(nullptr, LAYUP_EINVAL, "ctx is NULL");
  int rc = check_launchable(ctx, step, (cudaStream_t)cuda_stream);
  if (rc) return rc;
  for (int l = 0; l < ctx->L; ++l)
    if (ctx->next_step[l] != step)
      return fail(ctx, LAYUP_ESTATE, "layer %d expects step %lld, got %lld", l, (long long)ctx->next_step[l], (long long)step);
  LAYUP_ON_DEVICE(ctx);
  if (!ctx->capturing) ctx->last_order.clear();
  rc = issue(ctx, step, 0, ctx->L, (cudaStream_t)cuda_stream);
  if (rc == LAYUP_OK)
    for (int l = 0; l < ctx->L; ++l) ctx->next_step[l] = step + 1;
  return rc;
}

extern "C" int layup_round_host(layup_ctx *ctx, int64_t step, const float *g_host, float *x_host) {
  if (!ctx || !g_host) return fail(ctx, LAYUP_EINVAL, "ctx or g_host is NULL");
  if (ctx->capturing) return fail(ctx, LAYUP_ESTATE, "layup_round_host cannot be recorded into a graph");
  int rc = check_launchable(ctx, step, nullptr);
  if (rc) return rc;
  const int L = ctx->L, K = ctx->K;
  for (int l = 0; l < L; ++l)
    if (ctx->next_step[l] != step)
      return fail(ctx, LAYUP_ESTATE, "layer %d expects step %lld, got %lld", l, (long long)ctx->next_step[l], (long long)step);
  LAYUP_ON_DEVICE(ctx);
  if (!ctx->s_h2d) {
    CU_TRY(ctx, cudaStreamCreateWithFlags(&ctx->s_h2d, cudaStreamNonBlocking));
    CU_TRY(ctx, cudaStreamCreateWithFlags(&ctx->s_cmp, cudaStreamNonBlocking));
    CU_TRY(ctx, cudaStreamCreateWithFlags(&ctx->s_d2h, cudaStreamNonBlocking));
  }
  if ((int)ctx->ev_done.size() < L) {
    ctx->ev_h2d.reserve(L); ctx->ev_done.reserve(L);
    while ((int)ctx->ev_h2d.size() < L) {
      cudaEvent_t e;
      CU_TRY(ctx, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
      ctx->ev_h2d.push_back(e);
    }
    while ((int)ctx->ev_done.size() < L) {
      cudaEvent_t e;
      CU_TRY(ctx, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
      ctx->ev_done.push_back(e);
    }
  }
  std::vector<long long> hoff(L + 1, 0);                   // host offsets, layer-major, unpadded
  for (int l = 0; l < L; ++l) hoff[l + 1] = hoff[l] + (long long)K * ctx->layers[l].numel;
  float *gsec = ctx->arena + ctx->section;
  ctx->last_order.clear();
  // validate-then-commit: next_step moves only after the whole round is on the device and done
  auto pipeline = [&]() -> int {
    for (int l = L - 1; l >= 0; --l) {                     // output layer first
      const LayerDesc &d = ctx->layers[l];
      const size_t row = (size_t)d.numel * sizeof(float);
      CU_TRY(ctx, cudaMemcpy2DAsync(gsec + d.base, (size_t)d.pad * sizeof(float), g_host + hoff[l], row, row, K,
                                    cudaMemcpyHostToDevice, ctx->s_h2d));
      CU_TRY(ctx, cudaEventRecord(ctx->ev_h2d[l], ctx->s_h2d));
      CU_TRY(ctx, cudaStreamWaitEvent(ctx->s_cmp, ctx->ev_h2d[l], 0));
      const int pos = L - 1 - l;
      int r = issue(ctx, step, pos, pos + 1, ctx->s_cmp);
      if (r) return r;
      if (x_host) {
        CU_TRY(ctx, cudaEventRecord(ctx->ev_done[l], ctx->s_cmp));
        CU_TRY(ctx, cudaStreamWaitEvent(ctx->s_d2h, ctx->ev_done[l], 0));
        CU_TRY(ctx, cudaMemcpy2DAsync(x_host + hoff[l], row, ctx->arena + d.base, (size_t)d.pad * sizeof(float), row, K,
                                      cudaMemcpyDeviceToHost, ctx->s_d2h));
      }
    }
    CU_TRY(ctx, cudaStreamSynchronize(ctx->s_h2d));
    CU_TRY(ctx, cudaStreamSynchronize(ctx->s_cmp));
    CU_TRY(ctx, cudaStreamSynchronize(ctx->s_d2h));
    return LAYUP_OK;
  };
  rc = pipeline();
  if (rc != LAYUP_OK) {
    // the host buffers must not be in use when we return; the arena holds a partial round
    const std::string why = ctx->err;
    cudaStreamSynchronize(ctx->s_h2d);
    cudaStreamSynchronize(ctx->s_cmp);
    cudaStreamSynchronize(ctx->s_d2h);
    cudaGetLastError();
    ctx->poisoned = true;
    return fail(ctx, LAYUP_ECUDA, "layup_round_host failed mid-round, ctx poisoned: %s", why.c_str());
  }
  for (int l = 0; l < L; ++l) ctx->next_step[l] = step + 1;
  return LAYUP_OK;
}

extern "C" int layup_sync(layup_ctx *ctx) {
  if (!ctx) return fail(nullptr, LAYUP_EINVAL, "ctx is NULL");
  if (ctx->capturing) return fail(ctx, LAYUP_ESTATE, "a graph capture is open (layup_graph_end first)");
  LAYUP_ON_DEVICE(ctx);
  for (cudaStream_t s : ctx->streams) CU_TRY(ctx, cudaStreamSynchronize(s));
  CU_TRY(ctx, cudaGetLastError());
  // the device's round counters against the host's bookkeeping (graphs replay on the device's word)
  std::vector<uint32_t> dev(ctx->L);
  CU_TRY(ctx, cudaMemcpy(dev.data(), ctx->d_step, sizeof(uint32_t) * ctx->L, cudaMemcpyDeviceToHost));
  for (int l = 0; l < ctx->L; ++l)
    if (dev[l] != (uint32_t)ctx->next_step[l])
      return fail(ctx, LAYUP_ESTATE, "layer %d: device ran %u rounds, host expected %lld", l, dev[l], (long long)ctx->next_step[l]);
  return LAYUP_OK;
}

extern "C" int layup_peer(uint64_t seed, int64_t step, int32_t layer, int32_t replica, int32_t K, int32_t *peer) {
  if (!peer || K < 2 || replica < 0 || replica >= K || layer < -1) return fail(nullptr, LAYUP_EINVAL, "layup_peer: bad argument");
  *peer = draw_peer(seed, (uint32_t)step, layer < 0 ? kNoLayer : (uint32_t)layer, replica, K);
  return LAYUP_OK;
}

extern "C" int layup_schedule(layup_ctx *ctx, int64_t step, int32_t *peer, uint8_t *active) {
  if (!ctx || !peer || !active) return fail(ctx, LAYUP_EINVAL, "NULL argument");
  if (ctx->capturing) return fail(ctx, LAYUP_ESTATE, "a graph capture is open");
  if (step < 0 || step > 0xFFFFFFFFll) return fail(ctx, LAYUP_EINVAL, "step %lld outside [0, 2^32)", (long long)step);
  LAYUP_ON_DEVICE(ctx);
  CU_TRY(ctx, launch_peers_only(ctx->seed, (uint32_t)step, ctx->skip_thr, ctx->K, ctx->L, ctx->peer_mode,
                                ctx->delay_replica, ctx->delay_rounds, ctx->d_peer_scratch, ctx->d_active_scratch, ctx->own_stream));
  ctx->launches += 1;
  CU_TRY(ctx, cudaMemcpyAsync(peer, ctx->d_peer_scratch, sizeof(int32_t) * ctx->L * ctx->K, cudaMemcpyDeviceToHost, ctx->own_stream));
  CU_TRY(ctx, cudaMemcpyAsync(active, ctx->d_active_scratch, (size_t)ctx->K, cudaMemcpyDeviceToHost, ctx->own_stream));
  CU_TRY(ctx, cudaStreamSynchronize(ctx->own_stream));
  return LAYUP_OK;
}

extern "C" int layup_schedule_tables(layup_ctx *ctx, int32_t layer, int64_t *step_done, int32_t *peer, uint8_t *flags,
                                     int32_t *recv_off, int32_t *senders, float *alpha) {
  if (!ctx) return fail(nullptr, LAYUP_EINVAL, "ctx is NULL");
  if (layer < 0 || layer >= ctx->L) return fail(ctx, LAYUP_EINVAL, "layer %d out of range", layer);
  int rc = layup_sync(ctx);
  if (rc) return rc;
  LAYUP_ON_DEVICE(ctx);
  const int K = ctx->K;
  const size_t row = (size_t)layer * K;
  if (step_done) *step_done = ctx->last_event_step[layer];
  if (peer) CU_TRY(ctx, cudaMemcpy(peer, ctx->t.peer + row, sizeof(int32_t) * K, cudaMemcpyDeviceToHost));
  if (flags) CU_TRY(ctx, cudaMemcpy(flags, ctx->t.flags + row, (size_t)K, cudaMemcpyDeviceToHost));
  if (recv_off) CU_TRY(ctx, cudaMemcpy(recv_off, ctx->t.recv_off + (size_t)layer * (K + 1), sizeof(int32_t) * (K + 1), cudaMemcpyDeviceToHost));
  if (senders) CU_TRY(ctx, cudaMemcpy(senders, ctx->t.senders + row, sizeof(int32_t) * K, cudaMemcpyDeviceToHost));
  if (alpha) CU_TRY(ctx, cudaMemcpy(alpha, ctx->t.alpha + row, sizeof(float) * K, cudaMemcpyDeviceToHost));
  return LAYUP_OK;
}

extern "C" int layup_last_order(layup_ctx *ctx, int32_t *layers, int32_t *n) {
  if (!ctx || !layers || !n) return fail(ctx, LAYUP_EINVAL, "NULL argument");
  const size_t m = std::min(ctx->last_order.size(), (size_t)ctx->L);
  for (size_t k = 0; k < m; ++k) layers[k] = ctx->last_order[k];
  *n = (int32_t)m;
  return LAYUP_OK;
}

extern "C" int layup_trace(layup_ctx *ctx, int32_t enable) {
  if (!ctx) return fail(nullptr, LAYUP_EINVAL, "ctx is NULL");
  int rc = layup_sync(ctx);
  if (rc) return rc;
  LAYUP_ON_DEVICE(ctx);
  ctx->tracing = enable != 0;
  if (ctx->tracing) CU_TRY(ctx, cudaMemset(ctx->d_trace, 0xFF, sizeof(unsigned long long) * ctx->L));
  return LAYUP_OK;
}

extern "C" int layup_trace_read(layup_ctx *ctx, uint64_t *first_ns) {
  if (!ctx || !first_ns) return fail(ctx, LAYUP_EINVAL, "NULL argument");
  int rc = layup_sync(ctx);
  if (rc) return rc;
  LAYUP_ON_DEVICE(ctx);
  CU_TRY(ctx, cudaMemcpy(first_ns, ctx->d_trace, sizeof(uint64_t) * ctx->L, cudaMemcpyDeviceToHost));
  return LAYUP_OK;
}

extern "C" int layup_weights(layup_ctx *ctx, double *w) {
  if (!ctx || !w) return fail(ctx, LAYUP_EINVAL, "NULL argument");
  int rc = layup_sync(ctx);
  if (rc) return rc;
  LAYUP_ON_DEVICE(ctx);
  CU_TRY(ctx, cudaMemcpy(w, ctx->d_w, sizeof(double) * ctx->L * ctx->K, cudaMemcpyDeviceToHost));
  return LAYUP_OK;
}

extern "C" int layup_state_export(layup_ctx *ctx, double *w, double *bpow, int64_t *next_step) {
  if (!ctx || !w || !next_step) return fail(ctx, LAYUP_EINVAL, "NULL argument");
  if (ctx->opt == OPT_ADAMW && !bpow) return fail(ctx, LAYUP_EINVAL, "bpow is NULL but the optimizer is AdamW");
  int rc = layup_sync(ctx);
  if (rc) return rc;
  LAYUP_ON_DEVICE(ctx);
  const size_t n = (size_t)ctx->L * ctx->K;
  CU_TRY(ctx, cudaMemcpy(w, ctx->d_w, sizeof(double) * n, cudaMemcpyDeviceToHost));
  if (ctx->opt == OPT_ADAMW) CU_TRY(ctx, cudaMemcpy(bpow, ctx->d_bpow, sizeof(double) * 2 * n, cudaMemcpyDeviceToHost));
  for (int l = 0; l < ctx->L; ++l) next_step[l] = ctx->next_step[l];
  return LAYUP_OK;
}

extern "C" int layup_state_import(layup_ctx *ctx, const double *w, const double *bpow, const int64_t *next_step) {
  if (!ctx || !w || !next_step) return fail(ctx, LAYUP_EINVAL, "NULL argument");
  if (ctx->opt == OPT_ADAMW && !bpow) return fail(ctx, LAYUP_EINVAL, "bpow is NULL but the optimizer is AdamW");
  for (int l = 0; l < ctx->L; ++l)
    if (next_step[l] < 0 || next_step[l] > 0xFFFFFFFFll) return fail(ctx, LAYUP_EINVAL, "next_step[%d] outside [0, 2^32)", l);
  int rc = layup_sync(ctx);
  if (rc) return rc;
  LAYUP_ON_DEVICE(ctx);
  const size_t n = (size_t)ctx->L * ctx->K;
  CU_TRY(ctx, cudaMemcpy(ctx->d_w, w, sizeof(double) * n, cudaMemcpyHostToDevice));
  if (ctx->opt == OPT_ADAMW) CU_TRY(ctx, cudaMemcpy(ctx->d_bpow, bpow, sizeof(double) * 2 * n, cudaMemcpyHostToDevice));
  std::vector<uint32_t> dev(ctx->L);
  for (int l = 0; l < ctx->L; ++l) { ctx->next_step[l] = next_step[l]; dev[l] = (uint32_t)next_step[l]; }
  CU_TRY(ctx, cudaMemcpy(ctx->d_step, dev.data(), sizeof(uint32_t) * ctx->L, cudaMemcpyHostToDevice));
  return LAYUP_OK;
}

extern "C" int layup_disagreement(layup_ctx *ctx, int32_t weighted, double *dist, void *cuda_stream) {
  if (!ctx || !dist) return fail(ctx, LAYUP_EINVAL, "NULL argument");
  int rc = layup_sync(ctx);                       // everything this ctx issued, on whatever stream
  if (rc) return rc;
  LAYUP_ON_DEVICE(ctx);
  const int K = ctx->K, L = ctx->L;
  if (ctx->diag_C == 0) {
    cudaDeviceProp prop;
    CU_TRY(ctx, cudaGetDeviceProperties(&prop, ctx->device));
    rc = LAYUP_OK;
    int C = 0, smem = 0, ctas = 0, stages = 0;
    CU_TRY(ctx, diag_plan(K, (size_t)prop.sharedMemPerBlockOptin, &C, &stages, &smem, &ctas));
    if (ctas < 1) return fail(ctx, LAYUP_EINVAL, "K=%d does not fit the diagnostic kernel", K);
    ctx->diag_C = C; ctx->diag_smem = smem; ctx->diag_ctas = ctas; ctx->diag_stages = stages;
    while ((1 << ctx->diag_log2C) < C) ++ctx->diag_log2C;
    CU_TRY(ctx, cudaEventCreate(&ctx->diag_ev0));
    CU_TRY(ctx, cudaEventCreate(&ctx->diag_ev1));
  }
  cudaStream_t s = (cudaStream_t)cuda_stream;
  CU_TRY(ctx, cudaMemsetAsync(ctx->d_dist, 0, sizeof(double) * L * K, s));
  CU_TRY(ctx, cudaEventRecord(ctx->diag_ev0, s));
  const int C = ctx->diag_C;
  for (int q0 = 0; q0 < L;) {
    PosTable tab;
    int n = 0;
    tab.prefix[0] = 0;
    while (q0 + n < L && n < kMaxPos) {
      const LayerDesc &d = ctx->layers[L - 1 - (q0 + n)];
      tab.lay[n] = d;
      tab.layer[n] = L - 1 - (q0 + n);
      tab.prefix[n + 1] = tab.prefix[n] + (d.pad / 4 + C - 1) / C;
      ++n;
    }
    tab.n = n;
    const long long tiles = tab.prefix[n];
    const int grid = (int)std::min<long long>(tiles, (long long)ctx->n_sm * ctx->diag_ctas);
    CU_TRY(ctx, launch_disagreement(ctx->arena, weighted ? ctx->d_w : nullptr, ctx->d_dist, K, C, ctx->diag_log2C,
                                    ctx->diag_stages, tab, grid, ctx->diag_smem, s));
    ctx->launches += 1;
    q0 += n;
  }
  CU_TRY(ctx, cudaEventRecord(ctx->diag_ev1, s));
  CU_TRY(ctx, cudaMemcpyAsync(dist, ctx->d_dist, sizeof(double) * L * K, cudaMemcpyDeviceToHost, s));
  CU_TRY(ctx, cudaStreamSynchronize(s));
  ctx->diag_timed = true;
  return LAYUP_OK;
}

extern "C" int layup_disagreement_ms(layup_ctx *ctx, double *ms) {
  if (!ctx || !ms) return fail(ctx, LAYUP_EINVAL, "NULL argument");
  if (!ctx->diag_timed) return fail(ctx, LAYUP_ESTATE, "layup_disagreement has not run yet");
  LAYUP_ON_DEVICE(ctx);
  float f = 0.f;
  CU_TRY(ctx, cudaEventElapsedTime(&f, ctx->diag_ev0, ctx->diag_ev1));
  *ms = f;
  return LAYUP_OK;
}

// ---- CUDA-graph capture ---------------------------------------------------------------
extern "C" int layup_graph_begin(layup_ctx *ctx, void *cuda_stream) {
  if (!ctx) return fail(nullptr, LAYUP_EINVAL, "ctx is NULL");
  if (!cuda_stream) return fail(ctx, LAYUP_EINVAL, "the legacy default stream cannot be captured");
  if (ctx->capturing) return fail(ctx, LAYUP_ESTATE, "a graph capture is already open");
  if (ctx->poisoned) return fail(ctx, LAYUP_ECUDA, "ctx is poisoned");
  LAYUP_ON_DEVICE(ctx);
  CU_TRY(ctx, cudaStreamBeginCapture((cudaStream_t)cuda_stream, cudaStreamCaptureModeRelaxed));
  ctx->capturing = true;
  ctx->cap_stream = (cudaStream_t)cuda_stream;
  ctx->cap_next_step = ctx->next_step;           // nothing runs during capture: restored at the end
  ctx->cap_last_event = ctx->last_event_step;
  ctx->cap_order = ctx->last_order;
  ctx->cap_launches = ctx->launches;
  ctx->last_order.clear();
  return LAYUP_OK;
}

extern "C" int layup_graph_end(layup_ctx *ctx, layup_graph **out) {
  if (!ctx || !out) return fail(ctx, LAYUP_EINVAL, "NULL argument");
  if (!ctx->capturing) return fail(ctx, LAYUP_ESTATE, "no graph capture is open");
  LAYUP_ON_DEVICE(ctx);
  *out = nullptr;
  layup_graph *g = new layup_graph();
  g->owner = ctx;
  g->advance.resize(ctx->L);
  for (int l = 0; l < ctx->L; ++l) g->advance[l] = ctx->next_step[l] - ctx->cap_next_step[l];
  g->order = ctx->last_order;
  g->launches = ctx->launches - ctx->cap_launches;
  // roll the bookkeeping back: the recorded calls have not run
  ctx->next_step = ctx->cap_next_step;
  ctx->last_event_step = ctx->cap_last_event;
  ctx->last_order = ctx->cap_order;
  ctx->launches = ctx->cap_launches;
  ctx->capturing = false;
  cudaError_t e = cudaStreamEndCapture(ctx->cap_stream, &g->graph);
  if (e == cudaSuccess && !g->graph) e = cudaErrorStreamCaptureInvalidated;
  if (e == cudaSuccess) e = cudaGraphInstantiate(&g->exec, g->graph, 0);
  if (e != cudaSuccess) {
    if (g->graph) cudaGraphDestroy(g->graph);
    delete g;
    cudaGetLastError();
    return fail(ctx, LAYUP_ECUDA, "graph capture failed: %s", cudaGetErrorString(e));
  }
  *out = g;
  return LAYUP_OK;
}

extern "C" int layup_graph_launch(layup_ctx *ctx, layup_graph *g, void *cuda_stream) {
  if (!ctx || !g) return fail(ctx, LAYUP_EINVAL, "NULL argument");
  if (g->owner != ctx) return fail(ctx, LAYUP_EINVAL, "graph belongs to another ctx");
  if (ctx->capturing) return fail(ctx, LAYUP_ESTATE, "a graph capture is open");
  if (ctx->poisoned) return fail(ctx, LAYUP_ECUDA, "ctx is poisoned");
  for (int l = 0; l < ctx->L; ++l)
    if (ctx->next_step[l] + g->advance[l] > 0x100000000ll) return fail(ctx, LAYUP_EINVAL, "layer %d would pass step 2^32", l);
  LAYUP_ON_DEVICE(ctx);
  CU_TRY(ctx, cudaGraphLaunch(g->exec, (cudaStream_t)cuda_stream));
  for (int l = 0; l < ctx->L; ++l) {
    if (g->advance[l] > 0) ctx->last_event_step[l] = ctx->next_step[l] + g->advance[l] - 1;
    ctx->next_step[l] += g->advance[l];
  }
  ctx->last_order = g->order;
  ctx->launches += g->launches;
  note_stream(ctx, (cudaStream_t)cuda_stream);
  return LAYUP_OK;
}

extern "C" int layup_graph_destroy(layup_ctx *ctx, layup_graph *g) {
  if (!g) return LAYUP_OK;
  if (ctx && g->owner != ctx) return fail(ctx, LAYUP_EINVAL, "graph belongs to another ctx");
  if (ctx) {
    DeviceGuard guard(ctx->device);
    for (cudaStream_t s : ctx->streams) cudaStreamSynchronize(s);
    cudaGraphExecDestroy(g->exec);
    cudaGraphDestroy(g->graph);
  } else {
    cudaGraphExecDestroy(g->exec);
    cudaGraphDestroy(g->graph);
  }
  delete g;
  return LAYUP_OK;
}

extern "C" int layup_profile(layup_ctx *ctx, int32_t enable) {
  if (!ctx) return fail(nullptr, LAYUP_EINVAL, "ctx is NULL");
  ctx->profiling = enable != 0;
  return LAYUP_OK;
}

extern "C" int layup_profile_read(layup_ctx *ctx, int64_t *launches, double *total_ms) {
  if (!ctx || !launches || !total_ms) return fail(ctx, LAYUP_EINVAL, "NULL argument");
  int rc = layup_sync(ctx);
  if (rc) return rc;
  LAYUP_ON_DEVICE(ctx);
  double tot = 0.0;
  for (auto &pr : ctx->prof_pending) {
    float ms = 0.f;
    CU_TRY(ctx, cudaEventElapsedTime(&ms, pr.first, pr.second));
    tot += ms;
  }
  *launches = (int64_t)ctx->prof_pending.size();
  *total_ms = tot;
  ctx->prof_pool.insert(ctx->prof_pool.end(), ctx->prof_pending.begin(), ctx->prof_pending.end());
  ctx->prof_pending.clear();
  return LAYUP_OK;
}

extern "C" int layup_launch_count(layup_ctx *ctx, int64_t *launches) {
  if (!ctx || !launches) return fail(ctx, LAYUP_EINVAL, "NULL argument");
  *launches = ctx->launches;
  return LAYUP_OK;
}

extern "C" const char *layup_last_error(layup_ctx *ctx) {
  return ctx ? ctx->err.c_str() : g_err.c_str();
}
