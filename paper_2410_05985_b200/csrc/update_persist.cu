// Persistent form of the TMA-staged update kernel: a fixed grid of resident CTAs drains the
// reverse-layer-ordered work list (BASELINE.json north_star item 3, "a persistent grouped launch
// that drains many small layers from a work list") with a two-stage shared-memory pipeline: while
// a CTA computes and stores tile n out of one stage, the TMA engine fills the other stage with
// tile n + gridDim.x.  Same work item, same arithmetic (rule.cuh) and the same bits as
// update_tma.cu; the layer's schedule tables are reloaded only when the CTA crosses into another
// layer.
//
// Scope: every replica active, sender-list mixers (push-sum, lossy), schedule tables from the
// schedule kernel.  It is selected with LAYUP_PERSISTENT=1: on B200 the one-CTA-per-work-item
// launch measures faster, so this form is the measured alternative, not the default.
#include "layup_internal.cuh"
#include "rule.cuh"
#include "tma_ptx.cuh"

namespace layup {

namespace {

constexpr int kPsThreads = 256;

template <int OPT>
__global__ void __launch_bounds__(kPsThreads, 2)
    layup_update_persist(const __grid_constant__ UpdateParams p, const __grid_constant__ PosTable tab) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  constexpr int NARR = OptTraits<OPT>::kArrays;
  constexpr bool HAS_M = NARR >= 3, HAS_V = NARR >= 4;
  constexpr int THREADS = kPsThreads;
  const int K = p.K, C = p.C, log2C = p.log2C, tid = threadIdx.x;
  const int n_items = K << log2C;
  const size_t stage_f4 = (size_t)NARR * n_items;                            // float4 per stage
  float4 *stage0 = reinterpret_cast<float4 *>(smem_raw);
  uint64_t *bars = reinterpret_cast<uint64_t *>(stage0 + 2 * stage_f4);      // [2] one per stage
  int *s_begin = reinterpret_cast<int *>(bars + 2);                          // [K]
  int *s_cnt = s_begin + K;
  int *s_senders = s_cnt + K;
  float *s_alpha = reinterpret_cast<float *>(s_senders + K);
  float *s_c1 = s_alpha + K;                                                 // [K] (AdamW only)
  float *s_c2 = s_c1 + (HAS_V ? K : 0);

  const long long n_tiles = tab.prefix[tab.n];
  const bool boxed = p.tmaps != nullptr;
  constexpr int NW = THREADS / 32;
  const int slot0 = (tid & 31) * NW + (tid >> 5);

  auto locate = [&](long long tile) {
    int lo = 0, hi = tab.n;
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (tile >= tab.prefix[mid]) lo = mid; else hi = mid;
    }
    return lo;
  };
  // request tile `tile` into stage `s` (all threads call it; the copies are spread over the warps)
  auto issue_load = [&](long long tile, int s) {
    const int lo = locate(tile);
    const long long pad = tab.lay[lo].pad;
    const long long col0 = (tile - tab.prefix[lo]) << log2C;
    const long long cols_left = (pad >> 2) - col0;
    const uint32_t chunk = (uint32_t)(cols_left < C ? cols_left : C) * 16u;
    float4 *st = stage0 + (size_t)s * stage_f4;
    uint64_t *bar = bars + s;
    if (boxed) {
      if (tid == 0) {
        mbar_expect_tx(bar, (uint32_t)n_items * 16u * NARR);
        const unsigned char *tm = reinterpret_cast<const unsigned char *>(p.tmaps);
#pragma unroll
        for (int a = 0; a < NARR; ++a)
          tma_load_2d(st + a * n_items, tm + ((size_t)a * p.L + tab.layer[lo]) * 128, (int)(col0 << 2), 0, bar);
      }
    } else {
      if (tid == 0) mbar_expect_tx(bar, (uint32_t)K * NARR * chunk);
      const long long tile_off = tab.lay[lo].base + (col0 << 2);
      for (int c = slot0; c < K * NARR; c += THREADS) {
        const int i = c / NARR, a = c - i * NARR;
        const float *src = (a == 0 ? p.x : a == 1 ? p.g : a == 2 ? p.m : p.v) + tile_off + (long long)i * pad;
        bulk_g2s(st + a * n_items + (i << log2C), src, chunk, bar);
      }
    }
  };

  if (tid == 0) {
    mbar_init(bars, 1);
    mbar_init(bars + 1, 1);
  }
  __syncthreads();   // mbarriers visible

  long long tile = blockIdx.x;
  if (tile < n_tiles) issue_load(tile, 0);
  int cur_layer = -1;
  for (int it = 0; tile < n_tiles; tile += gridDim.x, ++it) {
    const int s = it & 1;
    // the other stage was released by the barrier that closed the previous iteration: prefetch
    if (tile + gridDim.x < n_tiles) issue_load(tile + gridDim.x, s ^ 1);

    const int lo = locate(tile);
    const int layer = tab.layer[lo];
    const long long pad = tab.lay[lo].pad;
    const long long col0 = (tile - tab.prefix[lo]) << log2C;
    const long long cols_left = (pad >> 2) - col0;
    const int ncols = cols_left < C ? (int)cols_left : C;
    const long long tile_off = tab.lay[lo].base + (col0 << 2);
    float *const xb = p.x + tile_off;
    float *const mb = HAS_M ? p.m + tile_off : nullptr;
    float *const vb = HAS_V ? p.v + tile_off : nullptr;
    if (layer != cur_layer) {
      if (cur_layer < 0) asm volatile("griddepcontrol.wait;" ::: "memory");   // tables of the schedule kernel
      const size_t row = (size_t)layer * K;
      for (int k = tid; k < K; k += THREADS) {
        s_senders[k] = p.t.senders[row + k];
        s_alpha[k] = p.t.alpha[row + k];
        const int b = p.t.recv_off[(size_t)layer * (K + 1) + k];
        s_begin[k] = b;
        s_cnt[k] = p.t.recv_off[(size_t)layer * (K + 1) + k + 1] - b;
        if (HAS_V) {
          s_c1[k] = p.t.c1[row + k];
          s_c2[k] = p.t.c2[row + k];
        }
      }
      cur_layer = layer;
      __syncthreads();
    }
    float4 *xs = stage0 + (size_t)s * stage_f4, *gs = xs + n_items;
    float4 *ms = HAS_M ? gs + n_items : gs, *vs = HAS_V ? ms + n_items : ms;
    mbar_wait(bars + s, (uint32_t)(it >> 1) & 1u);

    // ---- phase 1: local step; y overwrites x in place, m' (v') -> HBM
    for (int idx = tid; idx < n_items; idx += THREADS) {
      const int i = idx >> log2C, c = idx & (C - 1);
      if (c >= ncols) continue;
      float4 m = HAS_M ? ms[idx] : float4{0.f, 0.f, 0.f, 0.f};
      float4 v = HAS_V ? vs[idx] : float4{0.f, 0.f, 0.f, 0.f};
      const float4 y = local_step4<OPT>(xs[idx], gs[idx], m, v, p.s, HAS_V ? s_c1[i] : 0.f, HAS_V ? s_c2[i] : 0.f);
      const long long off = (long long)i * pad + (c << 2);
      if (HAS_M) st4(mb + off, m);
      if (HAS_V) st4(vb + off, v);
      xs[idx] = y;
    }
    __syncthreads();
    // ---- phase 2: each receiver folds its senders in ascending order; x written once
    for (int idx = tid; idx < n_items; idx += THREADS) {
      const int i = idx >> log2C, c = idx & (C - 1);
      if (c >= ncols) continue;
      float4 acc = xs[idx];
      const int k0 = s_begin[i], k_end = k0 + s_cnt[i];
      for (int k = k0; k < k_end; ++k) peer_update4(acc, xs[(s_senders[k] << log2C) + c], s_alpha[k]);
      st4(xb + (long long)i * pad + (c << 2), acc);
    }
    fence_proxy_async();   // the stage was written through the generic proxy; the TMA engine refills it next
    __syncthreads();       // this stage and the tables may be reused
  }
}

using PsFn = void (*)(const UpdateParams, const PosTable);
const PsFn kPs[3] = {layup_update_persist<OPT_SGD>, layup_update_persist<OPT_SGD_MOM>, layup_update_persist<OPT_ADAMW>};

}  // namespace

size_t persist_smem_bytes(int K, int C, int opt) {
  const int narr = opt == OPT_ADAMW ? 4 : opt == OPT_SGD_MOM ? 3 : 2;
  return 2 * (size_t)K * C * sizeof(float4) * narr + 16 + sizeof(int) * 3 * (size_t)K +
         sizeof(float) * K * (opt == OPT_ADAMW ? 3 : 1);
}

cudaError_t persist_kernel_setup(int opt, int smem_bytes, int *ctas_per_sm) {
  if (opt < 0 || opt > 2) return cudaErrorInvalidValue;
  cudaError_t e;
  if ((e = cudaFuncSetAttribute(kPs[opt], cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(kPs[opt], cudaFuncAttributePreferredSharedMemoryCarveout, 100)) != cudaSuccess) return e;
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas_per_sm, kPs[opt], kPsThreads, smem_bytes);
}

cudaError_t launch_update_persist(const UpdateParams &p, const PosTable &tab, int grid, int smem_bytes, bool pdl,
                                  cudaStream_t s) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid);
  cfg.blockDim = dim3((unsigned)kPsThreads);
  cfg.dynamicSmemBytes = (size_t)smem_bytes;
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kPs[p.opt], p, tab);
}

}  // namespace layup
