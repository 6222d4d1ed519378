// TMA-staged form of the fused local-step + gossip-mix kernel (see update.cu for the rule).
//
// Same work item -- (layer, tile of C float4 columns) for ALL K replicas, one CTA per item --
// but the K x {x, g, m} chunks of the tile are brought into shared memory by 1-D bulk
// copies (cp.async.bulk, the TMA engine; SASS UBLKCP) completing on one mbarrier, so the
// whole tile (K*C*16 B * 3) is in flight per CTA without holding registers.  The local step
// then runs out of shared memory, y overwrites x in place (the "send" is an on-chip read,
// PAPER.md:101), m' (and AdamW's v') go straight to HBM, and after one CTA barrier every
// receiver folds its senders and writes x once.  HBM traffic is unchanged: 12 B (SGD) / 20 B
// (momentum) / 28 B (AdamW) per parameter update.  Template parameters: OPT = local optimiser
// (rule.cuh), SYM = symmetric pairwise averaging instead of the push-sum fold.
#include "layup_internal.cuh"
#include "rule.cuh"

namespace layup {

namespace {

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// global -> shared::cta bulk copy, bytes % 16 == 0, both addresses 16-B aligned
__device__ __forceinline__ void bulk_g2s(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst_smem)),
               "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

// same copy with an L2 evict-first policy: every byte of the arena is touched once per round
__device__ __forceinline__ void bulk_g2s_ef(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar,
                                            uint64_t policy) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
          smem_u32(dst_smem)),
      "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
      : "memory");
}
__device__ __forceinline__ uint64_t policy_evict_first() {
  uint64_t pol;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}

// shared::cta -> global bulk copy (TMA store), bytes % 16 == 0; completion tracked by bulk groups
__device__ __forceinline__ void bulk_s2g(void *dst_gmem, const void *src_smem, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst_gmem), "r"(smem_u32(src_smem)),
               "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void bulk_commit_wait_read() {
  asm volatile("cp.async.bulk.commit_group;" ::: "memory");
  asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}
// generic-proxy writes to shared memory -> visible to the async proxy (TMA) before it reads them
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

__device__ __forceinline__ void st4(float *p, const float4 &v) { *reinterpret_cast<float4 *>(p) = v; }
__device__ __forceinline__ void st4_cs(float *p, const float4 &v) { __stcs(reinterpret_cast<float4 *>(p), v); }

template <int OPT, bool SYM, int THREADS, int MINB>
__global__ void __launch_bounds__(THREADS, MINB)
    layup_update_tma(const __grid_constant__ UpdateParams p, const __grid_constant__ PosTable tab) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  constexpr int NARR = OptTraits<OPT>::kArrays;
  constexpr bool HAS_M = NARR >= 3, HAS_V = NARR >= 4;
  const int K = p.K, C = p.C, log2C = p.log2C, tid = threadIdx.x;
  const int n_items = K << log2C;
  float4 *xs = reinterpret_cast<float4 *>(smem_raw);                       // [K*C]  x, then y in place
  float4 *gs = xs + n_items;                                                // [K*C]
  float4 *ms = HAS_M ? gs + n_items : gs;                                   // [K*C] (momentum / Adam m)
  float4 *vs = HAS_V ? ms + n_items : ms;                                   // [K*C] (Adam v)
  uint64_t *bar = reinterpret_cast<uint64_t *>(xs + NARR * n_items);
  int *s_recv_off = reinterpret_cast<int *>(bar + 1);                       // [K+1]
  int *s_senders = s_recv_off + (K + 1);                                    // [K]  (SYM: the peer table)
  float *s_alpha = reinterpret_cast<float *>(s_senders + K);                // [K]
  float *s_c1 = s_alpha + K;                                                // [K]  (AdamW only)
  float *s_c2 = s_c1 + (HAS_V ? K : 0);                                     // [K]  (AdamW only)
  unsigned char *s_flags = reinterpret_cast<unsigned char *>(s_c2 + (HAS_V ? K : 0));  // [K]

  // which layer does this work item belong to: binary search in the parameter table
  const long long tile = blockIdx.x;
  int lo = 0, hi = tab.n;
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (tile >= tab.prefix[mid]) lo = mid; else hi = mid;
  }
  const int layer = tab.layer[lo];
  const long long pad = tab.lay[lo].pad;
  const long long col0 = (tile - tab.prefix[lo]) << log2C;                  // first float4 column
  const long long cols_left = (pad >> 2) - col0;
  const int ncols = cols_left < C ? (int)cols_left : C;
  const long long tile_off = tab.lay[lo].base + (col0 << 2);
  float *const xb = p.x + tile_off;
  const float *const gb = p.g + tile_off;
  float *const mb = HAS_M ? p.m + tile_off : nullptr;
  float *const vb = HAS_V ? p.v + tile_off : nullptr;
  const uint32_t chunk = (uint32_t)ncols * 16u;

  if (tid == 0) {
    mbar_init(bar, 1);
    // no straggler this round: every replica is active, the byte count is known up front
    if (p.all_active) mbar_expect_tx(bar, (uint32_t)K * NARR * chunk);
  }
  __syncthreads();   // mbarrier visible

  // Bulk copies are issued one lane at a time within a warp, so spread them over all warps:
  // copy slot c = (replica, array) goes to warp c % NW, lane c / NW.
  constexpr int NW = THREADS / 32;
  const int slot0 = (tid & 31) * NW + (tid >> 5);
  auto issue_copies = [&](bool use_flags) {
    for (int c = slot0; c < K * NARR; c += THREADS) {
      const int i = c / NARR, a = c - i * NARR;
      if (use_flags) {
        const int f = s_flags[i];
        if (!f || (a > 0 && !(f & kFlagActive))) continue;
      }
      const long long off = (long long)i * pad;
      void *dst = xs + a * n_items + (i << log2C);
      const float *src = (a == 0 ? xb : a == 1 ? gb : a == 2 ? mb : vb) + off;
      if (p.hints & 1) bulk_g2s_ef(dst, src, chunk, bar, policy_evict_first());
      else bulk_g2s(dst, src, chunk, bar);
    }
  };
  if (p.all_active) issue_copies(false);

  // this layer's schedule -> shared memory (overlaps the bulk copies when all replicas are active)
  {
    const size_t row = (size_t)layer * K;
    for (int k = tid; k < K; k += THREADS) {
      s_senders[k] = SYM ? p.t.peer[row + k] : p.t.senders[row + k];
      s_alpha[k] = p.t.alpha[row + k];
      s_flags[k] = p.t.flags[row + k];
      if (HAS_V) {
        s_c1[k] = p.t.c1[row + k];
        s_c2[k] = p.t.c2[row + k];
      }
    }
    for (int k = tid; k <= K; k += THREADS) s_recv_off[k] = p.t.recv_off[(size_t)layer * (K + 1) + k];
  }
  __syncthreads();   // schedule visible

  if (!p.all_active) {
    // straggler round: the flags decide which chunks are touched at all
    if (tid < 32) {
      uint32_t bytes = 0;
      for (int i = tid; i < K; i += 32) {
        const int f = s_flags[i];
        bytes += f ? chunk * ((f & kFlagActive) ? (uint32_t)NARR : 1u) : 0u;
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) bytes += __shfl_xor_sync(0xFFFFFFFFu, bytes, o);
      if (tid == 0) mbar_expect_tx(bar, bytes);
    }
    __syncthreads();
    issue_copies(true);
  }
  mbar_wait(bar, 0);

  // ---- phase 1: local step out of shared memory; y overwrites x in place, m' (v') -> HBM
  const bool bulk_out = (p.hints & 4) != 0;     // outputs leave through TMA bulk stores instead of STG
  for (int idx = tid; idx < n_items; idx += THREADS) {
    const int i = idx >> log2C, c = idx & (C - 1);
    if (c >= ncols) continue;
    if (!(s_flags[i] & kFlagActive)) continue;                              // idle replica: y = x already there
    float4 m = HAS_M ? ms[idx] : float4{0.f, 0.f, 0.f, 0.f};
    float4 v = HAS_V ? vs[idx] : float4{0.f, 0.f, 0.f, 0.f};
    const float4 y = local_step4<OPT>(xs[idx], gs[idx], m, v, p.s, HAS_V ? s_c1[i] : 0.f, HAS_V ? s_c2[i] : 0.f);
    const long long off = (long long)i * pad + (c << 2);
    if (bulk_out) {
      if (HAS_M) ms[idx] = m;
      if (HAS_V) vs[idx] = v;
    } else {
      if (HAS_M) { if (p.hints & 2) st4_cs(mb + off, m); else st4(mb + off, m); }
      if (HAS_V) { if (p.hints & 2) st4_cs(vb + off, v); else st4(vb + off, v); }
    }
    xs[idx] = y;
  }
  if (bulk_out && HAS_M) fence_proxy_async();
  __syncthreads();
  if (bulk_out && HAS_M) {
    // m' (v') of every active replica: one bulk store per (replica, array), spread like the loads
    constexpr int NOUT = HAS_M ? NARR - 2 : 1;
    for (int c = slot0; c < K * NOUT; c += THREADS) {
      const int i = c / NOUT, a = 2 + (c - i * NOUT);
      if (!(s_flags[i] & kFlagActive)) continue;
      bulk_s2g((a == 2 ? mb : vb) + (long long)i * pad, xs + a * n_items + (i << log2C), chunk);
    }
  }

  if (SYM) {
    // ---- phase 2 (symmetric): every scalar column runs the K exchanges in worker order
    float *ysf = reinterpret_cast<float *>(xs);
    for (int e = tid; e < (ncols << 2); e += THREADS) symmetric_column(ysf, C << 2, e, K, s_senders);
    __syncthreads();
    for (int idx = tid; idx < n_items; idx += THREADS) {
      const int i = idx >> log2C, c = idx & (C - 1);
      if (c >= ncols || !s_flags[i]) continue;                              // idle and nobody's peer: 0 bytes
      st4(xb + (long long)i * pad + (c << 2), xs[idx]);
    }
  } else {
    // ---- phase 2: each receiver folds its senders in ascending order; x written once
    for (int idx = tid; idx < n_items; idx += THREADS) {
      const int i = idx >> log2C, c = idx & (C - 1);
      if (c >= ncols) continue;
      if (!s_flags[i]) continue;                                            // idle, no push received: 0 bytes
      float4 acc = xs[idx];
      const int k_end = s_recv_off[i + 1];
      for (int k = s_recv_off[i]; k < k_end; ++k) peer_update4(acc, xs[(s_senders[k] << log2C) + c], s_alpha[k]);
      if (bulk_out) gs[idx] = acc;                                          // g is dead: its tile carries x out
      else if (p.hints & 2) st4_cs(xb + (long long)i * pad + (c << 2), acc);
      else st4(xb + (long long)i * pad + (c << 2), acc);
    }
    if (bulk_out) {
      fence_proxy_async();
      __syncthreads();
      for (int i = slot0; i < K; i += THREADS)
        if (s_flags[i]) bulk_s2g(xb + (long long)i * pad, gs + (i << log2C), chunk);
    }
  }
  if (bulk_out) bulk_commit_wait_read();   // shared memory must outlive the stores' reads
}

using TmaFn = void (*)(const UpdateParams, const PosTable);
struct TmaVariant {
  int threads, minb;
  TmaFn fn[3][2];   // [OPT][SYM]
};
#define LAYUP_TMA_VARIANT(T, MB)                                                                              \
  TmaVariant {                                                                                                \
    T, MB, {                                                                                                  \
      {layup_update_tma<OPT_SGD, false, T, MB>, layup_update_tma<OPT_SGD, true, T, MB>},                      \
          {layup_update_tma<OPT_SGD_MOM, false, T, MB>, layup_update_tma<OPT_SGD_MOM, true, T, MB>},          \
          {layup_update_tma<OPT_ADAMW, false, T, MB>, layup_update_tma<OPT_ADAMW, true, T, MB>},              \
    }                                                                                                         \
  }
const TmaVariant kTma[] = {
    LAYUP_TMA_VARIANT(256, 4), LAYUP_TMA_VARIANT(128, 8), LAYUP_TMA_VARIANT(512, 2), LAYUP_TMA_VARIANT(256, 2),
};
constexpr int kNumTma = sizeof(kTma) / sizeof(kTma[0]);

}  // namespace

int tma_num_variants() { return kNumTma; }

size_t tma_smem_bytes(int K, int C, int opt) {
  const int narr = opt == OPT_ADAMW ? 4 : opt == OPT_SGD_MOM ? 3 : 2;
  return (size_t)K * C * sizeof(float4) * narr + 8 + sizeof(int) * (2 * (size_t)K + 1) +
         sizeof(float) * K * (opt == OPT_ADAMW ? 3 : 1) + (size_t)K;
}

cudaError_t tma_kernel_setup(int variant, int opt, bool symmetric, int smem_bytes, int *threads, int *ctas_per_sm) {
  if (variant < 0 || variant >= kNumTma || opt < 0 || opt > 2) return cudaErrorInvalidValue;
  const TmaVariant &v = kTma[variant];
  TmaFn f = v.fn[opt][symmetric ? 1 : 0];
  cudaError_t e;
  if ((e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(f, cudaFuncAttributePreferredSharedMemoryCarveout, 100)) != cudaSuccess) return e;
  int a = 0;
  if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&a, f, v.threads, smem_bytes)) != cudaSuccess) return e;
  *threads = v.threads;
  *ctas_per_sm = a;
  return cudaSuccess;
}

cudaError_t launch_update_tma(const UpdateParams &p, const PosTable &tab, int variant, int grid, int smem_bytes,
                              cudaStream_t s) {
  const TmaVariant &v = kTma[variant];
  v.fn[p.opt][p.symmetric ? 1 : 0]<<<grid, v.threads, smem_bytes, s>>>(p, tab);
  return cudaGetLastError();
}

}  // namespace layup
