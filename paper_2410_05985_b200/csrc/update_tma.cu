// TMA-staged form of the fused local-step + gossip-mix kernel (rule.cuh holds the arithmetic).
//
// Work item = (layer, tile of C float4 columns) for ALL K replicas, one CTA per item.  The tile
// of every array (x, g, m, v) is brought into shared memory by the TMA engine, completing on one
// mbarrier, so the whole tile (K*C*16 B per array) is in flight per CTA without holding registers:
//   - when every replica is active and the box fits the TMA limits: ONE 2-D tiled copy per array
//     (cp.async.bulk.tensor.2d, SASS UTMALDG.2D) through a tensor map that views a layer section
//     as [K rows][padded slice];
//   - otherwise K x arrays 1-D bulk copies (cp.async.bulk, SASS UBLKCP), spread over all warps,
//     skipping what an idle replica does not need.
// The local step then runs out of shared memory, y overwrites x in place (the "send" is an
// on-chip read), m' (and AdamW's v') go straight to HBM, and after one CTA barrier
// every receiver folds its senders and writes x once.  HBM traffic: 12 B (SGD) / 20 B (momentum) /
// 28 B (AdamW) per parameter update, nothing read or written twice.
// Template parameters: OPT = local optimiser (rule.cuh), SYM = symmetric pairwise averaging
// instead of the push-sum fold, FUSED = the schedule stage runs in this kernel (one launch).
#include "layup_internal.cuh"
#include "philox.cuh"
#include "rule.cuh"
#include "tma_ptx.cuh"

namespace layup {

namespace {

// FUSED: the schedule stage (schedule.cu) runs inside this kernel -- ONE launch per round or
// per layer event instead of two.  Every CTA of a layer recomputes that layer's O(K) schedule in
// shared memory from the same inputs (seed, step, w, beta powers), so all CTAs agree bit for bit;
// the CTA that is LAST to have read the state (a ticket per layer) writes the new w / beta powers
// back in place.  Used for launches of few tiles (launch-latency bound) and K <= kFusedMaxK.
template <int OPT, bool SYM, bool FUSED, int THREADS, int MINB>
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
  double *s_wh = reinterpret_cast<double *>(bar + 1);                       // [K]  FUSED only: halved weights
  double *s_wnew = s_wh + (FUSED ? K : 0);                                  // [K]  FUSED only: w after the round
  double *s_bp = s_wnew + (FUSED ? K : 0);                                  // [2K] FUSED + AdamW: new beta powers
  int *s_begin = reinterpret_cast<int *>(s_bp + (FUSED && HAS_V ? 2 * K : 0));   // [K] first sender slot
  int *s_cnt = s_begin + K;                                                 // [K]  senders of each receiver
  int *s_senders = s_cnt + K;                                               // [K]  (SYM: the peer table)
  int *s_peer = s_senders + K;                                              // [K]  FUSED only
  float *s_alpha = reinterpret_cast<float *>(s_peer + (FUSED ? K : 0));     // [K]
  float *s_c1 = s_alpha + K;                                                // [K]  (AdamW only)
  float *s_c2 = s_c1 + (HAS_V ? K : 0);                                     // [K]  (AdamW only)
  unsigned char *s_flags = reinterpret_cast<unsigned char *>(s_c2 + (HAS_V ? K : 0));  // [K]

  if (FUSED) {
    // Launched as a programmatic dependent of whatever kernel precedes it on the stream (in a graph
    // of L2-resident rounds: the previous round's launch of this same kernel): the CTAs are placed
    // and set up while that kernel drains, and only here wait for it to complete -- everything this
    // kernel reads (round counter, weights, x) may have been written by it.  The next launch may be
    // staged from now on; it will wait for THIS grid at the same point.
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  }
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

  trace_start(p.trace, layer);
  const bool boxed = p.all_active && p.tmaps != nullptr;   // whole-tile 2-D TMA loads, one per array
  if (tid == 0) {
    mbar_init(bar, 1);
    // no straggler this round: every replica is active, the byte count is known up front
    if (boxed) {
      mbar_expect_tx(bar, (uint32_t)n_items * 16u * NARR);                  // full boxes, zero fill included
      const unsigned char *tm = reinterpret_cast<const unsigned char *>(p.tmaps);
#pragma unroll
      for (int a = 0; a < NARR; ++a)
        tma_load_2d(xs + a * n_items, tm + ((size_t)a * p.L + layer) * 128, (int)(col0 << 2), 0, bar);
    } else if (p.all_active) {
      mbar_expect_tx(bar, (uint32_t)K * NARR * chunk);
    }
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
      bulk_g2s(dst, src, chunk, bar);
    }
  };
  if (p.all_active && !boxed) issue_copies(false);

  // this layer's schedule -> shared memory (overlaps the bulk copies when all replicas are active)
  int ticket = -1;
  if (FUSED) {
    // the schedule stage itself (same arithmetic as layup_schedule_kernel, K <= THREADS)
    const SchedParams &q = p.sched;
    const size_t row = (size_t)layer * K;
    const uint32_t step = q.step_dev[layer];                     // device state, advanced by the retiring CTA
    bool act = false;
    if (tid < K) {
      const int i = tid;
      act = draw_active(q.seed, step, i, q.skip_thr, q.delay_replica, q.delay_rounds);
      int peer = -1;
      double wh = q.w[row + i];
      if (act && K >= 2) {
        peer = draw_peer(q.seed, step, q.peer_mode == 0 ? (uint32_t)layer : kNoLayer, i, K);
        if (!SYM) wh = wh * 0.5;                                 // w_i <- w_i / 2 (exact)
      }
      if (HAS_V) {
        double p1 = q.bpow[2 * (row + i)], p2 = q.bpow[2 * (row + i) + 1];
        if (act) {
          p1 = __dmul_rn(p1, q.beta1);
          p2 = __dmul_rn(p2, q.beta2);
          s_c1[i] = (float)(q.lr / (1.0 - p1));
          s_c2[i] = (float)(1.0 / sqrt(1.0 - p2));
        }
        s_bp[2 * i] = p1;
        s_bp[2 * i + 1] = p2;
      }
      s_peer[i] = peer;
      s_wh[i] = wh;
    }
    __syncthreads();
    if (tid < K) {
      const int j = tid;
      int cnt = 0, below = 0, last = -1;
      for (int sdr = 0; sdr < K; ++sdr) {
        const int pr = s_peer[sdr];
        cnt += (pr == j);
        below += (pr >= 0 && pr < j);
        if (pr == j) last = sdr;
      }
      double W = s_wh[j];
      int n_list = 0;
      if (SYM) {
        s_senders[j] = s_peer[j];
        s_begin[j] = 0;
      } else if (q.mix_mode == kMixLossy) {
        // only the last writer lands; slot j is this receiver's own
        s_begin[j] = j;
        if (last >= 0) {
          const double ws = s_wh[last];
          s_senders[j] = last;
          s_alpha[j] = (float)(ws / (W + ws));
          W = W + ws;
          n_list = 1;
        }
      } else {
        int k = below;
        s_begin[j] = below;
        for (int sdr = 0; sdr < K; ++sdr) {
          if (s_peer[sdr] != j) continue;
          const double ws = s_wh[sdr];
          s_senders[k] = sdr;
          s_alpha[k] = (float)(ws / (W + ws));               // one rounding to fp32
          W = W + ws;                                        // w_j <- w_j + w_i
          ++k;
        }
        n_list = cnt;
      }
      s_cnt[j] = n_list;
      s_wnew[j] = W;
      s_flags[j] = (unsigned char)((act ? kFlagActive : 0) | (cnt > 0 ? kFlagRecv : 0));
    }
    __syncthreads();   // schedule visible; every read of step / w / bpow by this CTA has returned
    if (tid == 0) {
      // release: this CTA's reads of the old state are ordered before its ticket, so the CTA that
      // draws the last ticket (acquire below) may overwrite the state
      __threadfence();
      ticket = atomicAdd(q.ticket + layer, 1);
    }
  } else {
    // Programmatic dependent launch: this kernel may start while the schedule kernel in front of it
    // on the stream is still running (its tile loads above do not depend on it); the tables do.
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const size_t row = (size_t)layer * K;
    for (int k = tid; k < K; k += THREADS) {
      s_senders[k] = SYM ? p.t.peer[row + k] : p.t.senders[row + k];
      s_alpha[k] = p.t.alpha[row + k];
      s_flags[k] = p.t.flags[row + k];
      const int b = p.t.recv_off[(size_t)layer * (K + 1) + k];
      s_begin[k] = b;
      s_cnt[k] = p.t.recv_off[(size_t)layer * (K + 1) + k + 1] - b;
      if (HAS_V) {
        s_c1[k] = p.t.c1[row + k];
        s_c2[k] = p.t.c2[row + k];
      }
    }
    __syncthreads();   // schedule visible
  }

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
  for (int idx = tid; idx < n_items; idx += THREADS) {
    const int i = idx >> log2C, c = idx & (C - 1);
    if (c >= ncols) continue;
    if (!(s_flags[i] & kFlagActive)) continue;                              // idle replica: y = x already there
    float4 m = HAS_M ? ms[idx] : float4{0.f, 0.f, 0.f, 0.f};
    float4 v = HAS_V ? vs[idx] : float4{0.f, 0.f, 0.f, 0.f};
    const float4 y = local_step4<OPT>(xs[idx], gs[idx], m, v, p.s, HAS_V ? s_c1[i] : 0.f, HAS_V ? s_c2[i] : 0.f);
    const long long off = (long long)i * pad + (c << 2);
    if (HAS_M) st4(mb + off, m);
    if (HAS_V) st4(vb + off, v);
    xs[idx] = y;
  }
  __syncthreads();

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
      const int k0 = s_begin[i], k_end = k0 + s_cnt[i];
      for (int k = k0; k < k_end; ++k) peer_update4(acc, xs[(s_senders[k] << log2C) + c], s_alpha[k]);
      st4(xb + (long long)i * pad + (c << 2), acc);
    }
  }

  if (FUSED) {
    // the CTA that drew the last ticket of its layer knows every other CTA has read the old
    // state: it publishes the new push-sum weights / beta powers and re-arms the ticket
    __shared__ int s_last;
    const int tiles_in_layer = (int)(tab.prefix[lo + 1] - tab.prefix[lo]);
    if (tid == 0) {
      s_last = (ticket == tiles_in_layer - 1);
      if (s_last) __threadfence();   // acquire: every other CTA's ticket (and its reads before it) is behind us
    }
    __syncthreads();
    if (s_last) {
      const SchedParams &q = p.sched;
      const size_t row = (size_t)layer * K;
      if (tid < K) {
        if (!SYM) q.w[row + tid] = s_wnew[tid];
        if (HAS_V) {
          q.bpow[2 * (row + tid)] = s_bp[2 * tid];
          q.bpow[2 * (row + tid) + 1] = s_bp[2 * tid + 1];
          if (s_flags[tid] & kFlagActive) {
            q.t.c1[row + tid] = s_c1[tid];
            q.t.c2[row + tid] = s_c2[tid];
          }
        }
        // the schedule this launch consumed, for layup_schedule_tables (same layout as schedule.cu)
        q.t.peer[row + tid] = s_peer[tid];
        q.t.flags[row + tid] = s_flags[tid];
        // compact CSR by receiver (the lossy mixer keeps its one entry in slot j of shared memory)
        const int b = s_begin[tid], n = SYM ? 0 : s_cnt[tid];
        int off = 0;
        for (int r = 0; r < tid && !SYM; ++r) off += s_cnt[r];
        for (int k = 0; k < n; ++k) {
          q.t.senders[row + off + k] = s_senders[b + k];
          q.t.alpha[row + off + k] = s_alpha[b + k];
        }
        q.t.recv_off[(size_t)layer * (K + 1) + tid] = off;
        if (tid == K - 1) q.t.recv_off[(size_t)layer * (K + 1) + K] = off + n;
      }
      if (tid == 0) {
        q.step_dev[layer] = q.step_dev[layer] + 1u;
        q.ticket[layer] = 0;
      }
    }
  }
}

using TmaFn = void (*)(const UpdateParams, const PosTable);
struct TmaVariant {
  int threads, minb;
  TmaFn fn[3][2];       // [OPT][SYM]   schedule tables read from global memory (two launches)
  TmaFn fused[3][2];    // [OPT][SYM]   schedule computed in the kernel (one launch); nullptr = not built
};
#define LAYUP_TMA_ROW(O, F, T, MB) {layup_update_tma<O, false, F, T, MB>, layup_update_tma<O, true, F, T, MB>}
#define LAYUP_TMA_TABLE(F, T, MB) \
  {LAYUP_TMA_ROW(OPT_SGD, F, T, MB), LAYUP_TMA_ROW(OPT_SGD_MOM, F, T, MB), LAYUP_TMA_ROW(OPT_ADAMW, F, T, MB)}
#define LAYUP_TMA_NONE {{nullptr, nullptr}, {nullptr, nullptr}, {nullptr, nullptr}}
const TmaVariant kTma[] = {
    TmaVariant{256, 4, LAYUP_TMA_TABLE(false, 256, 4), LAYUP_TMA_TABLE(true, 256, 4)},
    TmaVariant{128, 8, LAYUP_TMA_TABLE(false, 128, 8), LAYUP_TMA_NONE},
    TmaVariant{512, 2, LAYUP_TMA_TABLE(false, 512, 2), LAYUP_TMA_NONE},
    TmaVariant{256, 2, LAYUP_TMA_TABLE(false, 256, 2), LAYUP_TMA_NONE},
    // tiles of >= 2048 items (K >= 32 without momentum): 16 warps per CTA, three CTAs per SM; measured on
    // configs[4] against the 256-thread shape: 0.819 -> 0.808 ms all active, 0.824 -> 0.777 ms with stragglers
    TmaVariant{512, 3, LAYUP_TMA_TABLE(false, 512, 3), LAYUP_TMA_TABLE(true, 512, 3)},
};
constexpr int kTmaBigTile = 4;
constexpr int kNumTma = sizeof(kTma) / sizeof(kTma[0]);

}  // namespace

int tma_num_variants() { return kNumTma; }
int tma_default_variant(int n_items, int n_sections) { return (n_items >= 2048 && n_sections == 2) ? kTmaBigTile : 0; }

size_t tma_smem_bytes(int K, int C, int opt, bool fused) {
  const int narr = opt == OPT_ADAMW ? 4 : opt == OPT_SGD_MOM ? 3 : 2;
  size_t b = (size_t)K * C * sizeof(float4) * narr + 8;                        // staged arrays + mbarrier
  if (fused) b += sizeof(double) * K * (opt == OPT_ADAMW ? 4 : 2) + sizeof(int) * K;   // wh, wnew (, beta powers), peer
  b += sizeof(int) * 3 * (size_t)K + sizeof(float) * K * (opt == OPT_ADAMW ? 3 : 1) + (size_t)K;
  return b;
}

bool tma_has_fused(int variant) { return variant >= 0 && variant < kNumTma && kTma[variant].fused[0][0] != nullptr; }

cudaError_t tma_kernel_setup(int variant, int opt, bool symmetric, int smem_bytes, int *threads, int *ctas_per_sm) {
  if (variant < 0 || variant >= kNumTma || opt < 0 || opt > 2) return cudaErrorInvalidValue;
  const TmaVariant &v = kTma[variant];
  cudaError_t e;
  int occ = 1 << 30;
  for (TmaFn f : {v.fn[opt][symmetric ? 1 : 0], v.fused[opt][symmetric ? 1 : 0]}) {
    if (!f) continue;
    if ((e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(f, cudaFuncAttributePreferredSharedMemoryCarveout, 100)) != cudaSuccess) return e;
    int a = 0;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&a, f, v.threads, smem_bytes)) != cudaSuccess) return e;
    occ = a < occ ? a : occ;
  }
  *threads = v.threads;
  *ctas_per_sm = occ;
  return cudaSuccess;
}

cudaError_t launch_update_tma(const UpdateParams &p, const PosTable &tab, int variant, bool fused, bool pdl, int grid,
                              int smem_bytes, cudaStream_t s) {
  const TmaVariant &v = kTma[variant];
  TmaFn f = (fused ? v.fused : v.fn)[p.opt][p.symmetric ? 1 : 0];
  if (!f) return cudaErrorInvalidValue;
  // two-launch path: behind the schedule kernel, programmatic stream serialization lets this kernel's
  // prologue and tile loads overlap it (griddepcontrol.wait above guards the tables);
  // single-launch path: the same attribute chains consecutive rounds (see the top of the kernel)
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid);
  cfg.blockDim = dim3((unsigned)v.threads);
  cfg.dynamicSmemBytes = (size_t)smem_bytes;
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, f, p, tab);
}

}  // namespace layup
