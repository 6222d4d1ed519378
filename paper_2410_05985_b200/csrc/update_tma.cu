// TMA-staged form of the fused local-step + gossip-mix kernel (rule.cuh holds the arithmetic).
//
// Work item = (layer, tile of C float4 columns) for ALL K replicas, one CTA per item.  The tile
// of every array (x, g, m, v) is brought into shared memory by the TMA engine, completing on one
// mbarrier, so the whole tile (K*C*16 B per array) is in flight per CTA without holding registers:
//   - when every replica is active and the box fits the TMA limits: ONE 2-D tiled copy per array
//     (cp.async.bulk.tensor.2d, SASS UTMALDG.2D) through a tensor map that views a layer section
//     as [K rows][padded slice];
//   - all active but no tensor map (K > 256, huge slices): K x arrays 1-D bulk copies (cp.async.bulk,
//     SASS UBLKCP), spread over all warps;
//   - straggler mode (STRAG): the rows a round needs -- x of every replica that is active or
//     receives, g / m / v of the active ones -- are only known on the device.  Every thread reads
//     the flag of its (replica, array) slot straight from the device table and issues that row's
//     bulk copy at once, posting its bytes on the barrier itself (one arrival per warp): no staging
//     of the flags, no CTA barrier in front of the loads; an idle replica costs no bytes.  With
//     one-row tensor maps (tiles whose rows are only 128 B long, or layup_tuning.tma2d = 1) the same
//     rows go out four at a time as cp.async.bulk.tensor.2d.tile::gather4 requests (SASS
//     UTMALDG.2D.GATHER4; a row the round does not need is given an out-of-range index, which
//     costs no HBM traffic and lands as zeros).
// The local step then runs out of shared memory, y overwrites x in place (the "send" is an
// on-chip read), m' (and AdamW's v') go straight to HBM, and after one CTA barrier
// every receiver folds its senders and writes x once.  HBM traffic: 12 B (SGD) / 20 B (momentum) /
// 28 B (AdamW) per parameter update, nothing read or written twice.
// Template parameters: OPT = local optimiser (rule.cuh), SYM = symmetric pairwise averaging
// instead of the push-sum fold, FUSED = the schedule stage runs in this kernel (one launch),
// STRAG = the ctx has a straggler mode (some replicas may idle in a round),
// REGA / U = split staging (below).
#include "layup_internal.cuh"
#include "philox.cuh"
#include "rule.cuh"
#include "tma_ptx.cuh"

namespace layup {

namespace {

__device__ __forceinline__ float4 ld4_stream(const float *p) {   // read once, by this thread only: keep it out of L1
  float4 v;
  asm volatile("ld.global.L1::no_allocate.v4.f32 {%0, %1, %2, %3}, [%4];"
               : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p) : "memory");
  return v;
}

// FUSED: the schedule stage (schedule.cu) runs inside this kernel -- ONE launch per round or
// per layer event instead of two.  Every CTA of a layer recomputes that layer's O(K) schedule in
// shared memory from the same inputs (seed, step, w, beta powers), so all CTAs agree bit for bit;
// the CTA that is LAST to have read the state (a ticket per layer) writes the new w / beta powers
// back in place.  Used for launches of few tiles (launch-latency bound) and K <= kFusedMaxK.
//
// REGA / U: split staging.  Only x has to be in shared memory (it becomes y, which the receivers
// of other replicas read); g, m and v are consumed once, by the thread that takes the local step
// of that element.  REGA > 0 brings the LAST REGA arrays of (x, g, m, v) into REGISTERS with plain
// 128-bit loads issued next to the TMA copies (each thread owns U items: idx = tid + u*THREADS),
// so a CTA needs less shared memory and one more CTA fits per SM (straggler rounds).
template <int OPT, bool SYM, bool FUSED, bool STRAG, int THREADS, int MINB, int REGA = 0, int U = 1>
__global__ void __launch_bounds__(THREADS, MINB)
    layup_update_tma(const __grid_constant__ UpdateParams p, const __grid_constant__ PosTable tab) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  constexpr int NARR = OptTraits<OPT>::kArrays;
  constexpr bool HAS_M = NARR >= 3, HAS_V = NARR >= 4;
  constexpr int RA = REGA < NARR ? REGA : NARR - 1;                         // arrays staged through registers
  constexpr int NS = NARR - RA;                                             // arrays staged in shared memory
  constexpr bool G_REG = NS <= 1, M_REG = HAS_M && NS <= 2, V_REG = HAS_V && NS <= 3;
  constexpr int NW = THREADS / 32;
  static_assert(!(FUSED && RA > 0), "the single-launch path stages every array in shared memory");
  const int K = p.K, C = p.C, log2C = p.log2C, tid = threadIdx.x;
  const int n_items = K << log2C;
  const int arr_items = STRAG && p.tmaps_g4 != nullptr ? ((K + 3) & ~3) << log2C : n_items;   // gather4: whole groups of four rows
  float4 *xs = reinterpret_cast<float4 *>(smem_raw);                       // [K*C]  x, then y in place
  float4 *gs = xs + arr_items;                                              // [K*C]  (unless G_REG)
  float4 *ms = HAS_M ? gs + arr_items : gs;                                 // [K*C] (momentum / Adam m; unless M_REG)
  float4 *vs = HAS_V ? ms + arr_items : ms;                                 // [K*C] (Adam v; unless V_REG)
  uint64_t *bar = reinterpret_cast<uint64_t *>(xs + NS * arr_items);
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
  unsigned char *s_flags = reinterpret_cast<unsigned char *>(s_c2 + (HAS_V ? K : 0));  // [K rounded up to 4], 4-byte aligned

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
  const bool boxed = !STRAG && p.tmaps != nullptr;         // whole-tile 2-D TMA loads, one per array
  if (tid == 0) {
    // STRAG: every warp posts the bytes of the copies it issues and then arrives (NW arrivals);
    // otherwise every replica is active, the byte count is known up front and thread 0 alone arrives
    mbar_init(bar, STRAG ? NW : 1);
    if (STRAG)
      for (int k = K; k < ((K + 3) & ~3); ++k) s_flags[k] = 0;              // the last group of four may be partial
    if (boxed) {
      mbar_expect_tx(bar, (uint32_t)n_items * 16u * NS);                    // full boxes, zero fill included
      const unsigned char *tm = reinterpret_cast<const unsigned char *>(p.tmaps);
#pragma unroll
      for (int a = 0; a < NS; ++a)
        tma_load_2d(xs + a * arr_items, tm + ((size_t)a * p.L + layer) * 128, (int)(col0 << 2), 0, bar);
    } else if (!STRAG) {
      mbar_expect_tx(bar, (uint32_t)K * NS * chunk);
    }
  }
  __syncthreads();   // mbarrier visible

  // Bulk copies are issued one lane at a time within a warp, so spread them over all warps:
  // copy slot c goes to warp c % NW, lane c / NW.
  const int slot0 = (tid & 31) * NW + (tid >> 5);
  if (!STRAG && !boxed) {
    for (int c = slot0; c < K * NS; c += THREADS) {
      const int i = c / NS, a = c - i * NS;
      const float *src = (a == 0 ? xb : a == 1 ? gb : a == 2 ? mb : vb) + (long long)i * pad;
      bulk_g2s(xs + a * arr_items + (i << log2C), src, chunk, bar);
    }
  }

  // Straggler mode, row copies: slot c = (replica i, array a) is fetched iff the round needs it -- x
  // of a replica that is active or receives, g / m / v of an active one (an idle replica costs no
  // bytes).  Every thread posts the bytes of its own copies on the barrier, and every warp arrives
  // once its lanes have posted, so the phase cannot complete before the last byte count is known.
  // With the one-row tensor maps (layup_tuning.tma2d = 1) the same rows go out four at a time as
  // tile::gather4 requests: slot c = (group q of four consecutive replicas, array a); a row the round
  // does not need gets the row index K, which does not exist: no HBM traffic, zeros in shared memory
  // (never read), and the four-row byte count still completes on the barrier.
  bool rows_issued = false;
  auto issue_rows = [&](auto flag_of) {
    if (p.tmaps_g4 != nullptr) {
      const int n_groups = (K + 3) >> 2;
      const unsigned char *tm = reinterpret_cast<const unsigned char *>(p.tmaps_g4);
      for (int c = slot0; c < n_groups * NS; c += THREADS) {
        const int q = c / NS, a = c - q * NS;
        int r4[4];
        bool any = false;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const int i = 4 * q + j;
          const int f = i < K ? flag_of(i) : 0;
          const bool need = a == 0 ? f != 0 : (f & kFlagActive) != 0;
          r4[j] = need ? i : K;
          any |= need;
        }
        if (!any) continue;
        mbar_post_tx(bar, 4u * (uint32_t)C * 16u);
        tma_gather4(xs + a * arr_items + ((4 * q) << log2C), tm + ((size_t)a * p.L + layer) * 128, (int)(col0 << 2),
                    r4[0], r4[1], r4[2], r4[3], bar);
      }
    } else {
      for (int c = slot0; c < K * NS; c += THREADS) {
        const int i = c / NS, a = c - i * NS;
        const int f = flag_of(i);
        if (!f || (a > 0 && !(f & kFlagActive))) continue;
        const float *src = (a == 0 ? xb : a == 1 ? gb : a == 2 ? mb : vb) + (long long)i * pad;
        mbar_post_tx(bar, chunk);
        bulk_g2s(xs + a * arr_items + (i << log2C), src, chunk, bar);
      }
    }
    __syncwarp();
    if ((tid & 31) == 0) mbar_arrive(bar);
  };

  // register-staged arrays: this thread's U items, requested while the TMA copies are in flight
  const float4 zero4 = float4{0.f, 0.f, 0.f, 0.f};
  float4 rg[RA > 0 ? U : 1], rm[RA > 0 ? U : 1], rv[RA > 0 ? U : 1];
  auto reg_loads = [&]() {
#pragma unroll
    for (int u = 0; u < (RA > 0 ? U : 0); ++u) {
      const int idx = tid + u * THREADS;
      const int i = idx >> log2C, c = idx & (C - 1);
      rg[u] = rm[u] = rv[u] = zero4;
      if (idx < n_items && c < ncols && (!STRAG || (s_flags[i] & kFlagActive))) {
        const long long off = (long long)i * pad + (c << 2);
        if (G_REG) rg[u] = ld4_stream(gb + off);
        if (M_REG) rm[u] = ld4_stream(mb + off);
        if (V_REG) rv[u] = ld4_stream(vb + off);
      }
    }
  };
  if (RA > 0 && !STRAG) reg_loads();

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
    if (STRAG) {
      // every copy depends on one flag (four for a gather4 request) only: read them straight from the
      // device table and issue, without waiting for the tables to be staged in shared memory
      issue_rows([&](int i) { return (int)p.t.flags[row + i]; });
      rows_issued = true;
    }
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

  if (STRAG) {
    if (!rows_issued) issue_rows([&](int i) { return (int)s_flags[i]; });   // single-launch path: the flags were computed here
    if (RA > 0) reg_loads();
  }
  mbar_wait(bar, 0);

  // ---- phase 1: local step out of shared memory; y overwrites x in place, m' (v') -> HBM
  auto step_item = [&](int idx, const float4 &g, float4 m, float4 v) {
    const int i = idx >> log2C, c = idx & (C - 1);
    const float4 y = local_step4<OPT>(xs[idx], g, m, v, p.s, HAS_V ? s_c1[i] : 0.f, HAS_V ? s_c2[i] : 0.f);
    const long long off = (long long)i * pad + (c << 2);
    if (HAS_M) st4(mb + off, m);
    if (HAS_V) st4(vb + off, v);
    xs[idx] = y;
  };
  if (RA == 0) {
    for (int idx = tid; idx < n_items; idx += THREADS) {
      if ((idx & (C - 1)) >= ncols) continue;
      if (STRAG && !(s_flags[idx >> log2C] & kFlagActive)) continue;        // idle replica: y = x already there
      step_item(idx, gs[idx], HAS_M ? ms[idx] : zero4, HAS_V ? vs[idx] : zero4);
    }
  } else {
#pragma unroll
    for (int u = 0; u < (RA > 0 ? U : 0); ++u) {
      const int idx = tid + u * THREADS;
      if (idx >= n_items || (idx & (C - 1)) >= ncols) continue;
      if (STRAG && !(s_flags[idx >> log2C] & kFlagActive)) continue;
      step_item(idx, G_REG ? rg[u] : gs[idx], HAS_M ? (M_REG ? rm[u] : ms[idx]) : zero4,
                HAS_V ? (V_REG ? rv[u] : vs[idx]) : zero4);
    }
  }
  __syncthreads();

  if (SYM) {
    // ---- phase 2 (symmetric): every scalar column runs the K exchanges in worker order
    float *ysf = reinterpret_cast<float *>(xs);
    for (int e = tid; e < (ncols << 2); e += THREADS) symmetric_column(ysf, C << 2, e, K, s_senders);
    __syncthreads();
    for (int idx = tid; idx < n_items; idx += THREADS) {
      const int i = idx >> log2C, c = idx & (C - 1);
      if (c >= ncols || (STRAG && !s_flags[i])) continue;                   // idle and nobody's peer: 0 bytes
      st4(xb + (long long)i * pad + (c << 2), xs[idx]);
    }
  } else {
    // ---- phase 2: each receiver folds its senders in ascending order; x written once
    for (int idx = tid; idx < n_items; idx += THREADS) {
      const int i = idx >> log2C, c = idx & (C - 1);
      if (c >= ncols) continue;
      if (STRAG && !s_flags[i]) continue;                                   // idle, no push received: 0 bytes
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
  int rega, items;      // split staging: arrays through registers, items per thread (0, 0 = everything in shared memory)
  TmaFn fn[2][3][2];    // [STRAG][OPT][SYM]   schedule tables read from global memory (two launches)
  TmaFn fused[2][3][2]; // [STRAG][OPT][SYM]   schedule computed in the kernel (one launch); nullptr = not built
};
#define LAYUP_TMA_ROW(O, F, ST, T, MB, R, UU) \
  {layup_update_tma<O, false, F, ST, T, MB, R, UU>, layup_update_tma<O, true, F, ST, T, MB, R, UU>}
#define LAYUP_TMA_OPTS(F, ST, T, MB, R, UU)                                                      \
  {LAYUP_TMA_ROW(OPT_SGD, F, ST, T, MB, R, UU), LAYUP_TMA_ROW(OPT_SGD_MOM, F, ST, T, MB, R, UU), \
   LAYUP_TMA_ROW(OPT_ADAMW, F, ST, T, MB, R, UU)}
#define LAYUP_TMA_TABLE(F, T, MB, R, UU) {LAYUP_TMA_OPTS(F, false, T, MB, R, UU), LAYUP_TMA_OPTS(F, true, T, MB, R, UU)}
#define LAYUP_TMA_NONE6 {{nullptr, nullptr}, {nullptr, nullptr}, {nullptr, nullptr}}
#define LAYUP_TMA_NONE {LAYUP_TMA_NONE6, LAYUP_TMA_NONE6}
const TmaVariant kTma[] = {
    TmaVariant{256, 4, 0, 0, LAYUP_TMA_TABLE(false, 256, 4, 0, 1), LAYUP_TMA_TABLE(true, 256, 4, 0, 1)},
    TmaVariant{128, 8, 0, 0, LAYUP_TMA_TABLE(false, 128, 8, 0, 1), LAYUP_TMA_NONE},
    TmaVariant{512, 2, 0, 0, LAYUP_TMA_TABLE(false, 512, 2, 0, 1), LAYUP_TMA_NONE},
    TmaVariant{256, 2, 0, 0, LAYUP_TMA_TABLE(false, 256, 2, 0, 1), LAYUP_TMA_NONE},
    // tiles of >= 2048 items (K >= 32 without momentum): 16 warps per CTA, three CTAs per SM; measured on
    // configs[4] against the 256-thread shape: 0.819 -> 0.808 ms all active, 0.824 -> 0.777 ms with stragglers
    TmaVariant{512, 3, 0, 0, LAYUP_TMA_TABLE(false, 512, 3, 0, 1), LAYUP_TMA_TABLE(true, 512, 3, 0, 1)},
    // split staging, five CTAs per SM: the last array (m, or AdamW's v) through registers.  The straggler-mode
    // default when the optimiser has state: configs[2] shapes with 25 % stragglers 13.56 -> 12.92 ms
    TmaVariant{256, 5, 1, 4, LAYUP_TMA_TABLE(false, 256, 5, 1, 4), LAYUP_TMA_NONE},
    // two staged arrays (SGD without momentum) and tiles of <= 1024 items (K <= 16): 32 KB per CTA, so six CTAs
    // fit per SM where the 64-register shape above stops at four (128 KB in flight per SM)
    TmaVariant{256, 6, 0, 0, LAYUP_TMA_TABLE(false, 256, 6, 0, 1), LAYUP_TMA_NONE},
    // split staging for tiles of 2048 items (K >= 32 with momentum): x and g staged (64 KB), m through registers,
    // three CTAs of 512 threads instead of two of 256 with 96 KB each; straggler rounds of 1024 x 1025 layers
    // K = 64: 1.507 -> 1.314 ms, K = 32: 1.370 -> 1.250 ms (all active it loses 1-2.5 %; AdamW would spill)
    TmaVariant{512, 3, 1, 4, LAYUP_TMA_TABLE(false, 512, 3, 1, 4), LAYUP_TMA_NONE},
};
constexpr int kTmaBigTile = 4, kTmaSplit = 5, kTmaSix = 6, kTmaSplitBig = 7;
constexpr int kNumTma = sizeof(kTma) / sizeof(kTma[0]);

}  // namespace

int tma_num_variants() { return kNumTma; }
int tma_default_variant(int n_items, int n_sections) { return (n_items >= 2048 && n_sections == 2) ? kTmaBigTile : 0; }
// the thread shape of the launches that are not latency bound, where it differs from the default (-1: it does not):
// straggler mode with optimiser state -> split staging; two arrays and small tiles -> six CTAs per SM
int tma_bulk_variant(int n_items, int n_sections, bool straggler_mode) {
  if (straggler_mode && n_sections >= 3 && n_items <= kTma[kTmaSplit].items * kTma[kTmaSplit].threads) return kTmaSplit;
  if (straggler_mode && n_sections == 3 && n_items <= kTma[kTmaSplitBig].items * kTma[kTmaSplitBig].threads) return kTmaSplitBig;
  if (n_sections == 2 && n_items <= 1024) return kTmaSix;
  return -1;
}
int tma_variant_rega(int variant, int opt) {
  const int narr = opt == OPT_ADAMW ? 4 : opt == OPT_SGD_MOM ? 3 : 2;
  const int r = variant >= 0 && variant < kNumTma ? kTma[variant].rega : 0;
  return r < narr ? r : narr - 1;
}
int tma_variant_max_items(int variant) {
  return variant >= 0 && variant < kNumTma && kTma[variant].rega > 0 ? kTma[variant].items * kTma[variant].threads : 0;
}

size_t tma_smem_bytes(int K, int C, int opt, bool fused, int rega, bool gather4) {
  const int narr = (opt == OPT_ADAMW ? 4 : opt == OPT_SGD_MOM ? 3 : 2) - rega;
  size_t b = (size_t)(gather4 ? (K + 3) / 4 * 4 : K) * C * sizeof(float4) * narr + 8;   // staged arrays (gather4: whole groups of four rows) + mbarrier
  if (fused) b += sizeof(double) * K * (opt == OPT_ADAMW ? 4 : 2) + sizeof(int) * K;   // wh, wnew (, beta powers), peer
  b += sizeof(int) * 3 * (size_t)K + sizeof(float) * K * (opt == OPT_ADAMW ? 3 : 1) + (size_t)K;
  b += 4;                                                                      // flags padded to whole groups of four
  return b;
}

bool tma_has_fused(int variant) { return variant >= 0 && variant < kNumTma && kTma[variant].fused[0][0][0] != nullptr; }

cudaError_t tma_kernel_setup(int variant, int opt, bool symmetric, bool strag, int smem_bytes, int *threads, int *ctas_per_sm) {
  if (variant < 0 || variant >= kNumTma || opt < 0 || opt > 2) return cudaErrorInvalidValue;
  const TmaVariant &v = kTma[variant];
  cudaError_t e;
  int occ = 1 << 30;
  for (TmaFn f : {v.fn[strag ? 1 : 0][opt][symmetric ? 1 : 0], v.fused[strag ? 1 : 0][opt][symmetric ? 1 : 0]}) {
    if (!f) continue;
    if ((e = allow_max_dynamic_smem((const void *)f, smem_bytes)) != cudaSuccess) return e;
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
  TmaFn f = (fused ? v.fused : v.fn)[p.all_active ? 0 : 1][p.opt][p.symmetric ? 1 : 0];
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
