// Persistent form of the TMA-staged update kernel: a fixed grid of resident CTAs drains the
// reverse-layer-ordered work list (BASELINE.json north_star item 3, "a persistent grouped launch
// that drains many small layers from a work list"; the per-layer event of PAPER.md:108-112 is most
// frequent exactly there).  Same work item, same arithmetic (rule.cuh) and the same bits as
// update_tma.cu.  Selected with layup_tuning.launch_shape = 2.
//
// Warp-specialised: every CTA is a few producer warps plus G consumer GROUPS of `gs` threads around
// an S-stage shared-memory ring (S >= 2, as deep as fits; layup_tuning.stages, G divides S).  The
// groups take the CTA's tiles in turn (iteration n uses stage n mod S and belongs to group n mod G),
// so G tiles are in different phases of their computation at once -- what G resident CTAs give the
// grouped launch -- while the ring keeps the next S-G tiles in flight (one group of 8 warps alone was
// measured issue-bound at 14 % of the SM's warp slots: profiles/r2_update_persist_gpt2m_k16_1group.txt).
// Because G divides S a stage is always consumed by the same group, so every waiter of an mbarrier
// sees each of its phases (a group that skipped a phase would mistake an older completion of the
// same parity for its own).
//   producers draw the CTA's next tile from a global ticket (one atomicAdd per tile by producer warp
//             0, passed to the other warps through the stage), so the list is drained in order,
//             output layer first, and an SM that runs slower simply takes fewer tiles (with a static
//             stride a quarter of the SMs finished 2.7 ms after the rest on configs[2]);
//             for each tile it waits for the stage's
//             "empty" mbarrier, copies the layer's schedule tables (held in its registers, reloaded
//             only when the list crosses into another layer) into the stage, and issues the tile's
//             TMA loads on the stage's "full" mbarrier: ONE 2-D tiled load per array when every
//             replica is active, else 1-D bulk copies of exactly the rows the flags ask for
//             (an idle replica costs nothing, an idle receiver only its x row) -- the flags are in
//             the producer's registers, so a straggler round's loads need no table round trip;
//   consumers (per group) wait for "full", take the local steps out of shared memory (y overwrites
//             x in place, m' / v' go to HBM), meet on a named barrier that only the group shares,
//             hand the g / m / v slots of the stage back ("empty" per array: they are refilled while
//             the mix runs), fold every receiver's senders, write x once and release the x slot.
//             No CTA-wide barrier exists, so the producers are never gated by the consumers' phases.
#include "layup_internal.cuh"
#include "rule.cuh"
#include "tma_ptx.cuh"

namespace layup {

namespace {

constexpr int kPsProducers = 4;                       // producer warps (row copies are issued one lane at a time per warp)
constexpr int kPsMaxConsumers = 768;                  // consumer threads per CTA, all groups together
constexpr int kPsMaxThreads = kPsMaxConsumers + 32 * kPsProducers;
constexpr int kPsMaxEntries = 4;                      // table entries per producer lane: K <= 128

__device__ __forceinline__ void group_barrier(int group, int threads) {
  asm volatile("bar.sync %0, %1;" ::"r"(group + 1), "r"(threads) : "memory");
}

// per-stage copy of a layer's schedule (what the consumers read)
struct StageTables {
  int *begin, *cnt, *senders;
  float *alpha, *c1, *c2;
  unsigned char *flags;
};
__host__ __device__ inline size_t tables_bytes(int K) { return ((size_t)K * 25 + 15) / 16 * 16; }
__device__ __forceinline__ StageTables carve_tables(unsigned char *base, int K) {
  StageTables t;
  t.begin = reinterpret_cast<int *>(base);
  t.cnt = t.begin + K;
  t.senders = t.cnt + K;
  t.alpha = reinterpret_cast<float *>(t.senders + K);
  t.c1 = t.alpha + K;
  t.c2 = t.c1 + K;
  t.flags = reinterpret_cast<unsigned char *>(t.c2 + K);
  return t;
}

template <int OPT, bool SYM>
__global__ void __launch_bounds__(kPsMaxThreads, 1)
    layup_update_persist(const __grid_constant__ UpdateParams p, const __grid_constant__ PosTable tab, const int S,
                         const int G) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  constexpr int NARR = OptTraits<OPT>::kArrays;
  constexpr bool HAS_M = NARR >= 3, HAS_V = NARR >= 4;
  const int K = p.K, C = p.C, log2C = p.log2C;
  const int n_consumers = (int)blockDim.x - 32 * kPsProducers, gthreads = n_consumers / G;   // threads per consumer group
  const int n_items = K << log2C;
  const size_t stage_f4 = (size_t)NARR * n_items;                            // float4 per stage
  float4 *ring = reinterpret_cast<float4 *>(smem_raw);                       // [S][NARR][K*C]
  // one full/empty pair per (stage, array): the g / m / v slots of a stage are handed back to the
  // producers right after the local step, only the x slot (it holds y) lives through the mix
  uint64_t *full = reinterpret_cast<uint64_t *>(ring + (size_t)S * stage_f4);    // [S][NARR]
  uint64_t *empty = full + S * NARR;                                         // [S][NARR]
  uint64_t *sched = empty + S * NARR;                                        // [S] "tile number of the stage is known"
  long long *tile_of = reinterpret_cast<long long *>(sched + S);             // [S] tile in the stage, -1 = list drained
  unsigned char *tables0 = reinterpret_cast<unsigned char *>(tile_of + S);   // [S] StageTables
  const size_t tb = tables_bytes(K);

  if (threadIdx.x == 0) {
    for (int s = 0; s < S * NARR; ++s) {
      mbar_init(full + s, 1);
      mbar_init(empty + s, gthreads / 32);                // a stage is consumed by one group
    }
    for (int s = 0; s < S; ++s) mbar_init(sched + s, 1);
  }
  __syncthreads();   // the only CTA-wide barrier: mbarriers visible

  const long long n_tiles = tab.prefix[tab.n];

  if ((int)threadIdx.x >= n_consumers) {
    // ------------------------------------------------------------------ producer warps
    // warp pw feeds array a = pw mod NARR; with two arrays the rows of a straggler round are split
    // between two warps per array (a warp issues its bulk copies one lane at a time, ~22 per us)
    constexpr int R = kPsProducers / NARR;              // warps per array: 2, 1, 1 for 2, 3, 4 arrays
    const int lane = ((int)threadIdx.x - n_consumers) & 31, pw = ((int)threadIdx.x - n_consumers) >> 5;
    const int a = pw % NARR, r = pw / NARR;
    const bool boxed = p.all_active && p.tmaps != nullptr;
    if (r >= R || (boxed && r > 0)) return;             // spare warp; whole-tile 2-D loads need one warp per array
    int r_begin[kPsMaxEntries], r_cnt[kPsMaxEntries], r_send[kPsMaxEntries], r_flag[kPsMaxEntries];
    float r_alpha[kPsMaxEntries], r_c1[kPsMaxEntries], r_c2[kPsMaxEntries];
    int pos = 0, cur_pos = -1, s = 0;
    uint32_t ph = 0;
    const float *const asrc = a == 0 ? p.x : a == 1 ? p.g : a == 2 ? p.m : p.v;
    // the schedule kernel in front of this launch wrote the tables and zeroed the ticket
    // (programmatic dependent launch: this kernel may have started under it)
    asm volatile("griddepcontrol.wait;" ::: "memory");
    int sentinels = 0;
    for (;;) {
      // ---- which tile goes into stage s: warp 0 draws the ticket once its x slot is free
      long long tile;
      if (pw == 0) {
        mbar_wait(empty + s * NARR, ph ^ 1u);             // the first trip round the ring is free
        long long t = 0;
        if (lane == 0) {
          t = sentinels == 0 ? (long long)(unsigned)atomicAdd(p.ps_ticket, 1) : n_tiles;
          if (t >= n_tiles) t = -1;
          tile_of[s] = t;
          mbar_arrive(sched + s);                            // release: the other producer warps may read it
        }
        tile = __shfl_sync(0xFFFFFFFFu, t, 0);
      } else {
        mbar_wait(sched + s, ph);
        tile = tile_of[s];
        if (tile < 0) return;                             // list drained
        mbar_wait(empty + s * NARR + a, ph ^ 1u);
      }
      if (tile < 0) {
        // one end marker per consumer group (consecutive iterations belong to different groups)
        __syncwarp();
        if (lane == 0) mbar_arrive(full + s * NARR);
        if (++sentinels == G) return;
        if (++s == S) { s = 0; ph ^= 1u; }
        continue;
      }
      while (tile >= tab.prefix[pos + 1]) ++pos;
      if (pos != cur_pos) {
        const int layer = tab.layer[pos];
        const size_t row = (size_t)layer * K;
#pragma unroll
        for (int e = 0; e < kPsMaxEntries; ++e) {
          const int k = lane + 32 * e;
          r_flag[e] = 0;
          if (k < K) {
            r_flag[e] = p.t.flags[row + k];
            if (pw == 0) {                                // only the x warp passes the tables on
              r_send[e] = SYM ? p.t.peer[row + k] : p.t.senders[row + k];
              r_alpha[e] = p.t.alpha[row + k];
              const int b = p.t.recv_off[(size_t)layer * (K + 1) + k];
              r_begin[e] = b;
              r_cnt[e] = p.t.recv_off[(size_t)layer * (K + 1) + k + 1] - b;
              r_c1[e] = HAS_V ? p.t.c1[row + k] : 0.f;
              r_c2[e] = HAS_V ? p.t.c2[row + k] : 0.f;
            }
          }
        }
        cur_pos = pos;
      }
      const long long pad = tab.lay[pos].pad;
      const long long col0 = (tile - tab.prefix[pos]) << log2C;
      const long long cols_left = (pad >> 2) - col0;
      const uint32_t chunk = (uint32_t)(cols_left < C ? cols_left : C) * 16u;
      uint64_t *const fbar = full + s * NARR + a;
      if (pw == 0) {
        // hand the layer's tables to the consumers through the stage (they acquire them with the x slot)
        const StageTables T = carve_tables(tables0 + (size_t)s * tb, K);
#pragma unroll
        for (int e = 0; e < kPsMaxEntries; ++e) {
          const int k = lane + 32 * e;
          if (k < K) {
            T.begin[k] = r_begin[e]; T.cnt[k] = r_cnt[e]; T.senders[k] = r_send[e]; T.alpha[k] = r_alpha[e];
            if (HAS_V) { T.c1[k] = r_c1[e]; T.c2[k] = r_c2[e]; }
            T.flags[k] = (unsigned char)r_flag[e];
          }
        }
      }
      float4 *dst = ring + (size_t)s * stage_f4 + (size_t)a * n_items;
      if (boxed) {
        // ONE 2-D tiled load for this array's tile; the arrays go out side by side from their warps
        __syncwarp();                                     // table stores of all lanes before lane 0's arrive (release)
        if (lane == 0) {
          mbar_expect_tx(fbar, (uint32_t)n_items * 16u);
          const unsigned char *tm = reinterpret_cast<const unsigned char *>(p.tmaps);
          tma_load_2d(dst, tm + ((size_t)a * p.L + tab.layer[pos]) * 128, (int)(col0 << 2), 0, fbar);
        }
      } else {
        // Row copies of exactly the rows the flags ask for: x for every replica that is active or
        // receives, g / m / v for the active ones.  Warp r == 0 of the array posts the byte count --
        // the only arrival the slot's "full" barrier expects, so the phase cannot complete before
        // it, whatever the other warp's copies have already delivered.
        uint32_t bytes = 0;
#pragma unroll
        for (int e = 0; e < kPsMaxEntries; ++e)
          if (lane + 32 * e < K && (a == 0 ? r_flag[e] != 0 : (r_flag[e] & kFlagActive) != 0)) bytes += chunk;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) bytes += __shfl_xor_sync(0xFFFFFFFFu, bytes, o);
        __syncwarp();
        if (lane == 0 && r == 0) mbar_expect_tx(fbar, bytes);
        __syncwarp();
        const long long tile_off = tab.lay[pos].base + (col0 << 2);
#pragma unroll
        for (int e = 0; e < kPsMaxEntries; ++e) {
          const int i = lane + 32 * e;
          if (i < K && (i % R) == r && (a == 0 ? r_flag[e] != 0 : (r_flag[e] & kFlagActive) != 0))
            bulk_g2s(dst + (i << log2C), asrc + tile_off + (long long)i * pad, chunk, fbar);
        }
      }
      if (++s == S) { s = 0; ph ^= 1u; }
    }
  }

  // -------------------------------------------------------------------- consumer groups
  const int NT = gthreads;
  const int group = (int)threadIdx.x / gthreads, tid = (int)threadIdx.x % gthreads;
  int pos = 0, cur_pos = -1;
  int s = group;                                        // this group's iterations: group, group + G, ... (G divides S)
  uint32_t ph = 0;
  for (;;) {
    mbar_wait(full + s * NARR, ph);                       // x slot, tables and the tile number have landed (acquire)
    const long long tile = tile_of[s];
    if (tile < 0) break;                                  // list drained
    while (tile >= tab.prefix[pos + 1]) ++pos;
    if (pos != cur_pos) {
      if (p.trace != nullptr && tid == 0) {             // layup_trace: first start of the layer on this GPU
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        atomicMin(p.trace + tab.layer[pos], t);
      }
      cur_pos = pos;
    }
    const long long pad = tab.lay[pos].pad;
    const long long col0 = (tile - tab.prefix[pos]) << log2C;
    const long long cols_left = (pad >> 2) - col0;
    const int ncols = cols_left < C ? (int)cols_left : C;
    const long long tile_off = tab.lay[pos].base + (col0 << 2);
    float *const xb = p.x + tile_off;
    float *const mb = HAS_M ? p.m + tile_off : nullptr;
    float *const vb = HAS_V ? p.v + tile_off : nullptr;
    float4 *xs = ring + (size_t)s * stage_f4, *gs = xs + n_items;
    float4 *ms = HAS_M ? gs + n_items : gs, *vs = HAS_V ? ms + n_items : ms;
    const StageTables T = carve_tables(tables0 + (size_t)s * tb, K);
#pragma unroll
    for (int a = 1; a < NARR; ++a) mbar_wait(full + s * NARR + a, ph);   // the other arrays of the tile

    // ---- phase 1: local step; y overwrites x in place, m' (v') -> HBM
    for (int idx = tid; idx < n_items; idx += NT) {
      const int i = idx >> log2C, c = idx & (C - 1);
      if (c >= ncols) continue;
      if (!(T.flags[i] & kFlagActive)) continue;          // idle replica: y = x already there (if it was loaded)
      float4 m = HAS_M ? ms[idx] : float4{0.f, 0.f, 0.f, 0.f};
      float4 v = HAS_V ? vs[idx] : float4{0.f, 0.f, 0.f, 0.f};
      const float4 y = local_step4<OPT>(xs[idx], gs[idx], m, v, p.s, HAS_V ? T.c1[i] : 0.f, HAS_V ? T.c2[i] : 0.f);
      const long long off = (long long)i * pad + (c << 2);
      if (HAS_M) st4(mb + off, m);
      if (HAS_V) st4(vb + off, v);
      xs[idx] = y;
    }
    group_barrier(group, gthreads);
    // every thread of the group is past its reads of g, m, v: those slots go back to the producers now
    if ((tid & 31) == 0) {
#pragma unroll
      for (int a = 1; a < NARR; ++a) mbar_arrive(empty + s * NARR + a);
    }
    if (SYM) {
      // ---- phase 2 (symmetric): every scalar column runs the K exchanges in worker order
      float *ysf = reinterpret_cast<float *>(xs);
      for (int e = tid; e < (ncols << 2); e += NT) symmetric_column(ysf, C << 2, e, K, T.senders);
      group_barrier(group, gthreads);
      for (int idx = tid; idx < n_items; idx += NT) {
        const int i = idx >> log2C, c = idx & (C - 1);
        if (c >= ncols || !T.flags[i]) continue;          // idle and nobody's peer: 0 bytes
        st4(xb + (long long)i * pad + (c << 2), xs[idx]);
      }
    } else {
      // ---- phase 2: each receiver folds its senders in ascending order; x written once
      for (int idx = tid; idx < n_items; idx += NT) {
        const int i = idx >> log2C, c = idx & (C - 1);
        if (c >= ncols) continue;
        if (!T.flags[i]) continue;                        // idle, no push received: 0 bytes
        float4 acc = xs[idx];
        const int k0 = T.begin[i], k_end = k0 + T.cnt[i];
        for (int k = k0; k < k_end; ++k) peer_update4(acc, xs[(T.senders[k] << log2C) + c], T.alpha[k]);
        st4(xb + (long long)i * pad + (c << 2), acc);
      }
    }
    fence_proxy_async();   // the x slot was written through the generic proxy; the TMA engine refills it next
    __syncwarp();
    if ((tid & 31) == 0) mbar_arrive(empty + s * NARR);     // this warp is done with the stage
    s += G;
    if (s >= S) { s -= S; ph ^= 1u; }
  }
}

using PsFn = void (*)(const UpdateParams, const PosTable, const int, const int);
const PsFn kPs[3][2] = {{layup_update_persist<OPT_SGD, false>, layup_update_persist<OPT_SGD, true>},
                        {layup_update_persist<OPT_SGD_MOM, false>, layup_update_persist<OPT_SGD_MOM, true>},
                        {layup_update_persist<OPT_ADAMW, false>, layup_update_persist<OPT_ADAMW, true>}};

size_t stage_bytes(int K, int C, int opt) {
  const int narr = opt == OPT_ADAMW ? 4 : opt == OPT_SGD_MOM ? 3 : 2;
  return (size_t)K * C * sizeof(float4) * narr + 16 * (size_t)narr + 16 + tables_bytes(K);   // arrays, mbarrier pairs, tile number + its barrier, tables
}

}  // namespace

int persist_max_k() { return 32 * kPsMaxEntries; }

// Ring depth: `want` stages if > 0, else as deep as `ctas` CTAs per SM allow (<= 8); 0 if fewer than 2 fit.
int persist_stages(int K, int C, int opt, size_t smem_optin, int ctas, int want) {
  if (ctas < 1) ctas = 1;
  size_t budget = (size_t)(226 * 1024) / ctas - 1024;
  if (budget > smem_optin) budget = smem_optin;
  int S = (int)(budget / stage_bytes(K, C, opt));
  if (S > 8) S = 8;
  if (want > 0 && want < S) S = want;
  return S >= 2 ? S : 0;
}

size_t persist_smem_bytes(int K, int C, int opt, int stages) { return stage_bytes(K, C, opt) * stages; }

cudaError_t persist_kernel_setup(int opt, bool symmetric, int smem_bytes, int *ctas_per_sm) {
  if (opt < 0 || opt > 2) return cudaErrorInvalidValue;
  cudaError_t e;
  PsFn f = kPs[opt][symmetric ? 1 : 0];
  if ((e = allow_max_dynamic_smem((const void *)f, smem_bytes)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(f, cudaFuncAttributePreferredSharedMemoryCarveout, 100)) != cudaSuccess) return e;
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas_per_sm, f, kPsMaxThreads, smem_bytes);
}

// Shape of the consumer side for a ring of *stages and a tile of `n_items` float4 items: G groups of
// gs threads.  G divides the ring depth (the depth is trimmed to a multiple of G) and every group
// keeps at least two stages, one computing and one in flight; gs is a multiple of 32, at most the
// tile, and G*gs <= kPsMaxConsumers.  want_groups / want_gs > 0: the caller's choice, made legal.
void persist_shape(int *stages, int n_items, int want_groups, int want_gs, int *groups, int *gs) {
  int g = want_groups > 0 ? want_groups : (*stages >= 4 ? 2 : 1);
  while (g > 1 && *stages / g < 2) --g;
  *stages -= *stages % g;
  // one group: 512 threads, 768 for tiles of >= 2048 items (configs[4], K = 64: 0.859 -> 0.826 ms)
  int t = want_gs > 0 ? want_gs : (g == 1 ? (n_items >= 2048 ? 768 : 512) : 256);
  t = t / 32 * 32;
  if (t < 32) t = 32;
  while (t > 32 && (t * g > kPsMaxConsumers || t > n_items)) t -= 32;
  *groups = g;
  *gs = t;
}

cudaError_t launch_update_persist(const UpdateParams &p, const PosTable &tab, int grid, int smem_bytes, int stages,
                                  int groups, int group_threads, bool pdl, cudaStream_t s) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid);
  cfg.blockDim = dim3((unsigned)(groups * group_threads + 32 * kPsProducers));
  cfg.dynamicSmemBytes = (size_t)smem_bytes;
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kPs[p.opt][p.symmetric ? 1 : 0], p, tab, stages, groups);
}

}  // namespace layup
