// Model-disagreement diagnostic: per (layer, replica) the squared distance
// to the consensus,  dist[l][i] = sum_e (x_i[e] - xbar[e])^2,  xbar = sum_i c_i x_i  with c_i = 1/K
// (the paper's plain average) or c_i = w_i (push-sum weighted consensus).
// PAPER.md:389-395 (Fig. A1 "model disagreement between workers"), eq. (9) PAPER.md:551.
//
// The only place on the path that needs norms, hence the only warp-level reductions.  Read-only:
// 4 B of HBM traffic per parameter, so the roofline is the HBM read rate.
//
// Ring kernel (K <= 64), warp specialised:
//   * four PRODUCER warps per CTA stream tiles (all K replicas x TF floats) into an S-stage shared
//     memory ring with 1-D TMA bulk copies (cp.async.bulk, SASS UBLKCP), one copy per replica row
//     spread over the warp's lanes, completing on the stage's "full" mbarrier; it re-arms a stage
//     as soon as the stage's "empty" mbarrier has seen every consumer warp;
//   * the CONSUMER warps (16 per CTA; 8 for K > 32, where the accumulators fill the register file)
//     never meet a CTA-wide barrier: a thread owns ONE scalar column of the tile for ALL K replicas,
//     so the consensus of its column and the K squared distances are register arithmetic (fp64),
//     with no exchange through shared memory.  For K <= 16 every element is converted to fp64 once
//     and kept in registers for both passes, and the stage is released right after the loads; for
//     larger K the second pass re-reads shared memory;
//   * a CTA walks a CONTIGUOUS range of the tile list, so it crosses a layer boundary only a few
//     times; the per-replica partial sums stay in registers until then and leave through warp
//     shuffles and one fp64 atomicAdd per (warp, replica).
// General kernel (K > 64): the earlier one-stage form, consensus through shared memory.
#include "layup_internal.cuh"
#include "tma_ptx.cuh"

namespace layup {

namespace {

struct DiagParams {
  const float *x;          // X section base
  const double *w;         // [L*K] push-sum weights, or nullptr for the plain mean
  double *dist;            // [L*K] output, zeroed before the launch
  int32_t K, C, log2C;     // C = float4 columns per tile
  int32_t stages;          // ring depth (ring kernel); 1 or 2 (general kernel)
};

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
  return v;
}

// KT: compile-time bound on K (loops fully unrolled, accumulators in registers)
// NCW: consumer warps; a thread owns ONE scalar column of the tile (tile row = NCW*32 floats)
// kDiagProducers producer warps share a tile's row copies (a warp issues its bulk copies one lane at a time)
// KEEP: keep the converted tile in registers between the two passes (one fp32->fp64 conversion per element)
// CPT: scalar columns per consumer thread (columns tid, tid + NC, ...): for K <= 8 two columns per thread
//      make the tile as large (32 KB) and the per-tile barrier traffic as rare as at K = 16
constexpr int kDiagProducers = 4;
template <int KT, bool KEEP, int NCW, int CPT = 1>
__global__ void __launch_bounds__(NCW * 32 + 32 * kDiagProducers, 1)
    layup_disagreement_kernel(const __grid_constant__ DiagParams p, const __grid_constant__ PosTable tab) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  constexpr int NC = NCW * 32;                                           // consumer threads
  constexpr int TF = NC * CPT;                                           // floats per replica row of a tile
  const int K = p.K, S = p.stages, tid = threadIdx.x;
  float *ring = reinterpret_cast<float *>(smem_raw);                    // [S][K][TF]
  uint64_t *full = reinterpret_cast<uint64_t *>(ring + (size_t)S * K * TF);   // [S]
  uint64_t *empty = full + S;                                           // [S]
  double *coef_all = reinterpret_cast<double *>(empty + S);             // [consumer warps][KT] weighted mode only
  if (tid == 0) {
    for (int s = 0; s < S; ++s) {
      mbar_init(full + s, 1);
      mbar_init(empty + s, NCW);
    }
  }
  __syncthreads();

  // contiguous share of the tile list (dealing the tiles round-robin over the CTAs was measured
  // slower, 3.51 vs 3.19 ms on configs[2]: every CTA then crosses every layer boundary)
  const long long n_tiles = tab.prefix[tab.n];
  const long long t0 = n_tiles * blockIdx.x / gridDim.x, t1 = n_tiles * (blockIdx.x + 1) / gridDim.x;
  if (t0 >= t1) return;
  int pos = 0;
  {
    int lo = 0, hi = tab.n;
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (t0 >= tab.prefix[mid]) lo = mid; else hi = mid;
    }
    pos = lo;
  }

  if (tid >= NC) {
    // ---------------- producer warps: row i of a tile goes to warp i mod kDiagProducers; warp 0 posts
    // the stage's byte count (the only arrival "full" expects, so the phase cannot complete before it)
    const int lane = (tid - NC) & 31, pw = (tid - NC) >> 5;
    int s = 0;
    uint32_t ph = 0;
    for (long long tile = t0; tile < t1; ++tile) {
      while (tile >= tab.prefix[pos + 1]) ++pos;
      const long long pad = tab.lay[pos].pad;
      const long long f0 = (tile - tab.prefix[pos]) * TF;               // first float of the tile in a slice
      const long long left = pad - f0;
      const uint32_t chunk = (uint32_t)(left < TF ? left : TF) * 4u;     // multiple of 128 B
      const float *src = p.x + tab.lay[pos].base + f0;
      mbar_wait(empty + s, ph ^ 1u);                                    // the first pass over the ring is free
      if (lane == 0 && pw == 0) mbar_expect_tx(full + s, chunk * (uint32_t)K);
      __syncwarp();
      float *dst = ring + (size_t)s * K * TF;
      for (int i = pw + kDiagProducers * lane; i < K; i += 32 * kDiagProducers)
        bulk_g2s(dst + (size_t)i * TF, src + (long long)i * pad, chunk, full + s);
      if (++s == S) { s = 0; ph ^= 1u; }
    }
    return;
  }

  // ---------------- consumers: thread owns column `tid` of the tile for all K replicas
  // consensus coefficients: the scalar 1/K, or this layer's push-sum weights in a per-warp copy
  // (warps cross layer boundaries at different times and never synchronise with each other)
  double acc[KT];
#pragma unroll
  for (int i = 0; i < KT; ++i) acc[i] = 0.0;
  const double inv_k = 1.0 / (double)K;
  double *coef = coef_all + (size_t)(tid >> 5) * KT;
  const bool weighted = p.w != nullptr;
  auto load_coef = [&](int q) {
    if (!weighted) return;
    __syncwarp();
    for (int i = tid & 31; i < KT; i += 32) coef[i] = i < K ? __ldg(p.w + (size_t)tab.layer[q] * K + i) : 0.0;
    __syncwarp();
  };
  auto flush = [&](int q) {
#pragma unroll
    for (int i = 0; i < KT; ++i) {
      if (i < K) {
        const double v = warp_sum(acc[i]);
        if ((tid & 31) == 0) atomicAdd(p.dist + (size_t)tab.layer[q] * K + i, v);
      }
      acc[i] = 0.0;
    }
  };
  load_coef(pos);
  int s = 0;
  uint32_t ph = 0;
  for (long long tile = t0; tile < t1; ++tile) {
    if (tile >= tab.prefix[pos + 1]) {
      flush(pos);
      while (tile >= tab.prefix[pos + 1]) ++pos;
      load_coef(pos);
    }
    const long long left = tab.lay[pos].pad - (tile - tab.prefix[pos]) * TF;
    const float *row0 = ring + (size_t)s * K * TF + tid;
    mbar_wait(full + s, ph);
    if (KEEP && K == KT && left >= TF) {
      // ---- whole tile, K == KT: no predicate anywhere; every element is converted once and kept in
      // registers for both passes, the stage is released right after the loads, and the consensus
      // sum of a column runs on four chains (two per column with two columns per thread)
      constexpr int CH = CPT == 1 ? 4 : 2;
      double xd[CPT][KT], mc[CPT][CH];
#pragma unroll
      for (int c = 0; c < CPT; ++c) {
#pragma unroll
        for (int h = 0; h < CH; ++h) mc[c][h] = 0.0;
#pragma unroll
        for (int i = 0; i < KT; ++i) {
          xd[c][i] = (double)row0[(size_t)i * TF + c * NC];
          mc[c][i % CH] = fma(weighted ? coef[i] : inv_k, xd[c][i], mc[c][i % CH]);
        }
      }
      __syncwarp();
      if ((tid & 31) == 0) mbar_arrive(empty + s);                      // the tile now lives in registers
#pragma unroll
      for (int c = 0; c < CPT; ++c) {
        const double m = CH == 4 ? (mc[c][0] + mc[c][1]) + (mc[c][2] + mc[c][3]) : mc[c][0] + mc[c][1];
#pragma unroll
        for (int i = 0; i < KT; ++i) {
          const double d = xd[c][i] - m;
          acc[i] = fma(d, d, acc[i]);
        }
      }
    } else {
      // ---- ragged tail of a layer, or K < KT: same arithmetic, predicated
#pragma unroll
      for (int c = 0; c < CPT; ++c) {
        const bool live = (long long)(tid + c * NC) < left;             // pads are part of the slice (zero in every replica)
        double m = 0.0;
        if (live) {
#pragma unroll
          for (int i = 0; i < KT; ++i)
            if (i < K) m = fma(weighted ? coef[i] : inv_k, (double)row0[(size_t)i * TF + c * NC], m);
#pragma unroll
          for (int i = 0; i < KT; ++i) {
            if (i < K) {
              const double d = (double)row0[(size_t)i * TF + c * NC] - m;
              acc[i] = fma(d, d, acc[i]);
            }
          }
        }
      }
      __syncwarp();
      if ((tid & 31) == 0) mbar_arrive(empty + s);
    }
    if (++s == S) { s = 0; ph ^= 1u; }
  }
  flush(pos);
}

// ---- split form (32 < K <= 64): eight lane groups of a warp share the warp's 16 columns.
// Lane l = (g, jj), g = l / 4, jj = l % 4, owns the four columns 4jj .. 4jj+3 of the warp's block (one
// float4) for the RPL = KT/8 replicas g*RPL .. g*RPL + RPL-1: one LDS.128 per replica.  The values
// stay in registers as fp32 (4*RPL registers), so the stage is handed back right after the loads --
// the whole ring is in flight, none of it parked under the two passes -- and the K accumulators of a
// column are spread over eight lanes (RPL fp64 registers each instead of KT), which leaves room for
// a tile row of only 128 floats: 32 KB stages at K = 64, six deep, where the one-column-per-thread
// form has three of 64 KB.  The partial consensus sums of the eight groups meet through three
// __shfl_xor_sync steps; no shared-memory exchange and no barrier besides the ring's mbarriers.
// (The two groups of a quarter-warp read the same 16 banks in different rows, a two-way conflict:
// shared memory then moves 64 B per clock per SM, still three times what HBM feeds an SM.)
// Slice pads are multiples of 32 floats, so a warp's 16-column block of a ragged last tile is
// either wholly inside the slice or wholly outside.

// fp32 -> fp64 of a value that was widened once already: `volatile` keeps the compiler from carrying the
// first pass's doubles (twice the registers of the fp32 tile) across to the second pass
__device__ __forceinline__ double widen_again(float f) {
  double d;
  asm volatile("cvt.f64.f32 %0, %1;" : "=d"(d) : "f"(f));
  return d;
}
__device__ __forceinline__ double shfl_add(double v, int mask) { return v + __shfl_xor_sync(0xFFFFFFFFu, v, mask); }

template <int KT, int NCW>
__global__ void __launch_bounds__(NCW * 32 + 32 * kDiagProducers, 1)
    layup_disagreement_split(const __grid_constant__ DiagParams p, const __grid_constant__ PosTable tab) {
  static_assert(KT % 8 == 0, "eight lane groups share the replicas");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  constexpr int NC = NCW * 32;                                           // consumer threads
  constexpr int TF = NCW * 16;                                           // floats per replica row of a tile
  constexpr int RPL = KT / 8;                                            // replicas per lane
  const int K = p.K, S = p.stages, tid = threadIdx.x;
  float *ring = reinterpret_cast<float *>(smem_raw);                    // [S][K][TF]
  uint64_t *full = reinterpret_cast<uint64_t *>(ring + (size_t)S * K * TF);   // [S]
  uint64_t *empty = full + S;                                           // [S]
  double *coef_all = reinterpret_cast<double *>(empty + S);             // [consumer warps][KT]
  if (tid == 0) {
    for (int s = 0; s < S; ++s) {
      mbar_init(full + s, 1);
      mbar_init(empty + s, NCW);
    }
  }
  __syncthreads();

  const long long n_tiles = tab.prefix[tab.n];
  const long long t0 = n_tiles * blockIdx.x / gridDim.x, t1 = n_tiles * (blockIdx.x + 1) / gridDim.x;
  if (t0 >= t1) return;
  int pos = 0;
  {
    int lo = 0, hi = tab.n;
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (t0 >= tab.prefix[mid]) lo = mid; else hi = mid;
    }
    pos = lo;
  }

  if (tid >= NC) {
    // ---------------- producer warps: as in the ring kernel above
    const int lane = (tid - NC) & 31, pw = (tid - NC) >> 5;
    int s = 0;
    uint32_t ph = 0;
    for (long long tile = t0; tile < t1; ++tile) {
      while (tile >= tab.prefix[pos + 1]) ++pos;
      const long long pad = tab.lay[pos].pad;
      const long long f0 = (tile - tab.prefix[pos]) * TF;
      const long long left = pad - f0;
      const uint32_t chunk = (uint32_t)(left < TF ? left : TF) * 4u;     // multiple of 128 B
      const float *src = p.x + tab.lay[pos].base + f0;
      mbar_wait(empty + s, ph ^ 1u);
      if (lane == 0 && pw == 0) mbar_expect_tx(full + s, chunk * (uint32_t)K);
      __syncwarp();
      float *dst = ring + (size_t)s * K * TF;
      for (int i = pw + kDiagProducers * lane; i < K; i += 32 * kDiagProducers)
        bulk_g2s(dst + (size_t)i * TF, src + (long long)i * pad, chunk, full + s);
      if (++s == S) { s = 0; ph ^= 1u; }
    }
    return;
  }

  // ---------------- consumers
  const int lane = tid & 31, g = lane >> 2, jj = lane & 3;
  const int wc0 = (tid >> 5) * 16;                                      // first column of this warp's block
  const int r0 = g * RPL;                                               // first replica of this lane group
  double acc[RPL];
#pragma unroll
  for (int k = 0; k < RPL; ++k) acc[k] = 0.0;
  const double inv_k = 1.0 / (double)K;
  double *coef = coef_all + (size_t)(tid >> 5) * KT;
  auto load_coef = [&](int qpos) {                                      // plain mean: the scalar 1/K, stored all the same
    __syncwarp();
    for (int i = lane; i < KT; i += 32)
      coef[i] = i < K ? (p.w != nullptr ? __ldg(p.w + (size_t)tab.layer[qpos] * K + i) : inv_k) : 0.0;
    __syncwarp();
  };
  auto flush = [&](int qpos) {
#pragma unroll
    for (int k = 0; k < RPL; ++k) {
      const double v = shfl_add(shfl_add(acc[k], 1), 2);                // the four lanes of a group: 16 columns
      if (jj == 0 && r0 + k < K) atomicAdd(p.dist + (size_t)tab.layer[qpos] * K + r0 + k, v);
      acc[k] = 0.0;
    }
  };
  load_coef(pos);
  int s = 0;
  uint32_t ph = 0;
  for (long long tile = t0; tile < t1; ++tile) {
    if (tile >= tab.prefix[pos + 1]) {
      flush(pos);
      while (tile >= tab.prefix[pos + 1]) ++pos;
      load_coef(pos);
    }
    const long long left = tab.lay[pos].pad - (tile - tab.prefix[pos]) * TF;
    const bool live = wc0 < left;                                       // warp-uniform: `left` is a multiple of 32
    const float *rows = ring + (size_t)s * K * TF + (size_t)r0 * TF + wc0 + 4 * jj;
    float4 xf[RPL];
    mbar_wait(full + s, ph);
    if (live) {
#pragma unroll
      for (int k = 0; k < RPL; ++k)
        xf[k] = (KT == K || r0 + k < K) ? *reinterpret_cast<const float4 *>(rows + (size_t)k * TF)
                                        : make_float4(0.f, 0.f, 0.f, 0.f);
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(empty + s);                              // the tile now lives in registers
    if (live) {
      double m[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
      for (int k = 0; k < RPL; ++k) {
        const double c = coef[r0 + k];                                  // 0 for replicas beyond K
        m[0] = fma(c, (double)xf[k].x, m[0]); m[1] = fma(c, (double)xf[k].y, m[1]);
        m[2] = fma(c, (double)xf[k].z, m[2]); m[3] = fma(c, (double)xf[k].w, m[3]);
      }
#pragma unroll
      for (int v = 0; v < 4; ++v) m[v] = shfl_add(shfl_add(shfl_add(m[v], 4), 8), 16);   // lanes with the same jj
#pragma unroll
      for (int k = 0; k < RPL; ++k) {
        if (KT == K || r0 + k < K) {
          double d;
          d = widen_again(xf[k].x) - m[0]; acc[k] = fma(d, d, acc[k]);
          d = widen_again(xf[k].y) - m[1]; acc[k] = fma(d, d, acc[k]);
          d = widen_again(xf[k].z) - m[2]; acc[k] = fma(d, d, acc[k]);
          d = widen_again(xf[k].w) - m[3]; acc[k] = fma(d, d, acc[k]);
        }
      }
    }
    if (++s == S) { s = 0; ph ^= 1u; }
  }
  flush(pos);
}

// ---- general form (K > 64): consensus of every column through shared memory, one or two stages
constexpr int kGenThreads = 256;
template <int MAXIT>
__global__ void __launch_bounds__(kGenThreads) layup_disagreement_general(const __grid_constant__ DiagParams p,
                                                                          const __grid_constant__ PosTable tab) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  constexpr int THREADS = kGenThreads;
  const int K = p.K, C = p.C, log2C = p.log2C, tid = threadIdx.x;
  const int n_items = K << log2C;
  const bool two_stage = p.stages >= 2;
  float4 *stage0 = reinterpret_cast<float4 *>(smem_raw);                          // [1 or 2][K*C]
  double *mean = reinterpret_cast<double *>(stage0 + (two_stage ? 2 : 1) * (size_t)n_items);   // [C*4]
  double *coef = mean + 4 * C;                                                    // [K]
  double *red = coef + K;                                                         // [K] per-layer CTA sums
  uint64_t *bars = reinterpret_cast<uint64_t *>(red + K);                         // [2]

  if (tid == 0) {
    mbar_init(bars, 1);
    mbar_init(bars + 1, 1);
  }
  for (int k = tid; k < K; k += THREADS) red[k] = 0.0;
  __syncthreads();

  const long long n_tiles = tab.prefix[tab.n];
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
  auto issue_load = [&](long long tile, int s) {
    const int lo = locate(tile);
    const long long pad = tab.lay[lo].pad;
    const long long col0 = (tile - tab.prefix[lo]) << log2C;
    const long long cols_left = (pad >> 2) - col0;
    const uint32_t chunk = (uint32_t)(cols_left < C ? cols_left : C) * 16u;
    const float *xb = p.x + tab.lay[lo].base + (col0 << 2);
    if (tid == 0) mbar_expect_tx(bars + s, (uint32_t)K * chunk);
    for (int i = slot0; i < K; i += THREADS)
      bulk_g2s(stage0 + (size_t)s * n_items + (i << log2C), xb + (long long)i * pad, chunk, bars + s);
  };

  double acc[MAXIT];
#pragma unroll
  for (int u = 0; u < MAXIT; ++u) acc[u] = 0.0;

  // this thread's partial sums of the layer at position `pos` -> red[] -> global, then reset
  auto flush = [&](int pos) {
    const int seg = C < 32 ? C : 32;                                              // lanes of a warp that share a replica
#pragma unroll
    for (int u = 0; u < MAXIT; ++u) {
      const int idx = u * THREADS + tid;
      double s = acc[u];
      acc[u] = 0.0;
      for (int o = seg >> 1; o > 0; o >>= 1) s += __shfl_xor_sync(0xFFFFFFFFu, s, o);
      if ((tid & (seg - 1)) == 0 && idx < n_items) atomicAdd(red + (idx >> log2C), s);
    }
    __syncthreads();
    for (int k = tid; k < K; k += THREADS) {
      atomicAdd(p.dist + (size_t)tab.layer[pos] * K + k, red[k]);
      red[k] = 0.0;
    }
  };

  long long tile = blockIdx.x;
  if (tile < n_tiles) issue_load(tile, 0);
  int cur = -1;
  for (int it = 0; tile < n_tiles; tile += gridDim.x, ++it) {
    const int s = two_stage ? (it & 1) : 0;
    if (two_stage && tile + gridDim.x < n_tiles) issue_load(tile + gridDim.x, s ^ 1);   // prefetch into the free stage
    const int pos = locate(tile);
    if (pos != cur) {
      // leaving a layer: flush this CTA's partial sums, load the next layer's coefficients
      if (cur >= 0) flush(cur);
      for (int k = tid; k < K; k += THREADS)
        coef[k] = p.w ? p.w[(size_t)tab.layer[pos] * K + k] : 1.0 / (double)K;
      cur = pos;
      __syncthreads();
    }
    const long long pad = tab.lay[pos].pad;
    const long long col0 = (tile - tab.prefix[pos]) << log2C;
    const long long cols_left = (pad >> 2) - col0;
    const int ncols = cols_left < C ? (int)cols_left : C;
    const float4 *xs = stage0 + (size_t)s * n_items;
    mbar_wait(bars + s, (uint32_t)(two_stage ? (it >> 1) : it) & 1u);

    // consensus of every column, then the distances, both out of shared memory
    // (pads are zero in every replica and contribute 0)
    for (int c = tid; c < ncols; c += THREADS) {
      double m0 = 0.0, m1 = 0.0, m2 = 0.0, m3 = 0.0;
      for (int i = 0; i < K; ++i) {
        const float4 v = xs[(i << log2C) + c];
        const double ci = coef[i];
        m0 += ci * (double)v.x; m1 += ci * (double)v.y; m2 += ci * (double)v.z; m3 += ci * (double)v.w;
      }
      mean[4 * c + 0] = m0; mean[4 * c + 1] = m1; mean[4 * c + 2] = m2; mean[4 * c + 3] = m3;
    }
    __syncthreads();

    // squared distances into this thread's register slots (slot u <-> item u*THREADS + tid)
#pragma unroll
    for (int u = 0; u < MAXIT; ++u) {
      const int idx = u * THREADS + tid;
      const int c = idx & (C - 1);
      if (idx < n_items && c < ncols) {
        const float4 v = xs[idx];
        const double d0 = (double)v.x - mean[4 * c + 0], d1 = (double)v.y - mean[4 * c + 1];
        const double d2 = (double)v.z - mean[4 * c + 2], d3 = (double)v.w - mean[4 * c + 3];
        acc[u] += d0 * d0 + d1 * d1 + d2 * d2 + d3 * d3;
      }
    }
    fence_proxy_async();
    __syncthreads();   // this stage and mean[] are reused
    if (!two_stage && tile + gridDim.x < n_tiles) issue_load(tile + gridDim.x, 0);
  }
  if (cur >= 0) flush(cur);
}

using DiagFn = void (*)(const DiagParams, const PosTable);
struct RingShape {
  int kt, ncw, cpt;     // a tile row is ncw * 32 * cpt floats
  DiagFn fn;
  bool exact;           // only for K == kt (its predicated path would be slower than a general shape's)
  int tf = 0;           // floats per tile row if not ncw * 32 * cpt (split form: ncw * 16)
};
int ring_tf(const RingShape *r) { return r->tf ? r->tf : r->ncw * 32 * r->cpt; }
// one CTA per SM: the registers go to the per-replica accumulators (and the fp64 copy of the tile),
// the shared memory to a deep ring; 16 consumer warps while the accumulators allow it (8 were measured
// issue-bound: profiles/r2_disagreement_gpt2m_k16_8warps.txt)
// K <= 16: one instantiation per K, so that K == KT always takes the unpredicated path (the predicated
// one runs at 4-5.8 TB/s where the exact one reaches 6.4-6.8); columns per thread chosen so that a
// thread keeps about 16 converted elements
#define LAYUP_DIAG(KT_, CPT_) {KT_, 16, CPT_, layup_disagreement_kernel<KT_, true, 16, CPT_>, false}
// 16 < K <= 32: the converted tile still fits in registers with 8 consumer warps (K = 32: 6.2 -> 6.8 TB/s)
#define LAYUP_DIAG8(KT_, KEEP_) {KT_, 8, 1, layup_disagreement_kernel<KT_, KEEP_, 8>, true}
#define LAYUP_DIAGQ(KT_) {KT_, 8, 1, layup_disagreement_split<KT_, 8>, false, 8 * 16}
const RingShape kRing[] = {
    LAYUP_DIAG(1, 8),  LAYUP_DIAG(2, 8),  LAYUP_DIAG(3, 4),  LAYUP_DIAG(4, 4),  LAYUP_DIAG(5, 3),  LAYUP_DIAG(6, 2),
    LAYUP_DIAG(7, 2),  LAYUP_DIAG(8, 2),  LAYUP_DIAG(9, 1),  LAYUP_DIAG(10, 1), LAYUP_DIAG(11, 1), LAYUP_DIAG(12, 1),
    LAYUP_DIAG(13, 1), LAYUP_DIAG(14, 1), LAYUP_DIAG(15, 1), LAYUP_DIAG(16, 1),
    LAYUP_DIAG8(20, true), LAYUP_DIAG8(24, true), LAYUP_DIAG8(28, true), LAYUP_DIAG8(32, true),
    {32, 16, 1, layup_disagreement_kernel<32, false, 16>, false},
    // 32 < K <= 64: the split form (eight lane groups share a 16-column block, tile in fp32 registers, 128-float rows)
    LAYUP_DIAGQ(40), LAYUP_DIAGQ(48), LAYUP_DIAGQ(56), LAYUP_DIAGQ(64),
};
const RingShape *ring_shape(int K) {
  for (const RingShape &r : kRing)
    if (K == r.kt) return &r;
  for (const RingShape &r : kRing)
    if (K <= r.kt && !r.exact) return &r;
  return nullptr;
}

size_t ring_smem(int K, int tf, int stages, int kt, int ncw) {
  return (size_t)stages * K * tf * sizeof(float) + 16 * (size_t)stages + sizeof(double) * ncw * (size_t)kt;
}
size_t general_smem(int K, int C, bool two_stage) {
  return (two_stage ? 2 : 1) * (size_t)K * C * sizeof(float4) + sizeof(double) * (4 * (size_t)C + 2 * (size_t)K) + 16;
}
int general_iters(int K, int C) { return (K * C + kGenThreads - 1) / kGenThreads; }

}  // namespace

// Picks the kernel shape for K: *C = float4 columns per tile, *stages = ring depth (general kernel: 1 or 2).
cudaError_t diag_plan(int K, size_t smem_optin, int *C, int *stages, int *smem_bytes, int *ctas_per_sm) {
  cudaError_t e;
  if (const RingShape *r = ring_shape(K)) {
    const int tf = ring_tf(r);
    // as deep as fits in the ~224 KB of shared memory of the SM's one CTA
    const size_t budget = (size_t)(224 * 1024) - 1024 - sizeof(double) * r->ncw * r->kt;
    int S = (int)((budget < smem_optin ? budget : smem_optin) / ((size_t)K * tf * sizeof(float) + 16));
    if (S > 14) S = 14;
    if (S >= 2) {
      *C = tf / 4;
      *stages = S;
      *smem_bytes = (int)ring_smem(K, tf, S, r->kt, r->ncw);
      if ((e = allow_max_dynamic_smem((const void *)r->fn, *smem_bytes)) != cudaSuccess) return e;
      if ((e = cudaFuncSetAttribute(r->fn, cudaFuncAttributePreferredSharedMemoryCarveout, 100)) != cudaSuccess) return e;
      return cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas_per_sm, r->fn, r->ncw * 32 + 32 * kDiagProducers, *smem_bytes);
    }
  }
  int c = 8;
  while ((long long)K * c * 2 <= 2048 && c < 256) c *= 2;
  const bool two = general_smem(K, c, true) <= smem_optin;
  *C = c;
  *stages = two ? 2 : 1;
  *smem_bytes = (int)general_smem(K, c, two);
  if (general_iters(K, c) > 32) return cudaErrorInvalidValue;
  auto f = general_iters(K, c) <= 8 ? layup_disagreement_general<8> : layup_disagreement_general<32>;
  if ((e = allow_max_dynamic_smem((const void *)f, *smem_bytes)) != cudaSuccess) return e;
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas_per_sm, f, kGenThreads, *smem_bytes);
}

cudaError_t launch_disagreement(const float *x, const double *w, double *dist, int K, int C, int log2C, int stages,
                                const PosTable &tab, int grid, int smem_bytes, cudaStream_t s) {
  DiagParams p{x, w, dist, K, C, log2C, stages};
  const RingShape *r = ring_shape(K);
  if (r && C * 4 == ring_tf(r) && stages >= 2 && (size_t)smem_bytes == ring_smem(K, C * 4, stages, r->kt, r->ncw)) {
    r->fn<<<grid, r->ncw * 32 + 32 * kDiagProducers, smem_bytes, s>>>(p, tab);
    return cudaGetLastError();
  }
  if (general_iters(K, C) <= 8) layup_disagreement_general<8><<<grid, kGenThreads, smem_bytes, s>>>(p, tab);
  else if (general_iters(K, C) <= 32) layup_disagreement_general<32><<<grid, kGenThreads, smem_bytes, s>>>(p, tab);
  else return cudaErrorInvalidValue;
  return cudaGetLastError();
}

}  // namespace layup

// =================================================================================================
// layup_disagreement_static (include/layup.h): the reduction above for callers that must not
// allocate device memory -- a monitoring hook inside the backward window (cudaMalloc / cudaFree
// wait for the whole device and would serialise the backward/gossip overlap of PAPER.md:108-112),
// a job whose HBM is fully handed out already, a process that only borrows an X section and
// never made a ctx (layup_init allocates).  The kernels and their launch plan are the ones
// layup_disagreement uses; only the home of the scratch differs:
//   ctx path:     ctx->d_dist / ctx->d_w, cudaMalloc'ed by layup_init;
//   static path:  g_static_scratch below, part of the library image on every device.
// =================================================================================================
#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "../../include/layup.h"

// [0, MAX_PAIRS): the fp64 sums the kernel atomicAdds into (must be zero at launch);
// [MAX_PAIRS, 2*MAX_PAIRS): this call's copy of the consensus coefficients w (weighted mode).
// 256 KiB per device, for as long as the library is loaded there.  The previous call's contents
// stay in it: every call clears / overwrites the part it is about to use, in stream order.
static __device__ __align__(256) double g_static_scratch[2 * LAYUP_STATIC_MAX_PAIRS];

namespace {

// In HOST code the name g_static_scratch is only the host-side shadow of the symbol -- not an
// address a kernel may dereference.  The real device address differs per device and comes from
// cudaGetSymbolAddress with that device current; it is looked up once per device and kept here.
constexpr int kStaticMaxDevices = 64;
struct StaticDevice {
  double *scratch = nullptr;     // device address of g_static_scratch on this device
  int n_sm = 0;
  size_t smem_optin = 0;
};
StaticDevice g_static_dev[kStaticMaxDevices];
std::mutex g_static_mu;           // set-up AND the whole call: all calls share the one array

int static_fail(int code, const char *fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  layup::note_error(buf);
  return code;
}
#define STATIC_CU(expr)                                                                          \
  do {                                                                                           \
    cudaError_t e__ = (expr);                                                                    \
    if (e__ != cudaSuccess)                                                                      \
      return static_fail(LAYUP_ECUDA, "%s: %s (%s:%d)", #expr, cudaGetErrorString(e__), __FILE__, __LINE__); \
  } while (0)

}  // namespace

extern "C" int layup_disagreement_static(const float *x_dev, int32_t K, int32_t L, const int64_t *numel,
                                         const double *w, double *dist, void *cuda_stream) {
  using namespace layup;
  // ---- arguments: everything is refused before a single CUDA call is enqueued
  if (!x_dev || !numel || !dist) return static_fail(LAYUP_EINVAL, "NULL argument");
  if (K < 1 || K > LAYUP_MAX_K) return static_fail(LAYUP_EINVAL, "K=%d outside [1,%d]", K, LAYUP_MAX_K);
  if (L < 1) return static_fail(LAYUP_EINVAL, "L=%d < 1", L);
  if ((long long)L * K > LAYUP_STATIC_MAX_PAIRS)
    return static_fail(LAYUP_EINVAL,
                       "L*K = %lld (layer, replica) pairs exceed LAYUP_STATIC_MAX_PAIRS = %d, the size of the "
                       "library's static scratch; use layup_disagreement (ctx-owned scratch) for this shape",
                       (long long)L * K, LAYUP_STATIC_MAX_PAIRS);
  if (reinterpret_cast<uintptr_t>(x_dev) % 128 != 0) return static_fail(LAYUP_EINVAL, "x_dev is not 128-byte aligned");
  long long section = 0;                                     // floats of the X section
  for (int l = 0; l < L; ++l) {
    if (numel[l] < 1) return static_fail(LAYUP_EINVAL, "numel[%d]=%lld < 1", l, (long long)numel[l]);
    section += (long long)K * ((numel[l] + 31) / 32 * 32);
  }
  int dev = -1;
  STATIC_CU(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kStaticMaxDevices) return static_fail(LAYUP_EINVAL, "device ordinal %d not supported (max %d)", dev, kStaticMaxDevices - 1);
  cudaPointerAttributes pa;
  STATIC_CU(cudaPointerGetAttributes(&pa, x_dev));
  if ((pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged) || (pa.type == cudaMemoryTypeDevice && pa.device != dev))
    return static_fail(LAYUP_EINVAL, "x_dev is not device memory of the current device %d", dev);

  std::lock_guard<std::mutex> lock(g_static_mu);             // held to the final synchronise (layup.h "Sharing")
  StaticDevice &sd = g_static_dev[dev];
  if (sd.scratch == nullptr) {
    // once per device, with that device current
    double *ptr = nullptr;
    STATIC_CU(cudaGetSymbolAddress(reinterpret_cast<void **>(&ptr), g_static_scratch));
    if (ptr == nullptr) return static_fail(LAYUP_ECUDA, "cudaGetSymbolAddress returned a null address");
    int n_sm = 0, optin = 0;
    STATIC_CU(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    STATIC_CU(cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    sd.n_sm = n_sm;
    sd.smem_optin = (size_t)optin;
    sd.scratch = ptr;
  }
  // the launch plan of layup_disagreement (function attributes + occupancy query: nothing is allocated)
  int C = 0, stages = 0, smem = 0, ctas = 0, log2C = 0;
  STATIC_CU(diag_plan(K, sd.smem_optin, &C, &stages, &smem, &ctas));
  if (ctas < 1) return static_fail(LAYUP_EINVAL, "K=%d does not fit the diagnostic kernel", K);
  while ((1 << log2C) < C) ++log2C;

  cudaStream_t s = (cudaStream_t)cuda_stream;
  const size_t n = (size_t)L * K;
  double *d_dist = sd.scratch, *d_w = sd.scratch + LAYUP_STATIC_MAX_PAIRS;
  STATIC_CU(cudaMemsetAsync(d_dist, 0, sizeof(double) * n, s));       // last call's sums are still there
  if (w) STATIC_CU(cudaMemcpyAsync(d_w, w, sizeof(double) * n, cudaMemcpyHostToDevice, s));
  // work list in reverse layer order, at most kMaxPos layers per launch, as in layup_disagreement;
  // layer offsets walked back from the end of the section (no host table is built)
  long long end = section;
  for (int q0 = 0; q0 < L;) {
    PosTable tab;
    int cnt = 0;
    tab.prefix[0] = 0;
    while (q0 + cnt < L && cnt < kMaxPos) {
      const int l = L - 1 - (q0 + cnt);
      const long long pad = (numel[l] + 31) / 32 * 32;
      end -= (long long)K * pad;
      tab.lay[cnt] = LayerDesc{end, pad, numel[l]};
      tab.layer[cnt] = l;
      tab.prefix[cnt + 1] = tab.prefix[cnt] + (pad / 4 + C - 1) / C;
      ++cnt;
    }
    tab.n = cnt;
    const long long tiles = tab.prefix[cnt];
    const long long resident = (long long)sd.n_sm * ctas;
    const int grid = (int)(tiles < resident ? tiles : resident);
    STATIC_CU(launch_disagreement(x_dev, w ? d_w : nullptr, d_dist, K, C, log2C, stages, tab, grid, smem, s));
    q0 += cnt;
  }
  STATIC_CU(cudaMemcpyAsync(dist, d_dist, sizeof(double) * n, cudaMemcpyDeviceToHost, s));
  STATIC_CU(cudaStreamSynchronize(s));
  return LAYUP_OK;
}
