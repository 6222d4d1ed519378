// Model-disagreement diagnostic: per (layer, replica) the squared distance
// to the consensus,  dist[l][i] = sum_e (x_i[e] - xbar[e])^2,  xbar = sum_i c_i x_i  with c_i = 1/K
// (the paper's plain average) or c_i = w_i (push-sum weighted consensus).
// PAPER.md:389-395 (Fig. A1 "model disagreement between workers"), eq. (9) PAPER.md:551.
//
// The only place on the path that needs norms, hence the only warp-level reductions.  Same tiling
// as the update kernel -- a CTA owns a tile of C float4 columns for ALL K replicas, staged by TMA
// bulk copies -- but read-only: 4 B of HBM traffic per parameter.  A persistent grid walks the
// work list with a static stride through a two-stage shared-memory pipeline (the next tile is in
// flight while this one is reduced).  A thread meets the same (replica, column) slots in every
// tile, so it keeps its partial sums in registers and the cross-thread reduction (warp shuffles,
// then one shared and one global fp64 atomic per replica) happens once per layer and CTA, not once
// per tile.  Everything is accumulated in fp64 (sums are order-dependent in the last bits).
#include "layup_internal.cuh"
#include "tma_ptx.cuh"

namespace layup {

namespace {

constexpr int kDiagThreads = 256;

struct DiagParams {
  const float *x;          // X section base
  const double *w;         // [L*K] push-sum weights, or nullptr for the plain mean
  double *dist;            // [L*K] output, zeroed before the launch
  int32_t K, C, log2C;
  int32_t two_stage;       // 1: prefetch the next tile into a second stage; 0: one stage (very large K)
};

// MAXIT >= ceil(K*C / kDiagThreads): register accumulators per thread
template <int MAXIT>
__global__ void __launch_bounds__(kDiagThreads) layup_disagreement_kernel(const __grid_constant__ DiagParams p,
                                                                          const __grid_constant__ PosTable tab) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  constexpr int THREADS = kDiagThreads;
  const int K = p.K, C = p.C, log2C = p.log2C, tid = threadIdx.x;
  const int n_items = K << log2C;
  float4 *stage0 = reinterpret_cast<float4 *>(smem_raw);                          // [1 or 2][K*C]
  double *mean = reinterpret_cast<double *>(stage0 + (p.two_stage ? 2 : 1) * (size_t)n_items);   // [C*4]
  double *psum = mean + 4 * C;                                                    // [THREADS*4] partial consensus sums
  double *coef = psum + 4 * THREADS;                                              // [K]
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
    const int s = p.two_stage ? (it & 1) : 0;
    if (p.two_stage && tile + gridDim.x < n_tiles) issue_load(tile + gridDim.x, s ^ 1);   // prefetch into the free stage
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
    mbar_wait(bars + s, (uint32_t)(p.two_stage ? (it >> 1) : it) & 1u);

    if (MAXIT <= 8 && C <= THREADS) {
      // Fast form: fp32 -> fp64 conversion is the scarce resource here (16 per clock and SM), so every
      // element is converted ONCE and kept in registers for both the consensus and the distance.
      // C divides THREADS: all items of a thread share the column c = tid & (C-1); the replicas of that
      // column are spread over the THREADS/C thread groups g = tid >> log2C, which exchange their
      // partial weighted sums through shared memory.
      double xd[MAXIT][4];
      double p0 = 0.0, p1 = 0.0, p2 = 0.0, p3 = 0.0;
      const int c = tid & (C - 1);
#pragma unroll
      for (int u = 0; u < MAXIT; ++u) {
        const int idx = u * THREADS + tid;
        float4 v = float4{0.f, 0.f, 0.f, 0.f};
        double ci = 0.0;
        if (idx < n_items && c < ncols) {
          v = xs[idx];
          ci = coef[idx >> log2C];
        }
        xd[u][0] = (double)v.x; xd[u][1] = (double)v.y; xd[u][2] = (double)v.z; xd[u][3] = (double)v.w;
        p0 += ci * xd[u][0]; p1 += ci * xd[u][1]; p2 += ci * xd[u][2]; p3 += ci * xd[u][3];
      }
      double *mine = psum + 4 * tid;                       // psum[g][c][4] with g*C + c == tid
      mine[0] = p0; mine[1] = p1; mine[2] = p2; mine[3] = p3;
      __syncthreads();
      double m0 = 0.0, m1 = 0.0, m2 = 0.0, m3 = 0.0;
      for (int g = 0; g < (THREADS >> log2C); ++g) {
        const double *q = psum + 4 * ((g << log2C) + c);
        m0 += q[0]; m1 += q[1]; m2 += q[2]; m3 += q[3];
      }
#pragma unroll
      for (int u = 0; u < MAXIT; ++u) {
        const int idx = u * THREADS + tid;
        if (idx < n_items && c < ncols) {
          const double d0 = xd[u][0] - m0, d1 = xd[u][1] - m1, d2 = xd[u][2] - m2, d3 = xd[u][3] - m3;
          acc[u] += d0 * d0 + d1 * d1 + d2 * d2 + d3 * d3;
        }
      }
      fence_proxy_async();
      __syncthreads();   // this stage and psum[] are reused
      if (!p.two_stage && tile + gridDim.x < n_tiles) issue_load(tile + gridDim.x, 0);
      continue;
    }

    // general form (very large K): consensus of every column, then the distances, both out of shared memory
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
    if (!p.two_stage && tile + gridDim.x < n_tiles) issue_load(tile + gridDim.x, 0);
  }
  if (cur >= 0) flush(cur);
}

}  // namespace

size_t diag_smem_bytes(int K, int C, bool two_stage) {
  return (two_stage ? 2 : 1) * (size_t)K * C * sizeof(float4) + sizeof(double) * (4 * (size_t)C + 4 * kDiagThreads + 2 * (size_t)K) + 16;
}

static int diag_iters(int K, int C) { return (K * C + kDiagThreads - 1) / kDiagThreads; }

cudaError_t diag_setup(int K, int C, int smem_bytes, int *ctas_per_sm) {
  cudaError_t e;
  auto f = diag_iters(K, C) <= 8 ? layup_disagreement_kernel<8> : layup_disagreement_kernel<32>;
  if ((e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes)) != cudaSuccess) return e;
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas_per_sm, f, kDiagThreads, smem_bytes);
}

cudaError_t launch_disagreement(const float *x, const double *w, double *dist, int K, int C, int log2C, bool two_stage,
                                const PosTable &tab, int grid, int smem_bytes, cudaStream_t s) {
  DiagParams p{x, w, dist, K, C, log2C, two_stage ? 1 : 0};
  if (diag_iters(K, C) <= 8) layup_disagreement_kernel<8><<<grid, kDiagThreads, smem_bytes, s>>>(p, tab);
  else if (diag_iters(K, C) <= 32) layup_disagreement_kernel<32><<<grid, kDiagThreads, smem_bytes, s>>>(p, tab);
  else return cudaErrorInvalidValue;
  return cudaGetLastError();
}

}  // namespace layup
