// Model-disagreement diagnostic: per (layer, replica) the squared distance
// to the consensus,  dist[l][i] = sum_e (x_i[e] - xbar[e])^2,  xbar = sum_i c_i x_i  with c_i = 1/K
// (the paper's plain average) or c_i = w_i (push-sum weighted consensus).
// PAPER.md:389-395 (Fig. A1 "model disagreement between workers"), eq. (9) PAPER.md:551.
//
// The only place on the path that needs norms, hence the only warp-level reductions.  Same tiling
// as the update kernel -- a CTA owns a tile of C float4 columns for ALL K replicas, staged by TMA
// bulk copies -- but read-only: 4 B of HBM traffic per parameter.  A persistent grid walks the
// work list with a static stride and keeps per-replica partial sums in shared memory while it
// stays inside a layer; everything is accumulated in fp64 (sums are order-dependent in the last
// bits: shared/global atomics).
#include "layup_internal.cuh"

namespace layup {

namespace {

constexpr int kDiagThreads = 256;

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
__device__ __forceinline__ void bulk_g2s(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst_smem)),
               "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

struct DiagParams {
  const float *x;          // X section base
  const double *w;         // [L*K] push-sum weights, or nullptr for the plain mean
  double *dist;            // [L*K] output, zeroed before the launch
  int32_t K, C, log2C;
};

__global__ void __launch_bounds__(kDiagThreads) layup_disagreement_kernel(const __grid_constant__ DiagParams p,
                                                                          const __grid_constant__ PosTable tab) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int K = p.K, C = p.C, log2C = p.log2C, tid = threadIdx.x;
  const int n_items = K << log2C;
  float4 *xs = reinterpret_cast<float4 *>(smem_raw);                              // [K*C]
  double *mean = reinterpret_cast<double *>(xs + n_items);                        // [C*4]
  double *coef = mean + 4 * C;                                                    // [K]
  double *acc = coef + K;                                                         // [K]
  uint64_t *bar = reinterpret_cast<uint64_t *>(acc + K);

  if (tid == 0) mbar_init(bar, 1);
  for (int k = tid; k < K; k += kDiagThreads) acc[k] = 0.0;
  __syncthreads();

  const long long n_tiles = tab.prefix[tab.n];
  int pos = 0, cur = -1;
  uint32_t parity = 0;
  for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    while (tile >= tab.prefix[pos + 1]) ++pos;
    if (pos != cur) {
      // leaving a layer: flush this CTA's partial sums, load the next layer's coefficients
      if (cur >= 0)
        for (int k = tid; k < K; k += kDiagThreads) {
          atomicAdd(p.dist + (size_t)tab.layer[cur] * K + k, acc[k]);
          acc[k] = 0.0;
        }
      for (int k = tid; k < K; k += kDiagThreads)
        coef[k] = p.w ? p.w[(size_t)tab.layer[pos] * K + k] : 1.0 / (double)K;
      cur = pos;
      __syncthreads();
    }
    const long long pad = tab.lay[pos].pad;
    const long long col0 = (tile - tab.prefix[pos]) << log2C;
    const long long cols_left = (pad >> 2) - col0;
    const int ncols = cols_left < C ? (int)cols_left : C;
    const float *xb = p.x + tab.lay[pos].base + (col0 << 2);
    const uint32_t chunk = (uint32_t)ncols * 16u;

    if (tid < 32) {
      if (tid == 0) mbar_expect_tx(bar, (uint32_t)K * chunk);
      __syncwarp();
      for (int i = tid; i < K; i += 32) bulk_g2s(xs + (i << log2C), xb + (long long)i * pad, chunk, bar);
    }
    mbar_wait(bar, parity);
    parity ^= 1u;

    // consensus of every column (pads are zero in every replica and contribute 0)
    for (int c = tid; c < ncols; c += kDiagThreads) {
      double m0 = 0.0, m1 = 0.0, m2 = 0.0, m3 = 0.0;
      for (int i = 0; i < K; ++i) {
        const float4 v = xs[(i << log2C) + c];
        const double ci = coef[i];
        m0 += ci * (double)v.x; m1 += ci * (double)v.y; m2 += ci * (double)v.z; m3 += ci * (double)v.w;
      }
      mean[4 * c + 0] = m0; mean[4 * c + 1] = m1; mean[4 * c + 2] = m2; mean[4 * c + 3] = m3;
    }
    __syncthreads();

    // squared distances; lanes that share a replica are reduced with shuffles before one shared atomic
    const int seg = C < 32 ? C : 32;                                              // lanes per replica in a warp
    for (int base = 0; base < n_items; base += kDiagThreads) {
      const int idx = base + tid;
      const int i = idx >> log2C, c = idx & (C - 1);
      double s = 0.0;
      if (idx < n_items && c < ncols) {
        const float4 v = xs[idx];
        const double d0 = (double)v.x - mean[4 * c + 0], d1 = (double)v.y - mean[4 * c + 1];
        const double d2 = (double)v.z - mean[4 * c + 2], d3 = (double)v.w - mean[4 * c + 3];
        s = d0 * d0 + d1 * d1 + d2 * d2 + d3 * d3;
      }
      for (int o = seg >> 1; o > 0; o >>= 1) s += __shfl_xor_sync(0xFFFFFFFFu, s, o);
      if ((tid & (seg - 1)) == 0 && idx < n_items) atomicAdd(acc + i, s);
    }
    __syncthreads();   // xs, mean are reused by the next tile
  }
  if (cur >= 0)
    for (int k = tid; k < K; k += kDiagThreads) atomicAdd(p.dist + (size_t)tab.layer[cur] * K + k, acc[k]);
}

}  // namespace

size_t diag_smem_bytes(int K, int C) {
  return (size_t)K * C * sizeof(float4) + sizeof(double) * (4 * (size_t)C + 2 * (size_t)K) + 8;
}

cudaError_t diag_setup(int smem_bytes, int *ctas_per_sm) {
  cudaError_t e;
  if ((e = cudaFuncSetAttribute(layup_disagreement_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                smem_bytes)) != cudaSuccess) return e;
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas_per_sm, layup_disagreement_kernel, kDiagThreads,
                                                       smem_bytes);
}

cudaError_t launch_disagreement(const float *x, const double *w, double *dist, int K, int C, int log2C,
                                const PosTable &tab, int grid, int smem_bytes, cudaStream_t s) {
  DiagParams p{x, w, dist, K, C, log2C};
  layup_disagreement_kernel<<<grid, kDiagThreads, smem_bytes, s>>>(p, tab);
  return cudaGetLastError();
}

}  // namespace layup
