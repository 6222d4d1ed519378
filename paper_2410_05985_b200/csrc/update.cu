// Fused local-step + gossip-mix kernel, sm_100a.
//
// One work item = (layer, tile of C float4 columns) for ALL K replicas.  A CTA that
// owns the tile for all K replicas reads every x, g, m once, takes the K local steps
//     m <- mu*m + g ; y = x - eta*m        ("Local Update", DESIGN R8)
// parks the post-step values y in shared memory (the "send", PAPER.md:101 -- an on-chip
// read here), folds each receiver's senders in ascending order
//     acc <- acc + alpha*(y_i - acc)       ("Peer Update")
// and writes every x, m once: 12 B (no momentum) / 20 B (momentum) of HBM traffic per
// parameter update, no second buffer, no inter-CTA hazard.
//
// The kernel is persistent: CTAs walk a reverse-layer-ordered work list (layer L-1
// first) with a static stride, so one launch serves a whole round
// (layup_round) or a single layer (layup_layer_update).
#include "layup_internal.cuh"

namespace layup {

namespace {

constexpr int U = 4;   // float4 items in flight per thread per batch

__device__ __forceinline__ float4 ld4(const float *p) { return *reinterpret_cast<const float4 *>(p); }
__device__ __forceinline__ void st4(float *p, const float4 &v) { *reinterpret_cast<float4 *>(p) = v; }

template <bool MOM>
__global__ void __launch_bounds__(kThreads) layup_update_kernel(const UpdateParams p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int K = p.K, C = p.C, log2C = p.log2C;
  const int n_items = K << log2C;
  float4 *ysm = reinterpret_cast<float4 *>(smem_raw);                       // [K*C]
  int *s_recv_off = reinterpret_cast<int *>(ysm + n_items);                 // [K+1]
  int *s_senders = s_recv_off + (K + 1);                                    // [K]
  float *s_alpha = reinterpret_cast<float *>(s_senders + K);                // [K]
  unsigned char *s_flags = reinterpret_cast<unsigned char *>(s_alpha + K);  // [K]

  const int tid = threadIdx.x;
  int pos = p.pos_begin;
  int loaded_pos = -1;
  long long pos_end_tile = p.tile_prefix[pos + 1];

  for (long long tile = p.tile_begin + blockIdx.x; tile < p.tile_end; tile += gridDim.x) {
    while (tile >= pos_end_tile) { ++pos; pos_end_tile = p.tile_prefix[pos + 1]; }
    const int layer = p.L - 1 - pos;
    if (pos != loaded_pos) {
      // new layer: bring its schedule (<= ~13 B per replica) into shared memory
      const size_t row = (size_t)layer * K;
      for (int k = tid; k < K; k += kThreads) {
        s_senders[k] = p.t.senders[row + k];
        s_alpha[k] = p.t.alpha[row + k];
        s_flags[k] = p.t.flags[row + k];
      }
      for (int k = tid; k <= K; k += kThreads) s_recv_off[k] = p.t.recv_off[(size_t)layer * (K + 1) + k];
      loaded_pos = pos;
      __syncthreads();
    }
    const LayerDesc lay = p.layers[layer];
    const long long col0 = (tile - p.tile_prefix[pos]) << log2C;            // first float4 column
    const long long cols_left = (lay.pad >> 2) - col0;
    const int ncols = cols_left < C ? (int)cols_left : C;

    // ---- phase 1: local step of every replica, y -> shared memory -----------------
    for (int base = 0; base < n_items; base += kThreads * U) {
      float4 xv[U], gv[U], mv[U];
      int fl[U];
      long long off[U];
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const int idx = base + u * kThreads + tid;
        const int i = idx >> log2C, c = idx & (C - 1);
        fl[u] = 0;
        if (idx < n_items && c < ncols) {
          fl[u] = s_flags[i] | 4;                                           // bit 2: item exists
          off[u] = lay.base + (long long)i * lay.pad + ((col0 + c) << 2);
          if (fl[u] & (kFlagActive | kFlagRecv)) xv[u] = ld4(p.x + off[u]);
          if (fl[u] & kFlagActive) {
            gv[u] = ld4(p.g + off[u]);
            if (MOM) mv[u] = ld4(p.m + off[u]);
          }
        }
      }
#pragma unroll
      for (int u = 0; u < U; ++u) {
        if (!(fl[u] & (kFlagActive | kFlagRecv))) continue;
        float4 y = xv[u];
        if (fl[u] & kFlagActive) {
          float4 d = gv[u];
          if (MOM) {
            d.x = __fmaf_rn(p.mu, mv[u].x, gv[u].x);
            d.y = __fmaf_rn(p.mu, mv[u].y, gv[u].y);
            d.z = __fmaf_rn(p.mu, mv[u].z, gv[u].z);
            d.w = __fmaf_rn(p.mu, mv[u].w, gv[u].w);
            st4(p.m + off[u], d);
          }
          y.x = __fmaf_rn(p.neg_lr, d.x, y.x);
          y.y = __fmaf_rn(p.neg_lr, d.y, y.y);
          y.z = __fmaf_rn(p.neg_lr, d.z, y.z);
          y.w = __fmaf_rn(p.neg_lr, d.w, y.w);
        }
        ysm[base + u * kThreads + tid] = y;
      }
    }
    __syncthreads();

    // ---- phase 2: each receiver folds its senders, x written once -----------------
    for (int idx = tid; idx < n_items; idx += kThreads) {
      const int i = idx >> log2C, c = idx & (C - 1);
      if (c >= ncols) continue;
      const int f = s_flags[i];
      if (!(f & (kFlagActive | kFlagRecv))) continue;                       // untouched: 0 bytes
      float4 acc = ysm[idx];
      const int k_end = s_recv_off[i + 1];
      for (int k = s_recv_off[i]; k < k_end; ++k) {
        const float a = s_alpha[k];
        const float4 ys = ysm[(s_senders[k] << log2C) + c];
        acc.x = __fmaf_rn(a, __fsub_rn(ys.x, acc.x), acc.x);
        acc.y = __fmaf_rn(a, __fsub_rn(ys.y, acc.y), acc.y);
        acc.z = __fmaf_rn(a, __fsub_rn(ys.z, acc.z), acc.z);
        acc.w = __fmaf_rn(a, __fsub_rn(ys.w, acc.w), acc.w);
      }
      st4(p.x + lay.base + (long long)i * lay.pad + ((col0 + c) << 2), acc);
    }
    __syncthreads();   // ysm and the schedule tables are reused by the next tile
  }
}

}  // namespace

size_t update_smem_bytes(int K, int C) {
  return (size_t)K * C * sizeof(float4) + sizeof(int) * (2 * (size_t)K + 1) + sizeof(float) * K + (size_t)K;
}

cudaError_t update_kernel_setup(int smem_bytes, int *ctas_per_sm) {
  cudaError_t e;
  if ((e = cudaFuncSetAttribute(layup_update_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                smem_bytes)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(layup_update_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                smem_bytes)) != cudaSuccess) return e;
  int a = 0, b = 0;
  if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&a, layup_update_kernel<true>, kThreads,
                                                         smem_bytes)) != cudaSuccess) return e;
  if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, layup_update_kernel<false>, kThreads,
                                                         smem_bytes)) != cudaSuccess) return e;
  *ctas_per_sm = a < b ? a : b;
  return cudaSuccess;
}

cudaError_t launch_update(const UpdateParams &p, int grid, int smem_bytes, cudaStream_t s) {
  if (p.m != nullptr)
    layup_update_kernel<true><<<grid, kThreads, smem_bytes, s>>>(p);
  else
    layup_update_kernel<false><<<grid, kThreads, smem_bytes, s>>>(p);
  return cudaGetLastError();
}

}  // namespace layup
