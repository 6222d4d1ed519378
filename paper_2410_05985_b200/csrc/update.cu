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
// The work list is ordered by reverse layer (layer L-1 first).  Two
// launch shapes over the same list:
//   grouped  : one CTA per work item; the hardware CTA scheduler drains the list in
//              order (measured fastest on B200 for HBM-sized layers);
//   persistent: a fixed grid of resident CTAs walks the list with a static stride
//              (many small layers, L2-resident rounds).
#include "layup_internal.cuh"

namespace layup {

namespace {

__device__ __forceinline__ float4 ld4(const float *p) { return *reinterpret_cast<const float4 *>(p); }
__device__ __forceinline__ void st4(float *p, const float4 &v) { *reinterpret_cast<float4 *>(p) = v; }

struct TileSmem {
  float4 *ysm;
  int *recv_off;
  int *senders;
  float *alpha;
  unsigned char *flags;
};

template <int THREADS>
__device__ __forceinline__ void load_schedule(const UpdateParams &p, const TileSmem &s, int layer) {
  const int K = p.K, tid = threadIdx.x;
  const size_t row = (size_t)layer * K;
  for (int k = tid; k < K; k += THREADS) {
    s.senders[k] = p.t.senders[row + k];
    s.alpha[k] = p.t.alpha[row + k];
    s.flags[k] = p.t.flags[row + k];
  }
  for (int k = tid; k <= K; k += THREADS) s.recv_off[k] = p.t.recv_off[(size_t)layer * (K + 1) + k];
}

// One tile: phase 1 (local steps, y -> smem), barrier, phase 2 (fold, x written once).
// The schedule of `layer` must already be in shared memory and visible.
template <bool MOM, int THREADS, int U>
__device__ __forceinline__ void process_tile(const UpdateParams &p, const TileSmem &s, const LayerDesc &lay,
                                             long long tile_in_layer) {
  const int K = p.K, C = p.C, log2C = p.log2C, tid = threadIdx.x;
  const int n_items = K << log2C;
  const long long col0 = tile_in_layer << log2C;                            // first float4 column
  const long long cols_left = (lay.pad >> 2) - col0;
  const int ncols = cols_left < C ? (int)cols_left : C;
  float *const xb = p.x + lay.base + (col0 << 2);
  const float *const gb = p.g + lay.base + (col0 << 2);
  float *const mb = MOM ? p.m + lay.base + (col0 << 2) : nullptr;

  for (int base = 0; base < n_items; base += THREADS * U) {
    float4 xv[U], gv[U], mv[U];
    int fl[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int idx = base + u * THREADS + tid;
      const int i = idx >> log2C, c = idx & (C - 1);
      fl[u] = 0;
      if (idx < n_items && c < ncols) {
        fl[u] = s.flags[i];
        const long long off = (long long)i * lay.pad + (c << 2);
        if (fl[u]) xv[u] = ld4(xb + off);
        if (fl[u] & kFlagActive) {
          gv[u] = ld4(gb + off);
          if (MOM) mv[u] = ld4(mb + off);
        }
      }
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      if (!fl[u]) continue;
      const int idx = base + u * THREADS + tid;
      float4 y = xv[u];
      if (fl[u] & kFlagActive) {
        float4 d = gv[u];
        if (MOM) {
          d.x = __fmaf_rn(p.mu, mv[u].x, gv[u].x);
          d.y = __fmaf_rn(p.mu, mv[u].y, gv[u].y);
          d.z = __fmaf_rn(p.mu, mv[u].z, gv[u].z);
          d.w = __fmaf_rn(p.mu, mv[u].w, gv[u].w);
          st4(mb + (long long)(idx >> log2C) * lay.pad + ((idx & (C - 1)) << 2), d);
        }
        y.x = __fmaf_rn(p.neg_lr, d.x, y.x);
        y.y = __fmaf_rn(p.neg_lr, d.y, y.y);
        y.z = __fmaf_rn(p.neg_lr, d.z, y.z);
        y.w = __fmaf_rn(p.neg_lr, d.w, y.w);
      }
      s.ysm[idx] = y;
    }
  }
  __syncthreads();

  for (int idx = tid; idx < n_items; idx += THREADS) {
    const int i = idx >> log2C, c = idx & (C - 1);
    if (c >= ncols) continue;
    if (!s.flags[i]) continue;                                              // idle, no push received: 0 bytes
    float4 acc = s.ysm[idx];
    const int k_end = s.recv_off[i + 1];
    for (int k = s.recv_off[i]; k < k_end; ++k) {
      const float a = s.alpha[k];
      const float4 ys = s.ysm[(s.senders[k] << log2C) + c];
      acc.x = __fmaf_rn(a, __fsub_rn(ys.x, acc.x), acc.x);
      acc.y = __fmaf_rn(a, __fsub_rn(ys.y, acc.y), acc.y);
      acc.z = __fmaf_rn(a, __fsub_rn(ys.z, acc.z), acc.z);
      acc.w = __fmaf_rn(a, __fsub_rn(ys.w, acc.w), acc.w);
    }
    st4(xb + (long long)i * lay.pad + (c << 2), acc);
  }
}

template <int THREADS>
__device__ __forceinline__ TileSmem carve(unsigned char *raw, int K, int n_items) {
  TileSmem s;
  s.ysm = reinterpret_cast<float4 *>(raw);
  s.recv_off = reinterpret_cast<int *>(s.ysm + n_items);
  s.senders = s.recv_off + (K + 1);
  s.alpha = reinterpret_cast<float *>(s.senders + K);
  s.flags = reinterpret_cast<unsigned char *>(s.alpha + K);
  return s;
}

// grouped launch: blockIdx.x = work item
template <bool MOM, int THREADS, int U, int MINB>
__global__ void __launch_bounds__(THREADS, MINB) layup_update_grouped(const UpdateParams p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const TileSmem s = carve<THREADS>(smem_raw, p.K, p.K << p.log2C);
  const long long tile = p.tile_begin + blockIdx.x;
  // position of this tile in the reverse-layer list: binary search of the prefix table
  int lo = p.pos_begin, hi = p.pos_end;                                     // tile in [prefix[lo], prefix[hi])
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (tile >= p.tile_prefix[mid]) lo = mid; else hi = mid;
  }
  const int layer = p.L - 1 - lo;
  load_schedule<THREADS>(p, s, layer);
  const LayerDesc lay = p.layers[layer];
  const long long t_in = tile - p.tile_prefix[lo];
  __syncthreads();
  process_tile<MOM, THREADS, U>(p, s, lay, t_in);
}

// persistent launch: resident CTAs stride over the list
template <bool MOM, int THREADS, int U, int MINB>
__global__ void __launch_bounds__(THREADS, MINB) layup_update_persistent(const UpdateParams p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const TileSmem s = carve<THREADS>(smem_raw, p.K, p.K << p.log2C);
  int pos = p.pos_begin, loaded_pos = -1;
  long long pos_end_tile = p.tile_prefix[pos + 1];
  for (long long tile = p.tile_begin + blockIdx.x; tile < p.tile_end; tile += gridDim.x) {
    while (tile >= pos_end_tile) { ++pos; pos_end_tile = p.tile_prefix[pos + 1]; }
    const int layer = p.L - 1 - pos;
    if (pos != loaded_pos) {
      load_schedule<THREADS>(p, s, layer);
      loaded_pos = pos;
      __syncthreads();
    }
    const LayerDesc lay = p.layers[layer];
    process_tile<MOM, THREADS, U>(p, s, lay, tile - p.tile_prefix[pos]);
    __syncthreads();   // ysm and the schedule tables are reused by the next tile
  }
}

using KernelFn = void (*)(const UpdateParams);

struct Variant {
  int threads, u, minb;
  KernelFn grouped[2], persistent[2];   // [MOM]
};

#define LAYUP_VARIANT(T, UU, MB)                                                                   \
  Variant {                                                                                        \
    T, UU, MB, {layup_update_grouped<false, T, UU, MB>, layup_update_grouped<true, T, UU, MB>},    \
        {layup_update_persistent<false, T, UU, MB>, layup_update_persistent<true, T, UU, MB>}      \
  }

const Variant kVariants[] = {
    LAYUP_VARIANT(256, 2, 4),   // default
    LAYUP_VARIANT(256, 4, 2), LAYUP_VARIANT(256, 4, 3), LAYUP_VARIANT(256, 2, 6), LAYUP_VARIANT(256, 1, 8),
    LAYUP_VARIANT(512, 2, 2),   LAYUP_VARIANT(512, 1, 4), LAYUP_VARIANT(128, 4, 8), LAYUP_VARIANT(128, 2, 12),
    LAYUP_VARIANT(1024, 1, 2),  LAYUP_VARIANT(128, 8, 4),
};
constexpr int kNumVariants = sizeof(kVariants) / sizeof(kVariants[0]);

}  // namespace

size_t update_smem_bytes(int K, int C) {
  return (size_t)K * C * sizeof(float4) + sizeof(int) * (2 * (size_t)K + 1) + sizeof(float) * K + (size_t)K;
}

int update_num_variants() { return kNumVariants; }

cudaError_t update_kernel_setup(int variant, int smem_bytes, int *threads, int *ctas_per_sm) {
  if (variant < 0 || variant >= kNumVariants) return cudaErrorInvalidValue;
  const Variant &v = kVariants[variant];
  cudaError_t e;
  int occ = 1 << 30;
  for (int mom = 0; mom < 2; ++mom) {
    for (KernelFn f : {v.grouped[mom], v.persistent[mom]}) {
      if ((e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes)) != cudaSuccess) return e;
      if ((e = cudaFuncSetAttribute(f, cudaFuncAttributePreferredSharedMemoryCarveout, 100)) != cudaSuccess) return e;
    }
    int a = 0;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&a, v.persistent[mom], v.threads, smem_bytes)) != cudaSuccess) return e;
    occ = a < occ ? a : occ;
  }
  *threads = v.threads;
  *ctas_per_sm = occ;
  return cudaSuccess;
}

cudaError_t launch_update(const UpdateParams &p, int variant, bool persistent, int grid, int smem_bytes, cudaStream_t s) {
  const Variant &v = kVariants[variant];
  const int mom = p.m != nullptr ? 1 : 0;
  if (persistent)
    v.persistent[mom]<<<grid, v.threads, smem_bytes, s>>>(p);
  else
    v.grouped[mom]<<<grid, v.threads, smem_bytes, s>>>(p);
  return cudaGetLastError();
}

}  // namespace layup
