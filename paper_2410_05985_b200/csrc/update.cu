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
//   persistent: a fixed grid of resident CTAs walks the list with a static stride.  This LDG
//              engine takes it only when asked for (layup_tuning.engine = 2 with launch_shape = 2)
//              or when a launch has more than 2^31 work items; the TMA engine's persistent form
//              is the ring kernel of update_persist.cu, which draws tiles from a ticket instead.
#include "layup_internal.cuh"
#include "rule.cuh"

namespace layup {

namespace {

__device__ __forceinline__ float4 ld4(const float *p) { return *reinterpret_cast<const float4 *>(p); }
__device__ __forceinline__ void st4(float *p, const float4 &v) { *reinterpret_cast<float4 *>(p) = v; }

struct TileSmem {
  float4 *ysm;
  int *recv_off;
  int *senders;          // SYM: the peer table
  float *alpha;
  float *c1, *c2;        // AdamW only
  unsigned char *flags;
};

template <int OPT, bool SYM, int THREADS>
__device__ __forceinline__ void load_schedule(const UpdateParams &p, const TileSmem &s, int layer) {
  const int K = p.K, tid = threadIdx.x;
  const size_t row = (size_t)layer * K;
  for (int k = tid; k < K; k += THREADS) {
    s.senders[k] = SYM ? p.t.peer[row + k] : p.t.senders[row + k];
    s.alpha[k] = p.t.alpha[row + k];
    s.flags[k] = p.t.flags[row + k];
    if (OPT == OPT_ADAMW) {
      s.c1[k] = p.t.c1[row + k];
      s.c2[k] = p.t.c2[row + k];
    }
  }
  for (int k = tid; k <= K; k += THREADS) s.recv_off[k] = p.t.recv_off[(size_t)layer * (K + 1) + k];
}

// One tile: phase 1 (local steps, y -> smem), barrier, phase 2 (fold, x written once).
// The schedule of `layer` must already be in shared memory and visible.
template <int OPT, bool SYM, int THREADS, int U>
__device__ __forceinline__ void process_tile(const UpdateParams &p, const TileSmem &s, const LayerDesc &lay,
                                             long long tile_in_layer) {
  constexpr bool HAS_M = OptTraits<OPT>::kArrays >= 3, HAS_V = OptTraits<OPT>::kArrays >= 4;
  const int K = p.K, C = p.C, log2C = p.log2C, tid = threadIdx.x;
  const int n_items = K << log2C;
  const long long col0 = tile_in_layer << log2C;                            // first float4 column
  const long long cols_left = (lay.pad >> 2) - col0;
  const int ncols = cols_left < C ? (int)cols_left : C;
  float *const xb = p.x + lay.base + (col0 << 2);
  const float *const gb = p.g + lay.base + (col0 << 2);
  float *const mb = HAS_M ? p.m + lay.base + (col0 << 2) : nullptr;
  float *const vb = HAS_V ? p.v + lay.base + (col0 << 2) : nullptr;

  for (int base = 0; base < n_items; base += THREADS * U) {
    float4 xv[U], gv[U], mv[U], vv[U];
    int fl[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int idx = base + u * THREADS + tid;
      const int i = idx >> log2C, c = idx & (C - 1);
      fl[u] = 0;
      mv[u] = vv[u] = float4{0.f, 0.f, 0.f, 0.f};
      if (idx < n_items && c < ncols) {
        fl[u] = s.flags[i];
        const long long off = (long long)i * lay.pad + (c << 2);
        if (fl[u]) xv[u] = ld4(xb + off);
        if (fl[u] & kFlagActive) {
          gv[u] = ld4(gb + off);
          if (HAS_M) mv[u] = ld4(mb + off);
          if (HAS_V) vv[u] = ld4(vb + off);
        }
      }
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      if (!fl[u]) continue;
      const int idx = base + u * THREADS + tid;
      float4 y = xv[u];
      if (fl[u] & kFlagActive) {
        const int i = idx >> log2C;
        y = local_step4<OPT>(xv[u], gv[u], mv[u], vv[u], p.s, HAS_V ? s.c1[i] : 0.f, HAS_V ? s.c2[i] : 0.f);
        const long long off = (long long)i * lay.pad + ((idx & (C - 1)) << 2);
        if (HAS_M) st4(mb + off, mv[u]);
        if (HAS_V) st4(vb + off, vv[u]);
      }
      s.ysm[idx] = y;
    }
  }
  __syncthreads();

  if (SYM) {
    float *ysf = reinterpret_cast<float *>(s.ysm);
    for (int e = tid; e < (ncols << 2); e += THREADS) symmetric_column(ysf, C << 2, e, K, s.senders);
    __syncthreads();
  }
  for (int idx = tid; idx < n_items; idx += THREADS) {
    const int i = idx >> log2C, c = idx & (C - 1);
    if (c >= ncols) continue;
    if (!s.flags[i]) continue;                                              // idle, no push received: 0 bytes
    float4 acc = s.ysm[idx];
    if (!SYM) {
      const int k_end = s.recv_off[i + 1];
      for (int k = s.recv_off[i]; k < k_end; ++k) peer_update4(acc, s.ysm[(s.senders[k] << log2C) + c], s.alpha[k]);
    }
    st4(xb + (long long)i * lay.pad + (c << 2), acc);
  }
}

template <int OPT>
__device__ __forceinline__ TileSmem carve(unsigned char *raw, int K, int n_items) {
  TileSmem s;
  s.ysm = reinterpret_cast<float4 *>(raw);
  s.recv_off = reinterpret_cast<int *>(s.ysm + n_items);
  s.senders = s.recv_off + (K + 1);
  s.alpha = reinterpret_cast<float *>(s.senders + K);
  s.c1 = s.alpha + K;
  s.c2 = s.c1 + (OPT == OPT_ADAMW ? K : 0);
  s.flags = reinterpret_cast<unsigned char *>(s.c2 + (OPT == OPT_ADAMW ? K : 0));
  return s;
}

// grouped launch: blockIdx.x = work item
template <int OPT, bool SYM, int THREADS, int U, int MINB>
__global__ void __launch_bounds__(THREADS, MINB) layup_update_grouped(const UpdateParams p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const TileSmem s = carve<OPT>(smem_raw, p.K, p.K << p.log2C);
  const long long tile = p.tile_begin + blockIdx.x;
  // position of this tile in the reverse-layer list: binary search of the prefix table
  int lo = p.pos_begin, hi = p.pos_end;                                     // tile in [prefix[lo], prefix[hi])
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (tile >= p.tile_prefix[mid]) lo = mid; else hi = mid;
  }
  const int layer = p.L - 1 - lo;
  trace_start(p.trace, layer);
  load_schedule<OPT, SYM, THREADS>(p, s, layer);
  const LayerDesc lay = p.layers[layer];
  const long long t_in = tile - p.tile_prefix[lo];
  __syncthreads();
  process_tile<OPT, SYM, THREADS, U>(p, s, lay, t_in);
}

// persistent launch: resident CTAs stride over the list
template <int OPT, bool SYM, int THREADS, int U, int MINB>
__global__ void __launch_bounds__(THREADS, MINB) layup_update_persistent(const UpdateParams p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const TileSmem s = carve<OPT>(smem_raw, p.K, p.K << p.log2C);
  int pos = p.pos_begin, loaded_pos = -1;
  long long pos_end_tile = p.tile_prefix[pos + 1];
  for (long long tile = p.tile_begin + blockIdx.x; tile < p.tile_end; tile += gridDim.x) {
    while (tile >= pos_end_tile) { ++pos; pos_end_tile = p.tile_prefix[pos + 1]; }
    const int layer = p.L - 1 - pos;
    if (pos != loaded_pos) {
      trace_start(p.trace, layer);
      load_schedule<OPT, SYM, THREADS>(p, s, layer);
      loaded_pos = pos;
      __syncthreads();
    }
    const LayerDesc lay = p.layers[layer];
    process_tile<OPT, SYM, THREADS, U>(p, s, lay, tile - p.tile_prefix[pos]);
    __syncthreads();   // ysm and the schedule tables are reused by the next tile
  }
}

using KernelFn = void (*)(const UpdateParams);

struct Variant {
  int threads, u, minb;
  KernelFn grouped[3][2], persistent[3][2];   // [OPT][SYM]
};

#define LAYUP_KROW(KERN, O, T, UU, MB) {KERN<O, false, T, UU, MB>, KERN<O, true, T, UU, MB>}
#define LAYUP_VARIANT(T, UU, MB)                                                                              \
  Variant {                                                                                                   \
    T, UU, MB,                                                                                                \
        {LAYUP_KROW(layup_update_grouped, OPT_SGD, T, UU, MB), LAYUP_KROW(layup_update_grouped, OPT_SGD_MOM, T, UU, MB), \
         LAYUP_KROW(layup_update_grouped, OPT_ADAMW, T, UU, MB)},                                             \
        {LAYUP_KROW(layup_update_persistent, OPT_SGD, T, UU, MB),                                             \
         LAYUP_KROW(layup_update_persistent, OPT_SGD_MOM, T, UU, MB),                                         \
         LAYUP_KROW(layup_update_persistent, OPT_ADAMW, T, UU, MB)}                                           \
  }

const Variant kVariants[] = {
    LAYUP_VARIANT(256, 2, 4),   // default
    LAYUP_VARIANT(256, 1, 8),   // the best LDG shape measured on B200
    LAYUP_VARIANT(512, 2, 2),
};
constexpr int kNumVariants = sizeof(kVariants) / sizeof(kVariants[0]);

}  // namespace

size_t update_smem_bytes(int K, int C) {
  return (size_t)K * C * sizeof(float4) + sizeof(int) * (2 * (size_t)K + 1) + sizeof(float) * 3 * K + (size_t)K;
}

int update_num_variants() { return kNumVariants; }

cudaError_t update_kernel_setup(int variant, int opt, bool symmetric, int smem_bytes, int *threads, int *ctas_per_sm) {
  if (variant < 0 || variant >= kNumVariants || opt < 0 || opt > 2) return cudaErrorInvalidValue;
  const Variant &v = kVariants[variant];
  cudaError_t e;
  const int sym = symmetric ? 1 : 0;
  for (KernelFn f : {v.grouped[opt][sym], v.persistent[opt][sym]}) {
    if ((e = allow_max_dynamic_smem((const void *)f, smem_bytes)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(f, cudaFuncAttributePreferredSharedMemoryCarveout, 100)) != cudaSuccess) return e;
  }
  int a = 0;
  if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&a, v.persistent[opt][sym], v.threads, smem_bytes)) != cudaSuccess) return e;
  *threads = v.threads;
  *ctas_per_sm = a;
  return cudaSuccess;
}

cudaError_t launch_update(const UpdateParams &p, int variant, bool persistent, int grid, int smem_bytes, cudaStream_t s) {
  const Variant &v = kVariants[variant];
  const int sym = p.symmetric ? 1 : 0;
  if (persistent)
    v.persistent[p.opt][sym]<<<grid, v.threads, smem_bytes, s>>>(p);
  else
    v.grouped[p.opt][sym]<<<grid, v.threads, smem_bytes, s>>>(p);
  return cudaGetLastError();
}

}  // namespace layup
