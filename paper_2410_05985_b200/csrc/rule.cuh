// The per-element arithmetic of the rule, shared by the two update kernels of the library
// (update_tma.cu, update.cu).  Every operation is spelled with a rounding-mode intrinsic so the
// compiler can neither contract nor reorder it: the results are bit-reproducible (DESIGN.md
// "Normative arithmetic").
//
//   OPT_SGD        y = x - eta*(g + wd*x)                         PAPER.md:78,101 "Local Update"
//   OPT_SGD_MOM    m <- mu*m + (g + wd*x);  y = x - eta*m         DESIGN.md R8, R21
//   OPT_ADAMW      x <- x(1 - eta*wd); m <- b1 m + (1-b1) g; v <- b2 v + (1-b2) g^2
//                  y = x - c1 * m / (sqrt(v)*c2 + eps)            PAPER.md:130, 469-491; R21
//                  c1 = eta/(1-b1^t), c2 = 1/sqrt(1-b2^t) come from the schedule kernel (fp64)
//   peer update    acc <- acc + alpha*(y_i - acc)                 PAPER.md:101 "Peer Update"
//   symmetric      x_i, x_j <- (x_i + x_j)/2                      PAPER.md:54 (AD-PSGD), R23
#pragma once
#include "layup_internal.cuh"

namespace layup {

constexpr int OPT_SGD = 0, OPT_SGD_MOM = 1, OPT_ADAMW = 2;

template <int OPT>
struct OptTraits {
  static constexpr int kArrays = OPT == OPT_ADAMW ? 4 : OPT == OPT_SGD_MOM ? 3 : 2;   // x, g (, m (, v))
};

template <int OPT>
__device__ __forceinline__ float local_step(float x, float g, float &m, float &v, const StepScalars &s,
                                            float c1, float c2) {
  if (OPT == OPT_ADAMW) {
    const float xd = __fmul_rn(x, s.decay);
    m = __fmaf_rn(s.b1, m, __fmul_rn(s.omb1, g));
    v = __fmaf_rn(s.b2, v, __fmul_rn(s.omb2, __fmul_rn(g, g)));
    const float den = __fmaf_rn(__fsqrt_rn(v), c2, s.eps);
    return __fmaf_rn(-c1, __fdiv_rn(m, den), xd);
  }
  float d = g;
  if (s.wd != 0.f) d = __fmaf_rn(s.wd, x, d);
  if (OPT == OPT_SGD_MOM) {
    d = __fmaf_rn(s.mu, m, d);
    m = d;
  }
  return __fmaf_rn(s.neg_lr, d, x);
}

template <int OPT>
__device__ __forceinline__ float4 local_step4(float4 x, const float4 &g, float4 &m, float4 &v, const StepScalars &s,
                                              float c1, float c2) {
  x.x = local_step<OPT>(x.x, g.x, m.x, v.x, s, c1, c2);
  x.y = local_step<OPT>(x.y, g.y, m.y, v.y, s, c1, c2);
  x.z = local_step<OPT>(x.z, g.z, m.z, v.z, s, c1, c2);
  x.w = local_step<OPT>(x.w, g.w, m.w, v.w, s, c1, c2);
  return x;
}

__device__ __forceinline__ void peer_update4(float4 &acc, const float4 &ys, float a) {
  acc.x = __fmaf_rn(a, __fsub_rn(ys.x, acc.x), acc.x);
  acc.y = __fmaf_rn(a, __fsub_rn(ys.y, acc.y), acc.y);
  acc.z = __fmaf_rn(a, __fsub_rn(ys.z, acc.z), acc.z);
  acc.w = __fmaf_rn(a, __fsub_rn(ys.w, acc.w), acc.w);
}

// Symmetric pairwise averaging of one scalar column held in shared memory for all K replicas:
// exchanges in ascending worker index, each seeing what the earlier ones left.  ys is the
// [K][stride] fp32 view of the y-tile; peer[i] < 0 means worker i does not exchange.
__device__ __forceinline__ void symmetric_column(float *ys, int stride, int e, int K, const int *peer) {
  for (int i = 0; i < K; ++i) {
    const int j = peer[i];
    if (j < 0) continue;
    const float avg = __fmul_rn(0.5f, __fadd_rn(ys[i * stride + e], ys[j * stride + e]));
    ys[i * stride + e] = avg;
    ys[j * stride + e] = avg;
  }
}

}  // namespace layup
