/*
 * layup_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, single-threaded CPU statement of the LayUp updater step
 * (arXiv 2410.05985, Algorithm 1 "Updater
 * Thread i"; weights PAPER.md:106; layer-wise order PAPER.md:23,25,112) for K
 * workers held as K replicas of every layer.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may call it.  It shares no
 * code, header, table or constant generator with paper_2410_05985_b200/csrc/.
 *
 * The paper's system is racy by design (lock-free overwrites);
 * the deterministic reading implemented here is the lock-step round of
 * DESIGN.md "Readings" R1-R10:
 *
 *   for one (step t, layer l):
 *   1. active[i]  : straggler mask, one draw per (t, i)          [PAPER.md:220,229]
 *   2. peer[i]    : j ~ Random(M-1), never i                     [PAPER.md:101]
 *      wh[i]      : w_i <- w_i / 2 for a sender                  [PAPER.md:101,106]
 *   3. local step : x^{i,l} <- x~^{i,l} - eta * grad             [PAPER.md:78,101]
 *                   (optional heavy-ball momentum, local only; reading R8)
 *   4. peer update: x^{j,l} <- w_j/(w_i+w_j) x^{j,l} + w_i/(w_i+w_j) x^{i,l}
 *                   w_j <- w_j + w_i                             [PAPER.md:101]
 *      applied once per sender of j, ascending sender index, every sender's
 *      value being its post-local-step, pre-mix value (readings R3, R4).
 *
 * Pins (tests/test_oracle_*.py): Philox against cuRAND's library routine run on
 * the host; worked examples W1/W2 (tests/golden/); mass conservation, weighted-
 * mean conservation, K=2 exact averaging, convexity, consensus contraction,
 * brute force over every peer map and mask on tiny layers against a dense
 * row-stochastic matrix product, K=1 against torch.optim.SGD.
 * Parity unpinned: the paper's real racy system (no deterministic definition
 * exists; R3).
 *
 * Build: gcc -O2 -ffp-contract=off -shared -fPIC (oracle/__init__.py).  All fp32
 * multiply-adds that the rule fuses are written as explicit fmaf().
 * The default build is single-threaded.  The SAME source built with -fopenmp
 * (oracle.build_omp(), bench.py's all-cores baseline) runs the element loops marked
 * ORACLE_PAR on all host cores: elements are independent, the statements and their
 * order per element are unchanged, so the results are bit-identical (asserted by
 * tests/test_oracle_omp.py).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef _OPENMP
#define ORACLE_PAR _Pragma("omp parallel for schedule(static) if (n >= 32768)")
#else
#define ORACLE_PAR
#endif

#define TAG_PEER 0u
#define TAG_SKIP 1u
#define FIELD_NONE 0xFFFFFFFFu

/* ---- Philox4x32 with 10 rounds (Salmon, Moraes, Dror, Shaw, SC'11) ---------
 * One round: two 32x32->64 products of counter words 0 and 2 with the two
 * multipliers; new counter = (hi1^c1^k0, lo1, hi0^c3^k1, lo0); the key is
 * bumped by the two Weyl constants between rounds.                          */
static void philox_round(uint32_t c[4], const uint32_t k[2]) {
  const uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c[0];
  const uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c[2];
  const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
  const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
  const uint32_t n0 = hi1 ^ c[1] ^ k[0];
  const uint32_t n2 = hi0 ^ c[3] ^ k[1];
  c[0] = n0; c[1] = lo1; c[2] = n2; c[3] = lo0;
}

void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c[4] = {ctr[0], ctr[1], ctr[2], ctr[3]};
  uint32_t k[2] = {key[0], key[1]};
  for (int r = 0; r < 10; ++r) {
    if (r > 0) { k[0] += 0x9E3779B9u; k[1] += 0xBB67AE85u; }
    philox_round(c, k);
  }
  out[0] = c[0]; out[1] = c[1]; out[2] = c[2]; out[3] = c[3];
}

/* first output word for key = seed, counter = (c0,c1,c2,c3) */
static uint32_t draw(uint64_t seed, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3) {
  const uint32_t ctr[4] = {c0, c1, c2, c3};
  const uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32)};
  uint32_t out[4];
  oracle_philox4x32_10(ctr, key, out);
  return out[0];
}

/* Reading R10: one skip draw per (step, replica); the layer field is unused so a
 * straggler idles for the whole round.  Threshold computed in
 * double from the fp32 probability, clamped to 2^32-1.                        */
int32_t oracle_active(uint64_t seed, int64_t step, int32_t replica, float skip_prob) {
  if (!(skip_prob > 0.0f)) return 1;
  double th = (double)skip_prob * 4294967296.0;
  if (th > 4294967295.0) th = 4294967295.0;
  const uint32_t thr = (uint32_t)th;
  const uint32_t r = draw(seed, (uint32_t)step, FIELD_NONE, (uint32_t)replica, TAG_SKIP);
  return r < thr ? 0 : 1;
}

/* Delay-mode straggler (reading R19; "one device (straggler) is caused to operate
 * slower ... by forcing it to idle. The idle time is chosen to be a multiple of the time required
 * ... to perform one forward and one backward pass ... delays are expressed in terms of the number
 * of iterations the straggler lags behind"): replica delay_replica completes one iteration every
 * delay_rounds+1 rounds -- it is active only in rounds t with (t+1) % (delay_rounds+1) == 0 -- and
 * idles (still receiving) in between.  delay_rounds == 0: off.  Combined with the
 * random mask by AND.                                                                        */
int32_t oracle_active_ex(uint64_t seed, int64_t step, int32_t replica, float skip_prob,
                         int32_t delay_replica, int32_t delay_rounds) {
  if (delay_rounds > 0 && replica == delay_replica && ((step + 1) % ((int64_t)delay_rounds + 1)) != 0) return 0;
  return oracle_active(seed, step, replica, skip_prob);
}

/* PAPER.md:101 "j ~ Random(M-1)": uniform over the K-1 other workers (R5).
 * uint32 -> [0, K-2] by multiply-high (R6), then skip over self.
 * peer_mode 0: a fresh peer per (step, layer, replica) (BASELINE.json north_star)
 * peer_mode 1: one peer per (step, replica), shared by all layers (Alg. 1).   */
int32_t oracle_peer(uint64_t seed, int64_t step, int32_t layer, int32_t replica,
                    int32_t K, int32_t peer_mode) {
  if (K < 2) return -1;
  const uint32_t lf = peer_mode == 0 ? (uint32_t)layer : FIELD_NONE;
  const uint32_t r = draw(seed, (uint32_t)step, lf, (uint32_t)replica, TAG_PEER);
  const uint32_t q = (uint32_t)(((uint64_t)r * (uint64_t)(K - 1)) >> 32);
  return (int32_t)(q + (q >= (uint32_t)replica ? 1u : 0u));
}

/* peer[l*K+i] = chosen peer, or -1 when replica i is inactive (or K == 1). */
void oracle_schedule(uint64_t seed, int64_t step, int32_t L, int32_t K, int32_t peer_mode,
                     float skip_prob, int32_t delay_replica, int32_t delay_rounds,
                     int32_t *peer, uint8_t *active) {
  for (int32_t i = 0; i < K; ++i)
    active[i] = (uint8_t)oracle_active_ex(seed, step, i, skip_prob, delay_replica, delay_rounds);
  for (int32_t l = 0; l < L; ++l)
    for (int32_t i = 0; i < K; ++i)
      peer[(size_t)l * K + i] = active[i] ? oracle_peer(seed, step, l, i, K, peer_mode) : -1;
}

/* ---- options of the widened rule -----------------------
 * optimizer 0: SGD, optional heavy-ball momentum mu (reading R8) and coupled weight decay
 *              wd (the "weight_decay" row of PAPER.md:416-443, Tables A5/A6; PyTorch's SGD
 *              convention d = g + wd*x, reading R21)
 * optimizer 1: AdamW (PAPER.md:130 + Tables A7/A8 PAPER.md:469-491 "optimizer AdamW"),
 *              decoupled decay, bias-corrected, PyTorch's convention (reading R21); the
 *              moments m, v and the step count are local to the worker, never gossiped
 * mix_mode 0 : push-sum fold, every colliding push applied (reading R3)
 * mix_mode 1 : contention as the paper describes its own race ("the parameters
 *              sent from one of the peers will be skipped", "not guaranteed that
 *              all the weights for the push sum will be used"): of the pushes colliding on one
 *              receiver only the LAST writer (highest sender index) lands, with its weight;
 *              the skipped senders have already halved their weight and that mass is lost
 *              (reading R22)
 * mix_mode 2 : AD-PSGD-style symmetric pairwise averaging ("enforced symmetric
 *              communication ... doubling the communication volume"): each active worker i, in
 *              ascending index, atomically averages with its peer j: x_i, x_j <- (x_i+x_j)/2;
 *              no push-sum weights (reading R23)
 * All scalars are doubles holding fp32-representable values; the fp32 path narrows them. */
typedef struct {
  int32_t optimizer;
  int32_t mix_mode;
  double lr, mu, wd, beta1, beta2, eps;
} oracle_opts;

enum { OPT_SGD = 0, OPT_ADAMW = 1 };
enum { MIX_PUSHSUM = 0, MIX_LOSSY = 1, MIX_SYMMETRIC = 2 };

/* steps 1-2 of the header: mask, peers, halved weights.  Symmetric averaging carries no
 * push-sum weight (R23), so nothing is halved there.                                     */
static void draw_schedule(int32_t K, const double *w, uint64_t seed, int64_t step, int32_t layer,
                          int32_t peer_mode, float skip_prob, int32_t delay_replica, int32_t delay_rounds,
                          int32_t mix_mode, const int32_t *peer_in, const uint8_t *active_in,
                          int32_t *peer, uint8_t *active, double *wh) {
  for (int32_t i = 0; i < K; ++i) {
    active[i] = active_in ? active_in[i]
                          : (uint8_t)oracle_active_ex(seed, step, i, skip_prob, delay_replica, delay_rounds);
    if (active[i] && K >= 2) {
      peer[i] = peer_in ? peer_in[i] : oracle_peer(seed, step, layer, i, K, peer_mode);
      wh[i] = mix_mode == MIX_SYMMETRIC ? w[i] : w[i] * 0.5;
    } else {
      peer[i] = -1;          /* inactive (or alone): no push, weight not halved */
      wh[i] = w[i];
    }
  }
}

/* ---- one (step, layer) of the updater, fp32 state, fp64 push-sum weights ----
 * x, g, m, v : [K][n] row-major fp32 (m NULL when unused: SGD with mu == 0; v NULL unless
 * AdamW);  w : [K] fp64;  bpow : [K][2] fp64 = (beta1^t_i, beta2^t_i), 1.0 before the first
 * step, AdamW only;  tcount : [K] steps worker i has taken on this layer, AdamW only.
 * peer_in/active_in: if non-NULL the schedule is taken from them instead of being drawn
 * (used by the brute-force tests to enumerate every schedule).
 * Returns 0, or -1 on allocation failure.                                    */
int oracle_layer_update_ex(int32_t K, int64_t n, float *x, const float *g, float *m, float *v, double *w,
                           double *bpow, int64_t *tcount, const oracle_opts *o,
                           uint64_t seed, int64_t step, int32_t layer,
                           int32_t peer_mode, float skip_prob, int32_t delay_replica, int32_t delay_rounds,
                           const int32_t *peer_in, const uint8_t *active_in) {
  int32_t *peer = (int32_t *)malloc(sizeof(int32_t) * (size_t)K);
  uint8_t *active = (uint8_t *)malloc((size_t)K);
  double *wh = (double *)malloc(sizeof(double) * (size_t)K);
  float *y = (float *)malloc(sizeof(float) * (size_t)K * (size_t)(n > 0 ? n : 1));
  float *acc = (float *)malloc(sizeof(float) * (size_t)(n > 0 ? n : 1));
  if (!peer || !active || !wh || !y || !acc) {
    free(peer); free(active); free(wh); free(y); free(acc);
    return -1;
  }
  const float lr = (float)o->lr, mu = (float)o->mu, wd = (float)o->wd;

  /* 1. straggler mask; 2. peer choice and weight halving */
  draw_schedule(K, w, seed, step, layer, peer_mode, skip_prob, delay_replica, delay_rounds, o->mix_mode,
                peer_in, active_in, peer, active, wh);

  /* 3. local step on the current copy */
  for (int32_t i = 0; i < K; ++i) {
    float *xi = x + (size_t)i * n;
    const float *gi = g + (size_t)i * n;
    float *yi = y + (size_t)i * n;
    if (!active[i]) {
      ORACLE_PAR
      for (int64_t e = 0; e < n; ++e) yi[e] = xi[e];
    } else if (o->optimizer == OPT_ADAMW) {
      /* AdamW (Loshchilov & Hutter), PyTorch's order of operations:
       *   x <- x (1 - eta wd);  m <- b1 m + (1-b1) g;  v <- b2 v + (1-b2) g^2
       *   x <- x - eta/(1-b1^t) * m / ( sqrt(v)/sqrt(1-b2^t) + eps )
       * the per-step scalars come from fp64, rounded once to fp32                          */
      float *mi = m + (size_t)i * n, *vi = v + (size_t)i * n;
      const float b1 = (float)o->beta1, b2 = (float)o->beta2, eps = (float)o->eps;
      const float omb1 = (float)(1.0 - (double)b1), omb2 = (float)(1.0 - (double)b2);
      const float decay = (float)(1.0 - (double)lr * (double)wd);
      bpow[2 * i + 0] *= (double)b1;                       /* beta1^t, t counted per worker  */
      bpow[2 * i + 1] *= (double)b2;
      tcount[i] += 1;
      const float c1 = (float)((double)lr / (1.0 - bpow[2 * i + 0]));
      const float c2 = (float)(1.0 / sqrt(1.0 - bpow[2 * i + 1]));
      ORACLE_PAR
      for (int64_t e = 0; e < n; ++e) {
        const float xd = xi[e] * decay;
        const float mm = fmaf(b1, mi[e], omb1 * gi[e]);
        const float gg = gi[e] * gi[e];
        const float vv = fmaf(b2, vi[e], omb2 * gg);
        const float den = fmaf(sqrtf(vv), c2, eps);
        mi[e] = mm;
        vi[e] = vv;
        yi[e] = fmaf(-c1, mm / den, xd);
      }
    } else {
      float *mi = mu != 0.0f ? m + (size_t)i * n : NULL;
      ORACLE_PAR
      for (int64_t e = 0; e < n; ++e) {
        float d = gi[e];
        if (wd != 0.0f) d = fmaf(wd, xi[e], d);      /* coupled decay: d = g + wd*x     */
        if (mi) {
          d = fmaf(mu, mi[e], d);                    /* m <- mu*m + d                   */
          mi[e] = d;
        }
        yi[e] = fmaf(-lr, d, xi[e]);                 /* y  = x - eta*(m | d)            */
      }
    }
  }

  if (o->mix_mode == MIX_SYMMETRIC) {
    /* 4''. symmetric pairwise averaging, one atomic exchange per active worker, ascending i;
     * each exchange sees the values the earlier ones left (a product of pairwise-averaging
     * matrices, Lian et al. 2018).  Weights stay as they are.                              */
    for (int32_t i = 0; i < K; ++i) {
      if (!(active[i] && peer[i] >= 0)) continue;
      float *yi = y + (size_t)i * n, *yj = y + (size_t)peer[i] * n;
      ORACLE_PAR
      for (int64_t e = 0; e < n; ++e) {
        const float avg = 0.5f * (yi[e] + yj[e]);
        yi[e] = avg;
        yj[e] = avg;
      }
    }
    memcpy(x, y, sizeof(float) * (size_t)K * (size_t)n);
  } else {
    /* 4. peer update, once per sender of j in ascending sender index; under contention
     * (MIX_LOSSY) only the last writer's push and weight land.                             */
    for (int32_t j = 0; j < K; ++j) {
      double W = wh[j];
      const float *yj = y + (size_t)j * n;
      int32_t last = -1;
      for (int32_t i = 0; i < K; ++i)
        if (active[i] && peer[i] == j) last = i;
      ORACLE_PAR
      for (int64_t e = 0; e < n; ++e) acc[e] = yj[e];
      for (int32_t i = 0; i < K; ++i) {
        if (!(active[i] && peer[i] == j)) continue;
        if (o->mix_mode == MIX_LOSSY && i != last) continue;  /* overwritten: skipped       */
        const float alpha = (float)(wh[i] / (W + wh[i]));   /* w_i/(w_i+w_j), one rounding */
        const float *yi = y + (size_t)i * n;
        ORACLE_PAR
        for (int64_t e = 0; e < n; ++e) {
          const float d = yi[e] - acc[e];
          acc[e] = fmaf(alpha, d, acc[e]);                  /* = (1-a)*x_j + a*x_i */
        }
        W = W + wh[i];                                      /* w_j <- w_j + w_i    */
      }
      float *xj = x + (size_t)j * n;
      ORACLE_PAR
      for (int64_t e = 0; e < n; ++e) xj[e] = acc[e];
      w[j] = W;
    }
  }

  free(peer); free(active); free(wh); free(y); free(acc);
  return 0;
}

/* ---- the scalar half of steps 2 and 4 on its own: for a given schedule (peer, active) and
 * weights w, the halved weights, then per receiver j in ascending sender index the coefficient
 * alpha = w_i/(w_i+w_j) of every push that lands ("Peer Update") and the weight
 * after it (w_j <- w_j + w_i).  Output as a CSR by receiver: entries [recv_off[j], recv_off[j+1])
 * of senders[] / alpha[] belong to receiver j.  The statements are those of step 4 of
 * oracle_layer_update_ex; tests compare this list with the tables the CUDA path consumed
 * (layup_schedule_tables) and pin it against oracle_layer_update_ex itself.  MIX_SYMMETRIC has no
 * sender list (recv_off all zero, weights unchanged).                                     */
void oracle_mix_tables(int32_t K, const double *w, const int32_t *peer, const uint8_t *active, int32_t mix_mode,
                       int32_t *recv_off, int32_t *senders, float *alpha, double *w_out) {
  int32_t k = 0;
  for (int32_t j = 0; j < K; ++j) {
    const double whj = (active[j] && K >= 2 && mix_mode != MIX_SYMMETRIC) ? w[j] * 0.5 : w[j];
    double W = whj;
    recv_off[j] = k;
    int32_t last = -1;
    for (int32_t i = 0; i < K; ++i)
      if (active[i] && peer[i] == j) last = i;
    for (int32_t i = 0; i < K && mix_mode != MIX_SYMMETRIC; ++i) {
      if (!(active[i] && peer[i] == j)) continue;
      if (mix_mode == MIX_LOSSY && i != last) continue;
      const double whi = w[i] * 0.5;                        /* a sender has halved its weight */
      senders[k] = i;
      alpha[k] = (float)(whi / (W + whi));
      W = W + whi;
      ++k;
    }
    w_out[j] = W;
  }
  recv_off[K] = k;
}

/* The rule of the header as first pinned: SGD (+ momentum), push-sum fold. */
int oracle_layer_update(int32_t K, int64_t n, float *x, const float *g, float *m, double *w,
                        float lr, float mu, uint64_t seed, int64_t step, int32_t layer,
                        int32_t peer_mode, float skip_prob, int32_t delay_replica, int32_t delay_rounds,
                        const int32_t *peer_in, const uint8_t *active_in) {
  const oracle_opts o = {OPT_SGD, MIX_PUSHSUM, (double)lr, (double)mu, 0.0, 0.0, 0.0, 0.0};
  return oracle_layer_update_ex(K, n, x, g, m, NULL, w, NULL, NULL, &o, seed, step, layer, peer_mode, skip_prob,
                                delay_replica, delay_rounds, peer_in, active_in);
}

/* ---- fp64 shadow: same schedule, every value in double, and the mix written in
 * its closed form  x_j <- (wh_j y_j + sum_i wh_i y_i) / (wh_j + sum_i wh_i)
 * (PAPER.md:101 applied once per sender telescopes to this weighted centroid); AdamW's bias
 * corrections from pow(beta, t) rather than running products.
 * Used for the 100-round error bound and as an independent statement of steps 3-4. */
int oracle_layer_update_ex_f64(int32_t K, int64_t n, double *x, const float *g, double *m, double *v, double *w,
                               double *bpow, int64_t *tcount, const oracle_opts *o,
                               uint64_t seed, int64_t step, int32_t layer,
                               int32_t peer_mode, float skip_prob, int32_t delay_replica, int32_t delay_rounds,
                               const int32_t *peer_in, const uint8_t *active_in) {
  (void)bpow;
  int32_t *peer = (int32_t *)malloc(sizeof(int32_t) * (size_t)K);
  uint8_t *active = (uint8_t *)malloc((size_t)K);
  double *wh = (double *)malloc(sizeof(double) * (size_t)K);
  double *y = (double *)malloc(sizeof(double) * (size_t)K * (size_t)(n > 0 ? n : 1));
  if (!peer || !active || !wh || !y) {
    free(peer); free(active); free(wh); free(y);
    return -1;
  }
  const double lr = o->lr, mu = o->mu, wd = o->wd;
  draw_schedule(K, w, seed, step, layer, peer_mode, skip_prob, delay_replica, delay_rounds, o->mix_mode,
                peer_in, active_in, peer, active, wh);
  for (int32_t i = 0; i < K; ++i) {
    double bc1 = 1.0, bc2 = 1.0;
    if (active[i] && o->optimizer == OPT_ADAMW) {
      tcount[i] += 1;
      bc1 = 1.0 - pow(o->beta1, (double)tcount[i]);
      bc2 = 1.0 - pow(o->beta2, (double)tcount[i]);
    }
    for (int64_t e = 0; e < n; ++e) {
      const size_t q = (size_t)i * n + e;
      if (!active[i]) {
        y[q] = x[q];
      } else if (o->optimizer == OPT_ADAMW) {
        const double gg = (double)g[q];
        m[q] = o->beta1 * m[q] + (1.0 - o->beta1) * gg;
        v[q] = o->beta2 * v[q] + (1.0 - o->beta2) * gg * gg;
        y[q] = x[q] * (1.0 - lr * wd) - (lr / bc1) * m[q] / (sqrt(v[q]) / sqrt(bc2) + o->eps);
      } else {
        double d = (double)g[q] + wd * x[q];
        if (mu != 0.0) {
          m[q] = mu * m[q] + d;
          d = m[q];
        }
        y[q] = x[q] - lr * d;
      }
    }
  }
  if (o->mix_mode == MIX_SYMMETRIC) {
    for (int32_t i = 0; i < K; ++i) {
      if (!(active[i] && peer[i] >= 0)) continue;
      for (int64_t e = 0; e < n; ++e) {
        const double avg = (y[(size_t)i * n + e] + y[(size_t)peer[i] * n + e]) / 2.0;
        y[(size_t)i * n + e] = avg;
        y[(size_t)peer[i] * n + e] = avg;
      }
    }
    memcpy(x, y, sizeof(double) * (size_t)K * (size_t)n);
  } else {
    for (int32_t j = 0; j < K; ++j) {
      int32_t last = -1;
      for (int32_t i = 0; i < K; ++i)
        if (active[i] && peer[i] == j) last = i;
      double W = wh[j];
      for (int32_t i = 0; i < K; ++i)
        if (active[i] && peer[i] == j && (o->mix_mode == MIX_PUSHSUM || i == last)) W += wh[i];
      for (int64_t e = 0; e < n; ++e) {
        double s = wh[j] * y[(size_t)j * n + e];
        for (int32_t i = 0; i < K; ++i)
          if (active[i] && peer[i] == j && (o->mix_mode == MIX_PUSHSUM || i == last)) s += wh[i] * y[(size_t)i * n + e];
        x[(size_t)j * n + e] = s / W;
      }
    }
    /* weights are updated after all receivers are done (wh is the pre-round view) */
    for (int32_t j = 0; j < K; ++j) {
      int32_t last = -1;
      for (int32_t i = 0; i < K; ++i)
        if (active[i] && peer[i] == j) last = i;
      double W = wh[j];
      for (int32_t i = 0; i < K; ++i)
        if (active[i] && peer[i] == j && (o->mix_mode == MIX_PUSHSUM || i == last)) W = W + wh[i];
      w[j] = W;
    }
  }
  free(peer); free(active); free(wh); free(y);
  return 0;
}

int oracle_layer_update_f64(int32_t K, int64_t n, double *x, const float *g, double *m, double *w,
                            double lr, double mu, uint64_t seed, int64_t step, int32_t layer,
                            int32_t peer_mode, float skip_prob, int32_t delay_replica, int32_t delay_rounds,
                            const int32_t *peer_in, const uint8_t *active_in) {
  const oracle_opts o = {OPT_SGD, MIX_PUSHSUM, lr, mu, 0.0, 0.0, 0.0, 0.0};
  return oracle_layer_update_ex_f64(K, n, x, g, m, NULL, w, NULL, NULL, &o, seed, step, layer, peer_mode,
                                    skip_prob, delay_replica, delay_rounds, peer_in, active_in);
}

/* ---- model disagreement (PAPER.md:389-395 Fig. A1; eq. (9)
 * E||xbar_t - x_t^i||^2 <= eta^2 B^2): per replica, the squared distance to the consensus
 *     dist[i] = sum_e (x_i[e] - xbar[e])^2 ,  xbar[e] = sum_i c_i x_i[e]
 * with c_i = 1/K (the paper's plain average, w == NULL) or c_i = w_i (push-sum weighted
 * consensus, sum_i w_i = 1).  x: [K][n] fp32; everything accumulated in fp64.             */
void oracle_disagreement(int32_t K, int64_t n, const float *x, const double *w, double *dist) {
  for (int32_t i = 0; i < K; ++i) dist[i] = 0.0;
  for (int64_t e = 0; e < n; ++e) {
    double xbar = 0.0;
    for (int32_t i = 0; i < K; ++i) xbar += (w ? w[i] : 1.0 / (double)K) * (double)x[(size_t)i * n + e];
    for (int32_t i = 0; i < K; ++i) {
      const double d = (double)x[(size_t)i * n + e] - xbar;
      dist[i] += d * d;
    }
  }
}
