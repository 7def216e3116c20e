/*
 * gsrq_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct CPU implementation of weighted Gain-Shape
 * K-means (GSKM) and Gain-Shape Residual Quantization (GSRQ), written from the
 * paper text only (/root/reference/PAPER.md at build time; citations below are
 * "PAPER.md:<line>" plus section / equation / algorithm).  It shares no code
 * with the CUDA path under paper_2607_01065_b200/csrc and neither includes nor
 * links anything from it.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.
 *
 * Arithmetic: every sum, dot product, norm, division and square root is in
 * IEEE double.  Inputs (rows, weights, codebooks) are fp32 values promoted to
 * double.  Codebooks are rounded to fp32 at the end of every update, so that
 * a GPU implementation scores against the same fp32 numbers (DESIGN.md
 * reading c-P).  The residual update and the decode sum are fp32 element-wise
 * (readings c-P, c-D).  There is no blocking, fusion or reordering: loops run
 * in the order the paper's equations are written.  OpenMP is used only over
 * rows in the assignment step (rows are independent there), so results do not
 * depend on the thread count.
 *
 * Parity pins: see tests/test_oracle_*.py (brute-force assignment, Eq. 4
 * identity, Eq. 7 maximiser, Eq. 8 closed form, weighted == replicated rows,
 * equal-norm case == textbook / scikit-learn Lloyd K-means, K = 1 closed form,
 * the hand-computed non-monotone example, equivariances, idempotence, RQ
 * identities, bf16 rounding vs torch, splitmix64 published vectors).
 * The full fit trajectory on the synthetic configs has no published value:
 * "parity unpinned" for that.
 *
 * One call handles ONE codebook group (one KV head) and ONE stage; the Python
 * wrapper oracle/gsrq_oracle.py loops over groups and stages.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define GSRQ_ORACLE_EPS 1e-12   /* y_i = x_i / (||x_i|| + eps)  PAPER.md:178; reading c-E */
#define GSRQ_ORACLE_DELTA 1e-8  /* "numerically close to zero" mean direction  PAPER.md:178; c-E */

/* ------------------------------------------------------------------ */
/* splitmix64 (public-domain generator by S. Vigna); used only to pick */
/* the K seeded initial rows (reading c-I).                            */
/* ------------------------------------------------------------------ */
uint64_t gsrq_oracle_splitmix64_next(uint64_t *state) {
  uint64_t z = (*state += 0x9E3779B97F4A7C15ULL);
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  return z ^ (z >> 31);
}

static double row_norm(const float *x, int d) {
  double n2 = 0.0;
  for (int j = 0; j < d; ++j) n2 += (double)x[j] * (double)x[j];
  return sqrt(n2);
}

/*
 * Initial shapes: "choose {s_k} on the unit sphere" (Alg. 1 l.1).
 * BASELINE.json config 0 fixes this to "K distinct input vectors chosen by
 * seed, normalised".  Reading c-I: a splitmix64 stream seeded with
 * seed XOR (0x9E3779B97F4A7C15 * (1 + group + G*stage)); candidate = next() mod N;
 * skip a candidate already chosen or with zero norm; take the first K.
 * Returns 0, or -1 if K distinct non-zero rows were not found within
 * 64*K + 4096 candidates (degenerate input).
 */
int gsrq_oracle_init_ids(const float *r, int64_t N, int d, int K, uint64_t seed,
                         int group, int G, int stage, int64_t *ids) {
  uint64_t st = seed ^ (0x9E3779B97F4A7C15ULL * (uint64_t)(1 + group + G * stage));
  int found = 0;
  int64_t limit = 64 * (int64_t)K + 4096;
  for (int64_t n = 0; n < limit && found < K; ++n) {
    int64_t c = (int64_t)(gsrq_oracle_splitmix64_next(&st) % (uint64_t)N);
    int dup = 0;
    for (int q = 0; q < found; ++q)
      if (ids[q] == c) { dup = 1; break; }
    if (dup) continue;
    if (row_norm(r + c * d, d) == 0.0) continue;
    ids[found++] = c;
  }
  return found == K ? 0 : -1;
}

/*
 * Assignment (Eq. 5):  k_i = argmax_k ( 2 g_k x_i^T s_k - g_k^2 ),
 * lowest k wins ties (reading c-T).  With g == NULL the score is the plain
 * projection x_i^T s_k (used once, for the initial gains: reading c-I).
 * best / second (optional) receive the top-2 scores of each row (second is
 * -inf when K == 1); the near-tie exemption of the parity protocol uses them.
 */
void gsrq_oracle_assign(const float *r, int64_t N, int d, const float *s, const float *g,
                        int K, int32_t *idx, double *best, double *second) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < N; ++i) {
    const float *x = r + i * d;
    double b1 = -INFINITY, b2 = -INFINITY;
    int32_t k1 = 0;
    for (int k = 0; k < K; ++k) {
      double dot = 0.0;
      for (int j = 0; j < d; ++j) dot += (double)x[j] * (double)s[(int64_t)k * d + j];
      double sc;
      if (g) {
        double gk = (double)g[k];
        sc = 2.0 * gk * dot - gk * gk;
      } else {
        sc = dot;
      }
      if (sc > b1) { b2 = b1; b1 = sc; k1 = k; }
      else if (sc > b2) { b2 = sc; }
    }
    idx[i] = k1;
    if (best) best[i] = b1;
    if (second) second[i] = b2;
  }
}

/*
 * Update (Eq. 6-8, weighted per reading c-W; safeguards
 * PAPER.md:178).  For each cluster k with members I_k:
 *   cnt_k = |I_k|,  W_k = sum w_i,  B_k = sum w_i y_i,  A_k = sum w_i x_i,
 *   y_i = x_i / (||x_i|| + eps);
 *   if cnt_k == 0 or W_k <= 0: keep (s_k, g_k);
 *   else: if ||B_k|| / W_k > delta: s_k = fl32(B_k / ||B_k||)      (Eq. 7)
 *         g_k = fl32(max(0, (A_k . s_k) / W_k))  with the UPDATED s_k (Eq. 8).
 * shapes_too == 0 updates gains only (Alg. 1 l.2 "Initialize gains by (8)").
 * Returns the number of empty clusters.  cnt_out (optional) gets |I_k|.
 */
int gsrq_oracle_update(const float *r, const float *w, int64_t N, int d, const int32_t *idx,
                       int K, float *s, float *g, int shapes_too, int64_t *cnt_out) {
  int64_t *cnt = (int64_t *)calloc((size_t)K, sizeof(int64_t));
  double *W = (double *)calloc((size_t)K, sizeof(double));
  double *A = (double *)calloc((size_t)K * d, sizeof(double));
  double *B = (double *)calloc((size_t)K * d, sizeof(double));
  for (int64_t i = 0; i < N; ++i) {
    const float *x = r + i * d;
    int k = idx[i];
    double wi = w ? (double)w[i] : 1.0;
    double n = row_norm(x, d);
    cnt[k] += 1;
    W[k] += wi;
    for (int j = 0; j < d; ++j) {
      double xj = (double)x[j];
      double yj = xj / (n + GSRQ_ORACLE_EPS);      /* Eq. 6 + safeguard */
      A[(int64_t)k * d + j] += wi * xj;
      B[(int64_t)k * d + j] += wi * yj;
    }
  }
  int n_empty = 0;
  for (int k = 0; k < K; ++k) {
    if (cnt[k] == 0) n_empty++;
    if (cnt[k] == 0 || !(W[k] > 0.0)) continue;    /* keep (g_k, s_k) */
    float *sk = s + (int64_t)k * d;
    if (shapes_too) {
      double bn2 = 0.0;
      for (int j = 0; j < d; ++j) bn2 += B[(int64_t)k * d + j] * B[(int64_t)k * d + j];
      double bn = sqrt(bn2);
      if (bn / W[k] > GSRQ_ORACLE_DELTA)           /* else keep previous s_k */
        for (int j = 0; j < d; ++j) sk[j] = (float)(B[(int64_t)k * d + j] / bn);
    }
    double proj = 0.0;
    for (int j = 0; j < d; ++j) proj += A[(int64_t)k * d + j] * (double)sk[j];
    double gk = proj / W[k];
    g[k] = (float)(gk > 0.0 ? gk : 0.0);
  }
  if (cnt_out) memcpy(cnt_out, cnt, (size_t)K * sizeof(int64_t));
  free(cnt); free(W); free(A); free(B);
  return n_empty;
}

/*
 * Weighted gain-shape distortion  J = sum_i w_i || x_i - g_{a_i} s_{a_i} ||^2
 * (the l2 distortion of Eq. 4/5, weighted per reading c-W),
 * written out directly (not via the expanded form).
 */
double gsrq_oracle_wdist(const float *r, const float *w, int64_t N, int d, const int32_t *idx,
                         const float *s, const float *g) {
  double J = 0.0;
  for (int64_t i = 0; i < N; ++i) {
    const float *x = r + i * d;
    int k = idx[i];
    double gk = (double)g[k], e2 = 0.0;
    for (int j = 0; j < d; ++j) {
      double e = (double)x[j] - gk * (double)s[(int64_t)k * d + j];
      e2 += e * e;
    }
    J += (w ? (double)w[i] : 1.0) * e2;
  }
  return J;
}

/*
 * GSKM, Algorithm 1, weighted:
 *   l.1   shapes = K seeded distinct rows, normalised       (gsrq_oracle_init_ids)
 *   l.2   gains by Eq. 8 under the max-projection assignment (reading c-I)
 *   l.3   for t = 1..iters:
 *   l.4-7   assignment, Eq. 5
 *   l.8-14  update, Eq. 6-8
 *   l.15-16 if assignments unchanged (vs. iteration t-1, t > 1): break
 *   l.19  return gains, shapes
 * Outputs: s[K][d], g[K]; idx_last[N] = assignment of the last iteration run;
 * J_assign[t-1] = weighted distortion right after iteration t's assignment
 * (with the codebook that produced it); changed[t-1] = #rows whose assignment
 * differs from the previous one (iteration 1 compares with the l.2
 * assignment); *iters_run; *n_empty_last; init_ids[K] (optional).
 * Returns 0, or -1 on degenerate input (see gsrq_oracle_init_ids).
 */
int gsrq_oracle_fit_stage(const float *r, const float *w, int64_t N, int d, int K, int iters,
                          uint64_t seed, int group, int G, int stage, float *s, float *g,
                          int32_t *idx_last, double *J_assign, int64_t *changed,
                          int32_t *iters_run, int32_t *n_empty_last, int64_t *init_ids) {
  int64_t *ids = (int64_t *)malloc((size_t)K * sizeof(int64_t));
  if (gsrq_oracle_init_ids(r, N, d, K, seed, group, G, stage, ids) != 0) { free(ids); return -1; }
  for (int k = 0; k < K; ++k) {
    const float *x = r + ids[k] * d;
    double n = row_norm(x, d);
    for (int j = 0; j < d; ++j) s[(int64_t)k * d + j] = (float)((double)x[j] / n);
    g[k] = 0.0f;
  }
  if (init_ids) memcpy(init_ids, ids, (size_t)K * sizeof(int64_t));
  free(ids);

  int32_t *a = (int32_t *)malloc((size_t)N * sizeof(int32_t));
  int32_t *a_prev = (int32_t *)malloc((size_t)N * sizeof(int32_t));
  gsrq_oracle_assign(r, N, d, s, NULL, K, a_prev, NULL, NULL);
  int n_empty = gsrq_oracle_update(r, w, N, d, a_prev, K, s, g, /*shapes_too=*/0, NULL);
  memcpy(a, a_prev, (size_t)N * sizeof(int32_t));

  int t_run = 0;
  for (int t = 1; t <= iters; ++t) {
    gsrq_oracle_assign(r, N, d, s, g, K, a, NULL, NULL);
    int64_t nch = 0;
    for (int64_t i = 0; i < N; ++i) nch += (a[i] != a_prev[i]);
    if (J_assign) J_assign[t - 1] = gsrq_oracle_wdist(r, w, N, d, a, s, g);
    if (changed) changed[t - 1] = nch;
    n_empty = gsrq_oracle_update(r, w, N, d, a, K, s, g, /*shapes_too=*/1, NULL);
    t_run = t;
    memcpy(a_prev, a, (size_t)N * sizeof(int32_t));
    if (t > 1 && nch == 0) break;
  }
  if (idx_last) memcpy(idx_last, a, (size_t)N * sizeof(int32_t));
  if (iters_run) *iters_run = t_run;
  if (n_empty_last) *n_empty_last = n_empty;
  free(a); free(a_prev);
  return 0;
}

/*
 * One RQ stage of the encoder ("each stage sequentially quantizes
 * the residual error of the previous stage"):
 *   a_i = argmax_k (2 g_k r_i.s_k - g_k^2)   (Eq. 5, double)
 *   c_k = fl32(g_k * s_k)                     (Eq. 3 centroid, fp32; reading c-P)
 *   r_i <- fl32(r_i - c_{a_i})                (fp32, element-wise, in place)
 */
void gsrq_oracle_encode_stage(float *r, int64_t N, int d, const float *s, const float *g, int K,
                              uint8_t *codes, double *best, double *second) {
  int32_t *a = (int32_t *)malloc((size_t)N * sizeof(int32_t));
  gsrq_oracle_assign(r, N, d, s, g, K, a, best, second);
  for (int64_t i = 0; i < N; ++i) {
    int k = a[i];
    codes[i] = (uint8_t)k;
    for (int j = 0; j < d; ++j) {
      volatile float c = g[k] * s[(int64_t)k * d + j];   /* fp32 product, rounded once */
      volatile float v = r[i * d + j] - c;               /* fp32 subtract, rounded once */
      r[i * d + j] = v;
    }
  }
  free(a);
}

/*
 * Decode (PAPER.md:56  x ~= sum_l C_l[i_l]; prefix of stages PAPER.md:25):
 *   xhat_i = ((c0[a0_i] + c1[a1_i]) + ...)  fp32, stage order 0..S_used-1
 * (reading c-D).  codes is [S][N] stage-major; s is [S][K][d]; g is [S][K].
 */
void gsrq_oracle_decode(const uint8_t *codes, int64_t N, int d, const float *s, const float *g,
                        int K, int S_used, float *out) {
  for (int64_t i = 0; i < N; ++i)
    for (int j = 0; j < d; ++j) {
      volatile float acc = 0.0f;
      for (int st = 0; st < S_used; ++st) {
        int k = codes[(int64_t)st * N + i];
        volatile float c = g[(int64_t)st * K + k] * s[((int64_t)st * K + k) * d + j];
        if (st == 0) acc = c; else acc = acc + c;
      }
      out[i * d + j] = acc;
    }
}

/* fp32 -> bf16 (upper 16 bits), round-to-nearest-even; NaN kept quiet. */
void gsrq_oracle_f32_to_bf16(const float *x, int64_t n, uint16_t *out) {
  for (int64_t i = 0; i < n; ++i) {
    uint32_t u; memcpy(&u, &x[i], 4);
    if ((u & 0x7F800000u) == 0x7F800000u && (u & 0x007FFFFFu)) { out[i] = (uint16_t)((u >> 16) | 0x40u); continue; }
    uint32_t lsb = (u >> 16) & 1u;
    u += 0x7FFFu + lsb;
    out[i] = (uint16_t)(u >> 16);
  }
}
