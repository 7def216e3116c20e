/*
 * km_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * The comparison baseline and the quality metrics of the paper's GSKM evaluation (section 6.1, :200-212; section 4,
 * :60-85), written from the paper text only, in plain IEEE double, sharing no code with the CUDA path:
 *   - standard (weighted) K-means, "KM": each vector is represented by a centroid mu and the squared euclidean distortion
 *     ||x - mu||^2 is minimised; the l2-optimal centroid of a cluster is the arithmetic mean of its points
 *     (Eq. 2) -- Lloyd's algorithm.  Weighted per PAPER.md:93 ("weighted K-means"): mu_k = sum w_i x_i / sum w_i.
 *   - metrics: MSE = E||x - xhat||^2, gain error E| ||x|| - ||xhat|| |, cosine similarity E cos(x, xhat);
 *     shrinkage ratio E||mu||^2 / E||x||^2, with the expectation over samples of their assigned centroid.
 * Readings where the paper is silent: ties go to the lowest index; an empty cluster keeps its centroid;
 * the initial centroids are K seeded distinct non-zero rows (the same rows as GSKM's initial shapes, reading c-I);
 * cos(x, xhat) = 0 when either vector is zero; centroids are rounded to fp32 after every update (reading c-P).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

int gsrq_oracle_init_ids(const float *r, int64_t N, int d, int K, uint64_t seed, int group, int G, int stage, int64_t *ids);

/* Assignment: k_i = argmin_k ||x_i - mu_k||^2, the distance written out directly; lowest k wins ties. */
void km_oracle_assign(const float *x, int64_t N, int d, const float *mu, int K, int32_t *idx, double *best) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < N; ++i) {
    double b = INFINITY;
    int32_t kb = 0;
    for (int k = 0; k < K; ++k) {
      double dist = 0.0;
      for (int j = 0; j < d; ++j) {
        double e = (double)x[i * d + j] - (double)mu[(int64_t)k * d + j];
        dist += e * e;
      }
      if (dist < b) { b = dist; kb = k; }
    }
    idx[i] = kb;
    if (best) best[i] = b;
  }
}

/* Update: mu_k = fl32(sum_{i in I_k} w_i x_i / sum w_i) (Eq. 2, weighted per :93); empty cluster keeps mu_k. */
int km_oracle_update(const float *x, const float *w, int64_t N, int d, const int32_t *idx, int K, float *mu) {
  double *A = (double *)calloc((size_t)K * d, sizeof(double));
  double *W = (double *)calloc((size_t)K, sizeof(double));
  int64_t *cnt = (int64_t *)calloc((size_t)K, sizeof(int64_t));
  for (int64_t i = 0; i < N; ++i) {
    int k = idx[i];
    double wi = w ? (double)w[i] : 1.0;
    cnt[k] += 1;
    W[k] += wi;
    for (int j = 0; j < d; ++j) A[(int64_t)k * d + j] += wi * (double)x[i * d + j];
  }
  int n_empty = 0;
  for (int k = 0; k < K; ++k) {
    if (cnt[k] == 0) n_empty++;
    if (cnt[k] == 0 || !(W[k] > 0.0)) continue;
    for (int j = 0; j < d; ++j) mu[(int64_t)k * d + j] = (float)(A[(int64_t)k * d + j] / W[k]);
  }
  free(A); free(W); free(cnt);
  return n_empty;
}

/* Weighted distortion J = sum_i w_i ||x_i - mu_{a_i}||^2. */
double km_oracle_wdist(const float *x, const float *w, int64_t N, int d, const int32_t *idx, const float *mu) {
  double J = 0.0;
  for (int64_t i = 0; i < N; ++i) {
    double e2 = 0.0;
    for (int j = 0; j < d; ++j) {
      double e = (double)x[i * d + j] - (double)mu[(int64_t)idx[i] * d + j];
      e2 += e * e;
    }
    J += (w ? (double)w[i] : 1.0) * e2;
  }
  return J;
}

/*
 * Lloyd's algorithm: init = K seeded distinct non-zero rows; for t = 1..iters: assign, update; stop when the assignment equals the
 * previous iteration's (t > 1).  Outputs mu[K][d], idx_last[N] (the assignment of the last iteration run), J_assign[t-1] (distortion
 * right after iteration t's assignment), changed[t-1] (vs. the previous assignment; iteration 1 compares with all-zero), *iters_run.
 */
int km_oracle_fit(const float *x, const float *w, int64_t N, int d, int K, int iters, uint64_t seed, float *mu, int32_t *idx_last,
                  double *J_assign, int64_t *changed, int32_t *iters_run, int32_t *n_empty_last) {
  int64_t *ids = (int64_t *)malloc((size_t)K * sizeof(int64_t));
  if (gsrq_oracle_init_ids(x, N, d, K, seed, 0, 1, 0, ids) != 0) { free(ids); return -1; }
  for (int k = 0; k < K; ++k) memcpy(mu + (int64_t)k * d, x + ids[k] * d, (size_t)d * sizeof(float));
  free(ids);
  int32_t *a = (int32_t *)calloc((size_t)N, sizeof(int32_t));
  int32_t *a_prev = (int32_t *)calloc((size_t)N, sizeof(int32_t));
  int t_run = 0, n_empty = 0;
  for (int t = 1; t <= iters; ++t) {
    km_oracle_assign(x, N, d, mu, K, a, NULL);
    int64_t nch = 0;
    for (int64_t i = 0; i < N; ++i) nch += (a[i] != a_prev[i]);
    if (J_assign) J_assign[t - 1] = km_oracle_wdist(x, w, N, d, a, mu);
    if (changed) changed[t - 1] = nch;
    n_empty = km_oracle_update(x, w, N, d, a, K, mu);
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
 * Metrics of a reconstruction xhat_i = proto[idx_i] (proto = the centroid mu_k for KM, fl32(g_k s_k) for GSKM), PAPER.md:202, :85:
 *   out[0] = MSE = mean_i ||x_i - xhat_i||^2, out[1] = mean_i | ||x_i|| - ||xhat_i|| |, out[2] = mean_i cos(x_i, xhat_i),
 *   out[3] = shrinkage ratio mean_i ||xhat_i||^2 / mean_i ||x_i||^2.
 */
void km_oracle_metrics(const float *x, int64_t N, int d, const float *proto, const int32_t *idx, double *out) {
  double mse = 0.0, ge = 0.0, cs = 0.0, p2 = 0.0, x2 = 0.0;
  for (int64_t i = 0; i < N; ++i) {
    const float *xi = x + i * d, *pi = proto + (int64_t)idx[i] * d;
    double e2 = 0.0, nx2 = 0.0, np2 = 0.0, dot = 0.0;
    for (int j = 0; j < d; ++j) {
      double a = (double)xi[j], b = (double)pi[j];
      e2 += (a - b) * (a - b);
      nx2 += a * a;
      np2 += b * b;
      dot += a * b;
    }
    double nx = sqrt(nx2), np = sqrt(np2);
    mse += e2;
    ge += fabs(nx - np);
    cs += (nx > 0.0 && np > 0.0) ? dot / (nx * np) : 0.0;
    p2 += np2;
    x2 += nx2;
  }
  out[0] = mse / (double)N;
  out[1] = ge / (double)N;
  out[2] = cs / (double)N;
  out[3] = p2 / x2;
}
