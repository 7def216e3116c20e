// k_prep.cuh -- per-stage preparation kernels: gather the fit rows, per-row 1/(||r||+eps),
// weighted energy, seeded initial rows (Alg. 1 l.1; reading c-I).
#pragma once
#include "gsrq_common.cuh"

namespace gsrq {

// Gather the fit rows of every group into a compact fp32 buffer Rf [G][Nf][D] and compute
// rinv[g][i] = 1 / (||r_i|| + eps) in fp64 (Eq. 6 with the safeguard of PAPER.md:178) and the
// compact per-fit-token weights wt [G][nf_tok].
template <int D>
__global__ void k_gather(RowSrc src, const float *__restrict__ w, long long w_stride_g,
                         const long long *__restrict__ fit_tokens, long long nf_tok,
                         float *__restrict__ Rf, double *__restrict__ rinv, float *__restrict__ wt) {
  const int g = blockIdx.y;
  const long long Nf = nf_tok * src.M;
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= Nf) return;
  const long long tl = i / src.M;
  const int m = (int)(i - tl * src.M);
  const long long tok = fit_tokens ? fit_tokens[(long long)g * nf_tok + tl] : tl;
  float x[D];
  if (src.rows) load_row_f32<D>(src.rows, (long long)g * src.rows_per_group + tok * src.M + m, x);
  else load_row_kv<D>(src.kv, src.dtype, (long long)g * src.stride_g + tok * src.stride_t + (long long)m * D, x);
  store_row_f32<D>(Rf, (long long)g * Nf + i, x);
  if (rinv) rinv[(long long)g * Nf + i] = 1.0 / (row_norm_f64<D>(x) + kEps);
  if (wt && m == 0) wt[(long long)g * nf_tok + tl] = w ? w[(long long)g * w_stride_g + tok] : 1.0f;
}

// Etot[g] = sum_i w_i ||r_i||^2 in fp64, fixed order (thread-strided partials + smem tree):
// the constant of Eq. 4 that turns sum of scores into the distortion J.
template <int D>
__global__ void __launch_bounds__(1024) k_energy(const float *__restrict__ Rf, const float *__restrict__ wt,
                                                 long long Nf, int M, double *__restrict__ Etot) {
  __shared__ double sh[1024];
  const int g = blockIdx.x;
  double acc = 0.0;
  for (long long i = threadIdx.x; i < Nf; i += 1024) {
    float x[D];
    load_row_f32<D>(Rf, (long long)g * Nf + i, x);
    double n2 = 0.0;
#pragma unroll
    for (int j = 0; j < D; ++j) n2 += (double)x[j] * (double)x[j];
    acc += (double)wt[(long long)g * (Nf / M) + i / M] * n2;
  }
  sh[threadIdx.x] = acc;
  __syncthreads();
  for (int s = 512; s > 0; s >>= 1) {
    if ((int)threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
    __syncthreads();
  }
  if (threadIdx.x == 0) Etot[g] = sh[0];
}

// Seeded initial rows.  Candidate n of group g is splitmix64(seed_g)[n] mod Nf; a candidate is
// accepted iff its row is non-zero and its value did not occur earlier in the stream; the first
// K accepted are the initial rows (same rule as "skip if already chosen or zero norm").
// One block of 512 threads per group evaluates 512 candidates per batch.
template <int D>
__global__ void __launch_bounds__(512) k_init_ids(const float *__restrict__ Rf, long long Nf, int K, int G, int stage,
                                                  uint64_t seed, long long *__restrict__ ids, DevStats *__restrict__ st) {
  __shared__ long long cand[512];
  __shared__ int ok[512];
  __shared__ int scan[512];
  __shared__ long long chosen[GSRQ_MAX_K];
  __shared__ int n_chosen;
  const int g = blockIdx.x, t = threadIdx.x;
  const uint64_t sg = seed ^ (kGamma * (uint64_t)(1 + g + G * stage));
  if (t == 0) n_chosen = 0;
  __syncthreads();
  const long long limit = 64LL * K + 4096;
  for (long long base = 0; base < limit; base += 512) {
    const long long n = base + t;
    long long c = (long long)(splitmix64_at(sg, (uint64_t)n) % (uint64_t)Nf);
    int good = n < limit;
    if (good) {
      float x[D];
      load_row_f32<D>(Rf, (long long)g * Nf + c, x);
      bool nz = false;
#pragma unroll
      for (int j = 0; j < D; ++j) nz |= (x[j] != 0.0f);
      good = nz;
    }
    cand[t] = c;
    __syncthreads();
    const int nc = n_chosen;
    if (good) {
      for (int q = 0; q < nc && good; ++q) good = (chosen[q] != c);
      for (int q = 0; q < t && good; ++q) good = (cand[q] != c);
    }
    ok[t] = good;
    scan[t] = good;
    __syncthreads();
    for (int off = 1; off < 512; off <<= 1) {  // inclusive Hillis-Steele scan (integers: exact)
      int v = (t >= off) ? scan[t - off] : 0;
      __syncthreads();
      scan[t] += v;
      __syncthreads();
    }
    const int pos = nc + scan[t] - ok[t];
    if (ok[t] && pos < K) chosen[pos] = c;
    __syncthreads();
    if (t == 0) n_chosen = min(K, nc + scan[511]);
    __syncthreads();
    if (n_chosen >= K) break;
  }
  if (n_chosen < K) {
    if (t == 0) st[g].err = GSRQ_EDEGENERATE;
    for (int k = t; k < K; k += 512) ids[(long long)g * K + k] = (k < n_chosen) ? chosen[k] : 0;
  } else {
    for (int k = t; k < K; k += 512) ids[(long long)g * K + k] = chosen[k];
  }
}

// s_k = fl32(r / ||r||) in fp64 for the K chosen rows; g_k = 0 (set by the first gain update).
template <int D>
__global__ void k_init_shapes(const float *__restrict__ Rf, long long Nf, int K, const long long *__restrict__ ids,
                              float *__restrict__ shapes, float *__restrict__ gains, long long cb_stride_g) {
  const int g = blockIdx.x;
  for (int k = threadIdx.x; k < K; k += blockDim.x) {
    float x[D];
    load_row_f32<D>(Rf, (long long)g * Nf + ids[(long long)g * K + k], x);
    const double n = row_norm_f64<D>(x);
    float *s = shapes + (long long)g * cb_stride_g * D + (long long)k * D;
#pragma unroll
    for (int j = 0; j < D; ++j) s[j] = (n > 0.0) ? (float)((double)x[j] / n) : 0.0f;
    gains[(long long)g * cb_stride_g + k] = 0.0f;
  }
}

}  // namespace gsrq
