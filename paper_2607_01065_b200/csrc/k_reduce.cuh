// k_reduce.cuh -- deterministic segmented weighted centroid reduction (Eq. 6-8 sums) and
// codeword renormalisation (Eq. 7, Eq. 8, safeguards of PAPER.md:178).
//
// Per cluster k the update needs  cnt_k, W_k = sum w_i, A_k = sum w_i r_i, B_k = sum w_i y_i,
// y_i = r_i/(||r_i||+eps).  No floating-point atomics: each CTA owns a chunk of kChunkRows
// consecutive rows of one group, buckets its rows by cluster with a shared-memory bitmap
// (integer atomicOr: order-independent), and one warp per cluster adds that cluster's rows in
// ascending row order (lanes = vector elements), writing a per-(chunk, cluster) partial.
// k_renorm merges the partials in chunk order.  All accumulation is fp64, so the sums equal
// the definition's row-order fp64 sums to ~1e-16 and the fp32-rounded codebook is, in
// practice, bit-identical to an fp64 reference.
#pragma once
#include "gsrq_common.cuh"

namespace gsrq {

constexpr int kReduceThreads = 512;
constexpr int kBmWords = kChunkRows / 32;


template <int D>
__global__ void k_rinv(const float *__restrict__ Rf, long long n_rows, double *__restrict__ rinv) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_rows) return;
  float x[D];
  load_row_f32<D>(Rf, i, x);
  rinv[i] = 1.0 / (row_norm_f64<D>(x) + kEps);
}

// grid = (C, G), block = 512.  part: [G][C][K][2D+2] fp64 = [A | B | W | cnt].
template <int D>
__global__ void __launch_bounds__(kReduceThreads) k_reduce(const float *__restrict__ Rf, const double *__restrict__ rinv,
                                                           const float *__restrict__ wt, const uint8_t *__restrict__ idx,
                                                           long long Nf, int M, int K, double *__restrict__ part,
                                                           const DevStats *__restrict__ st) {
  extern __shared__ __align__(16) unsigned int sm_u[];
  unsigned int *bm = sm_u;                                                        // [K][kBmWords]
  uint16_t *wl = reinterpret_cast<uint16_t *>(bm + (size_t)K * kBmWords);         // [16 warps][kChunkRows]
  const int g = blockIdx.y, c = blockIdx.x, C = gridDim.x;
  if (st && st[g].done) return;
  const long long base = (long long)c * kChunkRows;
  const int rows_here = (int)min((long long)kChunkRows, Nf - base);
  constexpr int P = 2 * D + 2;

  for (int e = threadIdx.x; e < K * kBmWords; e += kReduceThreads) bm[e] = 0u;
  __syncthreads();
  for (int i = threadIdx.x; i < rows_here; i += kReduceThreads) {
    const int k = idx[(long long)g * Nf + base + i];
    if (k < K) atomicOr(&bm[k * kBmWords + (i >> 5)], 1u << (i & 31));
  }
  __syncthreads();

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  uint16_t *my = wl + warp * kChunkRows;
  const int half = lane >> 4, jl = lane & 15;
  const float *rows = Rf + ((long long)g * Nf + base) * D;
  const double *ri = rinv + (long long)g * Nf + base;
  const float *wg = wt + (long long)g * (Nf / M);
  for (int k = warp; k < K; k += kReduceThreads / 32) {
    // expand the bitmap of cluster k into an ascending row list
    int n = 0;
#pragma unroll
    for (int h = 0; h < kBmWords / 32; ++h) {
      unsigned int word = bm[k * kBmWords + h * 32 + lane];
      int cnt = __popc(word), pre = cnt;
#pragma unroll
      for (int off = 1; off < 32; off <<= 1) {
        const int v = __shfl_up_sync(0xffffffffu, pre, off);
        if (lane >= off) pre += v;
      }
      const int tot = __shfl_sync(0xffffffffu, pre, 31);
      int o = n + pre - cnt;
      while (word) {
        const int b = __ffs(word) - 1;
        word &= word - 1;
        my[o++] = (uint16_t)((h * 32 + lane) * 32 + b);
      }
      n += tot;
    }
    __syncwarp();
    // add the cluster's rows in ascending order; lanes 0-15: A (coef w), lanes 16-31: B (coef w*rinv)
    double acc[(D + 15) / 16];
#pragma unroll
    for (int q = 0; q < (D + 15) / 16; ++q) acc[q] = 0.0;
    double Wk = 0.0;
    int o = 0;
    for (; o + 4 <= n; o += 4) {
      int r[4]; float wv[4]; double rv[4]; float xv[4][(D + 15) / 16];
#pragma unroll
      for (int u = 0; u < 4; ++u) r[u] = my[o + u];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        wv[u] = wg[(base + r[u]) / M];
        rv[u] = ri[r[u]];
#pragma unroll
        for (int q = 0; q < (D + 15) / 16; ++q)
          xv[u][q] = (jl + 16 * q < D) ? rows[(long long)r[u] * D + jl + 16 * q] : 0.0f;
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const double w = (double)wv[u];
        const double coef = half ? w * rv[u] : w;
        Wk += w;
#pragma unroll
        for (int q = 0; q < (D + 15) / 16; ++q) acc[q] += coef * (double)xv[u][q];
      }
    }
    for (; o < n; ++o) {
      const int r = my[o];
      const double w = (double)wg[(base + r) / M];
      const double coef = half ? w * ri[r] : w;
      Wk += w;
#pragma unroll
      for (int q = 0; q < (D + 15) / 16; ++q)
        if (jl + 16 * q < D) acc[q] += coef * (double)rows[(long long)r * D + jl + 16 * q];
    }
    double *out = part + (((long long)g * C + c) * K + k) * P;
#pragma unroll
    for (int q = 0; q < (D + 15) / 16; ++q)
      if (jl + 16 * q < D) out[half * D + jl + 16 * q] = acc[q];
    if (lane == 0) { out[2 * D] = Wk; out[2 * D + 1] = (double)n; }
    __syncwarp();
  }
}

// grid = G, block = 256 (thread k owns cluster k).  Merges the chunk partials in chunk order,
// records J_t = Etot - sum_k (2 g_k A_k.s_k - W_k g_k^2) with the codebook that produced the
// assignment (Eq. 4 summed over rows), then applies the update and the early-exit rule.
//   lloyd = 0: gains only (Alg. 1 l.2);  lloyd = 1: iteration t of Alg. 1 l.3-18.
template <int D>
__global__ void __launch_bounds__(256) k_renorm(const double *__restrict__ part, int C, int K, float *__restrict__ shapes,
                                                float *__restrict__ gains, long long cb_stride_g,
                                                const double *__restrict__ Etot, DevStats *__restrict__ st, int lloyd,
                                                int t) {
  __shared__ double term[256];
  __shared__ int n_empty;
  const int g = blockIdx.x, k = threadIdx.x;
  if (st[g].done) return;
  constexpr int P = 2 * D + 2;
  if (k == 0) n_empty = 0;
  __syncthreads();
  double tk = 0.0;
  if (k < K) {
    double acc[P];
#pragma unroll
    for (int p = 0; p < P; ++p) acc[p] = 0.0;
    for (int c = 0; c < C; ++c) {
      const double *in = part + (((long long)g * C + c) * K + k) * P;
#pragma unroll
      for (int p = 0; p < P; ++p) acc[p] += in[p];
    }
    float *s = shapes + ((long long)g * cb_stride_g + k) * D;
    float *gp = gains + (long long)g * cb_stride_g + k;
    const double W = acc[2 * D], cnt = acc[2 * D + 1];
    const double g_old = (double)*gp;
    double proj_old = 0.0;
#pragma unroll
    for (int j = 0; j < D; ++j) proj_old += acc[j] * (double)s[j];
    tk = 2.0 * g_old * proj_old - W * g_old * g_old;
    if (cnt == 0.0) atomicAdd(&n_empty, 1);
    if (cnt != 0.0 && W > 0.0) {
      float sn[D];
#pragma unroll
      for (int j = 0; j < D; ++j) sn[j] = s[j];
      if (lloyd) {
        double bn2 = 0.0;
#pragma unroll
        for (int j = 0; j < D; ++j) bn2 = __dadd_rn(bn2, __dmul_rn(acc[D + j], acc[D + j]));
        const double bn = sqrt(bn2);
        if (bn / W > kDelta) {
#pragma unroll
          for (int j = 0; j < D; ++j) { sn[j] = (float)(acc[D + j] / bn); s[j] = sn[j]; }
        }
      }
      double proj = 0.0;
#pragma unroll
      for (int j = 0; j < D; ++j) proj = __dadd_rn(proj, __dmul_rn(acc[j], (double)sn[j]));
      const double gk = proj / W;
      *gp = (float)(gk > 0.0 ? gk : 0.0);
    }
  }
  term[k] = tk;
  __syncthreads();
  if (k == 0) {
    if (lloyd) {
      double sum = 0.0;
      for (int q = 0; q < K; ++q) sum += term[q];
      st[g].J[t] = Etot[g] - sum;
      st[g].iters_run = t;
      st[g].n_empty = n_empty;
      if (t > 1 && st[g].changed[t] == 0) st[g].done = 1;
    }
  }
}

}  // namespace gsrq
