// k_prep.cuh -- per-stage preparation kernels: gather the fit rows with their per-row constants,
// operand planes and weighted energy; seeded initial rows and shapes (Alg. 1 l.1; reading c-I).
#pragma once
#include "gsrq_common.cuh"
#include "k_update.cuh"

namespace gsrq {

constexpr int kPrepRows = 1024;  // rows per CTA of k_prep_rows (256 threads x 4)

struct PrepParams {
  RowSrc src;
  const float *w;              // [.][T] per-token weights or nullptr (uniform)
  long long w_stride_g;
  const long long *fit_tokens; // [G][nf_tok] or nullptr
  long long nf_tok;
  float *Rf;                   // [G][Nf][D] compact fp32 rows (out; may alias src.rows)
  double2 *coef;               // [G][Nf] per-row {w_i, w_i/(||r_i||+eps)}  (Eq. 6 with the safeguard of PAPER.md:178), or nullptr
  double *wn;                  // [G][Nf] per-row w_i/(||r_i||+eps) alone (the fused fit kernel reads w_i from wt), or nullptr
  float *wt;                   // [G][nf_tok] compact per-fit-token weights (out)
  double *epart;               // [G][gridDim.x] partial sums of w_i ||r_i||^2 (Eq. 4's constant), or nullptr
  __nv_bfloat16 *ahi, *alo;    // [G][Nf][16] bf16 operand planes of the tensor-core filter (D == 16), or nullptr
  float *rnorm;                // [G][Nf] fp32 upper bound of ||r_i||, or nullptr
};

// One pass over the fit rows of every group: gather (through fit_tokens) into the compact fp32
// buffer, per-row constants, operand planes A_hi = bf16(r), A_lo = bf16(r - A_hi), and the CTA's
// partial of the weighted energy (fixed order: 4 rows per thread in row order, then a tree).
// grid = (ceil(Nf / kPrepRows), G), block = 256.
template <int D>
__global__ void __launch_bounds__(256) k_prep_rows(PrepParams p) {
  __shared__ double sh[256];
  const int g = blockIdx.y;
  const long long Nf = p.nf_tok * p.src.M;
  double e = 0.0;
#pragma unroll
  for (int u = 0; u < kPrepRows / 256; ++u) {
    const long long i = (long long)blockIdx.x * kPrepRows + u * 256 + threadIdx.x;
    if (i >= Nf) continue;
    const long long tl = i / p.src.M;
    const int m = (int)(i - tl * p.src.M);
    const long long tok = p.fit_tokens ? p.fit_tokens[(long long)g * p.nf_tok + tl] : tl;
    float x[D];
    if (p.src.rows) load_row_f32<D>(p.src.rows, (long long)g * p.src.rows_per_group + tok * p.src.M + m, x);
    else load_row_kv<D>(p.src.kv, p.src.dtype, (long long)g * p.src.stride_g + tok * p.src.stride_t + (long long)m * D, x);
    const long long gi = (long long)g * Nf + i;
    store_row_f32<D>(p.Rf, gi, x);
    const float wv = p.w ? p.w[(long long)g * p.w_stride_g + tok] : 1.0f;
    if (m == 0) p.wt[(long long)g * p.nf_tok + tl] = wv;
    double n2 = 0.0;
#pragma unroll
    for (int j = 0; j < D; ++j) n2 = __dadd_rn(n2, __dmul_rn((double)x[j], (double)x[j]));
    const double n = sqrt(n2);
    const double wnv = (double)wv * (1.0 / (n + kEps));
    if (p.coef) p.coef[gi] = make_double2((double)wv, wnv);
    if (p.wn) p.wn[gi] = wnv;
    e += (double)wv * n2;
    if (p.rnorm) p.rnorm[gi] = (float)n * 1.000001f;
    if (D == 16 && p.ahi) {
      uint32_t h[8], l[8];
#pragma unroll
      for (int j = 0; j < 16; j += 2) {
        const __nv_bfloat16 h0 = __float2bfloat16_rn(x[j]), h1 = __float2bfloat16_rn(x[j + 1]);
        const __nv_bfloat16 l0 = __float2bfloat16_rn(__fsub_rn(x[j], __bfloat162float(h0)));
        const __nv_bfloat16 l1 = __float2bfloat16_rn(__fsub_rn(x[j + 1], __bfloat162float(h1)));
        h[j / 2] = (uint32_t)__bfloat16_as_ushort(h0) | ((uint32_t)__bfloat16_as_ushort(h1) << 16);
        l[j / 2] = (uint32_t)__bfloat16_as_ushort(l0) | ((uint32_t)__bfloat16_as_ushort(l1) << 16);
      }
      uint4 *ph = reinterpret_cast<uint4 *>(p.ahi + gi * 16);
      ph[0] = make_uint4(h[0], h[1], h[2], h[3]);
      ph[1] = make_uint4(h[4], h[5], h[6], h[7]);
      if (p.alo) {
        uint4 *pl = reinterpret_cast<uint4 *>(p.alo + gi * 16);
        pl[0] = make_uint4(l[0], l[1], l[2], l[3]);
        pl[1] = make_uint4(l[4], l[5], l[6], l[7]);
      }
    }
  }
  if (!p.epart) return;
  sh[threadIdx.x] = e;
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if ((int)threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
    __syncthreads();
  }
  if (threadIdx.x == 0) p.epart[(long long)g * gridDim.x + blockIdx.x] = sh[0];
}

// Seeded initial rows.  Candidate n of group g is splitmix64(seed_g)[n] mod Nf; a candidate is
// accepted iff its row is non-zero and its value did not occur earlier in the stream; the first
// K accepted are the initial rows (same rule as "skip if already chosen or zero norm").
// One block of 512 threads per group evaluates 512 candidates per batch.  When shapes != nullptr
// the block goes on to Alg. 1 l.1: s_k = fl32(r / ||r||) (fp64 division) for the chosen rows, g_k = 0
// (set by the first gain update), and, when bimg != nullptr (D == 16), the projection-mode operand
// images of all 256 rows for the first scoring pass.
template <int D>
__global__ void __launch_bounds__(512) k_init_ids(const float *__restrict__ Rf, long long Nf, int K, int G, int stage,
                                                  uint64_t seed, long long *__restrict__ ids, DevStats *__restrict__ st,
                                                  float *__restrict__ shapes, float *__restrict__ gains,
                                                  long long cb_stride_g, uint8_t *__restrict__ bimg) {
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
      // no data-dependent exit and 8 comparisons per trip: the loads of a trip are independent, so the (in-order)
      // thread does not pay one shared-memory latency per comparison
      int dup = 0;
      for (int q = 0; q < nc; ++q) dup |= (chosen[q] == c);
      int q = 0;
      for (; q + 8 <= t; q += 8) {
        int d8 = 0;
#pragma unroll
        for (int u = 0; u < 8; ++u) d8 |= (cand[q + u] == c);
        dup |= d8;
      }
      for (; q < t; ++q) dup |= (cand[q] == c);
      good = !dup;
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
  if (!shapes) return;
  for (int k = t; k < GSRQ_MAX_K; k += 512) {
    float sv[D];
#pragma unroll
    for (int j = 0; j < D; ++j) sv[j] = 0.0f;
    if (k < K) {
      float x[D];
      load_row_f32<D>(Rf, (long long)g * Nf + (k < n_chosen ? chosen[k] : 0), x);
      const double n = row_norm_f64<D>(x);
#pragma unroll
      for (int j = 0; j < D; ++j) sv[j] = (n > 0.0) ? (float)((double)x[j] / n) : 0.0f;
      store_row_f32<D>(shapes + (long long)g * cb_stride_g * D, k, sv);
      gains[(long long)g * cb_stride_g + k] = 0.0f;
    }
    if (D == 16 && bimg) {
#pragma unroll
      for (int j = 0; j < D; ++j) write_bimg_elem(bimg + (size_t)g * 3 * kBImgBytesU, k, j, 1.0f, sv[j], 1, k >= K);
    }
  }
}

}  // namespace gsrq
