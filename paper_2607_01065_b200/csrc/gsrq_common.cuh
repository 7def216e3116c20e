// gsrq_common.cuh -- shared definitions of the CUDA path (no code shared with oracle/).
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "../../include/gsrq.h"

namespace gsrq {

constexpr double kEps = 1e-12;   // y = r / (||r|| + eps)            PAPER.md:178, reading c-E
constexpr double kDelta = 1e-8;  // "numerically close to zero"      PAPER.md:178, reading c-E
constexpr uint64_t kGamma = 0x9E3779B97F4A7C15ULL;

// Device-side statistics of one group (mirrors gsrq_fit_stats; slot 0 of changed[] is the
// init assignment, slot t the t-th Lloyd iteration).
struct DevStats {
  int done_iter;  // 0, or the iteration t at which Alg. 1 l.15-16 broke (kernels of passes > t skip the group)
  int err;
  int iters_run;  // filled by k_finish
  int pad;
  long long refined;
  long long changed[GSRQ_MAX_ITERS + 1];
  int n_empty[GSRQ_MAX_ITERS + 1];
  int gmax_bits[GSRQ_MAX_ITERS + 3];  // slot t: bit pattern of max_k g_k of the codebook scored at pass t
  double J[GSRQ_MAX_ITERS + 1];       // filled by k_finish
};

// Alg. 1 l.15-16 broke at an earlier iteration: the kernels of pass t leave the group alone.
__device__ __forceinline__ bool group_done(const DevStats *st, int g, int t) {
  return st && st[g].done_iter != 0 && st[g].done_iter < t;
}

// Where the rows of a pass come from.  Row i of group g:
//   src == kv  : element j at kv[g*stride_g + tok(i/M)*stride_t + (i%M)*d + j]
//   src == rows: element j at rows[(g*rows_per_group + ri(i))*d + j]
// tok()/ri() go through fit_tokens when the pass runs on a fit subset.
struct RowSrc {
  const void *kv;
  const float *rows;  // fp32 [G][rows_per_group][d] or nullptr
  int dtype;
  int M;
  int d;
  long long stride_g, stride_t;
  long long rows_per_group;  // of `rows`
};

void set_error(const char *fmt, ...);

#define GSRQ_CUDA_CHECK(expr)                                                       \
  do {                                                                              \
    cudaError_t _e = (expr);                                                        \
    if (_e != cudaSuccess) {                                                        \
      gsrq::set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(_e), __FILE__, __LINE__); \
      return GSRQ_ECUDA;                                                            \
    }                                                                               \
  } while (0)

__device__ __forceinline__ float bf16_bits_to_f32(uint16_t b) { return __uint_as_float(((uint32_t)b) << 16); }

// Load D contiguous elements of one sub-vector as fp32 (exact for bf16).
template <int D>
__device__ __forceinline__ void load_row_kv(const void *kv, int dtype, long long off, float (&x)[D]) {
  if (dtype == GSRQ_BF16) {
    const uint4 *p = reinterpret_cast<const uint4 *>(reinterpret_cast<const uint16_t *>(kv) + off);
#pragma unroll
    for (int q = 0; q < D / 8; ++q) {
      uint4 v = __ldg(p + q);
      uint32_t u[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        x[q * 8 + 2 * e] = __uint_as_float(u[e] << 16);
        x[q * 8 + 2 * e + 1] = __uint_as_float(u[e] & 0xFFFF0000u);
      }
    }
  } else {
    const float4 *p = reinterpret_cast<const float4 *>(reinterpret_cast<const float *>(kv) + off);
#pragma unroll
    for (int q = 0; q < D / 4; ++q) {
      float4 v = __ldg(p + q);
      x[q * 4] = v.x; x[q * 4 + 1] = v.y; x[q * 4 + 2] = v.z; x[q * 4 + 3] = v.w;
    }
  }
}

template <int D>
__device__ __forceinline__ void load_row_f32(const float *rows, long long row, float (&x)[D]) {
  const float4 *p = reinterpret_cast<const float4 *>(rows + row * D);
#pragma unroll
  for (int q = 0; q < D / 4; ++q) {
    float4 v = p[q];
    x[q * 4] = v.x; x[q * 4 + 1] = v.y; x[q * 4 + 2] = v.z; x[q * 4 + 3] = v.w;
  }
}

template <int D>
__device__ __forceinline__ void store_row_f32(float *rows, long long row, const float (&x)[D]) {
  float4 *p = reinterpret_cast<float4 *>(rows + row * D);
#pragma unroll
  for (int q = 0; q < D / 4; ++q) p[q] = make_float4(x[q * 4], x[q * 4 + 1], x[q * 4 + 2], x[q * 4 + 3]);
}

// fp64 norm of a row, summed in element order (matches the definition, not any blocking).
template <int D>
__device__ __forceinline__ double row_norm_f64(const float (&x)[D]) {
  double n2 = 0.0;
#pragma unroll
  for (int j = 0; j < D; ++j) n2 = __dadd_rn(n2, __dmul_rn((double)x[j], (double)x[j]));
  return sqrt(n2);
}

__device__ __forceinline__ uint64_t splitmix64_at(uint64_t seed, uint64_t n) {
  // n-th output (n = 0, 1, ...) of the splitmix64 stream started at `seed`
  uint64_t z = seed + (n + 1) * kGamma;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  return z ^ (z >> 31);
}

}  // namespace gsrq
