// k_variants.cuh -- small variants around the encoder:
//   * log-smoothed gradient weights  w~ = log(1 + lambda ||g||_2), lambda = tau / (median ||g||_2 + eps)   (PAPER.md:192 Eq. 9, :434 Eq. 10)
//   * per-vector fp16 gain codes (reading c-G's alternative; BASELINE.json config 0 "4-bit indices plus an fp16 gain")
//   * nibble packing of codes for K <= 16 (BASELINE.json config 0; "bit-packing")
#pragma once
#include <cuda_fp16.h>

#include "gsrq_common.cuh"

namespace gsrq {
namespace var {

// ||g_t||_2 per (head, token): warp per row of hd elements, fp64 sum of squares (fixed order), stored as fp32.
// grid = (ceil(T / 8), G), block = 256.
__global__ void __launch_bounds__(256) k_grad_norms(const void *__restrict__ grad, int dtype, int hd, long long T, long long stride_g,
                                                    long long stride_t, float *__restrict__ out) {
  const int g = blockIdx.y, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const long long t = (long long)blockIdx.x * 8 + warp;
  if (t >= T) return;
  const long long off = (long long)g * stride_g + t * stride_t;
  double n2 = 0.0;
  for (int e = lane; e < hd; e += 32) {
    const double x = (dtype == GSRQ_BF16) ? (double)bf16_bits_to_f32(reinterpret_cast<const uint16_t *>(grad)[off + e])
                                          : (double)reinterpret_cast<const float *>(grad)[off + e];
    n2 += x * x;
  }
  for (int o = 16; o; o >>= 1) n2 += __shfl_xor_sync(0xffffffffu, n2, o);
  if (lane == 0) out[(long long)g * T + t] = (float)sqrt(n2);
}

// The value of rank r (0-based, ascending) among n non-negative floats: radix select over the bit patterns, 8 bits per pass.
// All threads of the block call it together; hist is a shared array of 256 counters.
__device__ unsigned int block_select(const float *__restrict__ w, long long n, long long r, unsigned int *hist) {
  unsigned int prefix = 0, mask = 0;
  for (int shift = 24; shift >= 0; shift -= 8) {
    for (int b = threadIdx.x; b < 256; b += blockDim.x) hist[b] = 0u;
    __syncthreads();
    for (long long i = threadIdx.x; i < n; i += blockDim.x) {
      const unsigned int u = __float_as_uint(w[i]);
      if ((u & mask) == prefix) atomicAdd(&hist[(u >> shift) & 255u], 1u);
    }
    __syncthreads();
    __shared__ unsigned int s_digit;
    __shared__ long long s_rank;
    if (threadIdx.x == 0) {
      long long acc = 0;
      unsigned int dgt = 255;
      for (unsigned int b = 0; b < 256; ++b) {
        if (acc + hist[b] > r) { dgt = b; break; }
        acc += hist[b];
      }
      s_digit = dgt;
      s_rank = r - acc;
    }
    __syncthreads();
    prefix |= s_digit << shift;
    mask |= 255u << shift;
    r = s_rank;
    __syncthreads();
  }
  return prefix;
}

// Per group: median of the T norms (mean of the two middle values when T is even), lambda = tau / (median + eps), then
// w <- log(1 + lambda w) in place (double, stored as fp32).  grid = G, block = 1024.
__global__ void __launch_bounds__(1024) k_log_weights(float *__restrict__ w, long long T, double tau, double eps) {
  __shared__ unsigned int hist[256];
  float *wg = w + (long long)blockIdx.x * T;
  const float lo = __uint_as_float(block_select(wg, T, (T - 1) / 2, hist));
  const float hi = __uint_as_float(block_select(wg, T, T / 2, hist));
  const double med = 0.5 * ((double)lo + (double)hi);
  const double lam = tau / (med + eps);
  __syncthreads();
  for (long long i = threadIdx.x; i < T; i += blockDim.x) wg[i] = (float)log1p(lam * (double)wg[i]);
}

// ---- per-vector gain codes: after the projection arg-max (gsrq_assign, mode 1) of a stage ----
struct PvgParams {
  RowSrc src;               // rows of this stage: kv (stage 0) or the fp32 residual
  long long N;
  const float *shapes;      // stage slice, [G] stride cb_stride_g codewords
  long long cb_stride_g;
  const uint8_t *codes;     // [G][N] of this stage
  __half *gains;            // [G][N] out
  float *res_out;           // [G][N][D] out (may alias src.rows)
};

// gamma = fp16(max(0, r . s_k)) with the dot product in fp64 in element order (the oracle's arithmetic), one RN-even cast;
// r <- fl32(r - fl32(fl32(gamma) s_k)).  thread per row; grid = (ceil(N / 256), G).
template <int D>
__global__ void __launch_bounds__(256) k_pvg_finish(PvgParams p) {
  const int g = blockIdx.y;
  const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
  if (i >= p.N) return;
  float x[D];
  if (p.src.rows) load_row_f32<D>(p.src.rows, (long long)g * p.src.rows_per_group + i, x);
  else {
    const long long tok = i / p.src.M;
    const int m = (int)(i - tok * p.src.M);
    load_row_kv<D>(p.src.kv, p.src.dtype, (long long)g * p.src.stride_g + tok * p.src.stride_t + (long long)m * D, x);
  }
  const long long gi = (long long)g * p.N + i;
  const float *s = p.shapes + ((long long)g * p.cb_stride_g + p.codes[gi]) * D;
  double dot = 0.0;
#pragma unroll
  for (int j = 0; j < D; ++j) dot = __dadd_rn(dot, __dmul_rn((double)x[j], (double)s[j]));
  const __half gam = __double2half(dot > 0.0 ? dot : 0.0);
  p.gains[gi] = gam;
  const float gf = __half2float(gam);
#pragma unroll
  for (int j = 0; j < D; ++j) x[j] = __fsub_rn(x[j], __fmul_rn(gf, s[j]));
  store_row_f32<D>(p.res_out, gi, x);
}

struct PvgDecParams {
  const uint8_t *codes;     // [S][G][N]
  const __half *gains;      // [S][G][N]
  const float *shapes;      // [G][S][K][D]
  int S, K, G, n_stages, M;
  long long N;
  void *out;
  int dtype;
  long long stride_g, stride_t;
};

// xhat = sum over the stages of fl32(gamma s_k), fp32 in stage order, one RN-even cast.  thread per row.
template <int D>
__global__ void __launch_bounds__(256) k_pvg_decode(PvgDecParams p) {
  const int g = blockIdx.y;
  const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
  if (i >= p.N) return;
  float acc[D];
  for (int st = 0; st < p.n_stages; ++st) {
    const long long ci = ((long long)st * p.G + g) * p.N + i;
    const float gf = __half2float(p.gains[ci]);
    const float *s = p.shapes + (((long long)g * p.S + st) * p.K + min((int)p.codes[ci], p.K - 1)) * D;
#pragma unroll
    for (int j = 0; j < D; ++j) {
      const float c = __fmul_rn(gf, s[j]);
      acc[j] = (st == 0) ? c : __fadd_rn(acc[j], c);
    }
  }
  const long long tok = i / p.M;
  const int m = (int)(i - tok * p.M);
  const long long off = (long long)g * p.stride_g + tok * p.stride_t + (long long)m * D;
#pragma unroll
  for (int j = 0; j < D; ++j) {
    const float v = (p.n_stages > 0) ? acc[j] : 0.0f;
    if (p.dtype == GSRQ_BF16) reinterpret_cast<__nv_bfloat16 *>(p.out)[off + j] = __float2bfloat16_rn(v);
    else reinterpret_cast<float *>(p.out)[off + j] = v;
  }
}

// ---- nibble packing: plane of N codes (< 16) -> ceil(N / 2) bytes, row 2i in the low nibble ----
__global__ void __launch_bounds__(256) k_pack_nibbles(const uint8_t *__restrict__ codes, long long n_planes, long long N, uint8_t *__restrict__ packed) {
  const long long Np = (N + 1) / 2;
  for (long long e = (long long)blockIdx.x * 256 + threadIdx.x; e < n_planes * Np; e += (long long)gridDim.x * 256) {
    const long long pl = e / Np, i = e - pl * Np;
    const uint8_t lo = codes[pl * N + 2 * i] & 15, hi = (2 * i + 1 < N) ? (codes[pl * N + 2 * i + 1] & 15) : 0;
    packed[e] = (uint8_t)(lo | (hi << 4));
  }
}
__global__ void __launch_bounds__(256) k_unpack_nibbles(const uint8_t *__restrict__ packed, long long n_planes, long long N, uint8_t *__restrict__ codes) {
  const long long Np = (N + 1) / 2;
  for (long long e = (long long)blockIdx.x * 256 + threadIdx.x; e < n_planes * N; e += (long long)gridDim.x * 256) {
    const long long pl = e / N, i = e - pl * N;
    const uint8_t b = packed[pl * Np + (i >> 1)];
    codes[e] = (i & 1) ? (b >> 4) : (b & 15);
  }
}

}  // namespace var
}  // namespace gsrq
