// k_score.cuh -- CUDA-core scoring / arg-max / residual kernels (the exact path).
//
// Assignment (Eq. 5):  k_i = argmax_k (2 g_k r_i.s_k - g_k^2), lowest k on ties.
// Strategy "filter + exact refine": a fast filter computes every score
// with a rigorous per-row error bound E_i and keeps the top two; a row whose top-2 gap is
// <= 2 E_i is appended to a list and re-scored by k_encode_exact in fp64 with the operation order
// of the definition.  The assignment therefore equals the exact-arithmetic arg-max and the
// near-tie exemption of the parity protocol is never needed.
#pragma once
#include "gsrq_common.cuh"

namespace gsrq {

struct EncParams {
  RowSrc src;
  long long N;          // rows per group of this pass
  const float *shapes;  // [G][S][K][D]
  const float *gains;   // [G][S][K]
  int S, K;
  int s_first;          // exact path only: first stage applied to src (src holds the residual after stage s_first - 1)
  int s_begin, s_end;   // stages scored in this pass; stages < s_begin are replayed from codes
  int s_base;           // code plane index = s - s_base
  int mode;             // 0: Eq. 5 score, 1: plain projection (init assignment, reading c-I)
  int subtract;         // 1: r <- fl32(r - c_k) after each stage (encode); 0: assign only
  uint8_t *codes;       // plane p, group g, row i at codes[p*code_stride_s + g*N + i]
  long long code_stride_s;
  float *res_out;       // [G][N][D] or nullptr (may alias src.rows)
  DevStats *st;         // nullptr outside a fit
  int slot;             // st[g].changed[slot] counts rows whose code changed
  uint2 *list;          // rows for the exact path: {g*N + i, candidate-group mask | first undecided stage << 16}
  unsigned int *list_cnt;
};

template <int D>
__device__ __forceinline__ void load_src_row(const RowSrc &src, int g, long long i, float (&x)[D]) {
  if (src.rows) {
    load_row_f32<D>(src.rows, (long long)g * src.rows_per_group + i, x);
  } else {
    const long long tok = i / src.M;
    const int m = (int)(i - tok * src.M);
    load_row_kv<D>(src.kv, src.dtype, (long long)g * src.stride_g + tok * src.stride_t + (long long)m * D, x);
  }
}

constexpr float kU = 5.9604645e-8f;  // 2^-24, fp32 unit round-off

// Build the filter's operand tables of (group g, stage s) in shared memory:
//   c[k][j] = fl32(g_k s_kj)  (Eq. 3 centroid; also the vector subtracted by the encoder), b[k] = fl32(g_k^2);
//   projection mode: c = s, b = 0.  The filter's score is fl32(2 (r.c_k) - b_k).
// Error bound of that score against the exact 2 g (r.s) - g^2:  E = e1 ||r|| + e0 with
//   e1 = 1.05 u (2D+4) g_max,  e0 = 1.05 u 2 g_max^2   (derivation: DESIGN.md section 3).
template <int D>
__device__ __forceinline__ void build_tables(const EncParams &p, int g, int s, float *c_sh, float *b_sh, float *e_sh,
                                             int *gmax_bits) {
  const float *sh = p.shapes + ((long long)g * p.S + s) * p.K * D;
  const float *ga = p.gains + ((long long)g * p.S + s) * p.K;
  if (threadIdx.x == 0) *gmax_bits = 0;
  __syncthreads();
  for (int e = threadIdx.x; e < p.K * D; e += blockDim.x) {
    const int k = e / D;
    c_sh[e] = (p.mode == 0) ? __fmul_rn(ga[k], sh[e]) : sh[e];
  }
  for (int k = threadIdx.x; k < p.K; k += blockDim.x) {
    const float gk = ga[k];
    b_sh[k] = (p.mode == 0) ? __fmul_rn(gk, gk) : 0.0f;
    if (p.mode == 0) atomicMax(gmax_bits, __float_as_int(fmaxf(gk, 0.0f)));
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    const float gm = (p.mode == 0) ? __int_as_float(*gmax_bits) : 1.0f;
    e_sh[0] = 1.05f * kU * (2 * D + 4) * gm;
    e_sh[1] = (p.mode == 0) ? 1.05f * kU * 2.0f * gm * gm : 0.0f;
  }
  __syncthreads();
}

// Score one row against the K codewords in shared memory; returns best index, top-2 scores.
template <int D>
__device__ __forceinline__ int score_row(const float (&x)[D], const float *c_sh, const float *b_sh, int K, float &best,
                                         float &second) {
  best = -INFINITY;
  second = -INFINITY;
  int bi = 0;
  for (int k = 0; k < K; ++k) {
    const float4 *c4 = reinterpret_cast<const float4 *>(c_sh + k * D);
    float dot = 0.0f;
#pragma unroll
    for (int q = 0; q < D / 4; ++q) {
      const float4 c = c4[q];
      dot = fmaf(x[4 * q], c.x, dot);
      dot = fmaf(x[4 * q + 1], c.y, dot);
      dot = fmaf(x[4 * q + 2], c.z, dot);
      dot = fmaf(x[4 * q + 3], c.w, dot);
    }
    const float sc = fmaf(2.0f, dot, -b_sh[k]);
    if (sc > best) { second = best; best = sc; bi = k; }
    else if (sc > second) second = sc;
  }
  return bi;
}

// Filter kernel: thread per row, RPT rows per thread, stages [0, s_end) walked with one
// shared-memory table at a time.  grid = (ceil(N / (256*RPT)), G), block = 256.
template <int D, int RPT>
__global__ void __launch_bounds__(256) k_encode(EncParams p) {
  extern __shared__ __align__(16) float smem[];
  float *c_sh = smem;
  float *b_sh = c_sh + p.K * D;
  float *e_sh = b_sh + p.K;
  int *gmax_bits = reinterpret_cast<int *>(e_sh + 2);
  const int g = blockIdx.y;
  if (group_done(p.st, g, p.slot)) return;
  const long long i0 = (long long)blockIdx.x * (256 * RPT) + threadIdx.x;
  float x[RPT][D];
  bool live[RPT];
#pragma unroll
  for (int r = 0; r < RPT; ++r) {
    const long long i = i0 + r * 256;
    live[r] = i < p.N;
    if (live[r]) load_src_row<D>(p.src, g, i, x[r]);
  }
  unsigned int n_changed = 0;
  for (int s = 0; s < p.s_end; ++s) {
    if (s) __syncthreads();
    build_tables<D>(p, g, s, c_sh, b_sh, e_sh, gmax_bits);
#pragma unroll
    for (int r = 0; r < RPT; ++r) {
      if (!live[r]) continue;
      const long long i = i0 + r * 256;
      int k;
      if (s < p.s_begin) {
        k = p.codes[(long long)(s - p.s_base) * p.code_stride_s + (long long)g * p.N + i];
      } else {
        float best, second;
        k = score_row<D>(x[r], c_sh, b_sh, p.K, best, second);
        float n2 = 0.0f;
#pragma unroll
        for (int j = 0; j < D; ++j) n2 = fmaf(x[r][j], x[r][j], n2);
        const float E = fmaf(e_sh[0], sqrtf(n2) * 1.00001f, e_sh[1]);
        if (best - second <= 2.0f * E) {  // ambiguous: exact path decides this row (all stages)
          const unsigned int pos = atomicAdd(p.list_cnt, 1u);
          // stages before s are decided (their codes are stored); without a code plane the row restarts from 0
          p.list[pos] = make_uint2((uint32_t)((long long)g * p.N + i), 0xFFFFu | ((uint32_t)(p.codes ? s : 0) << 16));
          live[r] = false;
          continue;
        }
        if (p.codes) {
          uint8_t *cp = p.codes + (long long)(s - p.s_base) * p.code_stride_s + (long long)g * p.N + i;
          if (p.st) n_changed += (*cp != (uint8_t)k);
          *cp = (uint8_t)k;
        }
      }
      if (p.subtract) {
#pragma unroll
        for (int j = 0; j < D; ++j) x[r][j] = __fsub_rn(x[r][j], c_sh[k * D + j]);
      }
    }
  }
  if (p.res_out) {
#pragma unroll
    for (int r = 0; r < RPT; ++r)
      if (live[r]) store_row_f32<D>(p.res_out, (long long)g * p.N + i0 + r * 256, x[r]);
  }
  if (p.st) {
    for (int off = 16; off; off >>= 1) n_changed += __shfl_xor_sync(0xffffffffu, n_changed, off);
    if ((threadIdx.x & 31) == 0 && n_changed)
      atomicAdd(reinterpret_cast<unsigned long long *>(&p.st[g].changed[p.slot]), (unsigned long long)n_changed);
  }
}

// Exact fp64 scores of the codewords of the 16-codeword groups in `gmask` for row x; lowest k wins ties.
// fp64, dot product summed in element order without FMA contraction, score = (2 g)(r.s) - g g: the
// definition's own operation order.  Two groups (one per half-warp) per round.
template <int D>
__device__ __forceinline__ int exact_argmax_warp(const float (&x)[D], const float *__restrict__ sh, const float *__restrict__ ga,
                                                 int K, int mode, int lane, uint32_t gmask) {
  double best = -INFINITY;
  int bi = 0x7fffffff;
  while (gmask) {
    const int c0 = __ffs(gmask) - 1;
    gmask &= gmask - 1;
    int c1 = -1;
    if (gmask) { c1 = __ffs(gmask) - 1; gmask &= gmask - 1; }
    const int c = (lane < 16) ? c0 : c1;
    const int kk = 16 * c + (lane & 15);
    if (c >= 0 && kk < K) {
      float cwv[D];
      load_row_f32<D>(sh, kk, cwv);
      double dot = 0.0;
#pragma unroll
      for (int j = 0; j < D; ++j) dot = __dadd_rn(dot, __dmul_rn((double)x[j], (double)cwv[j]));
      double sc = dot;
      if (mode == 0) {
        const double gk = (double)ga[kk];
        sc = __dsub_rn(__dmul_rn(__dmul_rn(2.0, gk), dot), __dmul_rn(gk, gk));
      }
      if (sc > best || (sc == best && kk < bi)) { best = sc; bi = kk; }
    }
  }
  for (int off = 16; off; off >>= 1) {
    const double ob = __shfl_xor_sync(0xffffffffu, best, off);
    const int oi = __shfl_xor_sync(0xffffffffu, bi, off);
    if (ob > best || (ob == best && oi < bi)) { best = ob; bi = oi; }
  }
  return (bi == 0x7fffffff) ? 0 : bi;
}

// Exact arg-max of one row by a whole warp, cheap in the common case: fp32 filter across the warp
// (score = fl32(2 (r.c_k) - b_k), c = fl32(g s), b = fl32(g^2); 8 codewords per lane for K = 256) with the
// CUDA-core error bound, and fp64 over all codewords when its top-2 gap is within that bound.
template <int D>
__device__ __forceinline__ int warp_argmax_filtered(const float (&x)[D], const float *__restrict__ sh, const float *__restrict__ ga,
                                                    int K, int mode, int lane) {
  float best = -INFINITY, second = -INFINITY, gmx = 0.0f;
  int bi = 0x7fffffff;
  for (int kk = lane; kk < K; kk += 32) {
    const float gk = (mode == 0) ? ga[kk] : 1.0f;
    gmx = fmaxf(gmx, gk);
    float cwv[D];
    load_row_f32<D>(sh, kk, cwv);
    float dot = 0.0f;
#pragma unroll
    for (int j = 0; j < D; ++j) dot = fmaf(x[j], (mode == 0) ? __fmul_rn(gk, cwv[j]) : cwv[j], dot);
    const float sc = fmaf(2.0f, dot, (mode == 0) ? -__fmul_rn(gk, gk) : 0.0f);
    if (sc > best) { second = best; best = sc; bi = kk; }
    else if (sc > second) second = sc;
  }
  for (int off = 16; off; off >>= 1) {
    const float ob = __shfl_xor_sync(0xffffffffu, best, off), os = __shfl_xor_sync(0xffffffffu, second, off);
    const int oi = __shfl_xor_sync(0xffffffffu, bi, off);
    gmx = fmaxf(gmx, __shfl_xor_sync(0xffffffffu, gmx, off));
    if (ob > best || (ob == best && oi < bi)) { second = fmaxf(best, os); best = ob; bi = oi; }
    else second = fmaxf(second, ob);
  }
  float n2 = 0.0f;
#pragma unroll
  for (int j = 0; j < D; ++j) n2 = fmaf(x[j], x[j], n2);
  const float gm = (mode == 0) ? gmx : 1.0f;
  const float E = fmaf(1.05f * kU * (2 * D + 4) * gm, sqrtf(n2) * 1.00001f, (mode == 0) ? 1.05f * kU * 2.0f * gm * gm : 0.0f);
  if (best - second <= 2.0f * E) return exact_argmax_warp<D>(x, sh, ga, K, mode, lane, 0xFFFFu);
  return (bi == 0x7fffffff) ? 0 : bi;
}

// Exact path: one warp per listed row.  Stages before the entry's first undecided stage s* are replayed
// from their stored codes; stage s* is decided in fp64 among the entry's candidate groups (every
// codeword outside them is provably not the arg-max); later stages run the fp32 filter of k_encode
// across the warp (8 codewords per lane) and fall back to fp64 over all codewords when its top-2 gap
// is within the error bound.  The result equals the exact-arithmetic arg-max at every stage.
template <int D>
__global__ void __launch_bounds__(256) k_encode_exact(EncParams p) {
  const int lane = threadIdx.x & 31;
  const unsigned int n = *p.list_cnt;
  const unsigned int warp0 = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const unsigned int nwarps = (gridDim.x * blockDim.x) >> 5;
  for (unsigned int e = warp0; e < n; e += nwarps) {
    const uint2 en = p.list[e];
    const long long gi = en.x;
    const int s_star = (int)(en.y >> 16);
    const int g = (int)(gi / p.N);
    const long long i = gi - (long long)g * p.N;
    float x[D];
    load_src_row<D>(p.src, g, i, x);
    for (int s = p.s_first; s < p.s_end; ++s) {
      const float *sh = p.shapes + ((long long)g * p.S + s) * p.K * D;
      const float *ga = p.gains + ((long long)g * p.S + s) * p.K;
      int k;
      if (s < p.s_begin || s < s_star) {
        k = p.codes[(long long)(s - p.s_base) * p.code_stride_s + gi];
      } else {
        if (s == s_star) {
          k = exact_argmax_warp<D>(x, sh, ga, p.K, p.mode, lane, en.y & 0xFFFFu);
        } else {
          k = warp_argmax_filtered<D>(x, sh, ga, p.K, p.mode, lane);
        }
        if (lane == 0 && p.codes) {
          uint8_t *cp = p.codes + (long long)(s - p.s_base) * p.code_stride_s + gi;
          if (p.st && *cp != (uint8_t)k)
            atomicAdd(reinterpret_cast<unsigned long long *>(&p.st[g].changed[p.slot]), 1ull);
          *cp = (uint8_t)k;
        }
      }
      if (p.subtract) {
        const float gk = ga[k];
        float cwv[D];
        load_row_f32<D>(sh, k, cwv);
#pragma unroll
        for (int j = 0; j < D; ++j) x[j] = __fsub_rn(x[j], __fmul_rn(gk, cwv[j]));
      }
    }
    if (p.res_out && lane == 0) store_row_f32<D>(p.res_out, gi, x);
    if (p.st && lane == 0) atomicAdd(reinterpret_cast<unsigned long long *>(&p.st[g].refined), 1ull);
  }
}

// Encode-on-append (PAPER.md:443 (i): "residual quantization ... of newly generated KV vectors"): a handful of new
// tokens, one warp per sub-vector row, all stages with warp_argmax_filtered -- one small launch, no workspace.
// Row i of group g of the new tokens goes to codes[s*code_stride_s + g*plane_rows + row0 + i].
struct AppendParams {
  RowSrc src;           // the new tokens (kv view)
  long long N;          // new rows per group = n_new * M
  const float *shapes;  // [G][S][K][D]
  const float *gains;   // [G][S][K]
  int S, K, n_stages, G;
  uint8_t *codes;
  long long code_stride_s, plane_rows, row0;
};

template <int D>
__global__ void __launch_bounds__(256) k_encode_append(AppendParams p) {
  const int lane = threadIdx.x & 31;
  const long long total = (long long)p.G * p.N;
  for (long long gi = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5; gi < total; gi += ((long long)gridDim.x * blockDim.x) >> 5) {
    const int g = (int)(gi / p.N);
    const long long i = gi - (long long)g * p.N;
    float x[D];
    load_src_row<D>(p.src, g, i, x);
    for (int s = 0; s < p.n_stages; ++s) {
      const float *sh = p.shapes + ((long long)g * p.S + s) * p.K * D;
      const float *ga = p.gains + ((long long)g * p.S + s) * p.K;
      const int k = warp_argmax_filtered<D>(x, sh, ga, p.K, 0, lane);
      if (lane == 0) p.codes[(long long)s * p.code_stride_s + (long long)g * p.plane_rows + p.row0 + i] = (uint8_t)k;
      const float gk = ga[k];
      float cwv[D];
      load_row_f32<D>(sh, k, cwv);
#pragma unroll
      for (int j = 0; j < D; ++j) x[j] = __fsub_rn(x[j], __fmul_rn(gk, cwv[j]));
    }
  }
}

}  // namespace gsrq
