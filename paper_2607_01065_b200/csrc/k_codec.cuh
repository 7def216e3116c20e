// k_codec.cuh -- decode: xhat_i = ((c0[a0_i] + c1[a1_i]) + ...) in fp32, stage order, one
// RN-even cast to the output dtype (prefix of stages PAPER.md:25; reading c-D).
// HBM-bound: reads S bytes and writes 2d (bf16) bytes per sub-vector.  The scaled codeword
// tables c^(s)[K][D] = fl32(g_k s_k) live in shared memory; D/4 lanes cooperate on a row so
// that every store instruction of a warp covers one contiguous 256-byte span (bf16).
#pragma once
#include "gsrq_common.cuh"

namespace gsrq {

struct DecParams {
  const uint8_t *codes;  // [S][G][N]
  const float *shapes;   // [G][S][K][D]
  const float *gains;    // [G][S][K]
  int S, K, G;
  int n_stages;
  long long N;           // rows per group = T*M
  int M;
  void *out;
  int dtype;
  long long stride_g, stride_t;
  long long rows_per_cta;
  long long row_begin;   // generic kernel: first row it decodes (the tail after the fast kernel's chunks)
};

__device__ __forceinline__ uint32_t pack_bf16x2(float a, float b) {
  const __nv_bfloat16 lo = __float2bfloat16_rn(a), hi = __float2bfloat16_rn(b);
  return (uint32_t)__bfloat16_as_ushort(lo) | ((uint32_t)__bfloat16_as_ushort(hi) << 16);
}

// grid = (ceil(N / rows_per_cta), G), block = 256, dynamic smem = n_stages*K*D*4 (SMEM) or 0.
template <int D, bool SMEM, int U>
__global__ void __launch_bounds__(256) k_decode(DecParams p) {
  extern __shared__ __align__(16) float tab[];
  constexpr int LPR = D / 4;      // lanes per row
  constexpr int RPI = 256 / LPR;  // rows per CTA iteration
  const int g = blockIdx.y;
  if (SMEM) {
    for (int e = threadIdx.x; e < p.n_stages * p.K * D; e += 256) {
      const int s = e / (p.K * D), r = e - s * p.K * D;
      const long long cb = ((long long)g * p.S + s) * p.K;
      tab[e] = __fmul_rn(p.gains[cb + r / D], p.shapes[cb * D + r]);
    }
    __syncthreads();
  }
  const int sub = threadIdx.x % LPR, rl = threadIdx.x / LPR;
  const long long r0 = p.row_begin + (long long)blockIdx.x * p.rows_per_cta;
  const long long r1 = min(p.N, r0 + p.rows_per_cta);
  for (long long ib = r0 + rl; ib < r1; ib += (long long)RPI * U) {
    int code[U][GSRQ_MAX_STAGES > 8 ? 8 : GSRQ_MAX_STAGES];
    float4 acc[U];
#pragma unroll
    for (int u = 0; u < U; ++u) acc[u] = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int s0 = 0; s0 < p.n_stages; s0 += 8) {
      const int ns = min(8, p.n_stages - s0);
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const long long i = ib + (long long)u * RPI;
#pragma unroll
        for (int s = 0; s < 8; ++s)
          code[u][s] = (s < ns && i < r1) ? min((int)p.codes[((long long)(s0 + s) * p.G + g) * p.N + i], p.K - 1) : 0;   // a byte >= K (K < 256) stays inside the table
      }
#pragma unroll
      for (int s = 0; s < 8; ++s) {
        if (s >= ns) break;
#pragma unroll
        for (int u = 0; u < U; ++u) {
          float4 c;
          if (SMEM) {
            c = *reinterpret_cast<const float4 *>(tab + ((s0 + s) * p.K + code[u][s]) * D + sub * 4);
          } else {
            const long long cb = ((long long)g * p.S + s0 + s) * p.K + code[u][s];
            const float gk = p.gains[cb];
            const float4 sv = *reinterpret_cast<const float4 *>(p.shapes + cb * D + sub * 4);
            c = make_float4(__fmul_rn(gk, sv.x), __fmul_rn(gk, sv.y), __fmul_rn(gk, sv.z), __fmul_rn(gk, sv.w));
          }
          if (s0 + s == 0) acc[u] = c;
          else {
            acc[u].x = __fadd_rn(acc[u].x, c.x); acc[u].y = __fadd_rn(acc[u].y, c.y);
            acc[u].z = __fadd_rn(acc[u].z, c.z); acc[u].w = __fadd_rn(acc[u].w, c.w);
          }
        }
      }
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const long long i = ib + (long long)u * RPI;
      if (i >= r1) continue;
      const long long tok = i / p.M;
      const int m = (int)(i - tok * p.M);
      const long long off = (long long)g * p.stride_g + tok * p.stride_t + (long long)m * D + sub * 4;
      if (p.dtype == GSRQ_BF16) {
        uint2 v = make_uint2(pack_bf16x2(acc[u].x, acc[u].y), pack_bf16x2(acc[u].z, acc[u].w));
        *reinterpret_cast<uint2 *>(reinterpret_cast<uint16_t *>(p.out) + off) = v;
      } else {
        *reinterpret_cast<float4 *>(reinterpret_cast<float *>(p.out) + off) = acc[u];
      }
    }
  }
}

// ---- bandwidth path (D = 16, NS <= 4 stages, N % 16 == 0): full chunks of 256 rows ----
// HBM traffic is NS code bytes in and 32 (bf16) / 64 (fp32) bytes out per row; the per-row work
// that has to keep up with it is the table gather, NS x 64 bytes of shared-memory reads per row,
// so the table layout is what decides the speed.  Each codeword row is stored twice, as
// 128 bytes [c0 c1 c2 c3 | c0 c1 c2 c3] (16-byte chunks), and lane l reads the chunk at byte
// (l % 8) * 16 of its codeword's row: the 8 lanes of an LDS.128 phase always hit the 8 distinct
// 16-byte bank groups, whatever the codes are -- no bank conflicts for any data.
// Mapping: a warp owns 256 consecutive rows and decodes 8 consecutive rows per iteration, 4 lanes
// (one 4-element quarter each) per row.
constexpr int kDecThreads = 512;
constexpr int kDecTabBytes = 256 * 128;  // per stage (duplicated rows)
constexpr int kDecDeep = 12;             // stages of the single-copy variant (256 * 64 bytes per stage)

// DUP = true : NS = number of stages (1..4), duplicated table rows (128 bytes), conflict-free.
// DUP = false: NS = kDecDeep = upper bound, p.n_stages (5..kDecDeep) stages decoded; single-copy table rows (64 bytes:
//              two codewords of equal parity in one LDS phase conflict 2-way) so that 12 stages fit in shared memory.
// LAYOUT: 0 = any strided view; 1 = dense ([G][N][16] contiguous per group); 2 = M == 8 (a (head, token) slice is 8 rows = 128
// contiguous elements, e.g. head_dim 128 in either tensor layout): the warp's 8 rows of an iteration are one token.
// BF16: output dtype fixed at compile time (bf16 / fp32) so that the inner loop carries no dtype branch.
template <int NS, int LAYOUT, bool BF16, bool DUP = true>
__global__ void __launch_bounds__(kDecThreads) k_decode_fast(DecParams p, long long n_chunks) {
  extern __shared__ __align__(16) float tab[];
  constexpr int RS = DUP ? 32 : 16;  // floats per table row
  const int ns = DUP ? NS : p.n_stages;
  const int g = blockIdx.y;
  for (int e = threadIdx.x; e < ns * p.K * 16; e += kDecThreads) {
    const int s = e / (p.K * 16), r = e - s * p.K * 16, k = r >> 4, j = r & 15;
    const long long cb = ((long long)g * p.S + s) * p.K + k;
    const float v = __fmul_rn(p.gains[cb], p.shapes[cb * 16 + j]);
    float *row = tab + ((size_t)s * 256 + k) * RS;
    row[j] = v;
    if (DUP) row[16 + j] = v;
  }
  __syncthreads();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int slot = lane >> 2, c4 = lane & 3;
  const float *tl = tab + (DUP ? (lane & 7) : (lane & 3)) * 4;
  const int msh = ((p.M & (p.M - 1)) == 0) ? (31 - __clz(p.M)) : -1;
  const long long ch0 = (long long)blockIdx.x * (kDecThreads / 32) + warp, chs = (long long)gridDim.x * (kDecThreads / 32);
  // lane l holds the 8 code bytes of rows 8l..8l+7 of the chunk (one coalesced 256-byte load per stage), loaded one chunk ahead;
  // iteration u decodes rows 8u..8u+7 (slot = row within the 8), whose codes sit in lane u: two shuffles and a byte permute per
  // stage (a shared-memory strip of the code bytes instead of the shuffles was measured: no faster).  Every store instruction
  // writes 256 contiguous bytes (bf16).
  uint2 nx[NS];
  if (ch0 < n_chunks) {
#pragma unroll
    for (int s = 0; s < NS; ++s)
      if (s < ns) nx[s] = __ldcs(reinterpret_cast<const uint2 *>(p.codes + ((long long)s * p.G + g) * p.N + ch0 * 256) + lane);
  }
  uint16_t *out16 = reinterpret_cast<uint16_t *>(p.out) + (long long)g * p.stride_g;
  float *out32 = reinterpret_cast<float *>(p.out) + (long long)g * p.stride_g;
  for (long long ch = ch0; ch < n_chunks; ch += chs) {
    uint2 cw[NS];
#pragma unroll
    for (int s = 0; s < NS; ++s) cw[s] = nx[s];
    if (ch + chs < n_chunks) {
#pragma unroll
      for (int s = 0; s < NS; ++s)
        if (s < ns) nx[s] = __ldcs(reinterpret_cast<const uint2 *>(p.codes + ((long long)s * p.G + g) * p.N + (ch + chs) * 256) + lane);
    }
    // element offset of this lane's 4 values in iteration 0 and the step per iteration (LAYOUT 1 / 2: both warp-uniform + 4 lane)
    long long off0 = 0, step = 0;
    if (LAYOUT == 1) { off0 = ch * 4096 + lane * 4; step = 128; }
    if (LAYOUT == 2) { off0 = ch * 32 * p.stride_t + lane * 4; step = p.stride_t; }
#pragma unroll 8
    for (int u = 0; u < 32; ++u) {
      float4 acc;
#pragma unroll
      for (int s = 0; s < NS; ++s) {
        if (s >= ns) break;
        const uint32_t k = __byte_perm(__shfl_sync(0xffffffffu, cw[s].x, u), __shfl_sync(0xffffffffu, cw[s].y, u), slot) & 0xFFu;
        const float4 c = *reinterpret_cast<const float4 *>(tl + ((size_t)s * 256 + k) * RS);
        if (s == 0) acc = c;
        else {
          acc.x = __fadd_rn(acc.x, c.x); acc.y = __fadd_rn(acc.y, c.y);
          acc.z = __fadd_rn(acc.z, c.z); acc.w = __fadd_rn(acc.w, c.w);
        }
      }
      long long off;
      if (LAYOUT == 0) {
        const long long i = ch * 256 + u * 8 + slot;
        const long long tok = (msh >= 0) ? (i >> msh) : (i / p.M);
        off = tok * p.stride_t + (i - tok * p.M) * 16 + c4 * 4;
      } else {
        off = off0 + u * step;
      }
      if (BF16) __stcs(reinterpret_cast<uint2 *>(out16 + off), make_uint2(pack_bf16x2(acc.x, acc.y), pack_bf16x2(acc.z, acc.w)));
      else __stcs(reinterpret_cast<float4 *>(out32 + off), acc);
    }
  }
}

}  // namespace gsrq
